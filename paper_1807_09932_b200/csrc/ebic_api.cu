// ebic_api.cu -- host side of libebic.so: the C ABI declared in include/ebic.h.
// Links cudart only (no torch).  Product code: shares nothing with oracle/.
#include "../../include/ebic.h"

#include <cuda_runtime.h>
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ebic_device.cuh"
#include "extract_kernels.cuh"
#include "fitness_kernels.cuh"
#include "loader_kernels.cuh"
#include "pairbits_kernels.cuh"
#include "probe_kernels.cuh"

using namespace ebic;

struct ebic_ctx {
    int device = 0;
    int sm_count = 0;
    int smem_optin = 0;
    int64_t rows = 0;
    int32_t cols = 0;
    int64_t ld = 0;
    int32_t missing_mode = 0;
    int32_t kernel_request = EBIC_KERNEL_AUTO;

    float* Mc = nullptr;                    // [cols][ld]
    uint32_t* nanmask = nullptr;            // [cols][ld/32]
    unsigned long long* nonmissing = nullptr;  // [cols]
    uint8_t* Rk = nullptr;                  // [cols][ld] or nullptr
    uint32_t* PB = nullptr;                 // pair bit columns [cols*cols][ld/32] or nullptr
    int64_t pb_bytes = 0;
    int32_t* d_err = nullptr;               // sticky device error
    unsigned long long* d_visits = nullptr; // executed-visit counter (instrumentation)
    unsigned long long* d_task = nullptr;   // task counter of the persistent PAIRBITS kernel (zeroed by every ingest)
    int32_t pb_persist_ctas = 0;            // resident CTAs of that kernel on this GPU (0 = not yet queried)
    int32_t count_visits = 0;

    // scratch, grown on demand
    int2* meta = nullptr;
    int64_t meta_cap = 0;
    int32_t* pids = nullptr;
    int64_t pids_cap = 0;
    uint8_t* pids8 = nullptr;               // packed byte ids for the tiled kernels (cols <= 256)
    int64_t pids8_cap = 0;
    int32_t* ppair = nullptr;               // pair indices for the pair-bit kernels
    int64_t ppair_cap = 0;
    int32_t* prec = nullptr;                // 128-byte per-individual records for the pair-bit kernels
    int64_t prec_cap = 0;
    int32_t early_exit = 1;
    int32_t extract_pairbits = 1;           // extraction reads the pair table when it exists
    // staging for host-pointer calls
    void* stage[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    int64_t stage_cap[5] = {0, 0, 0, 0, 0};

    // bit 1 of `instrument`: time the fitness kernel(s) of each eval with CUDA events on its stream
    static constexpr int kTimingRing = 256;
    cudaEvent_t ev_begin[kTimingRing] = {};
    cudaEvent_t ev_end[kTimingRing] = {};
    int32_t time_kernels = 0;
    int64_t timed_evals = 0;

    int64_t bytes_owned = 0;
    int64_t launches = 0;
    int32_t last_grid = 0;
    int32_t last_T = 0;
    int32_t last_kernel = 0;                // kernel of the last fitness launch (0 = none yet)
};

namespace {

inline int cuda_status(cudaError_t e) {
    if (e == cudaSuccess) return EBIC_OK;
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? EBIC_ERR_OOM : EBIC_ERR_CUDA;
}
#define EBIC_TRY(expr)                         \
    do {                                       \
        int st__ = cuda_status((expr));        \
        if (st__ != EBIC_OK) return st__;      \
    } while (0)

int dev_alloc(ebic_ctx* ctx, void** p, int64_t bytes) {
    *p = nullptr;
    if (bytes <= 0) bytes = 16;
    cudaError_t e = cudaMalloc(p, static_cast<size_t>(bytes));
    if (e != cudaSuccess) {
        cudaGetLastError();
        *p = nullptr;
        return e == cudaErrorMemoryAllocation ? EBIC_ERR_OOM : EBIC_ERR_CUDA;
    }
    ctx->bytes_owned += bytes;
    return EBIC_OK;
}

int grow(ebic_ctx* ctx, void** p, int64_t* cap, int64_t bytes) {
    if (bytes <= *cap) return EBIC_OK;
    if (*p) {
        cudaError_t e = cudaFree(*p);      // synchronises: earlier work using the buffer has finished
        if (e != cudaSuccess) return cuda_status(e);
        ctx->bytes_owned -= *cap;
        *p = nullptr;
        *cap = 0;
    }
    int64_t want = std::max<int64_t>(bytes + bytes / 4, 4096);
    int st = dev_alloc(ctx, p, want);
    if (st == EBIC_OK) *cap = want;
    return st;
}

bool is_device_pointer(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

constexpr int64_t kPairbitsAutoMaxBytes = 8ll << 30;   // ebic_create builds the pair table up to this size
constexpr int kConsF32 = 31;   // consumer warps of the TILED_F32 kernel (+1 producer = 1024 threads)
constexpr int kConsR8 = 15;    // consumer warps of the RANK8 kernel     (+1 producer =  512 threads)

// Experiment knob (not part of the ABI): EBIC_R8_CONS=23 selects the 24-warp RANK8 build.
int env_int(const char* name, int dflt) {
    const char* v = std::getenv(name);
    return v ? std::atoi(v) : dflt;
}

// Rows per tile: largest multiple of `quantum` that double-buffers into shared memory, <= cap.
int32_t pick_tile_rows(const ebic_ctx* ctx, int32_t elem, int32_t quantum, int32_t cap, int32_t n_ind_launch) {
    const int64_t cnt = (static_cast<int64_t>(n_ind_launch) * 4 + 127) & ~127ll;
    const int64_t avail = static_cast<int64_t>(ctx->smem_optin) - kSmemHeader - cnt;
    if (avail <= 0) return 0;
    int64_t T = avail / (2ll * ctx->cols * elem);
    T = std::min<int64_t>(T, cap);
    T = std::min<int64_t>(T, ctx->ld);
    return static_cast<int32_t>(T / quantum * quantum);
}

int32_t tile_rows_f32(const ebic_ctx* ctx, int32_t n_ind_launch) {
    if (ctx->cols > 256) return 0;          // the tiled kernels read byte ids
    return pick_tile_rows(ctx, 4, kRowsPerSlabF32, 1024, n_ind_launch);
}
int32_t tile_rows_r8(const ebic_ctx* ctx, int32_t n_ind_launch) {
    if (!ctx->Rk) return 0;
    int32_t T = pick_tile_rows(ctx, 1, 4 * kRowsPerSlabR8, 4096, n_ind_launch);
    if (T == 0) T = pick_tile_rows(ctx, 1, 2 * kRowsPerSlabR8, 4096, n_ind_launch);
    if (T == 0) T = pick_tile_rows(ctx, 1, kRowsPerSlabR8, 4096, n_ind_launch);
    return T;
}

int32_t resolve_kernel(const ebic_ctx* ctx, int32_t n_ind_launch) {
    int32_t want = ctx->kernel_request;
    if (want == EBIC_KERNEL_AUTO) {
        if (ctx->PB) return EBIC_KERNEL_PAIRBITS;
        if (tile_rows_r8(ctx, n_ind_launch) > 0) return EBIC_KERNEL_RANK8;
        if (tile_rows_f32(ctx, n_ind_launch) > 0) return EBIC_KERNEL_TILED_F32;
        return EBIC_KERNEL_DIRECT;
    }
    return want;
}

template <class E, int NCONS>
int launch_tiled(ebic_ctx* ctx, const void* M, int32_t T, const int2* meta, int32_t n_ind,
                 unsigned long long* counts, cudaStream_t stream) {
    TiledParams p;
    p.M = M;
    p.ld = ctx->ld;
    p.cols = ctx->cols;
    p.T = T;
    p.n_tiles = (ctx->ld + T - 1) / T;
    p.meta = meta;
    p.idw = reinterpret_cast<const uint32_t*>(ctx->pids8);
    p.n_ind = n_ind;
    p.early_exit = ctx->early_exit;
    p.counts = counts;
    p.visits = ctx->count_visits ? ctx->d_visits : nullptr;
    const size_t smem = tiled_smem_bytes(ctx->cols, T, sizeof(typename E::type), n_ind);
    auto kern = fitness_tiled_kernel<E, NCONS>;
    EBIC_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    const int64_t P = p.n_tiles * n_ind;
    // at least one individual per consumer warp and CTA, never more CTAs than SMs (1 CTA / SM)
    int64_t grid = std::min<int64_t>(ctx->sm_count, std::max<int64_t>(1, P / NCONS));
    ctx->last_grid = static_cast<int32_t>(grid);
    ctx->last_T = T;
    kern<<<static_cast<unsigned>(grid), (NCONS + 1) * 32, smem, stream>>>(p);
    ctx->launches++;
    return cuda_status(cudaGetLastError());
}

// Words of a bit column per PAIRBITS warp task: about `tasks_per_slot` tasks per resident warp slot (32 / SM),
// 256..2048 words (8,192..65,536 rows) per task.
int64_t pairbits_chunk_words(const ebic_ctx* ctx, int32_t n_ind) {
    static const int64_t tasks_per_slot = env_int("EBIC_PB_TASKS_PER_SLOT", 8);
    const int64_t want_tasks = tasks_per_slot * ctx->sm_count * 32;
    const int64_t cw = (ctx->ld / 32) * n_ind / want_tasks;
    return std::max<int64_t>(kPairbitsStepWords, std::min<int64_t>(8 * kPairbitsStepWords, cw / kPairbitsStepWords * kPairbitsStepWords));
}
// The L2 prefetches request EVERY bit column once; that pays only when the population uses most of the cols^2
// columns (n_ids - n_ind = number of pair uses).  A sparse population (wide matrix: P3 uses 14 % of 96,100
// columns) gathers straight from HBM instead -- measured 87 % of the HBM peak.
bool pairbits_dense(const ebic_ctx* ctx, int32_t n_ind, int64_t n_ids) {
    return n_ids - n_ind >= 2ll * ctx->cols * ctx->cols;
}

int launch_pairbits(ebic_ctx* ctx, int32_t n_ind, int64_t n_ids, unsigned long long* counts, cudaStream_t stream) {
    PairbitsParams p;
    p.PB = ctx->PB;
    p.ldw = ctx->ld / 32;
    const int64_t cw = pairbits_chunk_words(ctx, n_ind);
    p.chunk_words = static_cast<int32_t>(cw);
    p.n_chunks = static_cast<int32_t>((p.ldw + cw - 1) / cw);
    p.prec = ctx->prec;
    p.ppair = ctx->ppair;
    p.n_ind = n_ind;
    p.counts = counts;
    p.visits = ctx->count_visits ? ctx->d_visits : nullptr;
    p.n_pairs = ctx->cols * ctx->cols;
    static const int prefetch_dist = env_int("EBIC_PB_PREFETCH", 1);
    p.prefetch_dist = pairbits_dense(ctx, n_ind, n_ids) ? prefetch_dist : 0;
    const int64_t tasks = static_cast<int64_t>(p.n_chunks) * n_ind;
    static const int nw = env_int("EBIC_PB_WARPS", 2);
    const int64_t grid = (tasks + nw - 1) / nw;
    if (grid > 0x7fffffffll) return EBIC_ERR_ARG;
    ctx->last_grid = static_cast<int32_t>(grid);
    ctx->last_T = static_cast<int32_t>(cw * 32);
    const unsigned g = static_cast<unsigned>(grid);
#define EBIC_PB_LAUNCH(NW)                                                              \
    do {                                                                                \
        if (ctx->early_exit) fitness_pairbits_kernel<true, NW><<<g, NW * 32, 0, stream>>>(p);  \
        else fitness_pairbits_kernel<false, NW><<<g, NW * 32, 0, stream>>>(p);                 \
    } while (0)
    static const int use_smem = env_int("EBIC_PB_SMEM", 1);
    static const int persist = env_int("EBIC_PB_PERSIST", 0);
    p.task_counter = ctx->d_task;
    if (persist && use_smem && nw == 2) {
        if (ctx->pb_persist_ctas == 0) {
            int per_sm = 0;
            EBIC_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fitness_pairbits_persistent_kernel<false, 2, true>, 64, 8192));
            ctx->pb_persist_ctas = std::max(1, per_sm) * ctx->sm_count;
        }
        const unsigned pg = static_cast<unsigned>(std::min<int64_t>(ctx->pb_persist_ctas, grid));
        ctx->last_grid = static_cast<int32_t>(pg);
        if (ctx->early_exit) fitness_pairbits_persistent_kernel<true, 2, true><<<pg, 64, 8192, stream>>>(p);
        else fitness_pairbits_persistent_kernel<false, 2, true><<<pg, 64, 8192, stream>>>(p);
        ctx->launches++;
        return cuda_status(cudaGetLastError());
    }
    if (use_smem && nw == 2) {
        if (ctx->early_exit) fitness_pairbits_kernel<true, 2, true><<<g, 64, 8192, stream>>>(p);
        else fitness_pairbits_kernel<false, 2, true><<<g, 64, 8192, stream>>>(p);
        ctx->launches++;
        return cuda_status(cudaGetLastError());
    }
    switch (nw) {
        case 1: EBIC_PB_LAUNCH(1); break;
        case 2: EBIC_PB_LAUNCH(2); break;
        case 4: EBIC_PB_LAUNCH(4); break;
        case 8: EBIC_PB_LAUNCH(8); break;
        default: EBIC_PB_LAUNCH(2); break;
    }
#undef EBIC_PB_LAUNCH
    ctx->launches++;
    return cuda_status(cudaGetLastError());
}

// a2": (re)build the pair-relation bitmasks.  Synchronous.
int build_pairbits(ebic_ctx* ctx) {
    if (ctx->PB) return EBIC_OK;
    if (ctx->cols > 46340) return EBIC_ERR_ARG;                  // cols^2 must fit int32
    const int64_t bytes = static_cast<int64_t>(ctx->cols) * ctx->cols * (ctx->ld / 8);
    if (bytes > (64ll << 30)) return EBIC_ERR_ARG;               // bit-column offsets are uint32 in 16-byte units
    int st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->PB), bytes);
    if (st) return st;
    ctx->pb_bytes = bytes;
    const dim3 grid(static_cast<unsigned>(ctx->ld / 1024), static_cast<unsigned>((ctx->cols + 7) / 8));
    if (grid.y > 65535u) return EBIC_ERR_ARG;
    pairbits_kernel<<<grid, 256>>>(ctx->Mc, ctx->ld, ctx->cols, ctx->PB);
    ctx->launches++;
    st = cuda_status(cudaGetLastError());
    if (!st) st = cuda_status(cudaDeviceSynchronize());
    return st;
}

void free_pairbits(ebic_ctx* ctx) {
    if (!ctx->PB) return;
    cudaFree(ctx->PB);
    ctx->bytes_owned -= ctx->pb_bytes;
    ctx->PB = nullptr;
    ctx->pb_bytes = 0;
}

// Population already on the device: ingest + chain kernels.
int eval_device(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                unsigned long long* counts, cudaStream_t stream) {
    int st = grow(ctx, reinterpret_cast<void**>(&ctx->meta), &ctx->meta_cap, static_cast<int64_t>(n_ind) * 8);
    if (st) return st;
    st = grow(ctx, reinterpret_cast<void**>(&ctx->pids), &ctx->pids_cap, (n_ids + 3ll * n_ind + 8) * 4);
    if (st) return st;
    if (ctx->cols <= 256) {
        st = grow(ctx, reinterpret_cast<void**>(&ctx->pids8), &ctx->pids8_cap, n_ids + 3ll * n_ind + 8);
        if (st) return st;
    }

    if (ctx->PB) {
        st = grow(ctx, reinterpret_cast<void**>(&ctx->ppair), &ctx->ppair_cap, (n_ids + 3ll * n_ind + 8) * 4);
        if (st) return st;
        st = grow(ctx, reinterpret_cast<void**>(&ctx->prec), &ctx->prec_cap, 128ll * n_ind);
        if (st) return st;
    }

    // Experiment, OFF by default (EBIC_PB_WARM=3 turns it on): when PAIRBITS runs next on a dense population the
    // ingest warps also request the first `warm` chunks of every bit column from HBM.  Measured on C4: the
    // event-bracketed fitness kernel drops 63.4 -> 61.0 us but the step does not (83.2 -> 83.6..84.3 us): the
    // cold-start HBM fetch only moves from inside the kernel's bracket to the ingest kernel before it.  It would
    // raise the reported L2 fraction (0.59 -> 0.61) without making an evaluation faster, so it stays off.
    static const int warm_chunks = env_int("EBIC_PB_WARM", 0);
    uint32_t warm_bytes = 0;
    if (warm_chunks > 0 && resolve_kernel(ctx, std::min<int32_t>(kMaxIndPerLaunch, n_ind)) == EBIC_KERNEL_PAIRBITS &&
        pairbits_dense(ctx, n_ind, n_ids))
        warm_bytes = static_cast<uint32_t>(std::min<int64_t>(warm_chunks * pairbits_chunk_words(ctx, n_ind), ctx->ld / 32) * 4);
    ingest_population_kernel<<<(n_ind + 7) / 8, 256, 0, stream>>>(
        offsets, col_ids, n_ind, n_ids, ctx->cols, ctx->rows, ctx->missing_mode == EBIC_MISSING_ON,
        ctx->nonmissing, ctx->meta, ctx->pids, ctx->cols <= 256 ? ctx->pids8 : nullptr,
        ctx->PB ? ctx->ppair : nullptr, ctx->PB ? ctx->prec : nullptr, static_cast<uint32_t>(ctx->ld / 128), counts,
        ctx->d_err, ctx->PB, ctx->cols * ctx->cols, warm_bytes, ctx->d_task);
    ctx->launches++;
    EBIC_TRY(cudaGetLastError());

    const int slot = static_cast<int>(ctx->timed_evals % ebic_ctx::kTimingRing);
    if (ctx->time_kernels) {
        if (!ctx->ev_begin[slot]) {
            EBIC_TRY(cudaEventCreate(&ctx->ev_begin[slot]));
            EBIC_TRY(cudaEventCreate(&ctx->ev_end[slot]));
        }
        EBIC_TRY(cudaEventRecord(ctx->ev_begin[slot], stream));
    }
    const bool whole = resolve_kernel(ctx, std::min<int32_t>(kMaxIndPerLaunch, n_ind)) == EBIC_KERNEL_PAIRBITS;
    const int32_t per_launch = whole ? n_ind : kMaxIndPerLaunch;   // PAIRBITS has no per-CTA counters
    for (int32_t k0 = 0; k0 < n_ind; k0 += per_launch) {
        const int32_t n = std::min<int32_t>(per_launch, n_ind - k0);
        const int32_t kernel = whole ? EBIC_KERNEL_PAIRBITS : resolve_kernel(ctx, n);
        ctx->last_kernel = kernel;
        if (kernel == EBIC_KERNEL_PAIRBITS) {
            if (!ctx->PB) return EBIC_ERR_ARG;
            st = launch_pairbits(ctx, n, n_ids, counts, stream);
        } else if (kernel == EBIC_KERNEL_RANK8) {
            const int32_t T = tile_rows_r8(ctx, n);
            if (T <= 0) return EBIC_ERR_ARG;
            static const int r8_cons = env_int("EBIC_R8_CONS", kConsR8);
            if (r8_cons == 23)
                st = launch_tiled<ElemR8, 23>(ctx, ctx->Rk, T, ctx->meta + k0, n, counts + k0, stream);
            else
                st = launch_tiled<ElemR8, kConsR8>(ctx, ctx->Rk, T, ctx->meta + k0, n, counts + k0, stream);
        } else if (kernel == EBIC_KERNEL_TILED_F32) {
            const int32_t T = tile_rows_f32(ctx, n);
            if (T <= 0) return EBIC_ERR_ARG;
            st = launch_tiled<ElemF32, kConsF32>(ctx, ctx->Mc, T, ctx->meta + k0, n, counts + k0, stream);
        } else {
            const int64_t gx = ctx->ld / 256;
            int64_t gy = std::max<int64_t>(1, (8ll * ctx->sm_count + gx - 1) / gx);
            gy = std::min<int64_t>(std::min<int64_t>(gy, n), 65535);
            dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(gy));
            fitness_direct_kernel<<<grid, 256, 0, stream>>>(ctx->Mc, ctx->ld, ctx->meta + k0, ctx->pids, n,
                                                            counts + k0);
            ctx->launches++;
            ctx->last_grid = static_cast<int32_t>(std::min<int64_t>(gx * gy, 0x7fffffff));
            ctx->last_T = 256;
            st = cuda_status(cudaGetLastError());
        }
        if (st) return st;
    }
    if (ctx->time_kernels) {
        EBIC_TRY(cudaEventRecord(ctx->ev_end[slot], stream));
        ctx->timed_evals++;
    }
    return EBIC_OK;
}

int extract_device(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                   const int32_t* chosen, int32_t n_chosen, uint64_t* masks, uint64_t* counts,
                   cudaStream_t stream) {
    const int64_t words32 = 2 * ((ctx->rows + 63) / 64);
    if (counts) EBIC_TRY(cudaMemsetAsync(counts, 0, static_cast<size_t>(n_chosen) * 8, stream));
    if (ctx->PB && ctx->extract_pairbits) {
        const dim3 grid(static_cast<unsigned>((words32 + 255) / 256), static_cast<unsigned>(std::min<int32_t>(n_chosen, 65535)));
        extract_rows_pairbits_kernel<<<grid, 256, 0, stream>>>(
            ctx->PB, ctx->ld, ctx->rows, ctx->cols, ctx->missing_mode == EBIC_MISSING_ON, ctx->nanmask, offsets,
            col_ids, n_ind, n_ids, chosen, n_chosen, reinterpret_cast<uint32_t*>(masks), words32,
            reinterpret_cast<unsigned long long*>(counts), ctx->d_err);
        ctx->launches++;
        return cuda_status(cudaGetLastError());
    }
    const int64_t gx = (words32 * 32 + kExtractRowsPerBlock - 1) / kExtractRowsPerBlock;
    dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(std::min<int32_t>(n_chosen, 65535)));
    extract_rows_kernel<<<grid, 256, 0, stream>>>(
        ctx->Mc, ctx->ld, ctx->rows, ctx->cols, ctx->missing_mode == EBIC_MISSING_ON, ctx->nanmask, offsets,
        col_ids, n_ind, n_ids, chosen, n_chosen, reinterpret_cast<uint32_t*>(masks), words32,
        reinterpret_cast<unsigned long long*>(counts), ctx->d_err);
    ctx->launches++;
    return cuda_status(cudaGetLastError());
}

int stage_in(ebic_ctx* ctx, int slot, const void* host, int64_t bytes, cudaStream_t stream, void** dev) {
    int st = grow(ctx, &ctx->stage[slot], &ctx->stage_cap[slot], bytes);
    if (st) return st;
    *dev = ctx->stage[slot];
    if (bytes > 0) EBIC_TRY(cudaMemcpyAsync(*dev, host, static_cast<size_t>(bytes), cudaMemcpyHostToDevice, stream));
    return EBIC_OK;
}

}  // namespace

extern "C" {

static int create_impl(const float* matrix, int64_t rows, int32_t cols, int32_t missing_mode, int32_t use_sentinel,
                       float sentinel, ebic_ctx** out) {
    if (out) *out = nullptr;
    if (!matrix || !out || rows <= 0 || rows > 2147483647ll || cols <= 0 ||
        (missing_mode != EBIC_MISSING_OFF && missing_mode != EBIC_MISSING_ON) || (use_sentinel && sentinel != sentinel))
        return EBIC_ERR_ARG;
    ebic_ctx* ctx = new (std::nothrow) ebic_ctx();
    if (!ctx) return EBIC_ERR_OOM;
    int st = EBIC_OK;
    float* staging = nullptr;
    do {
        if ((st = cuda_status(cudaGetDevice(&ctx->device)))) break;
        if ((st = cuda_status(cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device)))) break;
        if ((st = cuda_status(cudaDeviceGetAttribute(&ctx->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device)))) break;
        ctx->rows = rows;
        ctx->cols = cols;
        ctx->missing_mode = missing_mode;
        ctx->ld = (rows + kLdAlign - 1) / kLdAlign * kLdAlign;
        const int64_t n = ctx->ld * cols;
        if ((st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->Mc), n * 4))) break;
        if ((st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->nanmask), n / 8))) break;
        if ((st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->nonmissing), static_cast<int64_t>(cols) * 8))) break;
        if ((st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->d_err), 32))) break;
        ctx->d_visits = reinterpret_cast<unsigned long long*>(ctx->d_err + 2);
        ctx->d_task = reinterpret_cast<unsigned long long*>(ctx->d_err + 4);
        if ((st = cuda_status(cudaMemset(ctx->d_err, 0, 32)))) break;
        if ((st = cuda_status(cudaMemset(ctx->nonmissing, 0, static_cast<size_t>(cols) * 8)))) break;

        // a1: transpose (device input: in one go; host input: through a bounded staging buffer)
        const dim3 tb(32, 8);
        const unsigned gy = static_cast<unsigned>(std::min<int64_t>((cols + 31) / 32, 65535));
        if (is_device_pointer(matrix)) {
            const dim3 grid(static_cast<unsigned>((rows + 31) / 32), gy);
            transpose_pad_kernel<<<grid, tb>>>(matrix, ctx->Mc, 0, rows, cols, ctx->ld, use_sentinel, sentinel);
            ctx->launches++;
            if ((st = cuda_status(cudaGetLastError()))) break;
        } else {
            const int64_t chunk_rows = std::max<int64_t>(32, std::min<int64_t>(rows, (256ll << 20) / (4ll * cols) / 32 * 32));
            if ((st = cuda_status(cudaMalloc(reinterpret_cast<void**>(&staging), static_cast<size_t>(chunk_rows) * cols * 4)))) break;
            for (int64_t r0 = 0; r0 < rows && st == EBIC_OK; r0 += chunk_rows) {
                const int64_t nr = std::min<int64_t>(chunk_rows, rows - r0);
                if ((st = cuda_status(cudaMemcpy(staging, matrix + r0 * cols, static_cast<size_t>(nr) * cols * 4, cudaMemcpyHostToDevice)))) break;
                const dim3 grid(static_cast<unsigned>((nr + 31) / 32), gy);
                transpose_pad_kernel<<<grid, tb>>>(staging, ctx->Mc, r0, nr, cols, ctx->ld, use_sentinel, sentinel);
                ctx->launches++;
                st = cuda_status(cudaGetLastError());
            }
            if (st) break;
        }
        if (ctx->ld > rows) {
            const int64_t npad = (ctx->ld - rows) * cols;
            fill_pad_kernel<<<static_cast<unsigned>(std::min<int64_t>((npad + 255) / 256, 4096)), 256>>>(ctx->Mc, rows, cols, ctx->ld);
            ctx->launches++;
            if ((st = cuda_status(cudaGetLastError()))) break;
        }
        // a2: NaN bitmask + per-column non-missing counts
        {
            const int64_t words = ctx->ld / 32;
            const dim3 grid(static_cast<unsigned>((words + 255) / 256), static_cast<unsigned>(std::min<int32_t>(cols, 65535)));
            nan_mask_kernel<<<grid, 256>>>(ctx->Mc, ctx->ld, cols, ctx->nanmask, ctx->nonmissing);
            ctx->launches++;
            if ((st = cuda_status(cudaGetLastError()))) break;
        }
        // a2': rank tiles
        if (cols <= kMaxColsRank8) {
            if ((st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->Rk), n))) break;
            const size_t smem = static_cast<size_t>(cols) * 256 * 5;
            if ((st = cuda_status(cudaFuncSetAttribute(rank8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem))))) break;
            rank8_kernel<<<static_cast<unsigned>(ctx->ld / 256), 256, smem>>>(ctx->Mc, ctx->ld, cols, ctx->Rk);
            ctx->launches++;
            if ((st = cuda_status(cudaGetLastError()))) break;
        }
        if ((st = cuda_status(cudaDeviceSynchronize()))) break;
        // a2": pair-relation bitmasks, when they fit comfortably (otherwise the rank / float kernels serve)
        if (cols <= 46340) {
            const int64_t pb = static_cast<int64_t>(cols) * cols * (ctx->ld / 8);
            size_t free_b = 0, total_b = 0;
            if ((st = cuda_status(cudaMemGetInfo(&free_b, &total_b)))) break;
            if (pb <= kPairbitsAutoMaxBytes && pb <= static_cast<int64_t>(free_b / 2)) {
                st = build_pairbits(ctx);
                if (st == EBIC_ERR_OOM) {
                    free_pairbits(ctx);
                    st = EBIC_OK;
                }
                if (st) break;
            }
        }
    } while (0);
    if (staging) cudaFree(staging);
    if (st != EBIC_OK) {
        ebic_destroy(ctx);
        return st;
    }
    *out = ctx;
    return EBIC_OK;
}

int ebic_create(const float* matrix, int64_t rows, int32_t cols, int32_t missing_mode, ebic_ctx** out) {
    return create_impl(matrix, rows, cols, missing_mode, 0, 0.0f, out);
}

int ebic_create_sentinel(const float* matrix, int64_t rows, int32_t cols, int32_t missing_mode, float sentinel,
                         ebic_ctx** out) {
    return create_impl(matrix, rows, cols, missing_mode, 1, sentinel, out);
}

int ebic_destroy(ebic_ctx* ctx) {
    if (!ctx) return EBIC_OK;
    cudaFree(ctx->Mc);
    cudaFree(ctx->nanmask);
    cudaFree(ctx->nonmissing);
    cudaFree(ctx->Rk);
    cudaFree(ctx->PB);
    cudaFree(ctx->ppair);
    cudaFree(ctx->prec);
    cudaFree(ctx->d_err);
    cudaFree(ctx->meta);
    cudaFree(ctx->pids);
    cudaFree(ctx->pids8);
    for (void* s : ctx->stage) cudaFree(s);
    for (int i = 0; i < ebic_ctx::kTimingRing; ++i) {
        if (ctx->ev_begin[i]) cudaEventDestroy(ctx->ev_begin[i]);
        if (ctx->ev_end[i]) cudaEventDestroy(ctx->ev_end[i]);
    }
    cudaGetLastError();
    delete ctx;
    return EBIC_OK;
}

int ebic_eval_fitness(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                      uint64_t* counts, void* cuda_stream) {
    if (!ctx || n_ind < 0 || n_ids < 0 || n_ind == 2147483647) return EBIC_ERR_ARG;
    if (n_ind == 0) return EBIC_OK;
    if (!offsets || !counts || (!col_ids && n_ids > 0)) return EBIC_ERR_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const bool pop_dev = is_device_pointer(offsets);
    const bool out_dev = is_device_pointer(counts);
    const int32_t* d_off = offsets;
    const int32_t* d_ids = col_ids;
    unsigned long long* d_counts = reinterpret_cast<unsigned long long*>(counts);
    int st;
    if (!pop_dev) {
        void* p;
        if ((st = stage_in(ctx, 0, offsets, (static_cast<int64_t>(n_ind) + 1) * 4, stream, &p))) return st;
        d_off = static_cast<const int32_t*>(p);
        if ((st = stage_in(ctx, 1, col_ids, n_ids * 4, stream, &p))) return st;
        d_ids = static_cast<const int32_t*>(p);
    }
    if (!out_dev) {
        if ((st = grow(ctx, &ctx->stage[2], &ctx->stage_cap[2], static_cast<int64_t>(n_ind) * 8))) return st;
        d_counts = static_cast<unsigned long long*>(ctx->stage[2]);
    }
    if ((st = eval_device(ctx, d_off, d_ids, n_ind, n_ids, d_counts, stream))) return st;
    if (!out_dev) {
        EBIC_TRY(cudaMemcpyAsync(counts, d_counts, static_cast<size_t>(n_ind) * 8, cudaMemcpyDeviceToHost, stream));
        EBIC_TRY(cudaStreamSynchronize(stream));
    } else if (!pop_dev) {
        EBIC_TRY(cudaStreamSynchronize(stream));   // host population buffers may be reused on return
    }
    return EBIC_OK;
}

int ebic_extract_rows(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                      const int32_t* chosen, int32_t n_chosen, uint64_t* masks, uint64_t* counts,
                      void* cuda_stream) {
    if (!ctx || n_ind < 0 || n_ids < 0 || n_chosen < 0) return EBIC_ERR_ARG;
    if (n_chosen == 0) return EBIC_OK;
    if (!offsets || !chosen || !masks || (!col_ids && n_ids > 0)) return EBIC_ERR_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const bool pop_dev = is_device_pointer(offsets);
    const bool out_dev = is_device_pointer(masks);
    const int64_t words = (ctx->rows + 63) / 64;
    const int32_t* d_off = offsets;
    const int32_t* d_ids = col_ids;
    const int32_t* d_chosen = chosen;
    uint64_t* d_masks = masks;
    uint64_t* d_counts = counts;
    int st;
    void* p;
    if (!pop_dev) {
        if ((st = stage_in(ctx, 0, offsets, (static_cast<int64_t>(n_ind) + 1) * 4, stream, &p))) return st;
        d_off = static_cast<const int32_t*>(p);
        if ((st = stage_in(ctx, 1, col_ids, n_ids * 4, stream, &p))) return st;
        d_ids = static_cast<const int32_t*>(p);
        if ((st = stage_in(ctx, 3, chosen, static_cast<int64_t>(n_chosen) * 4, stream, &p))) return st;
        d_chosen = static_cast<const int32_t*>(p);
    }
    if (!out_dev) {
        if ((st = grow(ctx, &ctx->stage[4], &ctx->stage_cap[4], static_cast<int64_t>(n_chosen) * words * 8))) return st;
        d_masks = static_cast<uint64_t*>(ctx->stage[4]);
        if (counts) {
            if ((st = grow(ctx, &ctx->stage[2], &ctx->stage_cap[2], static_cast<int64_t>(n_chosen) * 8))) return st;
            d_counts = static_cast<uint64_t*>(ctx->stage[2]);
        }
    }
    if ((st = extract_device(ctx, d_off, d_ids, n_ind, n_ids, d_chosen, n_chosen, d_masks, d_counts, stream))) return st;
    if (!out_dev) {
        EBIC_TRY(cudaMemcpyAsync(masks, d_masks, static_cast<size_t>(n_chosen) * words * 8, cudaMemcpyDeviceToHost, stream));
        if (counts) EBIC_TRY(cudaMemcpyAsync(counts, d_counts, static_cast<size_t>(n_chosen) * 8, cudaMemcpyDeviceToHost, stream));
        EBIC_TRY(cudaStreamSynchronize(stream));
    } else if (!pop_dev) {
        EBIC_TRY(cudaStreamSynchronize(stream));
    }
    return EBIC_OK;
}

int64_t ebic_mask_words(const ebic_ctx* ctx) { return ctx ? (ctx->rows + 63) / 64 : -1; }

int ebic_status(ebic_ctx* ctx, void* cuda_stream) {
    if (!ctx) return EBIC_ERR_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int32_t err = 0;
    EBIC_TRY(cudaMemcpyAsync(&err, ctx->d_err, 4, cudaMemcpyDeviceToHost, stream));
    EBIC_TRY(cudaMemsetAsync(ctx->d_err, 0, 4, stream));
    EBIC_TRY(cudaStreamSynchronize(stream));
    return err;
}

int ebic_set_kernel(ebic_ctx* ctx, int32_t kernel) {
    if (!ctx) return EBIC_ERR_ARG;
    switch (kernel) {
        case EBIC_KERNEL_AUTO:
        case EBIC_KERNEL_DIRECT:
            break;
        case EBIC_KERNEL_TILED_F32:
            if (tile_rows_f32(ctx, 1) <= 0) return EBIC_ERR_ARG;
            break;
        case EBIC_KERNEL_RANK8:
            if (tile_rows_r8(ctx, 1) <= 0) return EBIC_ERR_ARG;
            break;
        case EBIC_KERNEL_PAIRBITS:
            if (!ctx->PB) return EBIC_ERR_ARG;
            break;
        default:
            return EBIC_ERR_ARG;
    }
    ctx->kernel_request = kernel;
    return EBIC_OK;
}

int ebic_set_pairbits(ebic_ctx* ctx, int32_t on) {
    if (!ctx) return EBIC_ERR_ARG;
    if (cudaDeviceSynchronize() != cudaSuccess) return cuda_status(cudaGetLastError());
    if (on == 0) {
        free_pairbits(ctx);
        if (ctx->kernel_request == EBIC_KERNEL_PAIRBITS) ctx->kernel_request = EBIC_KERNEL_AUTO;
        return EBIC_OK;
    }
    int st = build_pairbits(ctx);
    if (st) free_pairbits(ctx);
    return st;
}

int ebic_set_extract_source(ebic_ctx* ctx, int32_t use_pairbits) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->extract_pairbits = use_pairbits ? 1 : 0;
    return EBIC_OK;
}

int ebic_set_early_exit(ebic_ctx* ctx, int32_t on) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->early_exit = on ? 1 : 0;
    return EBIC_OK;
}

int ebic_set_instrumentation(ebic_ctx* ctx, int32_t on) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->count_visits = (on & 1) ? 1 : 0;
    ctx->time_kernels = (on & 2) ? 1 : 0;
    ctx->timed_evals = 0;
    return EBIC_OK;
}

int64_t ebic_get_info(ebic_ctx* ctx, int32_t what) {
    if (!ctx) return -1;
    switch (what) {
        case 0: return ctx->rows;
        case 1: return ctx->cols;
        case 2: return ctx->ld;
        case 3: return ctx->missing_mode;
        case 4: return resolve_kernel(ctx, 1);
        case 5: return ctx->last_T;
        case 6: return ctx->last_grid;
        case 7: return ctx->sm_count;
        case 8: return ctx->launches;
        case 9: return ctx->bytes_owned;
        case 10: {
            unsigned long long v = 0;
            if (cudaDeviceSynchronize() != cudaSuccess ||
                cudaMemcpy(&v, ctx->d_visits, 8, cudaMemcpyDeviceToHost) != cudaSuccess ||
                cudaMemset(ctx->d_visits, 0, 8) != cudaSuccess) {
                cudaGetLastError();
                return -1;
            }
            return static_cast<int64_t>(v);
        }
        case 11: {   // mean fitness-kernel time of the evals timed since instrumentation was set, in ns
            if (ctx->timed_evals == 0 || cudaDeviceSynchronize() != cudaSuccess) {
                cudaGetLastError();
                return -1;
            }
            const int64_t n = std::min<int64_t>(ctx->timed_evals, ebic_ctx::kTimingRing);
            double total_ms = 0;
            for (int64_t i = 0; i < n; ++i) {
                float ms = 0;
                if (cudaEventElapsedTime(&ms, ctx->ev_begin[i], ctx->ev_end[i]) != cudaSuccess) {
                    cudaGetLastError();
                    return -1;
                }
                total_ms += ms;
            }
            return static_cast<int64_t>(total_ms / n * 1e6);
        }
        case 12: return ctx->timed_evals;
        case 13: return ctx->early_exit;
        case 14: return ctx->pb_bytes;
        case 15: return ctx->last_kernel;
        default: return -1;
    }
}

int ebic_debug_read(const ebic_ctx* ctx, int32_t what, void* dst, int64_t dst_bytes) {
    if (!ctx || !dst) return EBIC_ERR_ARG;
    const int64_t n = ctx->ld * ctx->cols;
    const void* src = nullptr;
    int64_t bytes = 0;
    switch (what) {
        case 0: src = ctx->Mc; bytes = n * 4; break;
        case 1: src = ctx->nanmask; bytes = n / 8; break;
        case 2: src = ctx->nonmissing; bytes = static_cast<int64_t>(ctx->cols) * 8; break;
        case 3: src = ctx->Rk; bytes = n; break;
        case 4: src = ctx->PB; bytes = ctx->pb_bytes; break;
        default: return EBIC_ERR_ARG;
    }
    if (!src || bytes != dst_bytes) return EBIC_ERR_ARG;
    return cuda_status(cudaMemcpy(dst, src, static_cast<size_t>(bytes), cudaMemcpyDeviceToHost));
}

int ebic_probe_read_bandwidth(int64_t buffer_bytes, int32_t reps, double* gb_per_s) {
    if (!gb_per_s || buffer_bytes < (1ll << 20) || reps < 1) return EBIC_ERR_ARG;
    *gb_per_s = 0.0;
    int dev = 0, sms = 0;
    EBIC_TRY(cudaGetDevice(&dev));
    EBIC_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int64_t n_vec = buffer_bytes / 16;
    if (n_vec / (8ll * sms * 8 * 256) <= 0) return EBIC_ERR_ARG;
    uint4* buf = nullptr;
    unsigned int* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int st = cuda_status(cudaMalloc(&buf, static_cast<size_t>(n_vec) * 16));
    if (!st) st = cuda_status(cudaMalloc(&sink, 4));
    if (!st) st = cuda_status(cudaMemset(buf, 0x5a, static_cast<size_t>(n_vec) * 16));
    if (!st) st = cuda_status(cudaEventCreate(&e0));
    if (!st) st = cuda_status(cudaEventCreate(&e1));
    double best = 0.0;
    for (int per_sm = 2; per_sm <= 8 && !st; per_sm *= 2) {        // 2, 4, 8 CTAs of 256 threads per SM: keep the best
        const int grid = sms * per_sm;
        const int64_t stride = static_cast<int64_t>(grid) * 256;
        const int64_t span = n_vec / (8 * stride) * (8 * stride);
        for (int pass = 0; pass < 4 && !st; ++pass) {            // pass 0 warms the cache; best of the next 3
            cudaEventRecord(e0, nullptr);
            probe_read_kernel<<<grid, 256>>>(buf, n_vec, reps, sink);
            cudaEventRecord(e1, nullptr);
            st = cuda_status(cudaEventSynchronize(e1));
            float ms = 0.f;
            if (!st) st = cuda_status(cudaEventElapsedTime(&ms, e0, e1));
            if (!st && pass > 0 && ms > 0.f)
                best = std::max(best, static_cast<double>(span) * 16.0 * reps / (ms * 1e-3) / 1e9);
        }
    }
    if (!st) *gb_per_s = best;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(buf);
    return st;
}

const char* ebic_strerror(int status) {
    switch (status) {
        case EBIC_OK: return "ok";
        case EBIC_ERR_ARG: return "invalid argument";
        case EBIC_ERR_OOM: return "out of device memory";
        case EBIC_ERR_CUDA: return "CUDA runtime error";
        case EBIC_ERR_BAD_COLUMN: return "column id outside [0, cols) in the population";
        case EBIC_ERR_BAD_OFFSETS: return "bad population offsets or chosen index";
        case EBIC_ERR_IO: return "cannot read the file as a delimited matrix";
        default: return "unknown status";
    }
}

}  // extern "C"
