// ebic_api.cu -- host side of libebic.so: the boundary declared in include/ebic.h.
// Links cudart only (no torch).  Product code: shares nothing with oracle/.  No environment variables are read:
// the configuration is the set of defaults in ebic_ctx.hpp, changed only through include/ebic_debug.h.
#include "../../include/ebic.h"
#include "../../include/ebic_debug.h"

#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "ebic_ctx.hpp"
#include "ebic_device.cuh"
#include "extract_kernels.cuh"
#include "fitness_kernels.cuh"
#include "ingest_kernels.cuh"
#include "loader_kernels.cuh"
#include "pairbits_kernels.cuh"
#include "pairtile_kernels.cuh"
#include "prefix_kernels.cuh"
#include "union_kernels.cuh"

using namespace ebic;

#define EBIC_TRY(expr)                                  \
    do {                                                \
        int st__ = ebic_host::cuda_status((expr));      \
        if (st__ != EBIC_OK) return st__;               \
    } while (0)

namespace {

constexpr int64_t kPairbitsAutoMaxBytes = 32ll << 30;  // ebic_create builds the pair table up to this size (and half of the free memory)
constexpr int kConsF32 = 31;   // consumer warps of the TILED_F32 kernel (+1 producer = 1024 threads)
constexpr int kConsR8 = 15;    // consumer warps of the RANK8 kernel     (+1 producer =  512 threads)

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
    // A captured launch sequence (eval_extract_impl) has the addresses of the scratch buffers baked in.  Whatever call
    // makes one of them move -- typically one that is not replayed itself: host pointers, the default stream, a larger
    // population -- takes the graph with it; the next matching call starts over with a plain launch.
    if (ctx->graph_exec) {
        cudaGraphExecDestroy(ctx->graph_exec);
        ctx->graph_exec = nullptr;
        ctx->graph_state = 0;
    }
    if (*p) {
        cudaError_t e = cudaFree(*p);      // synchronises: earlier work using the buffer has finished
        if (e != cudaSuccess) return ebic_host::cuda_status(e);
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

// The context belongs to the device that was current in ebic_create; every later call must run on it.
bool on_ctx_device(const ebic_ctx* ctx) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return dev == ctx->device;
}

// Kernel launch with the programmatic-dependent-launch attribute: the kernel may begin while its predecessor on
// the stream is still running; it orders itself behind it with griddep_wait() (ebic_device.cuh).
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, bool pdl,
                       Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// Rows per tile: largest multiple of `quantum` that fits shared memory `nbuf` times, <= cap.
int32_t pick_tile_rows(const ebic_ctx* ctx, int32_t elem, int32_t quantum, int32_t cap, int32_t n_ind_launch, int32_t nbuf = 2) {
    const int64_t cnt = (static_cast<int64_t>(n_ind_launch) * 4 + 127) & ~127ll;
    const int64_t avail = static_cast<int64_t>(ctx->smem_optin) - kSmemHeader - cnt;
    if (avail <= 0) return 0;
    int64_t T = avail / (static_cast<int64_t>(nbuf) * ctx->cols * elem);
    T = std::min<int64_t>(T, cap);
    T = std::min<int64_t>(T, ctx->ld);
    return static_cast<int32_t>(T / quantum * quantum);
}

// TILED_F32 double-buffers its tiles when two of them fit; a matrix too wide for that (221 < cols <= 445) gets one
// 128-row tile: every individual of the population reuses it, so the load it can no longer hide is a few per cent.
int32_t tile_bufs_f32(const ebic_ctx* ctx, int32_t n_ind_launch) {
    return pick_tile_rows(ctx, 4, kRowsPerSlabF32, 1024, n_ind_launch, 2) > 0 ? 2 : 1;
}
int32_t tile_rows_f32(const ebic_ctx* ctx, int32_t n_ind_launch) {
    if (ctx->cols > 65535) return 0;        // the id records hold bytes (cols <= 256) or halfwords
    return pick_tile_rows(ctx, 4, kRowsPerSlabF32, 1024, n_ind_launch, tile_bufs_f32(ctx, n_ind_launch));
}
int32_t tile_rows_r8(const ebic_ctx* ctx, int32_t n_ind_launch) {
    if (ctx->cols > kMaxColsRank8) return 0;
    int32_t T = pick_tile_rows(ctx, 1, 4 * kRowsPerSlabR8, 4096, n_ind_launch);
    if (T == 0) T = pick_tile_rows(ctx, 1, 2 * kRowsPerSlabR8, 4096, n_ind_launch);
    if (T == 0) T = pick_tile_rows(ctx, 1, kRowsPerSlabR8, 4096, n_ind_launch);
    return T;
}
// UNION_F32: columns a staged 128-row tile can hold, double-buffered, next to the records of a 256-individual batch.
int32_t union_cap(const ebic_ctx* ctx) {
    if (ctx->cols > kUnionMaxCols) return 0;
    const int64_t avail = static_cast<int64_t>(ctx->smem_optin) - kSmemHeader - 2 * 256 * 40;
    return static_cast<int32_t>(std::min<int64_t>(std::min<int64_t>(avail / (2ll * kUnionTileRows * 4), 256), ctx->cols));
}
// Individuals per batch: the largest batch whose expected union, cols * (1 - exp(-batch * mean_L / cols)), still
// fits 85 % of the tile (the plan kernel evaluates whatever does not fit from global memory).
int32_t union_batch(const ebic_ctx* ctx, int32_t n_ind, int64_t n_ids) {
    if (ctx->union_batch > 0) return (ctx->union_batch + 1) & ~1;
    const double cap = 0.85 * union_cap(ctx), cols = ctx->cols;
    const double mean_l = std::max(2.0, static_cast<double>(n_ids) / std::max(n_ind, 1));
    double b = 128.0;
    if (cap < cols) b = -cols / mean_l * std::log(1.0 - cap / cols);
    return static_cast<int32_t>(std::max(4.0, std::min(128.0, b))) & ~1;       // even: the records are copied 16 bytes at a time
}

// PAIRTILE: a 1,024-row tile of all cols^2 bit columns next to one 4-byte counter per individual of the launch.
int64_t pairtile_smem(const ebic_ctx* ctx, int32_t n_ind_launch) {
    const int64_t n_groups = (n_ind_launch + 31) / 32;
    return kPtHeader + static_cast<int64_t>(ctx->cols) * ctx->cols * 128 + 4ll * n_groups * 32 + 4ll * ((n_groups + 3) & ~3ll);
}
// The record cache (entries 0..7 of every record, 16 bytes per sorted position) when it fits next to all that.
bool pairtile_rec_cache(const ebic_ctx* ctx, int32_t n_ind_launch) {
    return pairtile_smem(ctx, n_ind_launch) + 512ll * ((n_ind_launch + 31) / 32) <= ctx->smem_optin;
}
bool pairtile_fits(const ebic_ctx* ctx) { return ctx->cols <= 90 && pairtile_smem(ctx, 1024) <= ctx->smem_optin; }
// Individuals per launch: as many counters as fit next to the tile, at most kMaxIndPerLaunch.
int32_t pairtile_chunk(const ebic_ctx* ctx, int32_t n_ind) {
    const int64_t room = (static_cast<int64_t>(ctx->smem_optin) - pairtile_smem(ctx, 0)  - 16) / 132 * 32;   // 4 B + 1/8 int per individual
    return static_cast<int32_t>(std::min<int64_t>(std::min<int64_t>(n_ind, kMaxIndPerLaunch), room));
}

int32_t tile_rows(const ebic_ctx* ctx, int32_t kernel, int32_t n_ind_launch) {
    return kernel == EBIC_KERNEL_RANK8 ? tile_rows_r8(ctx, n_ind_launch) : tile_rows_f32(ctx, n_ind_launch);
}

// Individuals per launch of a tiled kernel: the per-CTA counters (4 bytes each) share the shared memory with the
// tiles, so a wide matrix gets a smaller population chunk rather than no tile at all.
int32_t tiled_chunk(const ebic_ctx* ctx, int32_t kernel, int32_t n_ind) {
    int32_t n = std::min<int32_t>(n_ind, kMaxIndPerLaunch);
    while (n > 1024 && tile_rows(ctx, kernel, n) <= 0) n = (n + 1) / 2;
    return n;
}

}  // namespace

namespace ebic_host {

// Elapsed GPU time of a synchronous build step on the legacy stream (CUDA events), into *ms.
struct BuildTimer {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float* ms;
    explicit BuildTimer(float* out) : ms(out) {
        if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess) cudaEventRecord(e0);
    }
    ~BuildTimer() {
        if (e0 && e1 && cudaEventRecord(e1) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess)
            cudaEventElapsedTime(ms, e0, e1);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
        cudaGetLastError();
    }
};

int cuda_status(cudaError_t e) {
    if (e == cudaSuccess) return EBIC_OK;
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? EBIC_ERR_OOM : EBIC_ERR_CUDA;
}

bool kernel_applies(const ebic_ctx* ctx, int32_t kernel) {
    switch (kernel) {
        case EBIC_KERNEL_AUTO:
        case EBIC_KERNEL_DIRECT: return true;
        case EBIC_KERNEL_TILED_F32: return tile_rows_f32(ctx, 1024) > 0;     // a tile next to >= 1,024 per-CTA counters
        case EBIC_KERNEL_RANK8: return tile_rows_r8(ctx, 1024) > 0;
        case EBIC_KERNEL_PAIRBITS:
        case EBIC_KERNEL_PREFIX: return ctx->PB != nullptr;
        case EBIC_KERNEL_PAIRTILE: return ctx->PBT != nullptr;
        case EBIC_KERNEL_UNION_F32: return union_cap(ctx) >= 2;
        default: return false;
    }
}

// PAIRTILE against PAIRBITS (both need the table; measured on 20 / 32 / 40 columns x 30 k .. 1.5 M rows x 128 .. 4,096
// individuals): staging whole tiles pays once (a) there are enough (tile, pair-use) units to keep
// every SM busy past the fixed cost of the extra launch, and (b) the population uses every staged bit column
// several times -- a small population reads only the columns it needs through PAIRBITS.
bool pairtile_pays(const ebic_ctx* ctx, int32_t n_ind, int64_t n_ids) {
    if (!ctx->PBT) return false;
    const int64_t tiles = ctx->ld / kPairTileRows, uses = std::max<int64_t>(n_ids - n_ind, 0);
    const int64_t n_pairs = static_cast<int64_t>(ctx->cols) * ctx->cols;
    if (ctx->pt_min_work > 0) return tiles * uses >= ctx->pt_min_work;
    const double reuse_penalty = std::max(1.0, 16.0 * n_pairs / static_cast<double>(std::max<int64_t>(uses, 1)));
    return static_cast<double>(tiles) * uses >= 4.0e6 * reuse_penalty;
}

int32_t resolve_kernel(const ebic_ctx* ctx, int32_t n_ind, int64_t n_ids) {
    if (ctx->kernel_request != EBIC_KERNEL_AUTO) return ctx->kernel_request;
    if (pairtile_pays(ctx, n_ind, n_ids)) return EBIC_KERNEL_PAIRTILE;
    if (ctx->PB) return EBIC_KERNEL_PAIRBITS;
    if (ctx->Rk && kernel_applies(ctx, EBIC_KERNEL_RANK8)) return EBIC_KERNEL_RANK8;
    if (kernel_applies(ctx, EBIC_KERNEL_TILED_F32)) return EBIC_KERNEL_TILED_F32;   // every column fits a tile
    if (kernel_applies(ctx, EBIC_KERNEL_UNION_F32)) return EBIC_KERNEL_UNION_F32;   // wider: a batch's column union
    return EBIC_KERNEL_DIRECT;
}

// a2': rank tiles (cols <= 127).  Synchronous.
int build_rank_tiles(ebic_ctx* ctx) {
    if (ctx->Rk) return EBIC_OK;
    if (ctx->cols > kMaxColsRank8) return EBIC_ERR_ARG;
    int st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->Rk), ctx->ld * ctx->cols);
    if (st) return st;
    BuildTimer timer(&ctx->create_ms[3]);                        // the kernel, not the allocation
    const size_t smem = static_cast<size_t>(ctx->cols) * 256 * 5;
    EBIC_TRY(cudaFuncSetAttribute(rank8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    rank8_kernel<<<static_cast<unsigned>(ctx->ld / 256), 256, smem>>>(ctx->Mc, ctx->ld, ctx->cols, ctx->Rk);
    ctx->launches++;
    st = cuda_status(cudaGetLastError());
    if (!st) st = cuda_status(cudaDeviceSynchronize());
    return st;
}

// a2": (re)build the pair-relation bitmasks.  Synchronous.
int build_pairbits(ebic_ctx* ctx) {
    if (ctx->PB) return EBIC_OK;
    if (ctx->cols > 46340) return EBIC_ERR_ARG;                  // cols^2 must fit int32
    const int64_t bytes = static_cast<int64_t>(ctx->cols) * ctx->cols * (ctx->ld / 8);
    if (bytes > (64ll << 30)) return EBIC_ERR_ARG;               // bit-column offsets are uint32 in 16-byte units
    const int64_t blocks = (ctx->ld / kPairTileRows) * ((ctx->cols + 15) / 16);
    if (blocks > 0x7fffffffll) return EBIC_ERR_ARG;
    const dim3 grid(static_cast<unsigned>(blocks));
    int st = dev_alloc(ctx, reinterpret_cast<void**>(&ctx->PB), bytes);
    if (st) return st;
    ctx->pb_bytes = bytes;
    // the tile-major copy for PAIRTILE, when a tile fits shared memory and the memory is there (never an error)
    if (ctx->pt_build && pairtile_fits(ctx)) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && bytes <= static_cast<int64_t>(free_b / 2) &&
            dev_alloc(ctx, reinterpret_cast<void**>(&ctx->PBT), bytes) == EBIC_OK)
            ctx->pbt_bytes = bytes;
        cudaGetLastError();
    }
    BuildTimer timer(&ctx->create_ms[2]);                        // the kernel, not the allocation
    EBIC_TRY(cudaFuncSetAttribute(pairbits_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * kPairStageBytes));
    pairbits_kernel<<<grid, 256, 2 * kPairStageBytes>>>(ctx->Mc, ctx->nanmask, ctx->ld, ctx->cols, ctx->PB, ctx->PBT);
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
    if (ctx->PBT) {
        cudaFree(ctx->PBT);
        ctx->bytes_owned -= ctx->pbt_bytes;
        ctx->PBT = nullptr;
        ctx->pbt_bytes = 0;
    }
}

}  // namespace ebic_host

namespace {

template <class E, int NCONS, class IW>
int launch_tiled(ebic_ctx* ctx, const void* M, int32_t T, int32_t k0, int32_t n_ind, const int32_t* col_ids,
                 unsigned long long* counts, cudaStream_t stream, bool pdl) {
    TiledParams p;
    p.M = M;
    p.ld = ctx->ld;
    p.cols = ctx->cols;
    p.T = T;
    p.nbuf = sizeof(typename E::type) == 4 ? tile_bufs_f32(ctx, n_ind) : 2;
    p.n_tiles = (ctx->ld + T - 1) / T;
    p.meta = ctx->meta + k0;
    p.idrec = ctx->idrec + static_cast<int64_t>(32 / IW::kPerWord) * k0;
    p.col_ids = col_ids;
    p.n_ind = n_ind;
    p.early_exit = ctx->early_exit;
    p.counts = counts + k0;
    p.visits = ctx->count_visits ? ctx->d_visits : nullptr;
    const size_t smem = tiled_smem_bytes(ctx->cols, T, sizeof(typename E::type), n_ind, p.nbuf);
    auto kern = fitness_tiled_kernel<E, NCONS, IW>;
    EBIC_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    const int64_t P = p.n_tiles * n_ind;
    // at least one individual per consumer warp and CTA, never more CTAs than SMs (1 CTA / SM)
    const int64_t grid = std::min<int64_t>(ctx->sm_count, std::max<int64_t>(1, P / NCONS));
    ctx->last_grid = static_cast<int32_t>(grid);
    ctx->last_T = T;
    ctx->launches++;
    return ebic_host::cuda_status(launch_pdl(kern, dim3(static_cast<unsigned>(grid)), dim3((NCONS + 1) * 32), smem, stream, pdl, p));
}

// Words of a bit column per PAIRBITS warp task: about `tasks_per_slot` tasks per resident warp slot (32 / SM),
// 256..2048 words (8,192..65,536 rows) per task.
int64_t pairbits_chunk_words(const ebic_ctx* ctx, int32_t n_ind) {
    const int64_t want_tasks = static_cast<int64_t>(ctx->pb_tasks_per_slot) * ctx->sm_count * 32;
    const int64_t cw = (ctx->ld / 32) * n_ind / want_tasks;
    int64_t words = std::max<int64_t>(kPairbitsStepWords, std::min<int64_t>(8 * kPairbitsStepWords, cw / kPairbitsStepWords * kPairbitsStepWords));
    // the row chunk is the grid's y axis (<= 65,535): a tiny population on a very long matrix gets longer chunks
    const int64_t ldw = ctx->ld / 32;
    const int64_t min_words = ((ldw + 65534) / 65535 + kPairbitsStepWords - 1) / kPairbitsStepWords * kPairbitsStepWords;
    return std::max(words, min_words);
}
// The L2 prefetches request EVERY bit column once; that pays only when the population uses most of the cols^2
// columns (n_ids - n_ind = number of pair uses).  A sparse population (wide matrix: P3 uses 14 % of 96,100
// columns) gathers straight from HBM instead -- measured 87 % of the HBM peak.
bool pairbits_dense(const ebic_ctx* ctx, int32_t n_ind, int64_t n_ids) {
    return n_ids - n_ind >= 2ll * ctx->cols * ctx->cols;
}

PairbitsParams pairbits_params(ebic_ctx* ctx, const int32_t* col_ids, int32_t n_ind, int64_t n_ids, unsigned long long* counts);

// Shared-prefix variant: plan (sort + groups) and the grouped evaluation.
int launch_prefix(ebic_ctx* ctx, const int32_t* col_ids, int32_t n_ind, int64_t n_ids, unsigned long long* counts,
                  cudaStream_t stream, bool pdl) {
    PrefixParams pp;
    pp.pb = pairbits_params(ctx, col_ids, n_ind, n_ids, counts);
    pp.pb.prefetch_dist = 0;                                 // groups walk the table in sorted-pair order, not all of it
    pp.groups = ctx->ubatch;
    pp.n_groups = ctx->ubatch + 8ll * n_ind;
    int32_t n_pow2 = 1;
    while (n_pow2 < n_ind) n_pow2 <<= 1;
    const size_t plan_smem = 13ull * n_pow2;
    EBIC_TRY(cudaFuncSetAttribute(prefix_plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan_smem)));
    ctx->launches += 2;
    EBIC_TRY(launch_pdl(prefix_plan_kernel, dim3(1), dim3(1024), plan_smem, stream, pdl, pp, n_pow2));
    const int64_t tasks = static_cast<int64_t>(pp.pb.n_chunks) * n_ind;          // worst case: every individual alone
    const int64_t grid = (tasks + kPairbitsWarps - 1) / kPairbitsWarps;
    if (grid > 0x7fffffffll) return EBIC_ERR_ARG;
    ctx->last_grid = static_cast<int32_t>(grid);
    ctx->last_T = pp.pb.chunk_words * 32;
    const dim3 g(static_cast<unsigned>(grid)), b(kPairbitsWarps * 32);
    return ebic_host::cuda_status(ctx->early_exit ? launch_pdl(fitness_prefix_kernel<true>, g, b, 0, stream, pdl, pp)
                                                  : launch_pdl(fitness_prefix_kernel<false>, g, b, 0, stream, pdl, pp));
}

PairbitsParams pairbits_params(ebic_ctx* ctx, const int32_t* col_ids, int32_t n_ind, int64_t n_ids, unsigned long long* counts) {
    PairbitsParams p;
    p.PB = ctx->PB;
    p.ldw = ctx->ld / 32;
    const int64_t cw = pairbits_chunk_words(ctx, n_ind);
    p.chunk_words = static_cast<int32_t>(cw);
    p.n_chunks = static_cast<int32_t>((p.ldw + cw - 1) / cw);
    p.prec = ctx->prec;
    p.meta = ctx->meta;
    p.col_ids = col_ids;
    p.cols = ctx->cols;
    p.pair_stride16 = static_cast<uint32_t>(ctx->ld / 128);
    p.n_ind = n_ind;
    p.counts = counts;
    p.visits = ctx->count_visits ? ctx->d_visits : nullptr;
    p.n_pairs = ctx->cols * ctx->cols;
    p.cols_per_task = (p.n_pairs + n_ind - 1) / std::max(n_ind, 1);
    p.prefetch_dist = pairbits_dense(ctx, n_ind, n_ids) ? ctx->pb_prefetch_dist : 0;
    p.prologue_chunks = std::max(p.prefetch_dist, p.prefetch_dist > 0 ? ctx->pb_prologue_chunks : 0);
    return p;
}

int launch_pairbits(ebic_ctx* ctx, const int32_t* col_ids, int32_t n_ind, int64_t n_ids, unsigned long long* counts,
                    cudaStream_t stream, bool pdl) {
    const PairbitsParams p = pairbits_params(ctx, col_ids, n_ind, n_ids, counts);
    const int64_t cw = p.chunk_words;
    const int64_t gx = (n_ind + kPairbitsWarps - 1) / kPairbitsWarps;
    if (p.n_chunks > 65535) return EBIC_ERR_ARG;                 // cannot happen: chunks grow to 65,536 rows (2^31 rows: 32,768)
    ctx->last_grid = static_cast<int32_t>(std::min<int64_t>(gx * p.n_chunks, 0x7fffffff));
    ctx->last_T = static_cast<int32_t>(cw * 32);
    const dim3 g(static_cast<unsigned>(gx), static_cast<unsigned>(p.n_chunks)), b(kPairbitsWarps * 32);
    cudaError_t e;
    if (ctx->pb_smem_ring) {
        const size_t smem = kPairbitsWarps * 4096;
        e = ctx->early_exit ? launch_pdl(fitness_pairbits_kernel<true, true>, g, b, smem, stream, pdl, p)
                            : launch_pdl(fitness_pairbits_kernel<false, true>, g, b, smem, stream, pdl, p);
    } else {
        e = ctx->early_exit ? launch_pdl(fitness_pairbits_kernel<true, false>, g, b, 0, stream, pdl, p)
                            : launch_pdl(fitness_pairbits_kernel<false, false>, g, b, 0, stream, pdl, p);
    }
    ctx->launches++;
    return ebic_host::cuda_status(e);
}

// PAIRTILE: plan (sort by length, transposed pair-slot records) + the persistent tile kernel, per population chunk.
int launch_pairtile(ebic_ctx* ctx, const int32_t* col_ids, int32_t k0, int32_t n_ind, unsigned long long* counts,
                    cudaStream_t stream, bool pdl_plan, bool pdl_fit, bool with_events, int slot) {
    PairtileParams p;
    p.PBT = ctx->PBT;
    p.n_tiles = ctx->ld / kPairTileRows;
    p.n_pairs = ctx->cols * ctx->cols;
    p.cols = ctx->cols;
    p.n_ind = n_ind;
    p.n_groups = (n_ind + 31) / 32;
    p.rec_cache = pairtile_rec_cache(ctx, n_ind) ? 1 : 0;
    p.meta = ctx->meta + k0;
    p.col_ids = col_ids;
    p.gmeta = static_cast<int2*>(ctx->tplan);
    p.tids = reinterpret_cast<uint4*>(static_cast<unsigned char*>(ctx->tplan) + 256ll * ((kMaxIndPerLaunch + 31) / 32));
    p.counts = counts + k0;
    p.visits = ctx->count_visits ? ctx->d_visits : nullptr;
    ctx->launches += 2;
    EBIC_TRY(launch_pdl(pairtile_plan_kernel, dim3((n_ind + kPtPlanThreads - 1) / kPtPlanThreads), dim3(kPtPlanThreads), 0,
                        stream, pdl_plan, p));
    if (with_events) EBIC_TRY(cudaEventRecord(ctx->ev_begin[slot], stream));
    const size_t smem = static_cast<size_t>(pairtile_smem(ctx, n_ind)) + (p.rec_cache ? 512ull * p.n_groups : 0);
    EBIC_TRY(cudaFuncSetAttribute(fitness_pairtile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    const int64_t items = p.n_tiles * p.n_groups;
    const int64_t grid = std::min<int64_t>(ctx->sm_count, items);
    ctx->last_grid = static_cast<int32_t>(grid);
    ctx->last_T = kPairTileRows;
    return ebic_host::cuda_status(launch_pdl(fitness_pairtile_kernel, dim3(static_cast<unsigned>(grid)), dim3(kPtWarps * 32), smem,
                                             stream, pdl_fit, p));
}

// Population already on the device: ingest + chain kernels.
int eval_device(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                unsigned long long* counts, cudaStream_t stream) {
    const int32_t kernel0 = ebic_host::resolve_kernel(ctx, n_ind, n_ids);
    ctx->last_n_ind = n_ind;
    ctx->last_n_ids = n_ids;
    if (!ebic_host::kernel_applies(ctx, kernel0)) return EBIC_ERR_ARG;
    const bool tiled = kernel0 == EBIC_KERNEL_RANK8 || kernel0 == EBIC_KERNEL_TILED_F32;
    if (kernel0 == EBIC_KERNEL_RANK8 && !ctx->Rk) {
        int st = ebic_host::build_rank_tiles(ctx);       // first use after ebic_set_pairbits(0): synchronous, once
        if (st) return st;
    }
    int st = grow(ctx, reinterpret_cast<void**>(&ctx->meta), &ctx->meta_cap, static_cast<int64_t>(n_ind) * 8);
    if (st) return st;
    const bool by_union = kernel0 == EBIC_KERNEL_UNION_F32;
    UnionParams up;
    if (tiled || by_union) {
        st = grow(ctx, reinterpret_cast<void**>(&ctx->idrec), &ctx->idrec_cap, (ctx->cols > 256 && tiled ? 64ll : 32ll) * n_ind);
        if (st) return st;
    }
    if (by_union) {
        up.batch = union_batch(ctx, n_ind, n_ids);
        up.n_batches = (n_ind + up.batch - 1) / up.batch;
        up.u_cap = union_cap(ctx);
        st = grow(ctx, reinterpret_cast<void**>(&ctx->ubatch), &ctx->ubatch_cap, 4ll * up.n_batches * (up.u_cap + 1));
        if (st) return st;
    }
    const bool by_tile = kernel0 == EBIC_KERNEL_PAIRTILE;
    if (by_tile) {                                          // gmeta (8 B) + four uint4 of pair slots (64 B) per sorted position
        st = grow(ctx, &ctx->tplan, &ctx->tplan_cap, (256ll + 2048ll) * ((kMaxIndPerLaunch + 31) / 32));
        if (st) return st;
    }
    const bool by_prefix = kernel0 == EBIC_KERNEL_PREFIX && n_ind <= kPrefixMaxInd;     // larger populations: plain PAIRBITS
    const bool by_pairs = kernel0 == EBIC_KERNEL_PAIRBITS || kernel0 == EBIC_KERNEL_PREFIX;
    if (by_pairs) {
        st = grow(ctx, reinterpret_cast<void**>(&ctx->prec), &ctx->prec_cap, 128ll * n_ind);
        if (st) return st;
    }
    if (by_prefix) {
        st = grow(ctx, reinterpret_cast<void**>(&ctx->ubatch), &ctx->ubatch_cap, 4ll * (8ll * n_ind + 4));
        if (st) return st;
    }

    IngestParams ip;
    ip.offsets = offsets;
    ip.col_ids = col_ids;
    ip.n_ind = n_ind;
    ip.n_ids = n_ids;
    ip.cols = ctx->cols;
    ip.rows = ctx->rows;
    ip.missing_on = ctx->missing_mode == EBIC_MISSING_ON;
    ip.sort_by_length = ctx->pb_sort;
    ip.nonmissing = ctx->nonmissing;
    ip.meta = ctx->meta;
    ip.idrec = tiled ? ctx->idrec : nullptr;
    ip.id_wide = ctx->cols > 256;
    ip.prec = by_pairs ? ctx->prec : nullptr;
    ip.pair_stride16 = static_cast<uint32_t>(ctx->ld / 128);
    ip.counts = counts;
    ip.err = ctx->d_err;
    if (by_pairs && !by_prefix && ctx->pb_ingest_prefetch > 0 && !pairbits_dense(ctx, n_ind, n_ids)) {
        ip.PB = ctx->PB;
        ip.prefetch_bytes = static_cast<uint32_t>(std::min<int64_t>(ctx->ld / 8, ctx->pb_ingest_prefetch)) & ~15u;
    }
    ingest_population_kernel<<<(n_ind + kIngestBlock - 1) / kIngestBlock, kIngestThreads, 0, stream>>>(ip);
    ctx->launches++;
    EBIC_TRY(cudaGetLastError());

    if (by_union) {                                         // a3, second half: the batches' column unions and local ids
        up.Mc = ctx->Mc;
        up.ld = ctx->ld;
        up.cols = ctx->cols;
        up.n_ind = n_ind;
        up.meta = ctx->meta;
        up.col_ids = col_ids;
        up.ucount = ctx->ubatch;
        up.ucols = ctx->ubatch + up.n_batches;
        up.urec = ctx->idrec;
        up.early_exit = ctx->early_exit;
        up.counts = counts;
        up.visits = ctx->count_visits ? ctx->d_visits : nullptr;
        const size_t plan_smem = 8ull * ((ctx->cols + 31) / 32);
        ctx->launches++;
        EBIC_TRY(launch_pdl(union_plan_kernel, dim3(static_cast<unsigned>(up.n_batches)), dim3(256), plan_smem, stream,
                            ctx->pdl != 0, up));
    }

    // With kernel timing on, an event sits between the ingest and the fitness kernel, so the two cannot overlap:
    // the timed kernel then includes its whole prologue (a conservative figure).
    bool pdl = ctx->pdl && !ctx->time_kernels;
    const int slot = static_cast<int>(ctx->timed_evals % ebic_ctx::kTimingRing);
    if (ctx->time_kernels) {
        if (!ctx->ev_begin[slot]) {
            EBIC_TRY(cudaEventCreate(&ctx->ev_begin[slot]));
            EBIC_TRY(cudaEventCreate(&ctx->ev_end[slot]));
        }
        if (!by_tile) EBIC_TRY(cudaEventRecord(ctx->ev_begin[slot], stream));   // PAIRTILE: behind its plan kernel (a3)
    }
    ctx->last_kernel = kernel0;
    if (by_tile) {
        const int32_t per_launch = pairtile_chunk(ctx, n_ind);
        for (int32_t k0 = 0; k0 < n_ind; k0 += per_launch) {
            const int32_t n = std::min<int32_t>(per_launch, n_ind - k0);
            // only the first chunk follows the ingest directly; later chunks reuse the plan buffers, so they are
            // ordered behind the previous chunk's kernel
            st = launch_pairtile(ctx, col_ids, k0, n, counts, stream, ctx->pdl && k0 == 0, pdl && k0 == 0,
                                 ctx->time_kernels && k0 == 0, slot);
            if (st) return st;
        }
    } else if (by_prefix) {
        st = launch_prefix(ctx, col_ids, n_ind, n_ids, counts, stream, pdl);
        if (st) return st;
    } else if (by_pairs) {
        ctx->last_kernel = EBIC_KERNEL_PAIRBITS;
        st = launch_pairbits(ctx, col_ids, n_ind, n_ids, counts, stream, pdl);   // any population size in one launch
        if (st) return st;
    } else if (tiled) {
        const int32_t per_launch = tiled_chunk(ctx, kernel0, n_ind);
        for (int32_t k0 = 0; k0 < n_ind; k0 += per_launch) {
            const int32_t n = std::min<int32_t>(per_launch, n_ind - k0);
            const int32_t T = tile_rows(ctx, kernel0, n);
            if (T <= 0) return EBIC_ERR_ARG;
            if (kernel0 == EBIC_KERNEL_RANK8)
                st = launch_tiled<ElemR8, kConsR8, IdWords>(ctx, ctx->Rk, T, k0, n, col_ids, counts, stream, pdl);
            else if (ctx->cols <= 256)
                st = launch_tiled<ElemF32, kConsF32, IdWords>(ctx, ctx->Mc, T, k0, n, col_ids, counts, stream, pdl);
            else
                st = launch_tiled<ElemF32, kConsF32, IdWords16>(ctx, ctx->Mc, T, k0, n, col_ids, counts, stream, pdl);
            if (st) return st;
            pdl = false;                                  // only the first launch directly follows the ingest
        }
    } else if (by_union) {
        const size_t smem = union_smem_bytes(up.u_cap, up.batch);
        auto kern = fitness_union_kernel<kUnionCons>;
        EBIC_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
        const int64_t P = (ctx->ld / kUnionTileRows) * up.n_batches;
        const int64_t grid = std::min<int64_t>(ctx->sm_count, P);
        ctx->last_grid = static_cast<int32_t>(grid);
        ctx->last_T = kUnionTileRows;
        ctx->launches++;
        EBIC_TRY(launch_pdl(kern, dim3(static_cast<unsigned>(grid)), dim3((kUnionCons + kUnionProd) * 32), smem, stream, pdl, up));
    } else {
        const int64_t gx = ctx->ld / 256;
        int64_t gy = std::max<int64_t>(1, (8ll * ctx->sm_count + gx - 1) / gx);
        gy = std::min<int64_t>(std::min<int64_t>(gy, n_ind), 65535);
        const dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(gy));
        ctx->launches++;
        ctx->last_grid = static_cast<int32_t>(std::min<int64_t>(gx * gy, 0x7fffffff));
        ctx->last_T = 256;
        EBIC_TRY(launch_pdl(fitness_direct_kernel, grid, dim3(256), 0, stream, pdl, ctx->Mc, ctx->ld, ctx->meta, col_ids,
                            n_ind, counts));
    }
    if (ctx->time_kernels) {
        EBIC_TRY(cudaEventRecord(ctx->ev_end[slot], stream));
        ctx->timed_evals++;
    }
    return EBIC_OK;
}

// `overlap`: the launch directly follows this library's own fitness kernel on `stream` and shares no buffer with
// it (ebic_eval_extract), so the two may run side by side; `counts` has been zeroed by the caller in that case.
int extract_device(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                   const int32_t* chosen, int32_t n_chosen, uint64_t* masks, uint64_t* counts,
                   cudaStream_t stream, bool overlap) {
    const int64_t words32 = 2 * ((ctx->rows + 63) / 64);
    if (counts && !overlap) EBIC_TRY(cudaMemsetAsync(counts, 0, static_cast<size_t>(n_chosen) * 8, stream));
    const int32_t ov = overlap ? 1 : 0;
    const bool pdl = ctx->pdl != 0;
    ctx->launches++;
    if (ctx->PB && ctx->extract_pairbits) {
        // about 16 CTAs per SM in total: a CTA's prologue (chosen -> offsets -> ids) is paid once for several blocks
        const int64_t n_wblocks = (words32 + 1023) / 1024;
        const int64_t gx = std::max<int64_t>(1, std::min<int64_t>(n_wblocks, (16ll * ctx->sm_count + n_chosen - 1) / n_chosen));
        const dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(std::min<int32_t>(n_chosen, 65535)));
        return ebic_host::cuda_status(launch_pdl(
            extract_rows_pairbits_kernel, grid, dim3(256), 0, stream, pdl, ctx->PB, ctx->ld, ctx->rows, ctx->cols,
            ctx->missing_mode == EBIC_MISSING_ON, ctx->nanmask, offsets, col_ids, n_ind, n_ids, chosen, n_chosen,
            reinterpret_cast<uint32_t*>(masks), words32, reinterpret_cast<unsigned long long*>(counts), ctx->d_err, ov));
    }
    const int64_t gx = (words32 * 32 + kExtractRowsPerBlock - 1) / kExtractRowsPerBlock;
    const dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(std::min<int32_t>(n_chosen, 65535)));
    return ebic_host::cuda_status(launch_pdl(
        extract_rows_kernel, grid, dim3(256), 0, stream, pdl, ctx->Mc, ctx->ld, ctx->rows, ctx->cols,
        ctx->missing_mode == EBIC_MISSING_ON, ctx->nanmask, offsets, col_ids, n_ind, n_ids, chosen, n_chosen,
        reinterpret_cast<uint32_t*>(masks), words32, reinterpret_cast<unsigned long long*>(counts), ctx->d_err, ov));
}

int stage_in(ebic_ctx* ctx, int slot, const void* host, int64_t bytes, cudaStream_t stream, void** dev) {
    int st = grow(ctx, &ctx->stage[slot], &ctx->stage_cap[slot], bytes);
    if (st) return st;
    *dev = ctx->stage[slot];
    if (bytes > 0) EBIC_TRY(cudaMemcpyAsync(*dev, host, static_cast<size_t>(bytes), cudaMemcpyHostToDevice, stream));
    return EBIC_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// ebic_eval_fitness_noalloc (include/ebic.h): the count of every individual, for hosts that may not allocate device
// memory after set-up.  The ingest kernel's products -- meta[k] (8 bytes) and, with the pair table, the 128-byte
// record prec[j] of every individual -- go into a fixed array that is part of the library image instead of the
// context's grown buffers.  Layout: [0, 8 * MAX) meta, [8 * MAX, 136 * MAX) prec; MAX = EBIC_NOALLOC_MAX_IND.
//
// `noalloc_scratch` below is a __device__ variable.  In HOST code that name is only the handle the runtime
// registered for it; it is not an address the GPU can use.  The device address differs per GPU and is asked for
// once per GPU with cudaGetSymbolAddress while that GPU is current (noalloc_scratch_for), and only that pointer is
// ever handed to a kernel.
// ------------------------------------------------------------------------------------------------
constexpr int64_t kNoAllocMetaBytes = 8ll * EBIC_NOALLOC_MAX_IND;
constexpr int64_t kNoAllocPrecBytes = 128ll * EBIC_NOALLOC_MAX_IND;
constexpr int kNoAllocMaxDevices = 64;

static __device__ __align__(256) unsigned char noalloc_scratch[kNoAllocMetaBytes + kNoAllocPrecBytes];

namespace {

std::mutex noalloc_mutex;
unsigned char* noalloc_addr[kNoAllocMaxDevices] = {};     // device address of noalloc_scratch on GPU i, nullptr = not asked yet

// Device address of the array on `device`, which must be the current device.  The first call per GPU asks the runtime.
int noalloc_scratch_for(int device, unsigned char** out) {
    if (device < 0 || device >= kNoAllocMaxDevices) return EBIC_ERR_ARG;
    std::lock_guard<std::mutex> lock(noalloc_mutex);
    if (!noalloc_addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return EBIC_ERR_CUDA;
        }
        noalloc_addr[device] = static_cast<unsigned char*>(p);
    }
    *out = noalloc_addr[device];
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
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // begin, transposed, masks, rank tiles, pair table
    do {
        if ((st = ebic_host::cuda_status(cudaGetDevice(&ctx->device)))) break;
        if ((st = ebic_host::cuda_status(cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device)))) break;
        if ((st = ebic_host::cuda_status(cudaDeviceGetAttribute(&ctx->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device)))) break;
        for (auto& e : ev)
            if ((st = ebic_host::cuda_status(cudaEventCreate(&e)))) break;
        if (st) break;
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
        if ((st = ebic_host::cuda_status(cudaMemset(ctx->d_err, 0, 32)))) break;
        if ((st = ebic_host::cuda_status(cudaMemset(ctx->nonmissing, 0, static_cast<size_t>(cols) * 8)))) break;
        cudaEventRecord(ev[0]);

        // a1: transpose (device input: in one go; host input: through a bounded staging buffer)
        const dim3 tb(32, 8);
        const unsigned gy = static_cast<unsigned>(std::min<int64_t>((cols + 31) / 32, 65535));
        if (is_device_pointer(matrix)) {
            const dim3 grid(static_cast<unsigned>((rows + 31) / 32), gy);
            transpose_pad_kernel<<<grid, tb>>>(matrix, ctx->Mc, 0, rows, cols, ctx->ld, use_sentinel, sentinel);
            ctx->launches++;
            if ((st = ebic_host::cuda_status(cudaGetLastError()))) break;
        } else {
            const int64_t chunk_rows = std::max<int64_t>(32, std::min<int64_t>(rows, (256ll << 20) / (4ll * cols) / 32 * 32));
            if ((st = ebic_host::cuda_status(cudaMalloc(reinterpret_cast<void**>(&staging), static_cast<size_t>(chunk_rows) * cols * 4)))) break;
            for (int64_t r0 = 0; r0 < rows && st == EBIC_OK; r0 += chunk_rows) {
                const int64_t nr = std::min<int64_t>(chunk_rows, rows - r0);
                if ((st = ebic_host::cuda_status(cudaMemcpy(staging, matrix + r0 * cols, static_cast<size_t>(nr) * cols * 4, cudaMemcpyHostToDevice)))) break;
                const dim3 grid(static_cast<unsigned>((nr + 31) / 32), gy);
                transpose_pad_kernel<<<grid, tb>>>(staging, ctx->Mc, r0, nr, cols, ctx->ld, use_sentinel, sentinel);
                ctx->launches++;
                st = ebic_host::cuda_status(cudaGetLastError());
            }
            if (st) break;
        }
        if (ctx->ld > rows) {
            const int64_t npad = (ctx->ld - rows) * cols;
            fill_pad_kernel<<<static_cast<unsigned>(std::min<int64_t>((npad + 255) / 256, 4096)), 256>>>(ctx->Mc, rows, cols, ctx->ld);
            ctx->launches++;
            if ((st = ebic_host::cuda_status(cudaGetLastError()))) break;
        }
        cudaEventRecord(ev[1]);
        // a2: NaN bitmask + per-column non-missing counts
        {
            const int64_t words = ctx->ld / 32;
            const dim3 grid(static_cast<unsigned>((words + 255) / 256), static_cast<unsigned>(std::min<int32_t>(cols, 65535)));
            nan_mask_kernel<<<grid, 256>>>(ctx->Mc, ctx->ld, cols, ctx->nanmask, ctx->nonmissing);
            ctx->launches++;
            if ((st = ebic_host::cuda_status(cudaGetLastError()))) break;
        }
        cudaEventRecord(ev[2]);
        if ((st = ebic_host::cuda_status(cudaDeviceSynchronize()))) break;
        // a2": pair-relation bitmasks, when they fit comfortably
        if (cols <= 46340) {
            const int64_t pb = static_cast<int64_t>(cols) * cols * (ctx->ld / 8);
            size_t free_b = 0, total_b = 0;
            if ((st = ebic_host::cuda_status(cudaMemGetInfo(&free_b, &total_b)))) break;
            if (pb <= kPairbitsAutoMaxBytes && pb <= static_cast<int64_t>(free_b / 2)) {
                st = ebic_host::build_pairbits(ctx);
                if (st == EBIC_ERR_OOM) {
                    ebic_host::free_pairbits(ctx);
                    st = EBIC_OK;
                }
                if (st) break;
            }
        }
        cudaEventRecord(ev[3]);
        // a2': rank tiles only when AUTO will run RANK8, i.e. when there is no pair table (ebic_set_kernel / a later
        // ebic_set_pairbits(0) build them on demand)
        if (!ctx->PB && cols <= kMaxColsRank8)
            if ((st = ebic_host::build_rank_tiles(ctx))) break;
        cudaEventRecord(ev[4]);
        if ((st = ebic_host::cuda_status(cudaDeviceSynchronize()))) break;
        cudaEventElapsedTime(&ctx->create_ms[0], ev[0], ev[1]);      // [2] pair table, [3] rank tiles: by their builders
        cudaEventElapsedTime(&ctx->create_ms[1], ev[1], ev[2]);
        cudaEventElapsedTime(&ctx->create_ms[4], ev[0], ev[4]);
        cudaGetLastError();
    } while (0);
    for (auto e : ev)
        if (e) cudaEventDestroy(e);
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
    cudaFree(ctx->PBT);
    cudaFree(ctx->tplan);
    cudaFree(ctx->prec);
    cudaFree(ctx->d_err);
    cudaFree(ctx->meta);
    cudaFree(ctx->idrec);
    cudaFree(ctx->ubatch);
    for (void* s : ctx->stage) cudaFree(s);
    if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_masks_ready) cudaEventDestroy(ctx->ev_masks_ready);
    if (ctx->ev_masks_copied) cudaEventDestroy(ctx->ev_masks_copied);
    for (int i = 0; i < ebic_ctx::kTimingRing; ++i) {
        if (ctx->ev_begin[i]) cudaEventDestroy(ctx->ev_begin[i]);
        if (ctx->ev_end[i]) cudaEventDestroy(ctx->ev_end[i]);
    }
    cudaGetLastError();
    delete ctx;
    return EBIC_OK;
}

// Shared by the three hot calls.  chosen == NULL: counts only; counts == NULL: masks only.
static int eval_extract_impl(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                             uint64_t* counts, const int32_t* chosen, int32_t n_chosen, uint64_t* masks,
                             uint64_t* mask_counts, void* cuda_stream, bool do_eval, bool do_extract) {
    if (!on_ctx_device(ctx)) return EBIC_ERR_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const bool pop_dev = is_device_pointer(offsets);
    const bool out_dev = is_device_pointer(do_eval ? static_cast<const void*>(counts) : static_cast<const void*>(masks));
    const int64_t words = (ctx->rows + 63) / 64;
    const int32_t* d_off = offsets;
    const int32_t* d_ids = col_ids;
    const int32_t* d_chosen = chosen;
    unsigned long long* d_counts = reinterpret_cast<unsigned long long*>(counts);
    uint64_t* d_masks = masks;
    uint64_t* d_mcnt = mask_counts;
    int st;
    void* p;
    if (!pop_dev) {
        if ((st = stage_in(ctx, 0, offsets, (static_cast<int64_t>(n_ind) + 1) * 4, stream, &p))) return st;
        d_off = static_cast<const int32_t*>(p);
        if ((st = stage_in(ctx, 1, col_ids, n_ids * 4, stream, &p))) return st;
        d_ids = static_cast<const int32_t*>(p);
        if (do_extract) {
            if ((st = stage_in(ctx, 3, chosen, static_cast<int64_t>(n_chosen) * 4, stream, &p))) return st;
            d_chosen = static_cast<const int32_t*>(p);
        }
    }
    if (!out_dev) {
        if (do_eval) {
            if ((st = grow(ctx, &ctx->stage[2], &ctx->stage_cap[2], static_cast<int64_t>(n_ind) * 8))) return st;
            d_counts = static_cast<unsigned long long*>(ctx->stage[2]);
        }
        if (do_extract) {
            if ((st = grow(ctx, &ctx->stage[4], &ctx->stage_cap[4], static_cast<int64_t>(n_chosen) * words * 8))) return st;
            d_masks = static_cast<uint64_t*>(ctx->stage[4]);
            if (mask_counts) {
                if ((st = grow(ctx, &ctx->stage[5], &ctx->stage_cap[5], static_cast<int64_t>(n_chosen) * 8))) return st;
                d_mcnt = static_cast<uint64_t*>(ctx->stage[5]);
            }
        }
    }
    const bool fused = do_eval && do_extract;
    // A GA loop calls this with the SAME device buffers every generation (only their contents change), so the launch
    // sequence is captured into a CUDA graph the second time a call repeats the previous one's arguments and replayed
    // from the third on: one graph launch instead of three or four kernel launches and a memset (the launch overhead
    // is a third of the step on the paper's dataset shapes).  Any change of a knob, a pointer or a size
    // starts over; instrumented calls, host pointers, the legacy default stream and a stream that is already being
    // captured by the caller always take the plain path.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    const bool graphable = ctx->use_graphs && pop_dev && out_dev && stream != nullptr && stream != cudaStreamLegacy &&
                           stream != cudaStreamPerThread && !ctx->time_kernels && !ctx->count_visits &&
                           cudaStreamIsCapturing(stream, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusNone;
    bool capture = false;
    if (graphable) {
        ebic_ctx::GraphKey key = {};                          // zeroed, padding included: compared with memcmp
        key.offsets = offsets; key.col_ids = col_ids; key.counts = counts; key.chosen = chosen; key.masks = masks;
        key.mask_counts = mask_counts; key.stream = stream; key.n_ids = n_ids; key.n_ind = n_ind; key.n_chosen = n_chosen;
        key.epoch = ctx->epoch; key.flags = (do_eval ? 1 : 0) | (do_extract ? 2 : 0);
        if (ctx->graph_state != 0 && std::memcmp(&key, &ctx->graph_key, sizeof(key)) == 0) {
            if (ctx->graph_exec) {
                ctx->launches += ctx->graph_launches;
                return ebic_host::cuda_status(cudaGraphLaunch(ctx->graph_exec, stream));
            }
            capture = ctx->graph_state == 1;                  // second sighting; 2 = capture failed once: stay plain
        } else {
            if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
            ctx->graph_exec = nullptr;
            ctx->graph_key = key;
            ctx->graph_state = 1;
        }
    } else {
        cudaGetLastError();
    }
    const int64_t launches0 = ctx->launches;
    if (capture && cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        capture = false;
        ctx->graph_state = 2;
    }
    if (capture) {
        // the buffers were grown by the identical plain call before this one: nothing allocates during the capture
        st = EBIC_OK;
        if (fused && d_mcnt) st = ebic_host::cuda_status(cudaMemsetAsync(d_mcnt, 0, static_cast<size_t>(n_chosen) * 8, stream));
        if (!st && do_eval) st = eval_device(ctx, d_off, d_ids, n_ind, n_ids, d_counts, stream);
        if (!st && do_extract) st = extract_device(ctx, d_off, d_ids, n_ind, n_ids, d_chosen, n_chosen, d_masks, d_mcnt, stream, fused);
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(stream, &graph);
        if (!st && e == cudaSuccess && graph && cudaGraphInstantiate(&ctx->graph_exec, graph, 0) != cudaSuccess) ctx->graph_exec = nullptr;
        if (graph) cudaGraphDestroy(graph);
        if (!st && e == cudaSuccess && ctx->graph_exec) {
            ctx->graph_launches = ctx->launches - launches0;
            return ebic_host::cuda_status(cudaGraphLaunch(ctx->graph_exec, stream));
        }
        cudaGetLastError();                                   // the capture did not work out: plain launches, now and later
        if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
        ctx->graph_exec = nullptr;
        ctx->graph_state = 2;
        ctx->launches = launches0;
    }
    if (fused && d_mcnt) EBIC_TRY(cudaMemsetAsync(d_mcnt, 0, static_cast<size_t>(n_chosen) * 8, stream));   // ahead of the kernel chain
    // One generation with HOST outputs: the masks are the large result (rows / 8 bytes per chosen individual) and the
    // extraction does not depend on the fitness kernel, so it runs FIRST and its device-to-host copy proceeds on the
    // context's copy stream while the fitness kernel works.
    const bool masks_first = fused && !out_dev;
    if (masks_first) {
        if (!ctx->copy_stream) {
            EBIC_TRY(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
            EBIC_TRY(cudaEventCreateWithFlags(&ctx->ev_masks_ready, cudaEventDisableTiming));
            EBIC_TRY(cudaEventCreateWithFlags(&ctx->ev_masks_copied, cudaEventDisableTiming));
        }
        if ((st = extract_device(ctx, d_off, d_ids, n_ind, n_ids, d_chosen, n_chosen, d_masks, d_mcnt, stream, false))) return st;
        EBIC_TRY(cudaEventRecord(ctx->ev_masks_ready, stream));
        EBIC_TRY(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_masks_ready, 0));
        EBIC_TRY(cudaMemcpyAsync(masks, d_masks, static_cast<size_t>(n_chosen) * words * 8, cudaMemcpyDeviceToHost, ctx->copy_stream));
        cudaError_t e = cudaSuccess;
        if (mask_counts) e = cudaMemcpyAsync(mask_counts, d_mcnt, static_cast<size_t>(n_chosen) * 8, cudaMemcpyDeviceToHost, ctx->copy_stream);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_masks_copied, ctx->copy_stream);
        if (e != cudaSuccess) {                                 // the first copy is already queued: wait it out
            cudaStreamSynchronize(ctx->copy_stream);
            return ebic_host::cuda_status(e);
        }
    }
    // From here on a copy into the caller's `masks` may be in flight on the copy stream: an error return must not
    // hand the buffer back while it is still being written, so every exit below drains that stream first.
    auto leave = [&](int status) {
        if (status != EBIC_OK && masks_first) {
            cudaStreamSynchronize(ctx->copy_stream);
            cudaGetLastError();
        }
        return status;
    };
    if (do_eval && (st = eval_device(ctx, d_off, d_ids, n_ind, n_ids, d_counts, stream))) return leave(st);
    if (do_extract && !masks_first &&
        (st = extract_device(ctx, d_off, d_ids, n_ind, n_ids, d_chosen, n_chosen, d_masks, d_mcnt, stream, fused)))
        return st;
    auto ok = [&](cudaError_t e) { return (st = ebic_host::cuda_status(e)) == EBIC_OK; };
    if (!out_dev) {
        if (do_eval && !ok(cudaMemcpyAsync(counts, d_counts, static_cast<size_t>(n_ind) * 8, cudaMemcpyDeviceToHost, stream))) return leave(st);
        if (do_extract && !masks_first) {
            EBIC_TRY(cudaMemcpyAsync(masks, d_masks, static_cast<size_t>(n_chosen) * words * 8, cudaMemcpyDeviceToHost, stream));
            if (mask_counts) EBIC_TRY(cudaMemcpyAsync(mask_counts, d_mcnt, static_cast<size_t>(n_chosen) * 8, cudaMemcpyDeviceToHost, stream));
        }
        if (masks_first && !ok(cudaStreamWaitEvent(stream, ctx->ev_masks_copied, 0))) return leave(st);
        if (!ok(cudaStreamSynchronize(stream))) return leave(st);
    } else if (!pop_dev) {
        EBIC_TRY(cudaStreamSynchronize(stream));   // host population buffers may be reused on return
    }
    return EBIC_OK;
}

int ebic_eval_fitness(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                      uint64_t* counts, void* cuda_stream) {
    if (!ctx || n_ind < 0 || n_ids < 0 || n_ind == 2147483647) return EBIC_ERR_ARG;
    if (n_ind == 0) return EBIC_OK;
    if (!offsets || !counts || (!col_ids && n_ids > 0)) return EBIC_ERR_ARG;
    return eval_extract_impl(ctx, offsets, col_ids, n_ind, n_ids, counts, nullptr, 0, nullptr, nullptr, cuda_stream, true, false);
}

int ebic_extract_rows(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                      const int32_t* chosen, int32_t n_chosen, uint64_t* masks, uint64_t* counts,
                      void* cuda_stream) {
    if (!ctx || n_ind < 0 || n_ids < 0 || n_chosen < 0) return EBIC_ERR_ARG;
    if (n_chosen == 0) return EBIC_OK;
    if (!offsets || !chosen || !masks || (!col_ids && n_ids > 0)) return EBIC_ERR_ARG;
    return eval_extract_impl(ctx, offsets, col_ids, n_ind, n_ids, nullptr, chosen, n_chosen, masks, counts, cuda_stream, false, true);
}

int ebic_eval_extract(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                      uint64_t* counts, const int32_t* chosen, int32_t n_chosen, uint64_t* masks,
                      uint64_t* mask_counts, void* cuda_stream) {
    if (!ctx || n_ind < 0 || n_ids < 0 || n_chosen < 0 || n_ind == 2147483647) return EBIC_ERR_ARG;
    if (n_ind == 0 && n_chosen == 0) return EBIC_OK;
    if (!offsets || (!col_ids && n_ids > 0) || (n_ind > 0 && !counts) || (n_chosen > 0 && (!chosen || !masks)))
        return EBIC_ERR_ARG;
    return eval_extract_impl(ctx, offsets, col_ids, n_ind, n_ids, counts, chosen, n_chosen, masks, mask_counts, cuda_stream,
                             n_ind > 0, n_chosen > 0);
}

int ebic_eval_fitness_noalloc(ebic_ctx* ctx, const int32_t* offsets, const int32_t* col_ids, int32_t n_ind, int64_t n_ids,
                              uint64_t* counts, void* cuda_stream) {
    if (!ctx || n_ind < 0 || n_ids < 0) return EBIC_ERR_ARG;
    if (n_ind > EBIC_NOALLOC_MAX_IND) return EBIC_ERR_LIMIT;         // the fixed array holds no more records than that
    if (n_ind == 0) return EBIC_OK;
    if (!offsets || !counts || (!col_ids && n_ids > 0)) return EBIC_ERR_ARG;
    if (!on_ctx_device(ctx)) return EBIC_ERR_ARG;
    // host buffers would have to be staged through device memory this call is not allowed to allocate
    if (!is_device_pointer(offsets) || !is_device_pointer(counts) || (n_ids > 0 && !is_device_pointer(col_ids))) return EBIC_ERR_ARG;
    unsigned char* scratch = nullptr;
    int st = noalloc_scratch_for(ctx->device, &scratch);
    if (st) return st;
    int2* meta = reinterpret_cast<int2*>(scratch);
    uint32_t* prec = reinterpret_cast<uint32_t*>(scratch + kNoAllocMetaBytes);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long* d_counts = reinterpret_cast<unsigned long long*>(counts);
    const bool by_pairs = ctx->PB != nullptr;

    // a3: validation + records, into the fixed array.  Every meta[k] and every record of 0 .. n_ind-1 is rewritten here,
    // so whatever the previous call left behind is never read; nothing has to be cleared.
    IngestParams ip;
    ip.offsets = offsets;
    ip.col_ids = col_ids;
    ip.n_ind = n_ind;
    ip.n_ids = n_ids;
    ip.cols = ctx->cols;
    ip.rows = ctx->rows;
    ip.missing_on = ctx->missing_mode == EBIC_MISSING_ON;
    ip.sort_by_length = ctx->pb_sort;
    ip.nonmissing = ctx->nonmissing;
    ip.meta = meta;
    ip.idrec = nullptr;
    ip.id_wide = 0;
    ip.prec = by_pairs ? prec : nullptr;
    ip.pair_stride16 = static_cast<uint32_t>(ctx->ld / 128);
    ip.counts = d_counts;
    ip.err = ctx->d_err;
    ingest_population_kernel<<<(n_ind + kIngestBlock - 1) / kIngestBlock, kIngestThreads, 0, stream>>>(ip);
    ctx->launches++;
    EBIC_TRY(cudaGetLastError());

    const bool pdl = ctx->pdl != 0;
    ctx->launches++;
    if (by_pairs) {
        PairbitsParams p = pairbits_params(ctx, col_ids, n_ind, n_ids, d_counts);
        p.prec = prec;                                               // the fixed array, not the context's buffers
        p.meta = meta;
        if (p.n_chunks > 65535) return EBIC_ERR_ARG;
        const dim3 g(static_cast<unsigned>((n_ind + kPairbitsWarps - 1) / kPairbitsWarps), static_cast<unsigned>(p.n_chunks));
        const dim3 b(kPairbitsWarps * 32);
        cudaError_t e;
        if (ctx->pb_smem_ring) {
            const size_t smem = kPairbitsWarps * 4096;
            e = ctx->early_exit ? launch_pdl(fitness_pairbits_kernel<true, true>, g, b, smem, stream, pdl, p)
                                : launch_pdl(fitness_pairbits_kernel<false, true>, g, b, smem, stream, pdl, p);
        } else {
            e = ctx->early_exit ? launch_pdl(fitness_pairbits_kernel<true, false>, g, b, 0, stream, pdl, p)
                                : launch_pdl(fitness_pairbits_kernel<false, false>, g, b, 0, stream, pdl, p);
        }
        return ebic_host::cuda_status(e);
    }
    const int64_t gx = ctx->ld / 256;
    int64_t gy = std::max<int64_t>(1, (8ll * ctx->sm_count + gx - 1) / gx);
    gy = std::min<int64_t>(std::min<int64_t>(gy, n_ind), 65535);
    const dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>(gy));
    return ebic_host::cuda_status(launch_pdl(fitness_direct_kernel, grid, dim3(256), 0, stream, pdl, ctx->Mc, ctx->ld,
                                             static_cast<const int2*>(meta), col_ids, n_ind, d_counts));
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

const char* ebic_strerror(int status) {
    switch (status) {
        case EBIC_OK: return "ok";
        case EBIC_ERR_ARG: return "invalid argument";
        case EBIC_ERR_OOM: return "out of device memory";
        case EBIC_ERR_CUDA: return "CUDA runtime error";
        case EBIC_ERR_BAD_COLUMN: return "column id outside [0, cols) in the population";
        case EBIC_ERR_BAD_OFFSETS: return "bad population offsets or chosen index";
        case EBIC_ERR_IO: return "cannot read the file as a delimited matrix";
        case EBIC_ERR_LIMIT: return "population larger than the fixed scratch of ebic_eval_fitness_noalloc (EBIC_NOALLOC_MAX_IND individuals)";
        default: return "unknown status";
    }
}

}  // extern "C"
