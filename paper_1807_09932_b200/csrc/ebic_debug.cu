// ebic_debug.cu -- the knobs, introspection, read-backs and measurement probes of include/ebic_debug.h.
// Same libebic.so as the boundary (ebic_api.cu); nothing here is a step of the path.
#include "../../include/ebic_debug.h"

#include <cuda_runtime.h>
#include <algorithm>

#include "ebic_ctx.hpp"
#include "probe_kernels.cuh"

using namespace ebic;
using ebic_host::cuda_status;

#define EBIC_TRY(expr)                         \
    do {                                       \
        int st__ = cuda_status((expr));        \
        if (st__ != EBIC_OK) return st__;      \
    } while (0)

extern "C" {

int ebic_set_kernel(ebic_ctx* ctx, int32_t kernel) {
    if (ctx) ctx->epoch++;
    if (!ctx || kernel < EBIC_KERNEL_AUTO || kernel > EBIC_KERNEL_PAIRTILE) return EBIC_ERR_ARG;
    if (!ebic_host::kernel_applies(ctx, kernel)) return EBIC_ERR_ARG;
    if (kernel == EBIC_KERNEL_RANK8) {
        if (cudaDeviceSynchronize() != cudaSuccess) return cuda_status(cudaGetLastError());
        int st = ebic_host::build_rank_tiles(ctx);
        if (st) return st;
    }
    ctx->kernel_request = kernel;
    return EBIC_OK;
}

int ebic_set_pairbits(ebic_ctx* ctx, int32_t on) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->epoch++;
    if (cudaDeviceSynchronize() != cudaSuccess) return cuda_status(cudaGetLastError());
    if (on == 0) {
        ebic_host::free_pairbits(ctx);
        if (ctx->kernel_request == EBIC_KERNEL_PAIRBITS || ctx->kernel_request == EBIC_KERNEL_PREFIX ||
            ctx->kernel_request == EBIC_KERNEL_PAIRTILE)
            ctx->kernel_request = EBIC_KERNEL_AUTO;
        if (ctx->cols <= 127) return ebic_host::build_rank_tiles(ctx);
        return EBIC_OK;
    }
    int st = ebic_host::build_pairbits(ctx);
    if (st) ebic_host::free_pairbits(ctx);
    return st;
}

int ebic_set_extract_source(ebic_ctx* ctx, int32_t use_pairbits) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->extract_pairbits = use_pairbits ? 1 : 0;
    ctx->epoch++;
    return EBIC_OK;
}

int ebic_set_early_exit(ebic_ctx* ctx, int32_t on) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->early_exit = on ? 1 : 0;
    ctx->epoch++;
    return EBIC_OK;
}

int ebic_set_tuning(ebic_ctx* ctx, int32_t knob, int32_t value) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->epoch++;
    switch (knob) {
        case 0:
            if (value < 1 || value > 64) return EBIC_ERR_ARG;
            ctx->pb_tasks_per_slot = value;
            return EBIC_OK;
        case 1:
            if (value < 0 || value > 8) return EBIC_ERR_ARG;
            ctx->pb_prefetch_dist = value;
            return EBIC_OK;
        case 2: ctx->pb_smem_ring = value ? 1 : 0; return EBIC_OK;
        case 3: ctx->pb_sort = value ? 1 : 0; return EBIC_OK;
        case 4: ctx->pdl = value ? 1 : 0; return EBIC_OK;
        case 5:
            if (value < 0 || value > 256) return EBIC_ERR_ARG;
            ctx->union_batch = value;
            return EBIC_OK;
        case 6: ctx->pt_build = value ? 1 : 0; return EBIC_OK;
        case 7:
            if (value < 0) return EBIC_ERR_ARG;
            ctx->pt_min_work = value;
            return EBIC_OK;
        case 8:
            if (value < 1 || value > 16) return EBIC_ERR_ARG;
            ctx->pb_prologue_chunks = value;
            return EBIC_OK;
        case 9: ctx->use_graphs = value ? 1 : 0; return EBIC_OK;
        case 10:
            if (value < 0 || value > (1 << 20) || (value & 15)) return EBIC_ERR_ARG;
            ctx->pb_ingest_prefetch = value;
            return EBIC_OK;
        default: return EBIC_ERR_ARG;
    }
}

int ebic_set_instrumentation(ebic_ctx* ctx, int32_t on) {
    if (!ctx) return EBIC_ERR_ARG;
    ctx->epoch++;
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
        case 4: return ebic_host::resolve_kernel(ctx, ctx->last_n_ind, ctx->last_n_ids);
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
        case 16: return ctx->Rk ? ctx->ld * ctx->cols : 0;
        case 17: return ctx->pbt_bytes;
        case 18: return ctx->graph_exec ? ctx->graph_launches : 0;
        case 20: case 21: case 22: case 23: case 24:
            return static_cast<int64_t>(static_cast<double>(ctx->create_ms[what - 20]) * 1e6);
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
        case 5: src = ctx->PBT; bytes = ctx->pbt_bytes; break;
        default: return EBIC_ERR_ARG;
    }
    if (!src || bytes != dst_bytes) return EBIC_ERR_ARG;
    return cuda_status(cudaMemcpy(dst, src, static_cast<size_t>(bytes), cudaMemcpyDeviceToHost));
}

// ---- probes ------------------------------------------------------------------------------------------------
namespace {
struct ProbeTimer {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int init() {
        int st = cuda_status(cudaEventCreate(&e0));
        if (!st) st = cuda_status(cudaEventCreate(&e1));
        return st;
    }
    ~ProbeTimer() {
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    }
    void begin() { cudaEventRecord(e0, nullptr); }
    int end(float* ms) {
        cudaEventRecord(e1, nullptr);
        int st = cuda_status(cudaEventSynchronize(e1));
        if (!st) st = cuda_status(cudaEventElapsedTime(ms, e0, e1));
        if (!st) st = cuda_status(cudaGetLastError());
        return st;
    }
};
int sm_count(int* sms) {
    int dev = 0;
    EBIC_TRY(cudaGetDevice(&dev));
    EBIC_TRY(cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev));
    return EBIC_OK;
}
}  // namespace

int ebic_probe_read_bandwidth(int64_t buffer_bytes, int32_t reps, double* gb_per_s) {
    if (!gb_per_s || buffer_bytes < (1ll << 20) || reps < 1) return EBIC_ERR_ARG;
    *gb_per_s = 0.0;
    int sms = 0;
    int st = sm_count(&sms);
    if (st) return st;
    const int64_t n_vec = buffer_bytes / 16;
    uint4* buf = nullptr;
    unsigned int* sink = nullptr;
    ProbeTimer t;
    st = cuda_status(cudaMalloc(&buf, static_cast<size_t>(n_vec) * 16));
    if (!st) st = cuda_status(cudaMalloc(&sink, 4));
    if (!st) st = cuda_status(cudaMemset(buf, 0x5a, static_cast<size_t>(n_vec) * 16));
    if (!st) st = t.init();
    double best = 0.0;
    for (int per_sm = 1; per_sm <= 8 && !st; per_sm *= 2) {       // 1, 2, 4, 8 CTAs of 256 threads per SM: keep the best
        const int grid = sms * per_sm;
        const int64_t stride = static_cast<int64_t>(grid) * 256;
        const int64_t span = n_vec / (kProbeUnroll * stride) * (kProbeUnroll * stride);
        if (span <= 0) continue;
        for (int pass = 0; pass < 4 && !st; ++pass) {             // pass 0 warms the cache; best of the next 3
            float ms = 0.f;
            t.begin();
            probe_read_kernel<<<grid, 256>>>(buf, span, reps, sink);
            st = t.end(&ms);
            if (!st && pass > 0 && ms > 0.f)
                best = std::max(best, static_cast<double>(span) * 16.0 * reps / (ms * 1e-3) / 1e9);
        }
    }
    if (!st) *gb_per_s = best;
    cudaFree(sink);
    cudaFree(buf);
    return st;
}

int ebic_probe_smem_bandwidth(double* gb_per_s) {
    if (!gb_per_s) return EBIC_ERR_ARG;
    *gb_per_s = 0.0;
    int sms = 0;
    int st = sm_count(&sms);
    if (st) return st;
    unsigned int* sink = nullptr;
    ProbeTimer t;
    st = cuda_status(cudaMalloc(&sink, 4));
    if (!st) st = t.init();
    if (!st) st = cuda_status(cudaFuncSetAttribute(probe_lds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));
    const int32_t iters = 4096;
    double best = 0.0;
    for (int pass = 0; pass < 4 && !st; ++pass) {
        float ms = 0.f;
        t.begin();
        probe_lds_kernel<<<sms, 1024, 65536>>>(iters, sink);
        st = t.end(&ms);
        if (!st && pass > 0 && ms > 0.f)
            best = std::max(best, static_cast<double>(sms) * 1024.0 * iters * 8 * 16 / (ms * 1e-3) / 1e9);
    }
    if (!st) *gb_per_s = best;
    cudaFree(sink);
    return st;
}

int ebic_probe_smem_gather(int32_t rotate, double* gb_per_s) {
    if (!gb_per_s) return EBIC_ERR_ARG;
    *gb_per_s = 0.0;
    int sms = 0;
    int st = sm_count(&sms);
    if (st) return st;
    unsigned int* sink = nullptr;
    ProbeTimer t;
    st = cuda_status(cudaMalloc(&sink, 4));
    if (!st) st = t.init();
    if (!st) st = cuda_status(cudaFuncSetAttribute(probe_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 131072));
    const int32_t iters = rotate ? 2048 : 256;
    double best = 0.0;
    for (int pass = 0; pass < 4 && !st; ++pass) {
        float ms = 0.f;
        t.begin();
        probe_gather_kernel<<<sms, 512, 131072>>>(iters, rotate ? 1 : 0, sink);
        st = t.end(&ms);
        if (!st && pass > 0 && ms > 0.f)     // 512 lanes x 8 slots x 128 bytes per iteration
            best = std::max(best, static_cast<double>(sms) * 512.0 * iters * 8 * 128 / (ms * 1e-3) / 1e9);
    }
    if (!st) *gb_per_s = best;
    cudaFree(sink);
    return st;
}

int ebic_probe_fsetp_rate(double* gcompares_per_s) {
    if (!gcompares_per_s) return EBIC_ERR_ARG;
    *gcompares_per_s = 0.0;
    int sms = 0;
    int st = sm_count(&sms);
    if (st) return st;
    unsigned int* sink = nullptr;
    ProbeTimer t;
    st = cuda_status(cudaMalloc(&sink, 4));
    if (!st) st = t.init();
    const int32_t iters = 2048;
    const int grid = sms * 8;
    double best = 0.0;
    for (int pass = 0; pass < 4 && !st; ++pass) {
        float ms = 0.f;
        t.begin();
        probe_fsetp_kernel<<<grid, 256>>>(iters, 1.0f, 2.0f, sink);
        st = t.end(&ms);
        if (!st && pass > 0 && ms > 0.f)
            best = std::max(best, static_cast<double>(grid) * 256.0 * iters * 48 / (ms * 1e-3) / 1e9);
    }
    if (!st) *gcompares_per_s = best;
    cudaFree(sink);
    return st;
}

}  // extern "C"
