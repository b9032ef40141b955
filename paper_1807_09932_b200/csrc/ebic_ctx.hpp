// ebic_ctx.hpp -- the context behind the opaque `ebic_ctx` of include/ebic.h, shared by the two translation units
// of libebic.so (ebic_api.cu: the boundary; ebic_debug.cu: the knobs / read-backs / probes of include/ebic_debug.h).
// Host-side only.  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct ebic_ctx {
    int device = 0;
    int sm_count = 0;
    int smem_optin = 0;
    int64_t rows = 0;
    int32_t cols = 0;
    int64_t ld = 0;
    int32_t missing_mode = 0;

    // ---- loader products
    float* Mc = nullptr;                       // [cols][ld]
    uint32_t* nanmask = nullptr;               // [cols][ld/32]
    unsigned long long* nonmissing = nullptr;  // [cols]
    uint8_t* Rk = nullptr;                     // [cols][ld] rank tiles, built when AUTO would use them or on request
    uint32_t* PB = nullptr;                    // pair bit columns [cols*cols][ld/32] or nullptr
    int64_t pb_bytes = 0;
    uint32_t* PBT = nullptr;                   // the same bits, tile-major [ld/1024][cols*cols][32 words] (PAIRTILE) or nullptr
    int64_t pbt_bytes = 0;
    int32_t* d_err = nullptr;                  // sticky device error (+ the executed-visit counter behind it)
    unsigned long long* d_visits = nullptr;

    // ---- per-call scratch, grown on demand; everything is keyed by the individual's index (ingest_kernels.cuh)
    int2* meta = nullptr;
    int64_t meta_cap = 0;
    uint32_t* idrec = nullptr;                 // 32 bytes per individual (cols <= 256)
    int64_t idrec_cap = 0;
    uint32_t* prec = nullptr;                  // 128 bytes per individual (pair table present)
    int64_t prec_cap = 0;
    void* tplan = nullptr;                     // PAIRTILE: sorted {k, n} and the transposed pair-slot records
    int64_t tplan_cap = 0;
    int32_t* ubatch = nullptr;                 // column-union kernel: per-batch column lists and remapped ids
    int64_t ubatch_cap = 0;
    void* stage[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // staging for host-pointer calls
    int64_t stage_cap[6] = {0, 0, 0, 0, 0, 0};
    // ---- the launch sequence of a repeated all-device call, captured once and replayed (ebic_api.cu eval_extract_impl)
    struct GraphKey {
        const void *offsets, *col_ids, *counts, *chosen, *masks, *mask_counts, *stream;
        int64_t n_ids;
        int32_t n_ind, n_chosen, epoch, flags;
    };
    GraphKey graph_key = {};
    int32_t graph_state = 0;                   // 0 nothing seen, 1 key seen once (plain call done), 2 capture failed for this key
    cudaGraphExec_t graph_exec = nullptr;
    int64_t graph_launches = 0;                // kernels in the captured sequence (the launch counter follows replays)
    int32_t epoch = 0;                         // bumped by every knob: a captured sequence never outlives its configuration
    int32_t use_graphs = 1;

    cudaStream_t copy_stream = nullptr;        // ebic_eval_extract with host outputs: the masks go back on this stream
    cudaEvent_t ev_masks_ready = nullptr;      // while the fitness kernel runs
    cudaEvent_t ev_masks_copied = nullptr;

    // ---- knobs (include/ebic_debug.h); the defaults are the product configuration
    int32_t kernel_request = 0;                // EBIC_KERNEL_AUTO
    int32_t early_exit = 1;
    int32_t extract_pairbits = 1;              // extraction reads the pair table when it exists
    int32_t pb_tasks_per_slot = 12;            // PAIRBITS: warp tasks per resident warp slot
    int32_t pb_prefetch_dist = 1;              // PAIRBITS: L2 prefetch distance in chunks (0 = off)
    int32_t pb_prologue_chunks = 1;            // PAIRBITS: row chunks requested into L2 by the kernel's prologue (>= the distance)
    int32_t pb_smem_ring = 1;                  // PAIRBITS: shared-memory landing ring for long chromosomes
    int32_t pt_build = 1;                      // build the tile-major copy of the pair table when a tile fits shared memory
    int32_t pt_min_work = 0;                   // AUTO picks PAIRTILE from this many (tile, pair-use) units on (0 = the rule of pairtile_pays)
    int32_t pb_sort = 1;                       // ingest sorts each 64-individual block by length
    int32_t pb_ingest_prefetch = 0;            // PAIRBITS, sparse populations: bytes of every used bit column the ingest requests into L2 (0 = off)
    int32_t pdl = 1;                           // programmatic dependent launch between ingest / fitness / extraction
    int32_t union_batch = 0;                   // UNION_F32: individuals per batch (0 = chosen from the shape)
    int32_t count_visits = 0;
    int32_t time_kernels = 0;

    // ---- instrumentation
    static constexpr int kTimingRing = 256;
    cudaEvent_t ev_begin[kTimingRing] = {};
    cudaEvent_t ev_end[kTimingRing] = {};
    int64_t timed_evals = 0;
    float create_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // h2d + transpose + padding, NaN mask, pair table, rank tiles, total

    int64_t bytes_owned = 0;
    int64_t launches = 0;
    int32_t last_grid = 0;
    int32_t last_T = 0;
    int32_t last_kernel = 0;                   // kernel of the last fitness launch (0 = none yet)
    int32_t last_n_ind = 1600;                 // shape of the last population (before any: the paper's typical 1,600
    int64_t last_n_ids = 17600;                // individuals, of 11 columns): what info(4) resolves AUTO for
};

namespace ebic_host {

int cuda_status(cudaError_t e);
int build_pairbits(ebic_ctx* ctx);             // synchronous; EBIC_OK if already built
void free_pairbits(ebic_ctx* ctx);
int build_rank_tiles(ebic_ctx* ctx);           // synchronous; EBIC_ERR_ARG if cols > 127
int32_t resolve_kernel(const ebic_ctx* ctx, int32_t n_ind, int64_t n_ids);
bool kernel_applies(const ebic_ctx* ctx, int32_t kernel);

}  // namespace ebic_host
