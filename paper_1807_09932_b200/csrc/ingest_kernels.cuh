// ingest_kernels.cuh -- SURVEY.md 8(a) row a3: population ingest + validation (a population
// of up to 65,535 individuals, 1,600 typical; BASELINE.json north_star (1): CSR offsets + int32 column ids).
//
// Everything the ingest writes is keyed by the individual's INDEX (or by a position inside the individual's own
// 64-individual block), never by the contents of `offsets`: two individuals can therefore never share scratch,
// whatever the offsets array holds (R8: an invalid individual leaves the valid ones unaffected).
//
//   meta[k]   = { b, L }: first entry of the chromosome in col_ids and its length; L = -1 = invalid individual
//               (offsets[k] < 0, offsets[k+1] < offsets[k], offsets[k+1] > n_ids, or an id outside [0, cols)).
//   idrec[k]  = the first 32 ids as bytes (cols <= 256: eight 32-bit words) or as halfwords (wider: sixteen words),
//               padded with the last id: the tiled kernels fetch four / two ids with one warp-uniform load.
//               Longer chromosomes continue from col_ids.
//   prec[j]   = (pair table present) one 128-byte record per individual, read by a warp with ONE coalesced load:
//               word 0 = L (-1 = invalid), word 1 = k, words 2..31 = the bit-column offsets of the first 30
//               consecutive pairs (id_i, id_{i+1}) in the pair table, in 16-byte units,
//               (id_i * cols + id_{i+1}) * pair_stride16, padded with the last pair (AND is idempotent).
//               Longer chromosomes continue from col_ids.  j = the individual's position inside its block of
//               64 consecutive individuals after sorting the block by DESCENDING length: the two warps of a
//               PAIRBITS CTA then work on chromosomes of (nearly) equal length and finish together.
//   counts[k] is initialised: rows (L = 0, or L = 1 in mode OFF), non-missing rows of the column (L = 1, mode
//               ON), else 0 -- the chain kernels then add to it (no separate memset launch).
//   err       sticky device error: atomicMax of EBIC_ERR_BAD_COLUMN (4) / EBIC_ERR_BAD_OFFSETS (5).
#pragma once
#include "ebic_device.cuh"

namespace ebic {

constexpr int kIngestBlock = 64;     // individuals per CTA = sorting block
constexpr int kIngestThreads = 1024; // 32 warps: two individuals per warp, so the id loads of a block all overlap
constexpr int kRecPairs = 30;        // pair offsets held in a record

struct IngestParams {
    const int32_t* offsets;
    const int32_t* col_ids;
    int32_t n_ind;
    int64_t n_ids;
    int32_t cols;
    int64_t rows;
    int32_t missing_on;
    int32_t sort_by_length;          // 0: records stay in population order
    const unsigned long long* nonmissing;
    int2* meta;
    uint32_t* idrec;                 // [n_ind][8] (byte ids) / [n_ind][16] (16-bit ids, id_wide) or nullptr
    int32_t id_wide;                 // cols > 256: the id record holds halfwords
    uint32_t* prec;                  // [n_ind][32] or nullptr
    uint32_t pair_stride16;          // 16-byte units per bit column = ld / 128
    unsigned long long* counts;
    int32_t* err;
    // Sparse populations on the pair table (a wide matrix: the population uses a small part of the cols^2 bit columns,
    // so the fitness kernel's prologue cannot afford to request all of them): the ingest, which forms every pair
    // offset anyway, asks L2 for the first `prefetch_bytes` of each bit column a record names (0 = off).  The fitness
    // kernel then finds its first loads in L2, or on their way, instead of starting a chain of HBM misses.
    const uint32_t* PB = nullptr;
    uint32_t prefetch_bytes = 0;     // multiple of 16, at most one bit column (ld / 8)
};

__global__ void __launch_bounds__(kIngestThreads)
ingest_population_kernel(const IngestParams p)
{
    __shared__ int32_t s_b[kIngestBlock];
    __shared__ int32_t s_L[kIngestBlock];      // -1 = bad offsets, -2 = beyond n_ind
    __shared__ int32_t s_pos[kIngestBlock];
    griddep_launch_dependents();                // the fitness kernel may start its (population-independent) prologue
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t k0 = blockIdx.x * kIngestBlock;
    if (tid < kIngestBlock) {
        const int32_t k = k0 + tid;
        int32_t b = 0, L = -2;
        if (k < p.n_ind) {
            b = p.offsets[k];
            const int32_t e = p.offsets[k + 1];
            L = (b < 0 || e < b || static_cast<int64_t>(e) > p.n_ids) ? -1 : e - b;
        }
        s_b[tid] = b;
        s_L[tid] = L;
    }
    __syncthreads();
    if (tid < kIngestBlock) {
        int32_t r = tid;
        if (p.sort_by_length) {                 // rank by descending L, ties in population order
            const int32_t mine = s_L[tid];
            r = 0;
            for (int u = 0; u < kIngestBlock; ++u) {
                const int32_t o = s_L[u];
                r += (o > mine || (o == mine && u < tid)) ? 1 : 0;
            }
        }
        s_pos[tid] = r;
    }
    __syncthreads();

    for (int t = warp; t < kIngestBlock; t += kIngestThreads / 32) {   // one warp per individual
        const int32_t L = s_L[t];
        if (L == -2) continue;                              // warp-uniform
        const int32_t k = k0 + t;
        const int64_t j = static_cast<int64_t>(k0) + s_pos[t];
        if (L == -1) {
            if (lane == 0) {
                p.meta[k] = make_int2(0, -1);
                p.counts[k] = 0;
                atomicMax(p.err, 5 /* EBIC_ERR_BAD_OFFSETS */);
            }
            if (p.prec != nullptr && lane < 2) p.prec[32 * j + lane] = lane == 0 ? 0xffffffffu : static_cast<uint32_t>(k);
            continue;
        }
        const int32_t b = s_b[t];
        const int32_t* ids = p.col_ids + b;
        bool bad = false;
        // lane i keeps id min(i, L-1) (ids outside [0, cols) become 0); ids beyond 32 are only validated here
        int32_t mine = 0;
        if (L > 0) {
            mine = ids[min(lane, L - 1)];
            if (mine < 0 || mine >= p.cols) { bad = true; mine = 0; }
        }
        for (int32_t i = 32 + lane; i < L; i += 32) {
            const int32_t id = ids[i];
            bad |= (id < 0 || id >= p.cols);
        }
        bad = __any_sync(0xffffffffu, bad);
        if (p.idrec != nullptr && p.id_wide) {              // two 16-bit ids per word, 16 words
            const uint32_t i0 = __shfl_sync(0xffffffffu, mine, (2 * lane) & 31), i1 = __shfl_sync(0xffffffffu, mine, (2 * lane + 1) & 31);
            if (lane < 16) p.idrec[16ll * k + lane] = i0 | (i1 << 16);
        } else if (p.idrec != nullptr) {                    // four byte ids per word, 8 words
            const uint32_t i0 = __shfl_sync(0xffffffffu, mine, (4 * lane) & 31), i1 = __shfl_sync(0xffffffffu, mine, (4 * lane + 1) & 31);
            const uint32_t i2 = __shfl_sync(0xffffffffu, mine, (4 * lane + 2) & 31), i3 = __shfl_sync(0xffffffffu, mine, (4 * lane + 3) & 31);
            if (lane < 8) p.idrec[8ll * k + lane] = i0 | (i1 << 8) | (i2 << 16) | (i3 << 24);
        }
        if (p.prec != nullptr) {
            // lane l >= 2 holds pair min(l - 2, L - 2) = (id_q, id_{q+1}); positions up to 30 live in lanes 0..30
            const int32_t q = max(0, min(lane - 2, L - 2));
            const uint32_t a = __shfl_sync(0xffffffffu, mine, q), c = __shfl_sync(0xffffffffu, mine, min(q + 1, 31));
            uint32_t v = (a * static_cast<uint32_t>(p.cols) + c) * p.pair_stride16;
            if (lane == 0) v = bad ? 0xffffffffu : static_cast<uint32_t>(L);
            if (lane == 1) v = static_cast<uint32_t>(k);
            p.prec[32 * j + lane] = v;                      // one coalesced 128-byte store
            if (p.prefetch_bytes != 0 && !bad && lane >= 2 && lane - 2 < L - 1)      // one request per pair of the record
                bulk_prefetch_l2(reinterpret_cast<const unsigned char*>(p.PB) + static_cast<int64_t>(v) * 16, p.prefetch_bytes);
        }
        if (lane != 0) continue;
        if (bad) {
            p.meta[k] = make_int2(b, -1);
            p.counts[k] = 0;
            atomicMax(p.err, 4 /* EBIC_ERR_BAD_COLUMN */);
            continue;
        }
        p.meta[k] = make_int2(b, L);
        unsigned long long c = 0;
        if (L == 0) c = static_cast<unsigned long long>(p.rows);
        else if (L == 1) c = p.missing_on ? p.nonmissing[mine] : static_cast<unsigned long long>(p.rows);
        p.counts[k] = c;
    }
}

}  // namespace ebic
