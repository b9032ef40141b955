// extract_kernels.cuh -- SURVEY.md 8(a) row a7: matched-row bitmask (and count) of chosen individuals.
// Both kernels are launched with programmatic dependent launch.  `overlap` = 0 (ebic_extract_rows): wait for the
// stream's earlier work before touching anything, so only the launch latency is hidden.  `overlap` = 1
// (ebic_eval_extract, where the library knows the predecessor is its own fitness kernel and that this kernel
// reads nothing it writes): run alongside the fitness kernel's last wave and wait for it only before exiting.
// results are biclusters = rows + columns; the rows of an individual are the rows
// for which ok(k,r) of include/ebic.h holds.  HBM-bound: reads 4*L bytes per row, writes 1/8 byte.
//
// Bit layout: row r <-> uint32 word r/32, bit r%32 (== little-endian uint64 word r/64, bit r%64).
// A warp covers 128 consecutive rows per step: lane l evaluates rows base + 32*w + l for w = 0..3, so
// the ballot of predicate w IS mask word w and every column load is one coalesced 128-byte request.
#pragma once
#include "ebic_device.cuh"

namespace ebic {

constexpr int kExtractMaxSmemIds = 1024;

// grid.x over row chunks (rows_per_block = 8 warps * 128 rows * kExtractSteps), grid.y over chosen.
constexpr int kExtractSteps = 4;
constexpr int kExtractRowsPerBlock = 8 * 128 * kExtractSteps;

__global__ void __launch_bounds__(256)
extract_rows_kernel(const float* __restrict__ Mc, int64_t ld, int64_t rows, int32_t cols, int32_t missing_on,
                    const uint32_t* __restrict__ nanmask, const int32_t* __restrict__ offsets,
                    const int32_t* __restrict__ col_ids, int32_t n_ind, int64_t n_ids,
                    const int32_t* __restrict__ chosen, int32_t n_chosen, uint32_t* __restrict__ masks32,
                    int64_t words32, unsigned long long* __restrict__ counts, int32_t* __restrict__ err,
                    int32_t overlap)
{
    if (!overlap) griddep_wait();                                  // stream order: everything before this launch is done
    __shared__ int32_t s_ids[kExtractMaxSmemIds];
    __shared__ int32_t s_bad;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t ldw = ld / 32;
    const int64_t w_block = static_cast<int64_t>(blockIdx.x) * (kExtractRowsPerBlock / 32);

    for (int32_t j = blockIdx.y; j < n_chosen; j += gridDim.y) {
        // ---- validate the chosen individual (every block does it; L is small) ----
        if (tid == 0) s_bad = 0;
        __syncthreads();
        const int32_t k = chosen[j];
        int32_t b = 0, L = -1;
        int bad = 0;
        if (k < 0 || k >= n_ind) {
            bad = 5;
        } else {
            b = offsets[k];
            const int32_t e = offsets[k + 1];
            if (b < 0 || e < b || static_cast<int64_t>(e) > n_ids) bad = 5;
            else L = e - b;
        }
        if (!bad) {
            for (int32_t i = tid; i < L; i += 256) {
                const int32_t id = col_ids[b + i];
                if (id < 0 || id >= cols) s_bad = 4;             // benign race: same value
                else if (i < kExtractMaxSmemIds) s_ids[i] = id;
            }
        }
        __syncthreads();
        if (!bad) bad = s_bad;
        if (bad && tid == 0 && blockIdx.x == 0) atomicMax(err, bad);
        const int32_t* gids = col_ids + b;

        uint32_t* out = masks32 + static_cast<int64_t>(j) * words32;
        unsigned int local = 0;
        for (int step = 0; step < kExtractSteps; ++step) {
            const int64_t w0 = w_block + (step * 8 + warp) * 4;   // first of this warp's 4 words
            if (w0 >= words32) break;
            unsigned int word = 0;                                 // lane w (< 4) ends up with word w
            if (bad) {
                word = 0;
            } else if (L >= 2) {
                const float* base = Mc + w0 * 32 + lane;
                const int32_t id0 = (0 < kExtractMaxSmemIds) ? s_ids[0] : gids[0];
                const float* c0 = base + static_cast<int64_t>(id0) * ld;
                float v0 = c0[0], v1 = c0[32], v2 = c0[64], v3 = c0[96];
                bool p0 = true, p1 = true, p2 = true, p3 = true;
                for (int32_t i = 1; i < L; ++i) {
                    const int32_t id = (i < kExtractMaxSmemIds) ? s_ids[i] : __ldg(&gids[i]);
                    const float* c = base + static_cast<int64_t>(id) * ld;
                    const float u0 = c[0], u1 = c[32], u2 = c[64], u3 = c[96];
                    p0 = p0 & (u0 >= v0);
                    p1 = p1 & (u1 >= v1);
                    p2 = p2 & (u2 >= v2);
                    p3 = p3 & (u3 >= v3);
                    v0 = u0; v1 = u1; v2 = u2; v3 = u3;
                }
                const unsigned int b0 = __ballot_sync(0xffffffffu, p0);
                const unsigned int b1 = __ballot_sync(0xffffffffu, p1);
                const unsigned int b2 = __ballot_sync(0xffffffffu, p2);
                const unsigned int b3 = __ballot_sync(0xffffffffu, p3);
                word = lane == 0 ? b0 : lane == 1 ? b1 : lane == 2 ? b2 : b3;
            } else if (lane < 4) {
                // L <= 1: closed form.  Valid rows of word w: [32w, min(rows, 32w+32)).
                const int64_t w = w0 + lane;
                const int64_t left = rows - w * 32;
                const unsigned int valid = left >= 32 ? 0xffffffffu : left <= 0 ? 0u : ((1u << left) - 1u);
                if (L == 1 && missing_on && w < ldw)
                    word = ~nanmask[static_cast<int64_t>(s_ids[0]) * ldw + w] & valid;
                else
                    word = valid;
            }
            if (lane < 4 && w0 + lane < words32) {
                out[w0 + lane] = word;
                local += __popc(word);
            }
        }
        if (counts != nullptr) {
            local = __reduce_add_sync(0xffffffffu, local);
            if (lane == 0 && local) atomicAdd(&counts[j], static_cast<unsigned long long>(local));
        }
        __syncthreads();                                           // s_ids / s_bad are reused for the next j
    }
    if (overlap) griddep_wait();                                   // this grid must not complete before its predecessor
}

// Extraction from the pair-relation bit columns (loader_kernels.cuh): for L >= 2 the mask IS the AND of
// the individual's L-1 bit columns, so a chosen individual costs (L-1) * rows / 8 bytes of HBM reads
// instead of 4 * L * rows -- 32x less.  One thread per FOUR 32-bit mask words (16-byte loads, four in flight per
// thread); a warp reads 512 contiguous bytes of a bit column per pair.  Padding rows are NaN, so bits >= rows are already zero.  L <= 1 as above.
// grid.x strided over blocks of 1,024 words (a CTA validates its individual once and then streams several blocks),
// grid.y over chosen (strided).
__global__ void __launch_bounds__(256)
extract_rows_pairbits_kernel(const uint32_t* __restrict__ PB, int64_t ld, int64_t rows, int32_t cols,
                             int32_t missing_on, const uint32_t* __restrict__ nanmask,
                             const int32_t* __restrict__ offsets, const int32_t* __restrict__ col_ids,
                             int32_t n_ind, int64_t n_ids, const int32_t* __restrict__ chosen, int32_t n_chosen,
                             uint32_t* __restrict__ masks32, int64_t words32,
                             unsigned long long* __restrict__ counts, int32_t* __restrict__ err, int32_t overlap)
{
    if (!overlap) griddep_wait();                                  // stream order: everything before this launch is done
    __shared__ int32_t s_pair[kExtractMaxSmemIds];
    __shared__ int32_t s_bad;
    __shared__ unsigned int s_cnt;
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t ldw = ld / 32;                                           // a multiple of 32: 16-byte units never straddle
    const int64_t ldw4 = ldw >> 2;
    const int64_t n_wblocks = (words32 + 1023) / 1024;                     // blocks of 1,024 mask words, strided over grid.x
    // 16-byte stores need every mask row 16-byte aligned: a row length that is a multiple of four words AND a
    // 16-byte-aligned base (include/ebic.h only promises uint64 alignment: the caller may pass an offset view)
    const bool vec_store = (words32 & 3) == 0 && (reinterpret_cast<uintptr_t>(masks32) & 15) == 0;

    for (int32_t j = blockIdx.y; j < n_chosen; j += gridDim.y) {
        if (tid == 0) {
            s_bad = 0;
            s_cnt = 0;
        }
        __syncthreads();
        const int32_t k = chosen[j];
        int32_t b = 0, L = -1;
        int bad = 0;
        if (k < 0 || k >= n_ind) {
            bad = 5;
        } else {
            b = offsets[k];
            const int32_t e = offsets[k + 1];
            if (b < 0 || e < b || static_cast<int64_t>(e) > n_ids) bad = 5;
            else L = e - b;
        }
        if (!bad) {
            for (int32_t i = tid; i < L; i += 256) {
                const int32_t id = col_ids[b + i];
                if (id < 0 || id >= cols) s_bad = 4;             // benign race: same value
                else if (i + 1 < L && i < kExtractMaxSmemIds) {
                    const int32_t nx = col_ids[b + i + 1];
                    s_pair[i] = (nx >= 0 && nx < cols) ? id * cols + nx : 0;
                }
            }
        }
        __syncthreads();
        if (!bad) bad = s_bad;
        if (bad && tid == 0 && blockIdx.x == 0) atomicMax(err, bad);

        unsigned int local = 0;
        for (int64_t wb = blockIdx.x; wb < n_wblocks; wb += gridDim.x) {
        const int64_t w = (wb * 256 + tid) * 4;                            // this thread's four mask words w .. w + 3
        const uint4* wbase = reinterpret_cast<const uint4*>(PB) + (min(w, ldw - 4) >> 2);   // + pair * (ldw / 4)
        uint4 word = make_uint4(0u, 0u, 0u, 0u);
        if (w < words32 && !bad) {
            if (L >= 2) {
                word = make_uint4(~0u, ~0u, ~0u, ~0u);
                const int32_t npr = L - 1;
                const int32_t ns = min(npr, kExtractMaxSmemIds);
                int32_t i = 0;
                for (; i + 4 <= ns; i += 4) {                   // four 16-byte loads in flight per thread
                    const uint4 v0 = __ldg(wbase + s_pair[i] * ldw4), v1 = __ldg(wbase + s_pair[i + 1] * ldw4);
                    const uint4 v2 = __ldg(wbase + s_pair[i + 2] * ldw4), v3 = __ldg(wbase + s_pair[i + 3] * ldw4);
                    word.x &= v0.x & v1.x & v2.x & v3.x; word.y &= v0.y & v1.y & v2.y & v3.y;
                    word.z &= v0.z & v1.z & v2.z & v3.z; word.w &= v0.w & v1.w & v2.w & v3.w;
                }
                for (; i < ns; ++i) {
                    const uint4 v = __ldg(wbase + s_pair[i] * ldw4);
                    word.x &= v.x; word.y &= v.y; word.z &= v.z; word.w &= v.w;
                }
                for (; i < npr; ++i) {                          // very long chromosomes: ids from global
                    const int64_t pr = static_cast<int64_t>(__ldg(&col_ids[b + i])) * cols + __ldg(&col_ids[b + i + 1]);
                    const uint4 v = __ldg(wbase + pr * ldw4);
                    word.x &= v.x; word.y &= v.y; word.z &= v.z; word.w &= v.w;
                }
            } else {
                unsigned int out[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int64_t left = rows - (w + c) * 32;
                    const unsigned int valid = left >= 32 ? 0xffffffffu : left <= 0 ? 0u : ((1u << left) - 1u);
                    out[c] = (L == 1 && missing_on) ? ~nanmask[static_cast<int64_t>(__ldg(&col_ids[b])) * ldw + w + c] & valid : valid;
                }
                word = make_uint4(out[0], out[1], out[2], out[3]);
            }
        }
        uint32_t* dst = masks32 + static_cast<int64_t>(j) * words32 + w;
        if (w + 3 < words32 && vec_store) {
            *reinterpret_cast<uint4*>(dst) = word;
        } else if (w < words32) {
            dst[0] = word.x;
            if (w + 1 < words32) dst[1] = word.y; else word.y = 0u;
            if (w + 2 < words32) dst[2] = word.z; else word.z = 0u;
            if (w + 3 < words32) dst[3] = word.w; else word.w = 0u;
        }
        local += __popc(word.x) + __popc(word.y) + __popc(word.z) + __popc(word.w);
        }
        if (counts != nullptr) {                                 // warp -> block -> one global atomic per block
            local = __reduce_add_sync(0xffffffffu, local);
            if (lane == 0 && local) atomicAdd(&s_cnt, local);
            __syncthreads();
            if (tid == 0 && s_cnt) atomicAdd(&counts[j], static_cast<unsigned long long>(s_cnt));
        }
        __syncthreads();
    }
    if (overlap) griddep_wait();                                   // this grid must not complete before its predecessor
}

}  // namespace ebic
