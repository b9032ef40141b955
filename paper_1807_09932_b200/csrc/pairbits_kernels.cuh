// pairbits_kernels.cuh -- a5/a6 on the pair-relation bit columns built by loader_kernels.cuh:
//   ok(k, r) = AND_{i < L-1} PB[(c_i, c_{i+1})] bit r          count[k] = popcount over rows.
// 1 bit per (row, pair): 8x fewer operand bytes than RANK8 and one LOP3 per 32 rows and pair.  Exact for
// every L >= 2 and both missing modes (an ordered >= is false on NaN; padding rows are NaN, bits 0).
//
// PAIRBITS (any cols): PB is pair-major, PB[pair][ld/32 words] -- the bit column of a pair is contiguous.
// No staging: a warp task = (individual, chunk of `chunk_words` words of rows).  Per step the warp covers
// 256 words (8,192 rows) and, per batch, 4 pairs: 8 independent LDG.128 per lane in flight before the
// first AND (two fully used 512-byte runs per pair).  Registers are the landing buffer; with 4 CTAs of 8
// warps per SM that is 32 warps x 4 KB of loads in flight per SM.  Tasks are ordered chunk-major, so the
// CTAs in flight walk the same few row chunks and the slice of PB they touch stays in the 126 MB L2;
// HBM sees every used bit column once per evaluation.  Bound: L2 -> SM bandwidth for the gathered
// bytes, HBM for the distinct bit columns.
// (Measured alternatives, round 1: gathering the same pieces with TMA bulk copies or per-lane cp.async
// into per-warp shared-memory rings was slower on every workload -- DESIGN.md 6.4.)
#pragma once
#include "ebic_device.cuh"

namespace ebic {

constexpr int kRecPairsPb = 30;      // pair indices held in an individual's 128-byte record (see ingest)
constexpr int kPairbitsWarps = 8;
constexpr int kPairbitsStepWords = 256;   // words (x32 rows) a warp covers per step: 2 x LDG.128 per lane and pair

struct PairbitsParams {
    const uint32_t* PB;              // [npairs][ldw]
    int64_t ldw;                     // words per bit column = ld / 32
    int32_t chunk_words;             // words per warp task, multiple of kPairbitsStepWords
    int32_t n_chunks;                // ceil(ldw / chunk_words)
    const int32_t* prec;             // [n_ind][32] records: L, slot4, 30 pair indices
    const int32_t* ppair;            // padded pair-index slots (chromosomes with more than 31 columns)
    int32_t n_ind;
    unsigned long long* counts;
    unsigned long long* visits;      // executed (row, pair) visits (instrumented) or nullptr
    int32_t n_pairs;                 // cols * cols bit columns in PB
    int32_t prefetch_dist;           // CTAs of chunk g prefetch a slice of the bit columns of chunk g + dist into L2 (0 = off)
};

__device__ __forceinline__ void and4(uint4& a, const uint4& v) {
    a.x &= v.x; a.y &= v.y; a.z &= v.z; a.w &= v.w;
}
__device__ __forceinline__ bool any4(const uint4& a) { return (a.x | a.y | a.z | a.w) != 0u; }

template <bool EARLY_EXIT>
__global__ void __launch_bounds__(kPairbitsWarps * 32)
fitness_pairbits_kernel(const PairbitsParams p)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t task = static_cast<int64_t>(blockIdx.x) * kPairbitsWarps + warp;
    const int64_t g = task / p.n_ind;
    const int32_t k = static_cast<int32_t>(task - g * p.n_ind);
    const int64_t w_begin = g * p.chunk_words;
    if (w_begin >= p.ldw) return;                                // warp-uniform
    if (p.prefetch_dist > 0 && warp == 0) {
        // Every bit column of a later chunk is requested from HBM exactly once, by one lane of one CTA of
        // this chunk, `prefetch_dist` chunks before the demand loads arrive: those then hit L2.
        const int64_t ctas_per_chunk = (static_cast<int64_t>(p.n_ind) + kPairbitsWarps - 1) / kPairbitsWarps;
        const int64_t j = blockIdx.x - g * p.n_ind / kPairbitsWarps; // position of this CTA inside its chunk (approx.)
        const int32_t per_cta = static_cast<int32_t>((p.n_pairs + ctas_per_chunk - 1) / ctas_per_chunk);
        const int64_t first = (g == 0) ? 1 : p.prefetch_dist;        // chunk 0 also covers the cold start
        for (int64_t d = first; d <= p.prefetch_dist; ++d) {
            const int64_t pw = (g + d) * p.chunk_words;
            if (pw >= p.ldw) break;
            const uint32_t bytes = static_cast<uint32_t>(min(static_cast<int64_t>(p.chunk_words), p.ldw - pw)) * 4u;
            for (int32_t q = lane; q < per_cta; q += 32) {
                const int64_t pair = j * per_cta + q;
                if (pair >= 0 && pair < p.n_pairs) bulk_prefetch_l2(p.PB + pair * p.ldw + pw, bytes);
            }
        }
    }
    const int32_t rec = __ldg(p.prec + 32ll * k + lane);         // the individual: one coalesced 128 B load
    const int32_t L = __shfl_sync(0xffffffffu, rec, 0);
    if (L < 2) return;
    const int32_t npr = L - 1;
    const int32_t n0 = min(npr, kRecPairsPb);
    const int32_t* pp = p.ppair + 4ll * __shfl_sync(0xffffffffu, rec, 1);
    const int64_t w_end = min(p.ldw, w_begin + p.chunk_words);
    const int64_t ldv = p.ldw / 4;                               // bit column length in uint4

    unsigned int cnt = 0;
    unsigned long long executed = 0;
    for (int64_t w0 = w_begin; w0 < w_end; w0 += kPairbitsStepWords) {
        const int64_t wa = w0 + lane * 4, wb = wa + 128;
        const bool va = wa < w_end, vb = wb < w_end;             // ldw is a multiple of 32: a lane's 4 words are all in or all out
        const uint4* base_a = reinterpret_cast<const uint4*>(p.PB + (va ? wa : w0));
        const uint4* base_b = reinterpret_cast<const uint4*>(p.PB + (vb ? wb : w0));
        uint4 acc_a = va ? make_uint4(~0u, ~0u, ~0u, ~0u) : make_uint4(0u, 0u, 0u, 0u);
        uint4 acc_b = vb ? make_uint4(~0u, ~0u, ~0u, ~0u) : make_uint4(0u, 0u, 0u, 0u);
        int32_t done = 0;
        int32_t i = 0;
        for (; i + 4 <= n0; i += 4) {
            const int64_t p0 = __shfl_sync(0xffffffffu, rec, i + 2) * ldv, p1 = __shfl_sync(0xffffffffu, rec, i + 3) * ldv;
            const int64_t p2 = __shfl_sync(0xffffffffu, rec, i + 4) * ldv, p3 = __shfl_sync(0xffffffffu, rec, i + 5) * ldv;
            const uint4 a0 = __ldg(base_a + p0), a1 = __ldg(base_a + p1), a2 = __ldg(base_a + p2), a3 = __ldg(base_a + p3);
            const uint4 b0 = __ldg(base_b + p0), b1 = __ldg(base_b + p1), b2 = __ldg(base_b + p2), b3 = __ldg(base_b + p3);
            and4(acc_a, a0); and4(acc_a, a1); and4(acc_a, a2); and4(acc_a, a3);
            and4(acc_b, b0); and4(acc_b, b1); and4(acc_b, b2); and4(acc_b, b3);
            done += 4;
            if (EARLY_EXIT && !__any_sync(0xffffffffu, any4(acc_a) || any4(acc_b))) goto step_done;
        }
        if (i < n0) {                                            // 1..3 pairs left: the record is padded with
            const int32_t r = n0 - i;                            // the last pair, so its entries are always valid
            const int64_t p0 = __shfl_sync(0xffffffffu, rec, i + 2) * ldv, p1 = __shfl_sync(0xffffffffu, rec, i + 3) * ldv;
            const int64_t p2 = __shfl_sync(0xffffffffu, rec, min(i + 4, 31)) * ldv;
            const uint4 a0 = __ldg(base_a + p0), b0 = __ldg(base_b + p0);
            and4(acc_a, a0); and4(acc_b, b0);
            if (r >= 2) {
                const uint4 a1 = __ldg(base_a + p1), b1 = __ldg(base_b + p1);
                and4(acc_a, a1); and4(acc_b, b1);
            }
            if (r >= 3) {
                const uint4 a2 = __ldg(base_a + p2), b2 = __ldg(base_b + p2);
                and4(acc_a, a2); and4(acc_b, b2);
            }
            done += r;
        }
        for (int32_t seg = kRecPairsPb; seg < npr; seg += 32) {  // chromosomes with more than 31 columns
            if (EARLY_EXIT && !__any_sync(0xffffffffu, any4(acc_a) || any4(acc_b))) break;
            const int32_t n = min(32, npr - seg);
            const int32_t mine = __ldg(pp + seg + min(lane, n - 1));
            for (int32_t j = 0; j < n; ++j) {
                const int64_t p0 = __shfl_sync(0xffffffffu, mine, j) * ldv;
                const uint4 a0 = __ldg(base_a + p0), b0 = __ldg(base_b + p0);
                and4(acc_a, a0); and4(acc_b, b0);
            }
            done += n;
        }
    step_done:
        cnt += __popc(acc_a.x) + __popc(acc_a.y) + __popc(acc_a.z) + __popc(acc_a.w);
        cnt += __popc(acc_b.x) + __popc(acc_b.y) + __popc(acc_b.z) + __popc(acc_b.w);
        executed += static_cast<unsigned long long>(done) *
                    (min(w_end - w0, static_cast<int64_t>(kPairbitsStepWords)) * 32);
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0) {
        if (cnt) atomicAdd(&p.counts[k], static_cast<unsigned long long>(cnt));
        if (p.visits != nullptr) atomicAdd(p.visits, executed);
    }
}

}  // namespace ebic
