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

constexpr int kRecPairsPb = 30;      // pair offsets held in an individual's 128-byte record (ingest_kernels.cuh)
constexpr int kPairbitsStepWords = 256;   // words (x32 rows) a warp covers per step: 2 x LDG.128 per lane and pair
constexpr int kPairbitsWarps = 2;    // warps per CTA: neighbours in the length-sorted record order

struct PairbitsParams {
    const uint32_t* PB;              // [npairs][ldw]
    int64_t ldw;                     // words per bit column = ld / 32
    int32_t chunk_words;             // words per warp task, multiple of kPairbitsStepWords
    int32_t n_chunks;                // ceil(ldw / chunk_words)
    const uint32_t* prec;            // [n_ind][32] records: L, k, 30 pair offsets (pair * ldw / 4, uint32)
    const int2* meta;                // [n_ind] {b, L}: only read for chromosomes with more than 31 columns
    const int32_t* col_ids;          // the caller's ids: pairs beyond the record are formed from them
    int32_t cols;
    uint32_t pair_stride16;          // 16-byte units per bit column = ldw / 4
    int32_t n_ind;
    unsigned long long* counts;
    unsigned long long* visits;      // executed (row, pair) visits (instrumented) or nullptr
    int32_t n_pairs;                 // cols * cols bit columns in PB
    int32_t cols_per_task;           // ceil(n_pairs / n_ind): bit columns a task requests for the prefetched chunk
    int32_t prefetch_dist;           // tasks of chunk g prefetch a slice of the bit columns of chunk g + dist into L2 (0 = off);
    int32_t prologue_chunks;         // chunks 0 .. prologue_chunks-1 (>= dist) are requested by the kernel's prologue,
                                     // before it waits for the ingest
};

__device__ __forceinline__ void and4(uint4& a, const uint4& v) {
    a.x &= v.x; a.y &= v.y; a.z &= v.z; a.w &= v.w;
}
__device__ __forceinline__ bool any4(const uint4& a) { return (a.x | a.y | a.z | a.w) != 0u; }

// One step of one chromosome: AND the 256-word slice [base_a, +128 words) / [base_b, +128 words) of each of its
// bit columns into acc_a / acc_b.  FULL: base_b == base_a + 32 uint4, so the second load of a pair is the
// first one's address + 512 bytes (an immediate).  Returns the number of pairs visited.
template <bool EARLY_EXIT, bool FULL, bool SMEM = false>
__device__ __forceinline__ int32_t pairbits_step(const uint4* __restrict__ base_a, const uint4* __restrict__ base_b,
                                                 uint32_t rec, int32_t n0, int32_t npr, const PairbitsParams& p, int32_t k,
                                                 int lane, uint4& acc_a, uint4& acc_b, uint32_t ring = 0)
{
    int32_t done = 0;
    int32_t i = 0;
    if (FULL && SMEM) {
        // 8 pairs per round: four land in registers (LDG.128), four in this lane's 16-byte cells of the warp's
        // 4 KB shared-memory ring (LDGSTS) -- twice the bytes in flight per warp for the same registers.
        for (; i + 8 <= n0; i += 8) {
            const uint4* q[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) q[j] = base_a + __shfl_sync(0xffffffffu, rec, i + 2 + j);
            // all sixteen requests leave before anything waits: eight register loads, then eight LDGSTS
            const uint4 a0 = ldg128_ordered(q[0]), a1 = ldg128_ordered(q[1]), a2 = ldg128_ordered(q[2]), a3 = ldg128_ordered(q[3]);
            const uint4 b0 = ldg128_ordered(q[0] + 32), b1 = ldg128_ordered(q[1] + 32);
            const uint4 b2 = ldg128_ordered(q[2] + 32), b3 = ldg128_ordered(q[3] + 32);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                cp_async16(ring + j * 1024 + lane * 16, q[4 + j]);
                cp_async16(ring + j * 1024 + 512 + lane * 16, q[4 + j] + 32);
            }
            cp_async_commit();
            and4(acc_a, a0); and4(acc_a, a1); and4(acc_a, a2); and4(acc_a, a3);
            and4(acc_b, b0); and4(acc_b, b1); and4(acc_b, b2); and4(acc_b, b3);
            cp_async_wait_all();
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint4 a = lds128(ring + j * 1024 + lane * 16), b = lds128(ring + j * 1024 + 512 + lane * 16);
                and4(acc_a, a); and4(acc_b, b);
            }
            done += 8;
            // Ring reuse: the next round's LDGSTS must not be issued before this round's LDS data has arrived.
            // Every lane reads and refills only its OWN 16-byte cells, so this is a same-thread, same-address
            // read-then-write in program order; __syncwarp() states it as a memory-ordering point the compiler
            // and the hardware must both honour, and `ring` is additionally made to depend on all eight
            // accumulator words (each holds the result of four of the LDS) so that the address of the next
            // LDGSTS does not exist before the loads have returned.
            __syncwarp();
            asm volatile("" : "+r"(ring) : "r"(acc_a.x), "r"(acc_a.y), "r"(acc_a.z), "r"(acc_a.w),
                                           "r"(acc_b.x), "r"(acc_b.y), "r"(acc_b.z), "r"(acc_b.w) : "memory");
            if (EARLY_EXIT && !__any_sync(0xffffffffu, any4(acc_a) || any4(acc_b))) return done;
        }
    }
    for (; i + 4 <= n0; i += 4) {
        const uint32_t p0 = __shfl_sync(0xffffffffu, rec, i + 2), p1 = __shfl_sync(0xffffffffu, rec, i + 3);
        const uint32_t p2 = __shfl_sync(0xffffffffu, rec, i + 4), p3 = __shfl_sync(0xffffffffu, rec, i + 5);
        const uint4 *q0 = base_a + p0, *q1 = base_a + p1, *q2 = base_a + p2, *q3 = base_a + p3;
        const uint4 *r0 = FULL ? q0 + 32 : base_b + p0, *r1 = FULL ? q1 + 32 : base_b + p1;
        const uint4 *r2 = FULL ? q2 + 32 : base_b + p2, *r3 = FULL ? q3 + 32 : base_b + p3;
        const uint4 a0 = __ldg(q0), a1 = __ldg(q1), a2 = __ldg(q2), a3 = __ldg(q3);
        const uint4 b0 = __ldg(r0), b1 = __ldg(r1), b2 = __ldg(r2), b3 = __ldg(r3);
        and4(acc_a, a0); and4(acc_a, a1); and4(acc_a, a2); and4(acc_a, a3);
        and4(acc_b, b0); and4(acc_b, b1); and4(acc_b, b2); and4(acc_b, b3);
        done += 4;
        if (EARLY_EXIT && !__any_sync(0xffffffffu, any4(acc_a) || any4(acc_b))) return done;
    }
    if (i < n0) {                                                // 1..3 pairs left: the record is padded with
        const int32_t r = n0 - i;                                // the last pair, so its entries are always valid
        const uint32_t p0 = __shfl_sync(0xffffffffu, rec, i + 2), p1 = __shfl_sync(0xffffffffu, rec, i + 3);
        const uint32_t p2 = __shfl_sync(0xffffffffu, rec, min(i + 4, 31));
        const uint4 *q0 = base_a + p0, *q1 = base_a + p1, *q2 = base_a + p2;
        const uint4 a0 = __ldg(q0), b0 = __ldg(FULL ? q0 + 32 : base_b + p0);
        and4(acc_a, a0); and4(acc_b, b0);
        if (r >= 2) {
            const uint4 a1 = __ldg(q1), b1 = __ldg(FULL ? q1 + 32 : base_b + p1);
            and4(acc_a, a1); and4(acc_b, b1);
        }
        if (r >= 3) {
            const uint4 a2 = __ldg(q2), b2 = __ldg(FULL ? q2 + 32 : base_b + p2);
            and4(acc_a, a2); and4(acc_b, b2);
        }
        done += r;
    }
    for (int32_t seg = kRecPairsPb; seg < npr; seg += 32) {      // chromosomes with more than 31 columns
        if (EARLY_EXIT && !__any_sync(0xffffffffu, any4(acc_a) || any4(acc_b))) break;
        // pair offsets beyond the 30 a record holds are formed from the caller's ids (a VALID individual: every
        // id is inside [0, cols)); pair q = (id_q, id_{q+1}), q + 1 <= L - 1
        const int32_t n = min(32, npr - seg);
        const int32_t* ids = p.col_ids + ld_produced(&p.meta[k]).x + seg + min(lane, n - 1);
        const uint32_t mine = (static_cast<uint32_t>(__ldg(ids)) * static_cast<uint32_t>(p.cols) +
                               static_cast<uint32_t>(__ldg(ids + 1))) * p.pair_stride16;
        for (int32_t j = 0; j < n; ++j) {
            const uint4* q0 = base_a + __shfl_sync(0xffffffffu, mine, j);
            const uint4 a0 = __ldg(q0), b0 = __ldg(FULL ? q0 + 32 : base_b + __shfl_sync(0xffffffffu, mine, j));
            and4(acc_a, a0); and4(acc_b, b0);
        }
        done += n;
    }
    return done;
}

// One warp task: record j (individual k = its word 1) on row chunk g.
// `rec` = this lane's word of the record.
template <bool EARLY_EXIT, bool SMEM>
__device__ __forceinline__ void pairbits_task(const PairbitsParams& p, int64_t g, int32_t j, uint32_t rec, int lane, uint32_t ring,
                                              unsigned long long& executed)
{
    const int64_t w_begin = g * p.chunk_words;
    if (w_begin >= p.ldw) return;                                // warp-uniform
    if (p.prefetch_dist > 0) {
        // Every bit column of chunk g + dist is requested from HBM exactly once, by one lane of one task of chunk g:
        // the demand loads that arrive `dist` chunks later then hit L2.  (Chunks 0 .. dist-1: the kernel's prologue.)
        const int32_t per = p.cols_per_task;                         // ceil(n_pairs / n_ind)
        const int64_t pw = (g + p.prefetch_dist) * p.chunk_words;
        if (pw < p.ldw && g + p.prefetch_dist >= p.prologue_chunks) {
            const uint32_t bytes = static_cast<uint32_t>(min(static_cast<int64_t>(p.chunk_words), p.ldw - pw)) * 4u;
            for (int32_t q = lane; q < per; q += 32) {
                const int64_t pair = static_cast<int64_t>(j) * per + q;
                if (pair < p.n_pairs) bulk_prefetch_l2(p.PB + pair * p.ldw + pw, bytes);
            }
        }
    }
    const int32_t L = static_cast<int32_t>(__shfl_sync(0xffffffffu, rec, 0));
    if (L < 2) return;                                           // L <= 1: closed form (ingest); -1: invalid
    const int32_t k = static_cast<int32_t>(__shfl_sync(0xffffffffu, rec, 1));
    const int32_t npr = L - 1;
    const int32_t n0 = min(npr, kRecPairsPb);
    const int64_t w_end = min(p.ldw, w_begin + p.chunk_words);
    const uint4* PB4 = reinterpret_cast<const uint4*>(p.PB);

    unsigned int cnt = 0;
    // Lane l holds words 4l .. 4l+3 of the step's first 128 words (acc_a) and the same words of its second 128
    // (acc_b).  Record entries are the bit columns' offsets into PB in uint4 units (< 2^32, host-checked).
    const int64_t n_full = (w_end - w_begin) / kPairbitsStepWords;
    const uint4* base = PB4 + (w_begin >> 2) + lane;
    for (int64_t s = 0; s < n_full; ++s, base += kPairbitsStepWords / 4) {
        uint4 acc_a = make_uint4(~0u, ~0u, ~0u, ~0u), acc_b = acc_a;
        const int32_t done = pairbits_step<EARLY_EXIT, true, SMEM>(base, base, rec, n0, npr, p, k, lane, acc_a, acc_b, ring);
        cnt += __popc(acc_a.x) + __popc(acc_a.y) + __popc(acc_a.z) + __popc(acc_a.w);
        cnt += __popc(acc_b.x) + __popc(acc_b.y) + __popc(acc_b.z) + __popc(acc_b.w);
        executed += static_cast<unsigned long long>(done) * (kPairbitsStepWords * 32);
    }
    const int64_t w0 = w_begin + n_full * kPairbitsStepWords;
    if (w0 < w_end) {                                            // ragged last step of a column (ldw % 256 != 0)
        const int64_t wa = w0 + lane * 4, wb = wa + 128;
        const bool va = wa < w_end, vb = wb < w_end;             // ldw % 32 == 0: a lane's 4 words are all in or all out
        const uint4* base_a = PB4 + ((va ? wa : w0) >> 2);
        const uint4* base_b = PB4 + ((vb ? wb : w0) >> 2);
        uint4 acc_a = va ? make_uint4(~0u, ~0u, ~0u, ~0u) : make_uint4(0u, 0u, 0u, 0u);
        uint4 acc_b = vb ? make_uint4(~0u, ~0u, ~0u, ~0u) : make_uint4(0u, 0u, 0u, 0u);
        const int32_t done = pairbits_step<EARLY_EXIT, false>(base_a, base_b, rec, n0, npr, p, k, lane, acc_a, acc_b);
        cnt += __popc(acc_a.x) + __popc(acc_a.y) + __popc(acc_a.z) + __popc(acc_a.w);
        cnt += __popc(acc_b.x) + __popc(acc_b.y) + __popc(acc_b.z) + __popc(acc_b.w);
        executed += static_cast<unsigned long long>(done) * ((w_end - w0) * 32);
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0 && cnt) atomicAdd(&p.counts[k], static_cast<unsigned long long>(cnt));
}

// One task per warp; grid = (ceil(n_ind / kPairbitsWarps), n_chunks): blockIdx.y is the row chunk, the CTA's warps
// take consecutive records of it (no division anywhere on the way to the first load), and the hardware block
// scheduler -- x fastest -- walks the chunks in order and balances the load.  Launched with programmatic dependent
// launch right behind the ingest kernel: the prologue (the HBM -> L2 requests for the first chunks of every bit
// column, which depend on the matrix only) overlaps the ingest; griddep_wait() then orders the record loads and the
// count atomics behind it.
template <bool EARLY_EXIT, bool SMEM>
__global__ void __launch_bounds__(kPairbitsWarps * 32)
fitness_pairbits_kernel(const PairbitsParams p)
{
    extern __shared__ __align__(16) unsigned char pb_ring[];     // SMEM: one 4 KB landing ring per warp
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    griddep_launch_dependents();                                 // a dependent extraction launch may be scheduled
    if (p.prefetch_dist > 0 && blockIdx.y == 0) {
        // chunks 0 .. prologue_chunks-1 of every bit column, each requested exactly once, spread over the first CTAs
        const int32_t n_pro = min(static_cast<int32_t>(gridDim.x), (p.n_pairs + 63) / 64);
        if (static_cast<int32_t>(blockIdx.x) < n_pro) {
            const uint32_t bytes = static_cast<uint32_t>(min(static_cast<int64_t>(p.prologue_chunks) * p.chunk_words, p.ldw)) * 4u;
            for (int32_t pair = blockIdx.x * 64 + threadIdx.x; pair < p.n_pairs; pair += n_pro * 64)
                bulk_prefetch_l2(p.PB + static_cast<int64_t>(pair) * p.ldw, bytes);
        }
    }
    griddep_wait();
    const int32_t j = blockIdx.x * kPairbitsWarps + warp;
    if (j >= p.n_ind) return;
    const uint32_t rec = ld_produced(p.prec + 32ll * j + lane);        // one coalesced 128 B load
    unsigned long long executed = 0;
    pairbits_task<EARLY_EXIT, SMEM>(p, blockIdx.y, j, rec, lane, SMEM ? smem_u32(pb_ring) + warp * 4096 : 0u, executed);
    if (lane == 0 && p.visits != nullptr && executed) atomicAdd(p.visits, executed);
}

}  // namespace ebic
