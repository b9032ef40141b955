// prefix_kernels.cuh -- SURVEY.md 8(f) NEXT-4, shared-prefix ("trie") evaluation on the pair-relation bit columns:
// individuals whose chromosomes start with the same columns share the AND of those columns' bit columns.
//   ok(k, r) = AND_{i < P} PB[(c_i, c_{i+1})] bit r  AND  AND_{P <= i < L-1} PB[(c_i, c_{i+1})] bit r
// and the first factor is the same for every member of a group with a common prefix of P pairs: a warp fetches the
// P shared bit columns once per 8,192-row step and finishes up to kPrefixGroup members from the shared accumulator.
// Results are bit-identical to PAIRBITS (AND is associative); only the number of bit-column fetches changes, and
// the executed-visit counter counts the fetches actually made.  A GA population that has converged is mostly
// near-duplicates (long shared prefixes); on the uniformly random populations of BASELINE.json only the first pair
// is shared by a few individuals (DESIGN.md 6.7 has the measured effect).
//
// prefix_plan_kernel (one CTA): sorts the ingest's records by their first two pair offsets (bitonic sort in shared
// memory, population <= kPrefixMaxInd), cuts every run of equal first pairs into groups of <= kPrefixGroup members,
// and writes for each group its members' record indices and P = the longest prefix (in pairs) common to all of them.
// Individuals with fewer than 2 or more than 31 columns become groups of one and run the plain PAIRBITS task.
#pragma once
#include "pairbits_kernels.cuh"

namespace ebic {

constexpr int kPrefixGroup = 4;              // members per group (each needs a record register and a counter)
constexpr int kPrefixMaxInd = 8192;          // the plan kernel sorts the whole population in shared memory

struct PrefixParams {
    PairbitsParams pb;               // the table, the records, the row chunking (tasks_* unused)
    int32_t* groups;                 // [n_ind][8]: {cnt | P << 8, record index of member 0..3, 0, 0, 0}
    int32_t* n_groups;               // device scalar written by the plan kernel
};

// ---- plan -------------------------------------------------------------------------------------------------
// dynamic shared memory: uint64 key[N], uint32 val[N], uint8 flag[N], N = population rounded up to a power of two
__global__ void __launch_bounds__(1024)
prefix_plan_kernel(const PrefixParams p, int32_t n_pow2)
{
    extern __shared__ __align__(16) unsigned char plan_mem[];
    unsigned long long* key = reinterpret_cast<unsigned long long*>(plan_mem);
    uint32_t* val = reinterpret_cast<uint32_t*>(plan_mem + 8ull * n_pow2);
    __shared__ int32_t s_scan[32];
    __shared__ int32_t s_total;
    griddep_wait();                                  // the records come from the ingest kernel
    griddep_launch_dependents();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t n = p.pb.n_ind;
    const uint32_t* prec = p.pb.prec;
    for (int32_t j = tid; j < n_pow2; j += 1024) {
        unsigned long long kk = ~0ull;
        if (j < n) {
            const int32_t L = static_cast<int32_t>(ld_produced(prec + 32ll * j));
            if (L >= 2 && L <= 31)                   // groupable: the whole chromosome lives in the record
                kk = (static_cast<unsigned long long>(ld_produced(prec + 32ll * j + 2)) << 32) | ld_produced(prec + 32ll * j + 3);
            else if (L >= 32)
                kk = ~0ull - 1;                      // evaluated, never grouped
        }
        key[j] = kk;
        val[j] = static_cast<uint32_t>(j);
    }
    __syncthreads();
    // bitonic sort, ascending by key
    for (int32_t size = 2; size <= n_pow2; size <<= 1) {
        for (int32_t stride = size >> 1; stride > 0; stride >>= 1) {
            for (int32_t t = tid; t < (n_pow2 >> 1); t += 1024) {
                const int32_t lo = 2 * t - (t & (stride - 1));           // index with bit `stride` clear
                const int32_t hi = lo + stride;
                const bool up = (lo & size) == 0;
                const unsigned long long a = key[lo], b = key[hi];
                if ((a > b) == up) {
                    key[lo] = b; key[hi] = a;
                    const uint32_t v = val[lo]; val[lo] = val[hi]; val[hi] = v;
                }
            }
            __syncthreads();
        }
    }
    // Sorted position i starts a group iff it starts a run of equal first pairs, or sits at a multiple of
    // kPrefixGroup inside its run, or cannot be grouped (key == ~0 - 1: more than 31 columns).  Positions whose key
    // is ~0 (fewer than 2 columns, invalid, beyond n) need no evaluation and start no group.
    uint8_t* flag = plan_mem + 12ull * n_pow2;                   // 1 = starts a group
    const int32_t per = (n_pow2 + 1023) / 1024;
    const int32_t i0 = tid * per, i1 = min(n_pow2, i0 + per);
    for (int32_t i = i0; i < i1; ++i) {
        const unsigned long long k = key[i];
        bool st = false;
        if (k == ~0ull - 1) {
            st = true;
        } else if (k != ~0ull) {
            const uint32_t fp = static_cast<uint32_t>(k >> 32);
            int32_t d = 0;                                       // distance to the start of the run of equal first pairs
            while (d < i && static_cast<uint32_t>(key[i - d - 1] >> 32) == fp && key[i - d - 1] < ~0ull - 1) ++d;
            st = (d % kPrefixGroup) == 0;
        }
        flag[i] = st ? 1 : 0;
    }
    __syncthreads();
    auto is_start = [&](int32_t i) -> bool { return flag[i] != 0; };
    int32_t mine = 0;
    for (int32_t i = i0; i < i1; ++i) mine += is_start(i) ? 1 : 0;
    // exclusive scan of `mine` over the 1,024 threads
    int32_t inc = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int32_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) s_scan[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int32_t w = s_scan[lane], winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int32_t t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        s_scan[lane] = winc - w;
        if (lane == 31) s_total = winc;
    }
    __syncthreads();
    int32_t g = s_scan[warp] + inc - mine;
    for (int32_t i = i0; i < i1; ++i) {
        if (!is_start(i)) continue;
        // members: i, i+1, ... while they are not starts themselves (and are groupable)
        int32_t cnt = 1;
        while (cnt < kPrefixGroup && i + cnt < n_pow2 && key[i + cnt] < ~0ull - 1 && !is_start(i + cnt)) ++cnt;
        int32_t P = 0;
        if (cnt > 1) {
            // longest prefix (in pairs) common to all members: compare each member with member 0
            P = 30;
            const uint32_t* r0 = prec + 32ll * val[i];
            for (int32_t m = 0; m < cnt; ++m) P = min(P, static_cast<int32_t>(ld_produced(prec + 32ll * val[i + m])) - 1);
            for (int32_t m = 1; m < cnt; ++m) {
                const uint32_t* rm = prec + 32ll * val[i + m];
                int32_t q = 0;
                while (q < P && ld_produced(r0 + 2 + q) == ld_produced(rm + 2 + q)) ++q;
                P = q;
            }
        }
        int32_t* out = p.groups + 8ll * g;
        out[0] = cnt | (P << 8);
        for (int32_t m = 0; m < kPrefixGroup; ++m) out[1 + m] = static_cast<int32_t>(val[i + min(m, cnt - 1)]);
        ++g;
    }
    if (tid == 0) *p.n_groups = s_total;
}

// ---- evaluation -------------------------------------------------------------------------------------------
// AND the 256-word slices of the bit columns named by entries [i0, i1) of `rec` into acc_a / acc_b, exactly.
__device__ __forceinline__ void prefix_and_range(const uint4* __restrict__ base, uint32_t rec, int32_t i0, int32_t i1,
                                                 uint4& acc_a, uint4& acc_b)
{
    int32_t i = i0;
    for (; i + 4 <= i1; i += 4) {
        const uint4 *q0 = base + __shfl_sync(0xffffffffu, rec, i + 2), *q1 = base + __shfl_sync(0xffffffffu, rec, i + 3);
        const uint4 *q2 = base + __shfl_sync(0xffffffffu, rec, i + 4), *q3 = base + __shfl_sync(0xffffffffu, rec, i + 5);
        const uint4 a0 = __ldg(q0), a1 = __ldg(q1), a2 = __ldg(q2), a3 = __ldg(q3);
        const uint4 b0 = __ldg(q0 + 32), b1 = __ldg(q1 + 32), b2 = __ldg(q2 + 32), b3 = __ldg(q3 + 32);
        and4(acc_a, a0); and4(acc_a, a1); and4(acc_a, a2); and4(acc_a, a3);
        and4(acc_b, b0); and4(acc_b, b1); and4(acc_b, b2); and4(acc_b, b3);
    }
    for (; i < i1; ++i) {                                        // warp-uniform
        const uint4* q0 = base + __shfl_sync(0xffffffffu, rec, i + 2);
        const uint4 a0 = __ldg(q0), b0 = __ldg(q0 + 32);
        and4(acc_a, a0); and4(acc_b, b0);
    }
}

__device__ __forceinline__ unsigned int popc8(const uint4& a, const uint4& b) {
    return __popc(a.x) + __popc(a.y) + __popc(a.z) + __popc(a.w) + __popc(b.x) + __popc(b.y) + __popc(b.z) + __popc(b.w);
}

// Task = (group, row chunk), chunk-major like PAIRBITS.  The grid is sized for the worst case (every individual its
// own group); blocks beyond n_groups * n_chunks exit.
template <bool EARLY_EXIT>
__global__ void __launch_bounds__(kPairbitsWarps * 32)
fitness_prefix_kernel(const PrefixParams pp)
{
    const PairbitsParams& p = pp.pb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    griddep_launch_dependents();
    griddep_wait();
    const int64_t n_groups = ld_produced(pp.n_groups);
    const int64_t task = static_cast<int64_t>(blockIdx.x) * kPairbitsWarps + warp;
    if (task >= n_groups * p.n_chunks) return;
    const int64_t g_chunk = task / n_groups;
    const int32_t g = static_cast<int32_t>(task - g_chunk * n_groups);
    const int32_t* grp = pp.groups + 8ll * g;
    const int32_t head = ld_produced(grp);
    const int32_t cnt = head & 0xff, P = head >> 8;
    unsigned long long executed = 0;
    if (cnt == 1) {                                              // not grouped: the plain task on this member's record
        const int32_t j = ld_produced(grp + 1);
        const uint32_t rec = ld_produced(p.prec + 32ll * j + lane);
        pairbits_task<EARLY_EXIT, false>(p, g_chunk, j, rec, lane, 0u, executed);
    } else {
        uint32_t rec[kPrefixGroup];
#pragma unroll
        for (int m = 0; m < kPrefixGroup; ++m) rec[m] = ld_produced(p.prec + 32ll * ld_produced(grp + 1 + m) + lane);
        const int64_t w_begin = g_chunk * p.chunk_words, w_end = min(p.ldw, w_begin + p.chunk_words);
        const uint4* PB4 = reinterpret_cast<const uint4*>(p.PB);
        unsigned int c[kPrefixGroup] = {0u, 0u, 0u, 0u};
        for (int64_t w0 = w_begin; w0 < w_end; w0 += kPairbitsStepWords) {
            // lane l: words 4l..4l+3 of the step's first 128 words and of its second 128 (clamped in the ragged last step)
            const int64_t wa = w0 + lane * 4, wb = wa + 128;
            const bool va = wa < w_end, vb = wb < w_end;
            const uint4* base = PB4 + ((va ? wa : w0) >> 2);
            const int64_t delta = ((vb ? wb : w0) >> 2) - ((va ? wa : w0) >> 2);   // 32 in every full step
            uint4 pa = va ? make_uint4(~0u, ~0u, ~0u, ~0u) : make_uint4(0u, 0u, 0u, 0u);
            uint4 pb = vb ? make_uint4(~0u, ~0u, ~0u, ~0u) : make_uint4(0u, 0u, 0u, 0u);
            if (w0 + kPairbitsStepWords <= w_end) {               // full step (warp-uniform): second halves at + 512 bytes
                prefix_and_range(base, rec[0], 0, P, pa, pb);
                executed += static_cast<unsigned long long>(P) * (min(static_cast<int64_t>(kPairbitsStepWords), w_end - w0) * 32);
                if (!(EARLY_EXIT && !__any_sync(0xffffffffu, any4(pa) || any4(pb)))) {
#pragma unroll
                    for (int m = 0; m < kPrefixGroup; ++m) {
                        if (m < cnt) {
                            const int32_t npr = static_cast<int32_t>(__shfl_sync(0xffffffffu, rec[m], 0)) - 1;
                            uint4 a = pa, b = pb;
                            prefix_and_range(base, rec[m], P, npr, a, b);
                            c[m] += popc8(a, b);
                            executed += static_cast<unsigned long long>(npr - P) * (kPairbitsStepWords * 32);
                        }
                    }
                }
            } else {
                // ragged last step of a column: second-half addresses are not base + 512 bytes; one column at a time
#pragma unroll
                for (int m = 0; m < kPrefixGroup; ++m) {
                    if (m < cnt) {
                        const int32_t npr = static_cast<int32_t>(__shfl_sync(0xffffffffu, rec[m], 0)) - 1;
                        uint4 a = pa, b = pb;
                        for (int32_t i = 0; i < npr; ++i) {
                            const uint4* q = base + __shfl_sync(0xffffffffu, rec[m], i + 2);
                            and4(a, __ldg(q));
                            and4(b, __ldg(q + delta));
                        }
                        c[m] += popc8(a, b);
                        executed += static_cast<unsigned long long>(npr) * ((w_end - w0) * 32);
                    }
                }
            }
        }
#pragma unroll
        for (int m = 0; m < kPrefixGroup; ++m) {
            if (m < cnt) {
                const unsigned int total = __reduce_add_sync(0xffffffffu, c[m]);
                const int32_t k = static_cast<int32_t>(__shfl_sync(0xffffffffu, rec[m], 1));
                if (lane == 0 && total) atomicAdd(&p.counts[k], static_cast<unsigned long long>(total));
            }
        }
    }
    if (lane == 0 && p.visits != nullptr && executed) atomicAdd(p.visits, executed);
}

}  // namespace ebic
