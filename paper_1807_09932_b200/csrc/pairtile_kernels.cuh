// pairtile_kernels.cuh -- a4/a5/a6 on TILES of the pair-relation table staged in shared memory (PAIRTILE):
//   ok(k, r) = AND_{i < L-1} PB[(c_i, c_{i+1})] bit r          count[k] = popcount over rows
// exactly as pairbits_kernels.cuh, but the bit columns come from shared memory instead of L2.  This is
// BASELINE.json north_star (3) -- "stages row tiles x all columns in shared memory via TMA, reuses each tile
// across a batch of individuals" -- applied to the 1-bit encoding: a tile = 1,024 rows of ALL cols^2 bit columns
// = cols^2 x 128 bytes, contiguous in the tile-major copy PBT[tile][pair][32 words] the loader writes next to the
// pair-major table (loader_kernels.cuh), so ONE TMA bulk copy stages it.  It applies while a tile fits shared
// memory next to the per-CTA counters (cols <= 42); narrow matrices with large populations (BASELINE config C5:
// 32 columns, 4,096 individuals, every bit column used 32 times per tile) are then bound by the shared-memory
// data pipe (128 B/clk/SM, 37 TB/s) instead of the L2 -> SM bandwidth (23 TB/s).
//
// Lane = individual.  A warp takes a GROUP of 32 individuals; lane l walks its own chromosome: for every pair it
// reads the pair's 128-byte slot (1,024 rows) as eight LDS.128 and ANDs them into 32 accumulator registers.  The
// lanes of a warp read DIFFERENT slots, so the 16-byte unit is rotated per lane: in step u lane l reads unit
// u ^ (l & 7) of its slot -- the eight lanes of every quarter-warp then hit eight different 16-byte bank groups
// whatever slots they picked (conflict-free; ebic_probe_smem_gather: 37.1 TB/s chip-wide with random slots, against
// 4.7 TB/s unrotated).  No cross-lane traffic at all: no shuffles, no ballots, no reductions -- the popcount of a lane's
// accumulators is its individual's count for the tile, added to a per-CTA shared counter the lane owns.
//
// An LDS.128 costs its four wavefronts whether or not all lanes are active (measured), so the groups must be
// uniform in length: pairtile_plan_kernel sorts the individuals by the number of pairs (counting sort, descending)
// and writes, for sorted position j = 32 g + l, gmeta[j] = {k, n} and the pair slots of the chromosome as 16-bit
// offsets (pair * 8, in 16-byte units), eight per uint4, in the transposed layout tids[g][chunk][l] a warp reads
// with coalesced 512-byte loads.  A record is padded to 32 entries with its last pair (AND is idempotent), so the
// group loop needs no per-lane predicate: every lane does max-over-the-group steps.  Chromosomes with more than 33
// columns continue from the caller's col_ids.
//
// Persistent CTAs, one per SM, 12 warps of 168 registers (no spill: 16 LDS.128 in flight per warp next to the 32
// accumulators; measured on C5: 8 / 10 / 12 / 14 / 16 / 20 warps = 2.38 / 2.22 / 2.15 / 2.18 / 2.17 / 2.38 ms).  Work = (tile, group) items in tile-major order cut into equal contiguous
// ranges (a tile is staged by at most two CTAs more than necessary); inside a tile the groups are handed out through
// a shared-memory cursor, alternately from the long and the short end of the sorted list.  One tile buffer (two
// tiles of 128 KB do not fit at 32 columns): while the warps work on tile t, tile t + 1 is requested into L2
// (cp.async.bulk.prefetch.L2); when the last warp is done the buffer is refilled from L2 with TMA bulk copies of 16
// KB, completion on an mbarrier.  (Measured and removed: a split buffer that staged the part of the next tile that
// fits a second time a whole tile ahead -- it did not change the kernel time.)
#pragma once
#include "ebic_device.cuh"

namespace ebic {

constexpr int kPtWarps = 12;
constexpr int kPtRecIds = 32;              // pair slots held per individual in tids (4 x uint4 of 8 halfwords)
constexpr int kPtPlanThreads = 1024;       // pairtile_plan_kernel: individuals per CTA
constexpr int kPtHeader = 128;             // shared-memory header (the mbarrier) in front of the tile
constexpr uint32_t kPtCopyBytes = 16384;   // bytes per TMA bulk copy / L2 prefetch request

struct PairtileParams {
    const uint32_t* PBT;             // [n_tiles][n_pairs][32 words]
    int64_t n_tiles;                 // ld / 1024
    int32_t n_pairs;                 // cols * cols
    int32_t cols;
    int32_t n_ind;                   // individuals of this launch
    int32_t n_groups;                // ceil(n_ind / 32)
    int32_t rec_cache;               // shared memory has room for entries 0..7 of every record (16 bytes per position)
    const int2* meta;                // [n_ind] {b, L} written by the ingest kernel (L = -1: invalid)
    const int32_t* col_ids;
    int2* gmeta;                     // [n_groups * 32] {k, n}: individual and its number of pairs (-1: nothing to do)
    uint4* tids;                     // [n_groups][4][32]: 8 x uint16 slot offsets (pair * 8) per lane and chunk
    unsigned long long* counts;      // [n_ind]
    unsigned long long* visits;      // executed (row, pair) visits (instrumented) or nullptr
};

// Sorting key: 0 = 32 pairs or more, ..., 31 = one pair, 32 = nothing to evaluate (L <= 1: closed form in the
// ingest kernel; L = -1: invalid), 33 = beyond n_ind (the CTA's idle threads).
__device__ __forceinline__ int32_t pairtile_key(int32_t L) { return L < 2 ? 32 : 32 - min(L - 1, 32); }

// a3, second half.  grid = ceil(n_ind / 1024), 1,024 threads, thread = individual.  Every CTA counts the keys of the
// whole launch (n_ind <= 8,192) and of the individuals in front of its block, so positions are global:
// pos = (individuals with a smaller key) + (same key, earlier block) + (same key, this block, drawn from a cursor).
__global__ void __launch_bounds__(kPtPlanThreads)
pairtile_plan_kernel(const PairtileParams p)
{
    __shared__ int32_t s_total[34], s_before[34], s_cursor[34], s_base[34];
    griddep_launch_dependents();                 // the fitness kernel may stage its first tile meanwhile
    const int tid = threadIdx.x, lane = tid & 31;
    if (tid < 34) { s_total[tid] = 0; s_before[tid] = 0; s_cursor[tid] = 0; }
    __syncthreads();
    griddep_wait();                              // meta comes from the ingest kernel
    const int32_t k_begin = blockIdx.x * kPtPlanThreads;
    const int32_t n_round = (p.n_ind + kPtPlanThreads - 1) / kPtPlanThreads * kPtPlanThreads;
    for (int32_t k = tid; k < n_round; k += kPtPlanThreads) {
        const int32_t key = k < p.n_ind ? pairtile_key(p.meta[k].y) : 33;
        const unsigned same = __match_any_sync(0xffffffffu, key);
        if (lane == __ffs(same) - 1) {
            atomicAdd(&s_total[key], __popc(same));
            if (k < k_begin) atomicAdd(&s_before[key], __popc(same));     // a warp never straddles a block boundary
        }
    }
    __syncthreads();
    if (tid == 0) {
        int32_t run = 0;
        for (int q = 0; q < 33; ++q) { s_base[q] = run; run += s_total[q]; }
        s_base[33] = run;
    }
    __syncthreads();
    const int32_t k = k_begin + tid;
    int2 m = make_int2(0, -1);
    if (k < p.n_ind) m = p.meta[k];
    const int32_t key = k < p.n_ind ? pairtile_key(m.y) : 33;
    const unsigned same = __match_any_sync(0xffffffffu, key);
    const int leader = __ffs(same) - 1;
    int32_t first = 0;
    if (lane == leader) first = atomicAdd(&s_cursor[key], __popc(same));
    first = __shfl_sync(0xffffffffu, first, leader);
    // the tail of the last group holds nobody: {0, -1}
    const int32_t n_slots = p.n_groups * 32;
    if (blockIdx.x == 0 && p.n_ind + tid < n_slots) {                  // n_slots - n_ind < 32
        const int32_t j = p.n_ind + tid;
        p.gmeta[j] = make_int2(0, -1);
        uint4* rec = p.tids + (static_cast<int64_t>(j >> 5) * 4) * 32 + (j & 31);
        const uint4 z = make_uint4(0u, 0u, 0u, 0u);                     // slot 0: a lane that idles reads valid memory
        rec[0] = z; rec[32] = z; rec[64] = z; rec[96] = z;
    }
    if (k >= p.n_ind) return;
    const int32_t pos = s_base[key] + s_before[key] + first + __popc(same & ((1u << lane) - 1u));
    const int32_t n = m.y < 2 ? -1 : m.y - 1;
    p.gmeta[pos] = make_int2(k, n);
    uint4* rec = p.tids + (static_cast<int64_t>(pos >> 5) * 4) * 32 + (pos & 31);
    if (n < 1) {
        const uint4 z = make_uint4(0u, 0u, 0u, 0u);
        rec[0] = z; rec[32] = z; rec[64] = z; rec[96] = z;
        return;
    }
    const int32_t* ids = p.col_ids + m.x;        // a VALID individual: every id is inside [0, cols)
    uint32_t w[16];
    int32_t a = ids[0];
#pragma unroll
    for (int i = 0; i < kPtRecIds; ++i) {
        // entry i = pair min(i, n - 1) = (id_q, id_{q+1})
        const int32_t q = min(i, n - 1);
        const int32_t a_q = (i < n) ? a : ids[q];
        const int32_t c_q = ids[q + 1];
        const uint32_t slot = static_cast<uint32_t>(a_q * p.cols + c_q) * 8u;      // < 65,536: n_pairs <= 1,783
        if (i & 1) w[i >> 1] |= slot << 16; else w[i >> 1] = slot;
        a = c_q;
    }
    rec[0] = make_uint4(w[0], w[1], w[2], w[3]);
    rec[32] = make_uint4(w[4], w[5], w[6], w[7]);
    rec[64] = make_uint4(w[8], w[9], w[10], w[11]);
    rec[96] = make_uint4(w[12], w[13], w[14], w[15]);
}

// AND the 1,024 rows of the slots at `off_a` / `off_b` (16-byte units from the tile start) into acc.  `lanebase` =
// shared address of the tile + 16 * (lane & 7): slot addresses are 128-byte aligned, so `^ (u << 4)` walks the eight
// 16-byte units of a slot starting at this lane's own unit.
__device__ __forceinline__ void pairtile_and2(uint4 (&acc)[8], uint32_t lanebase, uint32_t off_a, uint32_t off_b) {
    const uint32_t a = lanebase + off_a * 16u, b = lanebase + off_b * 16u;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const uint4 v = lds128(a ^ (u << 4)), w = lds128(b ^ (u << 4));
        acc[u].x &= v.x & w.x; acc[u].y &= v.y & w.y; acc[u].z &= v.z & w.z; acc[u].w &= v.w & w.w;
    }
}
__device__ __forceinline__ void pairtile_and1(uint4 (&acc)[8], uint32_t lanebase, uint32_t off_a) {
    const uint32_t a = lanebase + off_a * 16u;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const uint4 v = lds128(a ^ (u << 4));
        acc[u].x &= v.x; acc[u].y &= v.y; acc[u].z &= v.z; acc[u].w &= v.w;
    }
}

// Two record entries (the halfwords of `w`), of which `left` >= 1 (warp-uniform) are needed.
__device__ __forceinline__ void pairtile_step(uint4 (&acc)[8], uint32_t lanebase, uint32_t w, int32_t left) {
    if (left >= 2) pairtile_and2(acc, lanebase, w & 0xffffu, w >> 16);
    else pairtile_and1(acc, lanebase, w & 0xffffu);
}
// Eight record entries (one uint4 of halfwords), of which the first `n_left` (warp-uniform, >= 1) are needed.
__device__ __forceinline__ void pairtile_chunk(uint4 (&acc)[8], uint32_t lanebase, const uint4& ids, int32_t n_left) {
    pairtile_step(acc, lanebase, ids.x, n_left);
    if (n_left > 2) pairtile_step(acc, lanebase, ids.y, n_left - 2);
    if (n_left > 4) pairtile_step(acc, lanebase, ids.z, n_left - 4);
    if (n_left > 6) pairtile_step(acc, lanebase, ids.w, n_left - 6);
}

// Shared memory: [header: mbarrier + group cursors][tile: n_pairs slots of 128 bytes][counters: one per sorted
// position][gmax: per group, the longest chromosome in pairs = the group's loop count][record cache, when it fits:
// entries 0..7 of every record -- they are the same for every tile, so the per-group record load then stays on the SM].
__global__ void __launch_bounds__(kPtWarps * 32, 1)
fitness_pairtile_kernel(const PairtileParams p)
{
    extern __shared__ __align__(128) unsigned char pt_smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(pt_smem);
    int32_t* cursor = reinterpret_cast<int32_t*>(pt_smem + 32);                   // [2] next position of the even / odd tile
    unsigned char* tile = pt_smem + kPtHeader;
    const uint32_t tile_bytes = static_cast<uint32_t>(p.n_pairs) * 128u;
    uint32_t* counters = reinterpret_cast<uint32_t*>(tile + tile_bytes);          // [n_groups * 32]
    int32_t* s_gmax = reinterpret_cast<int32_t*>(counters + p.n_groups * 32);     // [n_groups rounded up to 4]
    uint4* s_ids0 = reinterpret_cast<uint4*>(s_gmax + ((p.n_groups + 3) & ~3));   // [n_groups * 32] if rec_cache
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // this CTA's contiguous range of (tile, position) items
    const int64_t items = p.n_tiles * p.n_groups;
    const int64_t per = (items + gridDim.x - 1) / gridDim.x;
    const int64_t i0 = per * blockIdx.x, i1 = min(items, i0 + per);
    griddep_launch_dependents();                 // a dependent extraction launch may be scheduled
    if (i0 >= i1) return;
    const int64_t t_first = i0 / p.n_groups, t_last = (i1 - 1) / p.n_groups;
    const unsigned char* table = reinterpret_cast<const unsigned char*>(p.PBT);

    auto stage = [&](int64_t t) {                // one thread: refill the tile buffer, completion on `full`
        const unsigned char* src = table + t * static_cast<int64_t>(tile_bytes);
        mbar_arrive_expect_tx(full, tile_bytes);
        for (uint32_t o = 0; o < tile_bytes; o += kPtCopyBytes)
            bulk_copy_g2s(tile + o, src + o, min(kPtCopyBytes, tile_bytes - o), full);
    };
    if (tid == 0) {
        mbar_init(full, 1);
        fence_mbar_init();
        stage(t_first);                          // the table depends on the matrix only: overlaps ingest + plan
        cursor[0] = static_cast<int32_t>(i0 - t_first * p.n_groups) + kPtWarps;
    }
    for (int32_t j = tid; j < p.n_groups * 32; j += kPtWarps * 32) counters[j] = 0;
    griddep_wait();                              // gmeta / tids (plan kernel), counts initialised (ingest kernel)
    for (int32_t grp = warp; grp < p.n_groups; grp += kPtWarps) {
        const int32_t mx = __reduce_max_sync(0xffffffffu, ld_produced(p.gmeta + grp * 32 + lane).y);
        if (lane == 0) s_gmax[grp] = mx;
        if (p.rec_cache) s_ids0[grp * 32 + lane] = ld_produced(p.tids + static_cast<int64_t>(grp) * 128 + lane);
    }
    __syncthreads();

    const uint32_t lanebase = smem_u32(tile) + ((lane & 7) << 4);
    unsigned long long executed = 0;
    // Position c of a tile's hand-out order -> group: alternately from the long and from the short end of the sorted
    // list, so that at any time the warps hold a mix of long and short groups.  (The fixed cost per group -- 32
    // popcounts, counter, cursor -- is poorly hidden while ALL warps work on one- or two-pair groups, as at the end of
    // a longest-first order: 2.24 -> 2.19 ms on C5; strided orders 2.20.)  The first kPtWarps positions of a tile go to
    // the warps statically, the rest through a shared cursor; a warp draws its next position, and requests the
    // group's records, before it evaluates the current one -- the first of the NEXT tile before the barrier that ends
    // this one, so that no warp starts a tile by waiting for its records.
    int32_t c = static_cast<int32_t>(i0 - t_first * p.n_groups) + warp;
    int32_t maxn = 0, grp_req = 0;
    uint4 ids0 = make_uint4(0u, 0u, 0u, 0u), ids1 = ids0;
    auto request = [&](int32_t pos) {            // loop count and record entries 0..15 of the group at position pos
        grp_req = (pos & 1) ? p.n_groups - 1 - (pos >> 1) : (pos >> 1);
        maxn = s_gmax[grp_req];
        const uint4* rec = p.tids + static_cast<int64_t>(grp_req) * 128 + lane;
        ids0 = p.rec_cache ? s_ids0[grp_req * 32 + lane] : ld_produced(rec);
        if (maxn > 8) ids1 = ld_produced(rec + 32);
    };
    if (c < (t_first == t_last ? static_cast<int32_t>(i1 - t_first * p.n_groups) : p.n_groups)) request(c);
    uint32_t phase = 0;
    for (int64_t t = t_first; t <= t_last; ++t) {
        const int q = static_cast<int>((t - t_first) & 1);
        const int32_t c_hi = t == t_last ? static_cast<int32_t>(i1 - t * p.n_groups) : p.n_groups;
        if (t < t_last && tid < 32) {            // next tile: HBM -> L2 while this one is evaluated
            const unsigned char* nxt = table + (t + 1) * static_cast<int64_t>(tile_bytes);
            for (uint32_t o = lane * kPtCopyBytes; o < tile_bytes; o += 32 * kPtCopyBytes)
                bulk_prefetch_l2(nxt + o, min(kPtCopyBytes, tile_bytes - o));
            if (lane == 0) cursor[q ^ 1] = kPtWarps;       // the next tile starts at position 0; nobody reads this cursor now
        }
        mbar_wait(full, phase);
        phase ^= 1;
        while (c < c_hi) {
            const int32_t maxn_cur = maxn, grp = grp_req;
            const uint4 cur0 = ids0, cur1 = ids1;
            int32_t c_next = 0;
            if (lane == 0) c_next = atomicAdd(&cursor[q], 1);
            c_next = __shfl_sync(0xffffffffu, c_next, 0);
            if (c_next < c_hi) request(c_next);  // in flight during this group's evaluation
            if (maxn_cur >= 1) {
                uint4 acc[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) acc[u] = make_uint4(~0u, ~0u, ~0u, ~0u);
                const int32_t m = min(maxn_cur, kPtRecIds);
                pairtile_chunk(acc, lanebase, cur0, m);
                if (m > 8) pairtile_chunk(acc, lanebase, cur1, m - 8);
                if (m > 16) {
                    const uint4* rec = p.tids + static_cast<int64_t>(grp) * 128 + lane;
                    const uint4 cur2 = ld_produced(rec + 64), cur3 = ld_produced(rec + 96);
                    pairtile_chunk(acc, lanebase, cur2, m - 16);
                    if (m > 24) pairtile_chunk(acc, lanebase, cur3, m - 24);
                }
                if (maxn_cur > kPtRecIds || p.visits != nullptr) {       // rare: a very long chromosome, or instrumented
                    const int2 gm = ld_produced(p.gmeta + grp * 32 + lane);
                    if (gm.y > kPtRecIds) {
                        // pairs beyond the record come from the caller's ids (a VALID individual)
                        const int32_t* ids_g = p.col_ids + ld_produced(&p.meta[gm.x]).x;
                        int32_t a = __ldg(ids_g + kPtRecIds);
                        for (int32_t j = kPtRecIds; j < gm.y; ++j) {
                            const int32_t b = __ldg(ids_g + j + 1);
                            pairtile_and1(acc, lanebase, static_cast<uint32_t>(a * p.cols + b) * 8u);
                            a = b;
                        }
                    }
                    if (gm.y >= 1) executed += static_cast<unsigned long long>(gm.y);
                }
                // A lane that holds no individual (or one with nothing to evaluate) walked slot 0 of an all-zero
                // record: its counter is never read back (the final loop checks gmeta).
                unsigned int cnt = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) cnt += __popc(acc[u].x) + __popc(acc[u].y) + __popc(acc[u].z) + __popc(acc[u].w);
                counters[grp * 32 + lane] += cnt;        // this lane is the only one that touches the counter now
            }
            c = c_next;
        }
        if (t < t_last) {                        // first position of the next tile (it starts at 0)
            c = warp;
            if (c < (t + 1 == t_last ? static_cast<int32_t>(i1 - t_last * p.n_groups) : p.n_groups)) request(c);
        }
        __syncthreads();                         // every warp is done with the tile (and with its counters)
        if (t < t_last && tid == 0) {
            fence_proxy_async_smem();            // the warps' LDS (generic proxy) before the refill's bulk-copy writes (async proxy)
            stage(t + 1);
        }
    }
    // one 64-bit global atomic per (CTA, individual)
    for (int32_t j = tid; j < p.n_groups * 32; j += kPtWarps * 32) {
        const uint32_t cnt = counters[j];
        const int2 gm = ld_produced(p.gmeta + j);
        if (cnt && gm.y >= 1) atomicAdd(&p.counts[gm.x], static_cast<unsigned long long>(cnt));
    }
    if (p.visits != nullptr) {
        for (int o = 16; o > 0; o >>= 1) executed += __shfl_down_sync(0xffffffffu, executed, o);
        if (lane == 0 && executed) atomicAdd(p.visits, executed * static_cast<unsigned long long>(kPairTileRows));
    }
}

}  // namespace ebic
