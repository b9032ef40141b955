// fitness_kernels.cuh -- SURVEY.md 8(a) rows a4 (tile staging), a5 (trend predicate) and a6 (count
// accumulation) on the float32 columns / the 8-bit rank tiles.  (a3, the ingest, is ingest_kernels.cuh.)
//
// Definition (include/ebic.h): count[k] = #{ r : AND_i M[r][c_{i+1}] >= M[r][c_i]
// and, in missing mode, no M[r][c_i] is NaN }.  For L >= 2 an ordered >= is already false on NaN, so
// the chain kernels need no NaN test and no mode; L <= 1 has a closed form from the loader's
// per-column non-missing counts and is resolved by the ingest kernel.  Padding rows are NaN / 0x7F.
#pragma once
#include "ebic_device.cuh"

namespace ebic {

// ------------------------------------------------------------------------------------------------
// DIRECT kernel: one thread per row, column-major global loads, ballot + popc, one global atomic
// per warp and individual.  Any shape; the simple GPU witness the tiled kernels are diffed against.
// grid.x = ld / 256 row blocks, grid.y = population slices.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
fitness_direct_kernel(const float* __restrict__ Mc, int64_t ld, const int2* meta,
                      const int32_t* __restrict__ col_ids, int32_t n_ind,
                      unsigned long long* __restrict__ counts)
{
    griddep_wait();                                              // meta / counts come from the ingest kernel
    const int64_t r = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;   // < ld; padding is NaN
    const int lane = threadIdx.x & 31;
    const int32_t per = (n_ind + gridDim.y - 1) / gridDim.y;
    const int32_t k_begin = blockIdx.y * per;
    const int32_t k_end = min(n_ind, k_begin + per);
    for (int32_t k = k_begin; k < k_end; ++k) {
        const int2 m = ld_produced(&meta[k]);
        if (m.y < 2) continue;
        const int32_t* ids = col_ids + m.x;                      // validated by the ingest: every id inside [0, cols)
        float prev = Mc[static_cast<int64_t>(__ldg(&ids[0])) * ld + r];
        bool ok = true;
        for (int32_t i = 1; i < m.y; ++i) {
            const float cur = Mc[static_cast<int64_t>(__ldg(&ids[i])) * ld + r];
            ok = ok & (cur >= prev);
            prev = cur;
        }
        const unsigned int c = __popc(__ballot_sync(0xffffffffu, ok));
        if (lane == 0 && c) atomicAdd(&counts[k], static_cast<unsigned long long>(c));
    }
}

// ------------------------------------------------------------------------------------------------
// Tiled kernels (TILED_F32 and RANK8): persistent CTAs, one per SM.
//
// Work space = (row tile t, individual k) pairs in tile-major order; CTA b owns the contiguous
// range [P*b/G, P*(b+1)/G), P = n_tiles * n_ind: equal shares whatever the shape, and every tile is
// loaded by at most (its share of CTAs) + 1 CTAs.  Warp `n_cons` is the producer: for every tile of
// the CTA's range it waits for the buffer to be released, arms the "full" mbarrier with the tile's
// byte count and issues one TMA bulk copy per column (T contiguous rows of a column-major column).
// Consumer warps wait on "full", each takes every n_cons-th individual of the tile's range,
// evaluates it on all slabs of the tile, warp-reduces the count and adds it to the CTA's
// shared-memory counter of that individual; then releases the buffer ("empty" mbarrier, one arrival
// per consumer warp).  Counters are flushed with one 64-bit global atomic per (CTA, individual).
// Per-CTA counters are uint32: a CTA sees < 2^31 rows, so they cannot overflow.
// ------------------------------------------------------------------------------------------------
struct TiledParams {
    const void* M;                   // column-major [cols][ld] (float or uint8 rank codes)
    int64_t ld;
    int32_t cols;
    int32_t T;                       // rows per tile (multiple of the slab size)
    int32_t nbuf;                    // tile buffers: 2 (the next tile travels while this one is evaluated), or 1 when a
                                     // tile of all columns only fits once (wide matrices: loading is a few % of the work)
    int64_t n_tiles;                 // ceil(ld / T)
    const int2* meta;                // [n_ind] of this launch's population chunk
    const uint32_t* idrec;           // [n_ind][8] / [n_ind][16]: the first 32 ids of each individual as bytes / halfwords
    const int32_t* col_ids;          // the caller's ids: chromosomes with more than 32 columns continue from them
    int32_t n_ind;                   // individuals in this launch (<= kMaxIndPerLaunch)
    int32_t early_exit;              // stop a chain once no row of the warp's slab group is alive
    unsigned long long* counts;      // [n_ind]
    unsigned long long* visits;      // executed column visits (instrumented build) or nullptr
};

constexpr int kMaxIndPerLaunch = 8192;
constexpr int kRecIds = 32;          // ids held in an individual's id record (ingest_kernels.cuh)
constexpr int kSmemHeader = 128;     // 4 mbarriers, padded

__host__ __device__ inline size_t tiled_smem_bytes(int32_t cols, int32_t T, int32_t elem, int32_t n_ind, int32_t nbuf) {
    size_t cnt = (static_cast<size_t>(n_ind) * 4 + 127) & ~static_cast<size_t>(127);
    return kSmemHeader + cnt + nbuf * static_cast<size_t>(cols) * T * elem;
}

__device__ __forceinline__ uint32_t id_byte(uint32_t w, int b) {   // b is a compile-time constant: one PRMT
    return __byte_perm(w, 0, 0x4440 + b);
}

// ---- a5 on float32: 4 rows per lane and slab: one LDS.128 + 4 FSETP.GE.AND per column -----------
struct ChainF32 {
    uint32_t base;                   // shared address of tile + (slab * 128 + lane * 4) * 4
    uint32_t stride;                 // bytes between columns of the tile = T * 4
    float4 prev;
    bool p0, p1, p2, p3;
    __device__ __forceinline__ float4 load(uint32_t id) const {
        const uint4 v = lds128(id * stride + base);
        return make_float4(__uint_as_float(v.x), __uint_as_float(v.y), __uint_as_float(v.z), __uint_as_float(v.w));
    }
    __device__ __forceinline__ void init(uint32_t id) {
        prev = load(id);
        p0 = p1 = p2 = p3 = true;
    }
    __device__ __forceinline__ void step(uint32_t id) {
        const float4 cur = load(id);
        p0 = p0 & (cur.x >= prev.x);
        p1 = p1 & (cur.y >= prev.y);
        p2 = p2 & (cur.z >= prev.z);
        p3 = p3 & (cur.w >= prev.w);
        prev = cur;
    }
    __device__ __forceinline__ bool alive() const { return p0 | p1 | p2 | p3; }
    __device__ __forceinline__ int count() const {
        return static_cast<int>(p0) + static_cast<int>(p1) + static_cast<int>(p2) + static_cast<int>(p3);
    }
};

// ---- a5 on rank codes: 16 rows per lane and slab, NS slabs per id fetch -------------------------
// code = 0x80|rank (rank <= 126) or 0x7F (missing).  Per byte t = cur - prev + 0x80 stays in [1, 255] for
// every code pair, so the 32-bit IADD3 never carries between bytes.  Bit 7 of t:
//   value, value   : 0x80 + rank(cur) - rank(prev)      -> set iff rank(cur) >= rank(prev)
//   missing, value : 0x7F - rank(prev) in [1, 127]       -> clear (the pair fails, as an ordered >= does)
//   value, missing : 0x81 + rank(cur)                    -> set, but the chain has already failed:
//   missing,missing: 0x80                                -> set,  the FIRST missing column of a chain is
//                    either column 0 (acc starts as its code, bit 7 clear) or follows a value (case 2).
// acc = AND of all t (and the first code): bit 7 of each byte = ok(k, r) for that row.
template <int NS>
struct ChainR8 {
    static constexpr unsigned int H = 0x80808080u;
    uint32_t base;                   // shared address of tile + slab * 512 + lane * 16
    uint32_t stride;                 // bytes between columns of the tile = T
    uint4 prev[NS], acc[NS];
    __device__ __forceinline__ void init(uint32_t id) {
        const uint32_t col = id * stride + base;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            prev[s] = lds128(col + s * kRowsPerSlabR8);
            acc[s] = prev[s];
        }
    }
    __device__ __forceinline__ void step(uint32_t id) {
        const uint32_t col = id * stride + base;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const uint4 cur = lds128(col + s * kRowsPerSlabR8);
            acc[s].x &= cur.x - prev[s].x + H;
            acc[s].y &= cur.y - prev[s].y + H;
            acc[s].z &= cur.z - prev[s].z + H;
            acc[s].w &= cur.w - prev[s].w + H;
            prev[s] = cur;
        }
    }
    __device__ __forceinline__ bool alive() const {
        unsigned int any = 0;
#pragma unroll
        for (int s = 0; s < NS; ++s) any |= acc[s].x | acc[s].y | acc[s].z | acc[s].w;
        return (any & H) != 0;
    }
    __device__ __forceinline__ int count() const {
        int total = 0;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const unsigned int m = (acc[s].x & H) | ((acc[s].y & H) >> 1) | ((acc[s].z & H) >> 2) | ((acc[s].w & H) >> 3);
            total += __popc(m);
        }
        return total;
    }
};

// The ids of one individual.  Its id record (ingest_kernels.cuh) holds the first 32 ids, four per 32-bit word
// (cols <= 256) or two per word (wider matrices): one warp-uniform load per word.  A chromosome longer than the
// record continues, id by id, from the caller's int32 ids (a valid individual: every id is inside [0, cols)); that
// tail is kept out of the record loop so that the common case pays nothing for it.
struct IdWords {
    static constexpr int kPerWord = 4;
    const uint32_t* rec;             // idrec + 8 * k
    const int32_t* ids;              // col_ids + b
    __device__ __forceinline__ uint32_t word(int32_t j) const { return ld_produced(rec + j); }
    __device__ __forceinline__ uint32_t tail_id(int32_t i) const { return static_cast<uint32_t>(__ldg(ids + i)); }
};
struct IdWords16 {
    static constexpr int kPerWord = 2;
    const uint32_t* rec;             // idrec + 16 * k
    const int32_t* ids;
    __device__ __forceinline__ uint32_t word(int32_t j) const { return ld_produced(rec + j); }
    __device__ __forceinline__ uint32_t tail_id(int32_t i) const { return static_cast<uint32_t>(__ldg(ids + i)); }
};
// An id record that has been staged in shared memory (UNION_F32: admitted individuals have L <= 32, no tail).
struct IdWordsShared {
    static constexpr int kPerWord = 4;
    const uint32_t* rec;
    __device__ __forceinline__ uint32_t word(int32_t j) const { return rec[j]; }
    __device__ __forceinline__ uint32_t tail_id(int32_t) const { return 0u; }
};

// One chromosome on one slab group; w0 = first word of the id record (already loaded).  Full words run
// branch-free; the ragged last word goes id by id.  Returns the number of matching rows; adds the number of
// columns actually visited to `steps`.
// TAIL = false: the caller guarantees L <= kRecIds (the instantiation the hot path runs: the tail's code, when
// present in the same loop nest, cost the float32 kernel 6 % -- measured in round 2).
template <bool TAIL, class C, class IW>
__device__ __forceinline__ int run_chain(C& c, const IW& iw, uint32_t w0, int32_t L,
                                         bool early_exit, int32_t& steps)
{
    const int32_t Lr = TAIL ? min(L, kRecIds) : L;        // ids that live in the record
    int32_t done;
    bool dead = false;
    if constexpr (IW::kPerWord == 2) {                    // 16-bit ids, two per word
        uint32_t w = w0;
        uint32_t wn = (Lr > 2) ? iw.word(1) : 0u;
        c.init(w & 0xffffu);
        c.step(w >> 16);
        int32_t rem = Lr - 2, j = 1;
        done = 2;
        while (rem > 0) {
            if (early_exit && (j & 1) && !__any_sync(0xffffffffu, c.alive())) { dead = true; break; }
            w = wn;
            if (rem > 2) wn = iw.word(j + 1);
            ++j;
            c.step(w & 0xffffu);
            if (rem >= 2) c.step(w >> 16);
            done += min(rem, 2);
            rem -= 2;
        }
    } else {
        uint32_t w = w0;
        uint32_t wn = (Lr > 4) ? iw.word(1) : 0u;
        c.init(id_byte(w, 0));
        int32_t rem = Lr - 1;                             // steps still to do inside the record; L >= 2
        done = 1;
        {                                                 // bytes 1..3 of word 0
            c.step(id_byte(w, 1));
            if (rem >= 2) c.step(id_byte(w, 2));
            if (rem >= 3) c.step(id_byte(w, 3));
            const int32_t n0 = min(rem, 3);
            rem -= n0;
            done += n0;
        }
        int32_t j = 1;
        while (rem > 0) {
            if (early_exit && !__any_sync(0xffffffffu, c.alive())) { dead = true; break; }
            w = wn;
            if (rem > 4) wn = iw.word(j + 1);
            ++j;
            if (rem >= 4) {
                c.step(id_byte(w, 0));
                c.step(id_byte(w, 1));
                c.step(id_byte(w, 2));
                c.step(id_byte(w, 3));
                rem -= 4;
                done += 4;
            } else {
                c.step(id_byte(w, 0));
                if (rem >= 2) c.step(id_byte(w, 1));
                if (rem >= 3) c.step(id_byte(w, 2));
                done += rem;
                rem = 0;
            }
        }
    }
    if (TAIL && L > kRecIds && !dead) {                   // rare: the chromosome continues beyond its record
        for (int32_t i = kRecIds; i < L; ++i) {
            if (early_exit && (i & 3) == 0 && !__any_sync(0xffffffffu, c.alive())) break;
            c.step(iw.tail_id(i));
            ++done;
        }
    }
    steps += done;
    return c.count();
}

struct ElemF32 {
    using type = float;
    static constexpr int kSlabRows = kRowsPerSlabF32;
};
struct ElemR8 {
    using type = uint8_t;
    static constexpr int kSlabRows = kRowsPerSlabR8;
};

// All slabs of the tile for one individual.  Returns matches; `visited` += rows * columns actually visited.
template <bool TAIL, class IW>
__device__ __forceinline__ int eval_individual_on_tile(ElemF32, const float* tile, int32_t T, int32_t nslabs, int lane,
                                                        const IW& iw, uint32_t w0, int32_t L,
                                                        bool early_exit, unsigned long long& visited)
{
    int cnt = 0;
    int32_t steps = 0;
    for (int32_t s = 0; s < nslabs; ++s) {
        ChainF32 c;
        c.base = smem_u32(tile) + (s * kRowsPerSlabF32 + lane * 4) * 4;
        c.stride = static_cast<uint32_t>(T) * 4;
        cnt += run_chain<TAIL>(c, iw, w0, L, early_exit, steps);
    }
    visited += static_cast<unsigned long long>(steps) * kRowsPerSlabF32;
    return cnt;
}

template <bool TAIL, class IW>
__device__ __forceinline__ int eval_individual_on_tile(ElemR8, const uint8_t* tile, int32_t T, int32_t nslabs, int lane,
                                                        const IW& iw, uint32_t w0, int32_t L,
                                                        bool early_exit, unsigned long long& visited)
{
    int cnt = 0;
    int32_t s = 0;
    int32_t steps4 = 0, steps2 = 0, steps1 = 0;
    for (; s + 4 <= nslabs; s += 4) {
        ChainR8<4> c;
        c.base = smem_u32(tile) + s * kRowsPerSlabR8 + lane * 16;
        c.stride = static_cast<uint32_t>(T);
        cnt += run_chain<TAIL>(c, iw, w0, L, early_exit, steps4);
    }
    for (; s + 2 <= nslabs; s += 2) {
        ChainR8<2> c;
        c.base = smem_u32(tile) + s * kRowsPerSlabR8 + lane * 16;
        c.stride = static_cast<uint32_t>(T);
        cnt += run_chain<TAIL>(c, iw, w0, L, early_exit, steps2);
    }
    for (; s < nslabs; ++s) {
        ChainR8<1> c;
        c.base = smem_u32(tile) + s * kRowsPerSlabR8 + lane * 16;
        c.stride = static_cast<uint32_t>(T);
        cnt += run_chain<TAIL>(c, iw, w0, L, early_exit, steps1);
    }
    visited += static_cast<unsigned long long>(4 * steps4 + 2 * steps2 + steps1) * kRowsPerSlabR8;
    return cnt;
}

// IW = IdWords (byte ids, cols <= 256) or IdWords16 (16-bit ids, wider matrices).
template <class E, int NCONS, class IW>
__global__ void __launch_bounds__((NCONS + 1) * 32, 1)
fitness_tiled_kernel(const TiledParams p)
{
    constexpr int kRecWords = 32 / IW::kPerWord;                 // words of an id record
    using elem_t = typename E::type;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);          // [2]
    uint64_t* empty = full + 2;                                  // [2]
    uint32_t* s_cnt = reinterpret_cast<uint32_t*>(smem + kSmemHeader);
    const size_t cnt_bytes = (static_cast<size_t>(p.n_ind) * 4 + 127) & ~static_cast<size_t>(127);
    elem_t* tiles = reinterpret_cast<elem_t*>(smem + kSmemHeader + cnt_bytes);
    const size_t tile_elems = static_cast<size_t>(p.cols) * p.T;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t P = p.n_tiles * p.n_ind;
    const int64_t pb = P * blockIdx.x / gridDim.x;
    const int64_t pe = P * (blockIdx.x + 1) / gridDim.x;
    if (pb >= pe) return;                                        // CTA-uniform
    const int64_t t0 = pb / p.n_ind, t1 = (pe - 1) / p.n_ind;
    const int32_t ntl = static_cast<int32_t>(t1 - t0 + 1);

    for (int32_t k = tid; k < p.n_ind; k += blockDim.x) s_cnt[k] = 0;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_init(&empty[0], NCONS);
        mbar_init(&empty[1], NCONS);
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == NCONS) {
        // ---------------- producer warp (a4) ----------------
        const elem_t* M = reinterpret_cast<const elem_t*>(p.M);
        for (int32_t j = 0; j < ntl; ++j) {
            const int buf = j % p.nbuf;
            mbar_wait(&empty[buf], ((j / p.nbuf) & 1) ^ 1);      // passes immediately for j < nbuf
            const int64_t r0 = (t0 + j) * p.T;
            const int32_t nrows = static_cast<int32_t>(min(static_cast<int64_t>(p.T), p.ld - r0));
            const uint32_t col_bytes = static_cast<uint32_t>(nrows) * sizeof(elem_t);
            if (lane == 0) mbar_arrive_expect_tx(&full[buf], col_bytes * static_cast<uint32_t>(p.cols));
            __syncwarp();
            elem_t* dst = tiles + buf * tile_elems;
            for (int32_t c = lane; c < p.cols; c += 32)
                bulk_copy_g2s(dst + static_cast<size_t>(c) * p.T, M + static_cast<int64_t>(c) * p.ld + r0, col_bytes,
                              &full[buf]);
        }
        griddep_wait();                                          // before the count flush below
    } else {
        // ---------------- consumer warps (a5, a6) ----------------
        griddep_wait();                                          // meta / idrec / counts come from the ingest kernel;
                                                                 // the producer warp is already staging tiles
        unsigned long long visited = 0;
        const bool early_exit = p.early_exit != 0;
        for (int32_t j = 0; j < ntl; ++j) {
            const int buf = j % p.nbuf;
            const int64_t r0 = (t0 + j) * p.T;
            const int32_t nrows = static_cast<int32_t>(min(static_cast<int64_t>(p.T), p.ld - r0));
            const int32_t nslabs = nrows / E::kSlabRows;
            const int32_t ka = (j == 0) ? static_cast<int32_t>(pb - t0 * p.n_ind) : 0;
            const int32_t kb = (j == ntl - 1) ? static_cast<int32_t>(pe - t1 * p.n_ind) : p.n_ind;
            const elem_t* tile = tiles + buf * tile_elems;
            // software pipeline over this warp's individuals: meta and first id word one ahead
            int32_t k = ka + warp;
            int2 m_cur = make_int2(0, 0);
            uint32_t w_cur = 0;
            if (k < kb) {
                m_cur = ld_produced(&p.meta[k]);
                w_cur = ld_produced(p.idrec + static_cast<int64_t>(kRecWords) * k);
            }
            mbar_wait(&full[buf], (j / p.nbuf) & 1);
            for (; k < kb; k += NCONS) {
                const int2 m = m_cur;
                const uint32_t w0 = w_cur;
                if (k + NCONS < kb) {
                    m_cur = ld_produced(&p.meta[k + NCONS]);
                    w_cur = ld_produced(p.idrec + static_cast<int64_t>(kRecWords) * (k + NCONS));
                }
                if (m.y < 2) continue;
                const IW iw{p.idrec + static_cast<int64_t>(kRecWords) * k, p.col_ids + m.x};
                int cnt = (m.y <= kRecIds)                       // warp-uniform
                              ? eval_individual_on_tile<false>(E{}, tile, p.T, nslabs, lane, iw, w0, m.y, early_exit, visited)
                              : eval_individual_on_tile<true>(E{}, tile, p.T, nslabs, lane, iw, w0, m.y, early_exit, visited);
                cnt = __reduce_add_sync(0xffffffffu, cnt);
                if (lane == 0 && cnt) atomicAdd(&s_cnt[k], static_cast<unsigned int>(cnt));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[buf]);
        }
        if (p.visits != nullptr && lane == 0 && visited) atomicAdd(p.visits, visited);
    }
    __syncthreads();
    for (int32_t k = tid; k < p.n_ind; k += blockDim.x) {
        const unsigned int c = s_cnt[k];
        if (c) atomicAdd(&p.counts[k], static_cast<unsigned long long>(c));
    }
}

}  // namespace ebic
