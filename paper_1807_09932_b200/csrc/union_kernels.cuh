// union_kernels.cuh -- a4/a5/a6 for matrices too wide to stage whole: the COLUMN UNION of a batch of
// individuals (BASELINE.json north_star (3): "stages row tiles x all columns (or the population's column union)
// in shared memory"; the paper's 310-column shape).
//
// The population is cut into batches of `batch` consecutive individuals.  union_plan_kernel (one CTA per batch)
// walks the batch in order and admits an individual while the union of the admitted individuals' columns stays
// <= u_cap; it writes the batch's sorted column list, and for every admitted individual a 32-byte record of LOCAL
// column indices (position in that list).  An individual that is not admitted -- the union is full, or its
// chromosome is longer than the record's 32 ids -- is evaluated by the same warps straight from global memory.
// fitness_union_kernel: persistent CTAs (one per SM) over (row tile, batch) items in tile-major order, so the
// tile's columns stay in L2 while the batches pass over it and HBM reads the matrix about once.  Per item the
// producer warp stages the batch's U columns x kUnionTileRows rows, and the batch's id records, with 16-byte
// cp.async copies whose completion is counted on an mbarrier (double-buffered, full/empty pairs); each consumer warp takes every n_cons-th individual of the batch and runs the same
// float32 chain as the TILED_F32 kernel (4 rows per lane, LDS.128 + 4 FSETP.GE.AND per column) on local ids.
// Counts: warp reduce -> one global 64-bit atomic per (item, individual) with a non-zero count.
#pragma once
#include "ebic_device.cuh"
#include "fitness_kernels.cuh"

namespace ebic {

constexpr int kUnionTileRows = 128;          // one slab of the float32 chain: 4 rows per lane
constexpr int kUnionMaxCols = 65536;         // the plan kernel keeps a bit per column in shared memory
constexpr int kUnionCons = 16;               // consumer warps
constexpr int kUnionProd = 16;                // producer warps (512 threads in all)

struct UnionParams {
    const float* Mc;
    int64_t ld;
    int32_t cols;
    int32_t n_ind;
    int32_t batch;                   // individuals per batch
    int32_t n_batches;
    int32_t u_cap;                   // columns a staged tile can hold (double-buffered)
    const int2* meta;                // [n_ind] {b, L}; L = -1 invalid
    const int32_t* col_ids;
    int32_t* ucount;                 // [n_batches] columns of the batch's union
    int32_t* ucols;                  // [n_batches][u_cap] sorted column ids
    uint32_t* urec;                  // [n_ind][8]: 32 local byte ids; word 0 = 0xffffffff when not admitted
    int32_t early_exit;
    unsigned long long* counts;
    unsigned long long* visits;
};

// One CTA (256 threads) per batch.
__global__ void __launch_bounds__(256)
union_plan_kernel(const UnionParams p)
{
    extern __shared__ uint32_t plan_smem[];          // bitmap[words] then prefix[words]
    const int32_t words = (p.cols + 31) / 32;
    uint32_t* bitmap = plan_smem;
    uint32_t* prefix = plan_smem + words;
    __shared__ int32_t s_u;
    __shared__ uint8_t s_admit[256];
    griddep_wait();                                  // meta comes from the ingest kernel
    griddep_launch_dependents();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t k0 = blockIdx.x * p.batch, k1 = min(p.n_ind, k0 + p.batch);
    for (int32_t i = tid; i < words; i += 256) bitmap[i] = 0;
    if (tid == 0) s_u = 0;
    __syncthreads();
    if (warp == 0) {
        // in population order: admit while the union fits.  Newly set bits are rolled back when it does not.
        int32_t u = 0;
        for (int32_t k = k0; k < k1; ++k) {
            const int2 m = ld_produced(&p.meta[k]);
            bool admit = m.y >= 2 && m.y <= 32;
            if (admit) {
                const int32_t id = (lane < m.y) ? __ldg(p.col_ids + m.x + lane) : -1;
                bool fresh = false;
                if (id >= 0) {
                    const uint32_t bit = 1u << (id & 31);
                    fresh = !(atomicOr(&bitmap[id >> 5], bit) & bit);      // duplicates inside a chromosome: one wins
                }
                const int32_t n_new = __popc(__ballot_sync(0xffffffffu, fresh));
                if (u + n_new > p.u_cap) {
                    if (fresh) atomicAnd(&bitmap[id >> 5], ~(1u << (id & 31)));
                    admit = false;
                } else {
                    u += n_new;
                }
                __syncwarp();
            }
            if (lane == 0) s_admit[k - k0] = admit ? 1 : 0;
        }
        if (lane == 0) s_u = u;
    }
    __syncthreads();
    // exclusive prefix of the bitmap's popcounts (one warp; words <= 2,048)
    if (warp == 0) {
        int32_t run = 0;
        for (int32_t base = 0; base < words; base += 32) {
            const int32_t i = base + lane;
            const int32_t c = (i < words) ? __popc(bitmap[i]) : 0;
            int32_t inc = c;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int32_t t = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += t;
            }
            if (i < words) prefix[i] = run + inc - c;
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();
    if (tid == 0) p.ucount[blockIdx.x] = s_u;
    int32_t* ucols = p.ucols + static_cast<int64_t>(blockIdx.x) * p.u_cap;
    for (int32_t i = tid; i < words; i += 256) {
        uint32_t wbits = bitmap[i];
        int32_t pos = prefix[i];
        while (wbits) {
            const int b = __ffs(wbits) - 1;
            ucols[pos++] = i * 32 + b;
            wbits &= wbits - 1;
        }
    }
    // local ids: position of the column in the sorted list = set bits below it
    for (int32_t k = k0 + warp; k < k1; k += 8) {
        uint32_t local = 0;
        const bool admit = s_admit[k - k0] != 0;
        if (admit) {
            const int2 m = ld_produced(&p.meta[k]);
            const int32_t id = __ldg(p.col_ids + m.x + min(lane, m.y - 1));          // padded with the last id
            local = prefix[id >> 5] + __popc(bitmap[id >> 5] & ((1u << (id & 31)) - 1u));
        }
        const uint32_t i0 = __shfl_sync(0xffffffffu, local, (4 * lane) & 31), i1 = __shfl_sync(0xffffffffu, local, (4 * lane + 1) & 31);
        const uint32_t i2 = __shfl_sync(0xffffffffu, local, (4 * lane + 2) & 31), i3 = __shfl_sync(0xffffffffu, local, (4 * lane + 3) & 31);
        uint32_t word = i0 | (i1 << 8) | (i2 << 16) | (i3 << 24);
        if (!admit) word = 0xffffffffu;
        if (lane < 8) p.urec[8ll * k + lane] = word;
    }
}

// Shared memory of one buffer: the tile, then the batch's id records (32 bytes each) and meta entries (8 bytes
// each), which travel with the tile so that the consumers never wait on a global load.
__host__ __device__ inline size_t union_buffer_bytes(int32_t u_cap, int32_t batch) {
    return static_cast<size_t>(u_cap) * kUnionTileRows * sizeof(float) + static_cast<size_t>(batch) * 40;
}
__host__ __device__ inline size_t union_smem_bytes(int32_t u_cap, int32_t batch) {
    return kSmemHeader + 2 * union_buffer_bytes(u_cap, batch);
}

// Chain of one individual on 128 rows read straight from global memory (not admitted to its batch's union).
__device__ __forceinline__ int union_direct_chain(const float* __restrict__ Mc, int64_t ld, int64_t r0, int lane,
                                                  const int32_t* __restrict__ ids, int32_t L, bool early_exit, int32_t& steps)
{
    const float* base = Mc + r0 + lane * 4;
    float4 prev = __ldg(reinterpret_cast<const float4*>(base + static_cast<int64_t>(__ldg(ids)) * ld));
    bool p0 = true, p1 = true, p2 = true, p3 = true;
    int32_t i = 1;
    for (; i < L; ++i) {
        if (early_exit && (i & 3) == 0 && !__any_sync(0xffffffffu, p0 | p1 | p2 | p3)) break;
        const float4 cur = __ldg(reinterpret_cast<const float4*>(base + static_cast<int64_t>(__ldg(ids + i)) * ld));
        p0 = p0 & (cur.x >= prev.x);
        p1 = p1 & (cur.y >= prev.y);
        p2 = p2 & (cur.z >= prev.z);
        p3 = p3 & (cur.w >= prev.w);
        prev = cur;
    }
    steps += i;
    return static_cast<int>(p0) + static_cast<int>(p1) + static_cast<int>(p2) + static_cast<int>(p3);
}

template <int NCONS>
__global__ void __launch_bounds__((NCONS + kUnionProd) * 32, 1)
fitness_union_kernel(const UnionParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);          // [2]
    uint64_t* empty = full + 2;                                  // [2]
    unsigned char* buffers = smem + kSmemHeader;
    const size_t tile_bytes = static_cast<size_t>(p.u_cap) * kUnionTileRows * sizeof(float);
    const size_t buf_bytes = union_buffer_bytes(p.u_cap, p.batch);     // tile | records [batch][8] | meta [batch]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t n_tiles = p.ld / kUnionTileRows;
    const int64_t P = n_tiles * p.n_batches;                     // items, tile-major
    const int64_t pb = P * blockIdx.x / gridDim.x;
    const int64_t pe = P * (blockIdx.x + 1) / gridDim.x;
    if (tid == 0) {
        mbar_init(&full[0], kUnionProd * 32);                    // one arrival per producer lane, when its copies have landed
        mbar_init(&full[1], kUnionProd * 32);
        mbar_init(&empty[0], NCONS);
        mbar_init(&empty[1], NCONS);
        fence_mbar_init();
    }
    __syncthreads();
    griddep_wait();                                              // the plan (and the ingest before it) has completed

    if (warp >= NCONS) {
        const int pw = warp - NCONS;                             // producer warp pw copies columns pw, pw + 4, ...
        // ---------------- producer warps (a4): the batch's columns of this tile + the batch's records ----------------
        // 16-byte cp.async copies (LDGSTS), one 512-byte column run per warp instruction: 64 B/clk/SM, the rate of the
        // SM's L2 port.  (TMA bulk copies of 512 bytes were measured at ~64 cycles each, 8 B/clk: the round-2 first
        // version of this kernel spent 6.7 us per item in them.)
        for (int64_t it = pb; it < pe; ++it) {
            const int32_t j = static_cast<int32_t>(it - pb);
            const int buf = j & 1;
            const int64_t t = it / p.n_batches;
            const int32_t b = static_cast<int32_t>(it - t * p.n_batches);
            const int32_t U = ld_produced(&p.ucount[b]);
            const int32_t k0 = b * p.batch;
            const int32_t nb = min(p.n_ind, k0 + p.batch) - k0;
            mbar_wait(&empty[buf], ((j >> 1) & 1) ^ 1);          // passes immediately for j < 2
            const int32_t* ucols = p.ucols + static_cast<int64_t>(b) * p.u_cap;
            unsigned char* buffer = buffers + buf * buf_bytes;
            const uint32_t dst = smem_u32(buffer) + lane * 16;
            const float* src = p.Mc + t * kUnionTileRows + lane * 4;
            for (int32_t c0 = pw * 32; c0 < U; c0 += kUnionProd * 32) {
                const int32_t mine = (c0 + lane < U) ? ld_produced(ucols + c0 + lane) : 0;
                const int32_t n = min(32, U - c0);
                for (int32_t i = 0; i < n; ++i)
                    cp_async16(dst + (c0 + i) * (kUnionTileRows * 4), src + static_cast<int64_t>(__shfl_sync(0xffffffffu, mine, i)) * p.ld);
            }
            const uint32_t rec_dst = smem_u32(buffer + tile_bytes), meta_dst = rec_dst + p.batch * 32;
            const unsigned char* rec_src = reinterpret_cast<const unsigned char*>(p.urec + 8ll * k0);
            const unsigned char* meta_src = reinterpret_cast<const unsigned char*>(p.meta + k0);
            if (pw == 0) {
                for (int32_t u = lane; u < nb * 2; u += 32) cp_async16(rec_dst + u * 16, rec_src + u * 16);
                for (int32_t u = lane; u < (nb + 1) / 2; u += 32) cp_async16(meta_dst + u * 16, meta_src + u * 16);
            }
            cp_async_arrive_on(&full[buf]);
        }
    } else {
        // ---------------- consumer warps (a5, a6) ----------------
        unsigned long long visited = 0;
        const bool early_exit = p.early_exit != 0;
        for (int64_t it = pb; it < pe; ++it) {
            const int32_t j = static_cast<int32_t>(it - pb);
            const int buf = j & 1;
            const int64_t t = it / p.n_batches;
            const int32_t b = static_cast<int32_t>(it - t * p.n_batches);
            const int32_t k0 = b * p.batch, k1 = min(p.n_ind, k0 + p.batch);
            const unsigned char* buffer = buffers + buf * buf_bytes;
            const float* tile = reinterpret_cast<const float*>(buffer);
            const uint32_t* s_rec = reinterpret_cast<const uint32_t*>(buffer + tile_bytes);
            const int2* s_meta = reinterpret_cast<const int2*>(buffer + tile_bytes + static_cast<size_t>(p.batch) * 32);
            mbar_wait(&full[buf], (j >> 1) & 1);
            for (int32_t k = k0 + warp; k < k1; k += NCONS) {
                const int2 m = s_meta[k - k0];
                if (m.y < 2) continue;
                const IdWordsShared iw{s_rec + 8 * (k - k0)};                           // admitted: L <= 32, words 0..7 only
                const uint32_t w0 = iw.word(0);
                int cnt;
                int32_t steps = 0;
                if (w0 != 0xffffffffu) {
                    ChainF32 c;
                    c.base = smem_u32(tile) + lane * 16;
                    c.stride = kUnionTileRows * 4;
                    cnt = run_chain<false>(c, iw, w0, m.y, early_exit, steps);
                } else {
                    cnt = union_direct_chain(p.Mc, p.ld, t * kUnionTileRows, lane, p.col_ids + m.x, m.y, early_exit, steps);
                }
                visited += static_cast<unsigned long long>(steps) * kUnionTileRows;
                cnt = __reduce_add_sync(0xffffffffu, cnt);
                if (lane == 0 && cnt) atomicAdd(&p.counts[k], static_cast<unsigned long long>(cnt));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[buf]);
        }
        if (p.visits != nullptr && lane == 0 && visited) atomicAdd(p.visits, visited);
    }
}

}  // namespace ebic
