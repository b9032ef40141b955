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
// producer warp stages the batch's U columns x kUnionTileRows rows with TMA bulk copies (double-buffered,
// mbarrier full/empty pairs); each consumer warp takes every n_cons-th individual of the batch and runs the same
// float32 chain as the TILED_F32 kernel (4 rows per lane, LDS.128 + 4 FSETP.GE.AND per column) on local ids.
// Counts: warp reduce -> one global 64-bit atomic per (item, individual) with a non-zero count.
#pragma once
#include "ebic_device.cuh"
#include "fitness_kernels.cuh"

namespace ebic {

constexpr int kUnionTileRows = 128;          // one slab of the float32 chain: 4 rows per lane
constexpr int kUnionMaxCols = 65536;         // the plan kernel keeps a bit per column in shared memory
constexpr int kUnionCons = 15;               // consumer warps (+1 producer = 512 threads)

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
            const int2 m = __ldg(&p.meta[k]);
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
            const int2 m = __ldg(&p.meta[k]);
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

__host__ __device__ inline size_t union_smem_bytes(int32_t u_cap) {
    return kSmemHeader + 2 * static_cast<size_t>(u_cap) * kUnionTileRows * sizeof(float);
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
__global__ void __launch_bounds__((NCONS + 1) * 32, 1)
fitness_union_kernel(const UnionParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);          // [2]
    uint64_t* empty = full + 2;                                  // [2]
    float* tiles = reinterpret_cast<float*>(smem + kSmemHeader);
    const size_t tile_elems = static_cast<size_t>(p.u_cap) * kUnionTileRows;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t n_tiles = p.ld / kUnionTileRows;
    const int64_t P = n_tiles * p.n_batches;                     // items, tile-major
    const int64_t pb = P * blockIdx.x / gridDim.x;
    const int64_t pe = P * (blockIdx.x + 1) / gridDim.x;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_init(&empty[0], NCONS);
        mbar_init(&empty[1], NCONS);
        fence_mbar_init();
    }
    __syncthreads();
    griddep_wait();                                              // the plan (and the ingest before it) has completed

    if (warp == NCONS) {
        // ---------------- producer warp (a4): the batch's columns of this tile ----------------
        for (int64_t it = pb; it < pe; ++it) {
            const int32_t j = static_cast<int32_t>(it - pb);
            const int buf = j & 1;
            const int64_t t = it / p.n_batches;
            const int32_t b = static_cast<int32_t>(it - t * p.n_batches);
            const int32_t U = __ldg(&p.ucount[b]);
            mbar_wait(&empty[buf], ((j >> 1) & 1) ^ 1);          // passes immediately for j < 2
            if (lane == 0) mbar_arrive_expect_tx(&full[buf], static_cast<uint32_t>(U) * kUnionTileRows * 4u);
            __syncwarp();
            const int32_t* ucols = p.ucols + static_cast<int64_t>(b) * p.u_cap;
            float* dst = tiles + buf * tile_elems;
            const float* src = p.Mc + t * kUnionTileRows;
            for (int32_t c = lane; c < U; c += 32)
                bulk_copy_g2s(dst + static_cast<size_t>(c) * kUnionTileRows, src + static_cast<int64_t>(__ldg(ucols + c)) * p.ld,
                              kUnionTileRows * 4u, &full[buf]);
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
            const float* tile = tiles + buf * tile_elems;
            mbar_wait(&full[buf], (j >> 1) & 1);
            for (int32_t k = k0 + warp; k < k1; k += NCONS) {
                const int2 m = __ldg(&p.meta[k]);
                if (m.y < 2) continue;
                const uint32_t w0 = __ldg(p.urec + 8ll * k);
                int cnt;
                int32_t steps = 0;
                if (w0 != 0xffffffffu) {
                    ChainF32 c;
                    c.base = smem_u32(tile) + lane * 16;
                    c.stride = kUnionTileRows * 4;
                    const IdWords iw{p.urec + 8ll * k, p.col_ids + m.x, m.y};          // admitted: L <= 32, words 0..7 only
                    cnt = run_chain(c, iw, w0, m.y, early_exit, steps);
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
