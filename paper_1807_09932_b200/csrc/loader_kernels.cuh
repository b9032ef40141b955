// loader_kernels.cuh -- SURVEY.md 8(a) rows a1/a2 (+ the rank tiles of the RANK8 path).
//   a1  transpose the user's row-major float32 matrix to column-major Mc[cols][ld], ld = rows
//       rounded up to 1024, padding rows = NaN (so padding can never match an L >= 2 chromosome);
//   a2  packed NaN bitmask uint32[cols][ld/32] and per-column non-missing counts (PAPER.md line 60:
//       missing values must not count);
//   a2' rank tiles uint8[cols][ld]: per row, code(c) = 0x80 | #{c' : M[r][c'] < M[r][c]} for a value,
//       0x7F for NaN.  a >= b on float32 (ordered)  <=>  both codes have bit 7 set and
//       code(a) >= code(b): the trend predicate depends only on the within-row order, so the
//       fitness kernel can compare 4 rows per 32-bit word.
//   a2" pair-relation bit columns PB[pair][ld/32 words], pair (a,b) = a*cols + b (pair-major: the bit
//       column of a pair is contiguous): bit (r % 32) of word r / 32 = ( M[r][b] >= M[r][a] ), ordered
//       float32 >=.  An L >= 2 chromosome matches row r iff all its L-1 consecutive pair bits are set, so
//       the fitness kernel ANDs bit columns: 1 bit per (row, pair) instead of an 8-bit rank per (row,
//       column).  The diagonal (a,a) is "not NaN"; padding rows are NaN, so their bits are 0.
// All HBM-bound, run once per ebic_create.
#pragma once
#include "ebic_device.cuh"

namespace ebic {

// block (32, 8); tile = 32 rows x 32 cols.  src: row-major chunk [chunk_rows][cols], whose first row is
// global row `row0`.  grid.x = ceil(chunk_rows / 32), grid.y = ceil(cols / 32).
__global__ void __launch_bounds__(256)
transpose_pad_kernel(const float* __restrict__ src, float* __restrict__ Mc, int64_t row0,
                     int64_t chunk_rows, int32_t cols, int64_t ld, int32_t use_sentinel, float sentinel)
{
    __shared__ float tile[32][33];
    const int64_t r0 = static_cast<int64_t>(blockIdx.x) * 32;
    for (int32_t c0 = blockIdx.y * 32; c0 < cols; c0 += gridDim.y * 32) {
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
            const int64_t r = r0 + threadIdx.y + j;
            const int32_t c = c0 + threadIdx.x;
            if (r < chunk_rows && c < cols) {
                // a file marks missing cells with a numeric value (e.g. 0 or 999); here it becomes
                // NaN, the ABI's missing marker (float ==, so a sentinel of 0 also maps -0)
                const float v = src[r * cols + c];
                tile[threadIdx.y + j][threadIdx.x] = (use_sentinel && v == sentinel) ? __uint_as_float(0x7fc00000u) : v;
            }
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
            const int32_t c = c0 + threadIdx.y + j;
            const int64_t r = r0 + threadIdx.x;
            if (r < chunk_rows && c < cols) Mc[static_cast<int64_t>(c) * ld + row0 + r] = tile[threadIdx.x][threadIdx.y + j];
        }
        __syncthreads();
    }
}

// Padding rows [rows, ld) of every column <- NaN.  One thread per (column, padding row).
__global__ void __launch_bounds__(256)
fill_pad_kernel(float* __restrict__ Mc, int64_t rows, int32_t cols, int64_t ld)
{
    const int64_t pad = ld - rows;
    const int64_t n = pad * cols;
    for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n;
         i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        const int64_t c = i / pad, r = rows + i % pad;
        Mc[c * ld + r] = __uint_as_float(0x7fc00000u);
    }
}

// One warp per 32 rows of one column: ballot of the NaN test -> one mask word.
// grid.x over row chunks of 256*32 rows, grid.y over columns (strided).
__global__ void __launch_bounds__(256)
nan_mask_kernel(const float* __restrict__ Mc, int64_t ld, int32_t cols, uint32_t* __restrict__ mask,
                unsigned long long* __restrict__ nonmissing)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t words = ld / 32;
    for (int32_t c = blockIdx.y; c < cols; c += gridDim.y) {
        const float* col = Mc + static_cast<int64_t>(c) * ld;
        unsigned int present = 0;
        const int64_t w_begin = static_cast<int64_t>(blockIdx.x) * 256 + warp * 32;
        for (int64_t w = w_begin; w < w_begin + 32 && w < words; ++w) {
            const bool nan = is_nan_bits(col[w * 32 + lane]);
            const unsigned int bits = __ballot_sync(0xffffffffu, nan);
            if (lane == 0) mask[static_cast<int64_t>(c) * words + w] = bits;
            present += 32 - __popc(bits);
        }
        if (lane == 0 && present) atomicAdd(&nonmissing[c], static_cast<unsigned long long>(present));
    }
}

// Rank tiles.  Block = 256 threads = 256 consecutive rows; dynamic smem = cols*256*4 (values)
// + cols*256 (codes).  grid.x = ld / 256.
__global__ void __launch_bounds__(256)
rank8_kernel(const float* __restrict__ Mc, int64_t ld, int32_t cols, uint8_t* __restrict__ Rk)
{
    extern __shared__ __align__(16) unsigned char rk_smem[];
    float* vals = reinterpret_cast<float*>(rk_smem);                 // [cols][256]
    uint8_t* codes = rk_smem + static_cast<size_t>(cols) * 256 * 4;   // [cols][256]
    const int tid = threadIdx.x;
    const int64_t r0 = static_cast<int64_t>(blockIdx.x) * 256;
    for (int c = 0; c < cols; ++c) vals[c * 256 + tid] = Mc[static_cast<int64_t>(c) * ld + r0 + tid];
    // each thread only reads back its own column of `vals`: no barrier needed before this loop
    for (int c = 0; c < cols; ++c) {
        const float v = vals[c * 256 + tid];
        unsigned int below = 0;
        for (int c2 = 0; c2 < cols; ++c2) below += (vals[c2 * 256 + tid] < v) ? 1u : 0u;  // ordered <: NaN never counts
        codes[c * 256 + tid] = is_nan_bits(v) ? static_cast<uint8_t>(kRankNaN) : static_cast<uint8_t>(0x80u | below);
    }
    __syncthreads();
    // coalesced write-out, 4 codes per thread per step
    const uint32_t* codes32 = reinterpret_cast<const uint32_t*>(codes);
    for (int i = tid; i < cols * 64; i += 256) {
        const int c = i >> 6, w = i & 63;
        reinterpret_cast<uint32_t*>(Rk + static_cast<int64_t>(c) * ld + r0)[w] = codes32[c * 64 + w];
    }
}

// Pair bit columns (a2").  A lane OWNS one output word: lane l of a warp produces the word of rows
// [1024 t + 32 l, + 32) of the bit column of pair (a, b), so a warp's 32 words are one coalesced 128-byte store
// -- no ballots.  A bit costs two instructions on two different pipes: d = b - a (FADD) and a funnel shift that
// moves d's sign bit into the word (SHF).  Why the sign of the float32 difference IS the ordered comparison
// (DESIGN.md section 5): for two numbers b - a is negative iff b < a -- the subtraction is exact in sign (no
// flush-to-zero: two distinct floats never give 0), inf - inf is the positive canonical NaN (">=" holds), and
// the one wrong case, (-0) - (+0) = -0, is removed by turning every zero of the `a` column into -0 once
// ((+0) - (-0) = (-0) - (-0) = +0).  A NaN operand is taken from the loader's NaN bitmask (one 128-byte load per
// column and warp): the word is ANDed with "both present".  A warp keeps its two `a` columns in registers
// (32 consecutive rows per lane each) and walks every column b; the b columns of the tile are staged through
// shared memory in groups of kPairCB with cp.async, double-buffered, in a padded layout (a lane's 128 bytes start
// every 144 bytes) that makes the lanes' 16-byte reads conflict-free.
// Block = 8 warps = 16 `a` columns on one 1,024-row tile; grid = (ld / 1024) * ceil(cols / 16) blocks, the `a`
// group fastest, so the blocks that share a tile's b columns run together and HBM sees the matrix about once.
constexpr int kPairCB = 8;                       // b columns per stage
constexpr int kPairLaneStride = 144;             // bytes between two lanes' 32-row runs in the staged copy
constexpr int kPairColBytes = 32 * kPairLaneStride;          // 4,608
constexpr int kPairStageBytes = kPairCB * kPairColBytes;     // 36,864; two stages

// `va0` / `va1`: zeros already turned into -0.  w0 / w1 bit j = !(vb[j] < va[j]) for numbers (garbage where either
// is NaN).  The two words are built together: two independent FADD -> SHF chains per warp.
__device__ __forceinline__ void pair_words(const float (&va0)[32], const float (&va1)[32], const float (&vb)[32],
                                           uint32_t& w0, uint32_t& w1) {
    uint32_t x0 = 0, x1 = 0;
#pragma unroll
    for (int j = 31; j >= 0; --j) {
        x0 = __funnelshift_l(__float_as_uint(vb[j] - va0[j]), x0, 1);          // x = x << 1 | sign(b - a)
        x1 = __funnelshift_l(__float_as_uint(vb[j] - va1[j]), x1, 1);
    }
    w0 = ~x0;
    w1 = ~x1;
}

__global__ void __launch_bounds__(256, 2)
pairbits_kernel(const float* __restrict__ Mc, const uint32_t* __restrict__ nanmask, int64_t ld, int32_t cols,
                uint32_t* __restrict__ PB, uint32_t* __restrict__ PBT)
{
    extern __shared__ __align__(16) unsigned char pb_stage[];   // 2 x kPairStageBytes
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t n_groups = (cols + 15) / 16;
    const int64_t t = blockIdx.x / n_groups;
    const int32_t a0 = static_cast<int32_t>(blockIdx.x % n_groups) * 16 + 2 * warp, a1 = a0 + 1;
    const float* tile = Mc + t * kPairTileRows;
    const int64_t ldw = ld / 32;

    float va0[32], va1[32];
    {
        const float4* c0 = reinterpret_cast<const float4*>(tile + static_cast<int64_t>(min(a0, cols - 1)) * ld) + 8 * lane;
        const float4* c1 = reinterpret_cast<const float4*>(tile + static_cast<int64_t>(min(a1, cols - 1)) * ld) + 8 * lane;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const float4 x = __ldg(c0 + q), y = __ldg(c1 + q);
            va0[4 * q] = x.x; va0[4 * q + 1] = x.y; va0[4 * q + 2] = x.z; va0[4 * q + 3] = x.w;
            va1[4 * q] = y.x; va1[4 * q + 1] = y.y; va1[4 * q + 2] = y.z; va1[4 * q + 3] = y.w;
        }
#pragma unroll
        for (int j = 0; j < 32; ++j) {                           // +0 / -0 -> -0 (see the header)
            va0[j] = (va0[j] == 0.0f) ? -0.0f : va0[j];
            va1[j] = (va1[j] == 0.0f) ? -0.0f : va1[j];
        }
    }
    // "present" words of this lane's 32 rows: the NaN bitmask is [cols][ld / 32], bit set = missing
    const uint32_t* nan_t = nanmask + t * 32 + lane;
    const uint32_t pa0 = ~__ldg(nan_t + static_cast<int64_t>(min(a0, cols - 1)) * ldw);
    const uint32_t pa1 = ~__ldg(nan_t + static_cast<int64_t>(min(a1, cols - 1)) * ldw);
    const uint32_t stage0 = smem_u32(pb_stage);
    // thread `tid` copies 16-byte unit `tid` (rows 4 tid .. 4 tid + 3) of each staged column
    const uint32_t my_dst = (tid >> 3) * kPairLaneStride + (tid & 7) * 16;
    auto stage = [&](int32_t b0, int buf) {
#pragma unroll
        for (int c = 0; c < kPairCB; ++c)
            if (b0 + c < cols)
                cp_async16(stage0 + buf * kPairStageBytes + c * kPairColBytes + my_dst,
                           tile + static_cast<int64_t>(b0 + c) * ld + 4 * tid);
        cp_async_commit();
    };
    // running pointers: the words of pairs (a0, b) / (a1, b) and the NaN word of column b, b = 0, 1, 2, ...
    uint32_t* out0 = PB + static_cast<int64_t>(min(a0, cols - 1)) * cols * ldw + t * 32 + lane;
    uint32_t* out1 = PB + static_cast<int64_t>(min(a1, cols - 1)) * cols * ldw + t * 32 + lane;
    // optional second copy, TILE-major PBT[tile][pair][32 words] (pairtile_kernels.cuh stages whole tiles): the
    // same 128-byte store, 128 bytes further on for every b
    const bool tiled = PBT != nullptr;
    uint32_t* tout0 = PBT + (t * cols * cols + static_cast<int64_t>(min(a0, cols - 1)) * cols) * 32 + lane;
    uint32_t* tout1 = PBT + (t * cols * cols + static_cast<int64_t>(min(a1, cols - 1)) * cols) * 32 + lane;
    const uint32_t* nan_b = nan_t;
    const bool do0 = a0 < cols, do1 = a1 < cols;
    const int32_t n_stage = (cols + kPairCB - 1) / kPairCB;
    stage(0, 0);
    uint32_t pb_next = ~__ldg(nan_b);                            // "present" word of column b, fetched one column ahead
    for (int32_t s = 0; s < n_stage; ++s) {
        if (s + 1 < n_stage) {
            stage((s + 1) * kPairCB, (s + 1) & 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            cp_async_wait_all();
        }
        __syncthreads();                                         // every thread's share of stage s has landed
        uint32_t src = stage0 + (s & 1) * kPairStageBytes + lane * kPairLaneStride;
        const int32_t b_end = min(kPairCB, cols - s * kPairCB);
        for (int32_t c = 0; c < b_end; ++c, src += kPairColBytes, out0 += ldw, out1 += ldw, tout0 += 32, tout1 += 32, nan_b += ldw) {
            float vb[32];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const uint4 x = lds128(src + q * 16);
                vb[4 * q] = __uint_as_float(x.x); vb[4 * q + 1] = __uint_as_float(x.y);
                vb[4 * q + 2] = __uint_as_float(x.z); vb[4 * q + 3] = __uint_as_float(x.w);
            }
            const uint32_t pb = pb_next;
            if (s * kPairCB + c + 1 < cols) pb_next = ~__ldg(nan_b + ldw);
            uint32_t w0, w1;
            pair_words(va0, va1, vb, w0, w1);
            w0 &= pa0 & pb;
            w1 &= pa1 & pb;
            if (do0) *out0 = w0;
            if (do1) *out1 = w1;
            if (tiled && do0) *tout0 = w0;
            if (tiled && do1) *tout1 = w1;
        }
        __syncthreads();                                         // stage s may be overwritten by stage s + 2
    }
}

}  // namespace ebic
