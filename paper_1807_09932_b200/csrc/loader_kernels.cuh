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

// Pair bit columns.  Block = 8 warps; warp w of block (t, y) owns column a = 8*y + w on the 1024-row
// tile t: it keeps the tile's 1024 values of column a in registers (32 per lane, lane = row % 32) and
// walks every column b (coalesced 128 B loads, served by L1 for the other 7 warps of the block), turning
// each 32-row comparison into one ballot word; lane j keeps word j and the 32 words go out as one 128 B
// store into the bit column of pair (a, b).  grid = (ld / 1024, ceil(cols / 8)).
__global__ void __launch_bounds__(256)
pairbits_kernel(const float* __restrict__ Mc, int64_t ld, int32_t cols, uint32_t* __restrict__ PB)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t a = blockIdx.y * 8 + warp;
    if (a >= cols) return;
    const int64_t t = blockIdx.x;
    const float* tile = Mc + t * kPairTileRows + lane;
    float va[32];
    const float* ca = tile + static_cast<int64_t>(a) * ld;
#pragma unroll
    for (int j = 0; j < 32; ++j) va[j] = ca[32 * j];
    const int64_t ldw = ld / 32;
    uint32_t* out = PB + static_cast<int64_t>(a) * cols * ldw + t * 32 + lane;
    for (int32_t b = 0; b < cols; ++b) {
        const float* cb = tile + static_cast<int64_t>(b) * ld;
        unsigned int mine = 0;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            const unsigned int w = __ballot_sync(0xffffffffu, cb[32 * j] >= va[j]);
            if (lane == j) mine = w;
        }
        out[static_cast<int64_t>(b) * ldw] = mine;
    }
}

}  // namespace ebic
