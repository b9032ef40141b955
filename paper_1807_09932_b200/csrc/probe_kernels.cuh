// probe_kernels.cuh -- measurement utilities, not steps of the path (include/ebic_debug.h).  They measure the
// ceilings DESIGN.md 6.1 uses as roofline denominators on the GPU the benchmark runs on:
//   probe_read_kernel  L2 -> SM (buffer inside the 126 MB L2) or HBM (buffer far larger) read bandwidth with
//                      plain coalesced 128-bit loads that bypass L1, 16 independent loads per thread in flight;
//   probe_lds_kernel   conflict-free LDS.128 rate: the 128 B/clk/SM shared-memory data pipe of the tiled kernels;
//   probe_fsetp_kernel issue rate of ordered float32 compares (FSETP.GE), the other pipe of the TILED_F32 kernel;
//   probe_gather_kernel the PAIRTILE access pattern on its own: every lane reads its own pseudo-random 128-byte slot
//                      of a 128 KB shared-memory tile as eight LDS.128, the 16-byte unit rotated per lane (or not:
//                      `rotate` = 0 shows the 8-way bank conflicts the rotation removes), AND + popcount as in the
//                      kernel, no staging and no records.
#pragma once
#include "ebic_device.cuh"

namespace ebic {

constexpr int kProbeUnroll = 16;

// volatile: ptxas may neither drop a repeated read of the same shared address nor narrow the vector
__device__ __forceinline__ uint4 probe_lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

// Thread i of the grid reads vectors i, i + S, i + 2S, ... (S = grid size) of buf[0, n_vec): every pass reads the
// whole buffer exactly once, each warp 512 contiguous bytes per load.  n_vec must be a multiple of kProbeUnroll * S.
__global__ void __launch_bounds__(256)
probe_read_kernel(const uint4* __restrict__ buf, int64_t n_vec, int32_t reps, unsigned int* __restrict__ sink)
{
    const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
    const uint4* mine = buf + static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int64_t iters = n_vec / (kProbeUnroll * stride);
    unsigned int acc = 0;
    for (int32_t r = 0; r < reps; ++r) {
        const uint4* p = mine;
        for (int64_t j = 0; j < iters; ++j, p += kProbeUnroll * stride) {
            uint4 v[kProbeUnroll];
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u) v[u] = __ldcg(p + u * stride);   // L2 only: never allocates in L1
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
        }
    }
    if (acc == 0x9e3779b9u) *sink = acc;                        // keeps the loads alive
}

// 1,024 threads, 64 KB of shared memory; lane l of warp w reads 16 bytes at w * 2048 + u * 512 + l * 16 (+ a
// per-iteration rotation): a warp's request is 512 contiguous bytes = 4 conflict-free wavefronts.  8 independent
// LDS.128 per iteration, every loaded word used (ptxas narrows a vector load whose components are dead).
__global__ void __launch_bounds__(1024, 1)
probe_lds_kernel(int32_t iters, unsigned int* __restrict__ sink)
{
    extern __shared__ __align__(16) unsigned char probe_smem[];
    uint4* s = reinterpret_cast<uint4*>(probe_smem);
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) s[i] = make_uint4(i, i + 1, i + 2, i + 3);
    __syncthreads();
    const uint32_t a0 = smem_u32(probe_smem) + (threadIdx.x & 31) * 16 + (threadIdx.x >> 5) * 2048;
    const uint32_t a1 = smem_u32(probe_smem) + (threadIdx.x & 31) * 16 + ((threadIdx.x >> 5) ^ 16) * 2048;
    uint4 acc = make_uint4(0u, 0u, 0u, 0u);
    for (int32_t it = 0; it < iters; it += 2) {
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = probe_lds128(a0 + u * 512);
#pragma unroll
        for (int u = 0; u < 4; ++u) v[4 + u] = probe_lds128(a1 + u * 512);
#pragma unroll
        for (int u = 0; u < 8; u += 2) { acc.x ^= v[u].x ^ v[u + 1].x; acc.y ^= v[u].y ^ v[u + 1].y; acc.z ^= v[u].z ^ v[u + 1].z; acc.w ^= v[u].w ^ v[u + 1].w; }
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = probe_lds128(a1 + u * 512);
#pragma unroll
        for (int u = 0; u < 4; ++u) v[4 + u] = probe_lds128(a0 + u * 512);
#pragma unroll
        for (int u = 0; u < 8; u += 2) { acc.x ^= v[u].x ^ v[u + 1].x; acc.y ^= v[u].y ^ v[u + 1].y; acc.z ^= v[u].z ^ v[u + 1].z; acc.w ^= v[u].w ^ v[u + 1].w; }
    }
    if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x9e3779b9u) *sink = acc.x;
}

// 512 threads, 128 KB of shared memory = 1,024 slots of 128 bytes.  Per iteration a lane ANDs the 1,024 "rows" of
// 8 slots (two per step, as fitness_pairtile_kernel does) into 32 accumulator registers and popcounts them.
__global__ void __launch_bounds__(512, 1)
probe_gather_kernel(int32_t iters, int32_t rotate, unsigned int* __restrict__ sink)
{
    extern __shared__ __align__(128) unsigned char probe_smem[];
    for (int i = threadIdx.x; i < 32768; i += blockDim.x) reinterpret_cast<uint32_t*>(probe_smem)[i] = ~0u ^ ((i * 2654435761u) >> 31);
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const uint32_t base = smem_u32(probe_smem) + (rotate ? ((lane & 7) << 4) : 0u);
    uint32_t state = threadIdx.x * 747796405u + blockIdx.x * 2891336453u + 1u;
    unsigned int cnt = 0;
    for (int32_t it = 0; it < iters; ++it) {
        uint4 acc[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] = make_uint4(~0u, ~0u, ~0u, ~0u);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            state = state * 1664525u + 1013904223u;
            const uint32_t a = base + ((state >> 12) & 1023u) * 128u, b = base + ((state >> 22) & 1023u) * 128u;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint4 v = lds128(a ^ (u << 4)), w = lds128(b ^ (u << 4));
                acc[u].x &= v.x & w.x; acc[u].y &= v.y & w.y; acc[u].z &= v.z & w.z; acc[u].w &= v.w & w.w;
            }
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) cnt += __popc(acc[u].x) + __popc(acc[u].y) + __popc(acc[u].z) + __popc(acc[u].w);
    }
    if (cnt == 0x9e3779b9u) *sink = cnt;
}

// Six independent chains of setp.ge.and.f32 (the form of the TILED_F32 inner loop: p = p & (cur >= prev)) per
// thread -- the hardware has seven predicate registers --, unrolled 8 times; 256 threads per block.
__global__ void __launch_bounds__(256)
probe_fsetp_kernel(int32_t iters, float a, float b, unsigned int* __restrict__ sink)
{
    const float x = a + threadIdx.x, y = b + threadIdx.x;
    unsigned int res;
#define EBIC_FSETP6 \
        "setp.ge.and.f32 p0, fx, fy, p0;\n\t setp.ge.and.f32 p1, fy, fx, p1;\n\t setp.ge.and.f32 p2, fx, fz, p2;\n\t" \
        "setp.ge.and.f32 p3, fz, fx, p3;\n\t setp.ge.and.f32 p4, fy, fz, p4;\n\t setp.ge.and.f32 p5, fz, fy, p5;\n\t"
    asm volatile(
        "{\n\t"
        ".reg .pred p<6>;\n\t"
        ".reg .pred q;\n\t"
        ".reg .s32 n;\n\t"
        ".reg .f32 fx, fy, fz;\n\t"
        "mov.s32 n, %1;\n\t"
        "mov.f32 fx, %2;\n\t"
        "mov.f32 fy, %3;\n\t"
        "add.f32 fz, fx, fy;\n\t"
        "setp.ge.f32 p0, fx, fy;\n\t setp.ge.f32 p1, fy, fx;\n\t setp.ge.f32 p2, fx, fz;\n\t"
        "setp.ge.f32 p3, fz, fx;\n\t setp.ge.f32 p4, fy, fz;\n\t setp.ge.f32 p5, fz, fy;\n\t"
        "PROBE_FSETP_LOOP:\n\t"
        EBIC_FSETP6 EBIC_FSETP6 EBIC_FSETP6 EBIC_FSETP6 EBIC_FSETP6 EBIC_FSETP6 EBIC_FSETP6 EBIC_FSETP6
        "add.f32 fx, fx, 0f3F800000;\n\t"
        "sub.s32 n, n, 1;\n\t"
        "setp.gt.s32 q, n, 0;\n\t"
        "@q bra PROBE_FSETP_LOOP;\n\t"
        "and.pred p0, p0, p1;\n\t and.pred p2, p2, p3;\n\t and.pred p4, p4, p5;\n\t"
        "and.pred p0, p0, p2;\n\t and.pred p0, p0, p4;\n\t"
        "selp.u32 %0, 1, 0, p0;\n\t"
        "}"
        : "=r"(res)
        : "r"(iters), "f"(x), "f"(y));
#undef EBIC_FSETP6
    if (res != 0u) atomicAdd(sink, res);                        // data-dependent: the chains cannot be dropped
}

}  // namespace ebic
