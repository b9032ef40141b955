// probe_kernels.cuh -- measurement utilities, not steps of the path (include/ebic_debug.h).  They measure the
// ceilings DESIGN.md 6.1 uses as roofline denominators on the GPU the benchmark runs on:
//   probe_read_kernel  L2 -> SM (buffer inside the 126 MB L2) or HBM (buffer far larger) read bandwidth with
//                      plain coalesced 128-bit loads that bypass L1, 16 independent loads per thread in flight;
//   probe_lds_kernel   conflict-free LDS.128 rate: the 128 B/clk/SM shared-memory data pipe of the tiled kernels;
//   probe_fsetp_kernel issue rate of ordered float32 compares (FSETP.GE), the other pipe of the TILED_F32 kernel.
#pragma once
#include "ebic_device.cuh"

namespace ebic {

constexpr int kProbeUnroll = 16;

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

// 1,024 threads, 64 KB of shared memory; lane l of every warp reads 16 bytes at (l * 16 + k * 512) mod 64 KB:
// a warp's request is 512 contiguous bytes = 4 conflict-free wavefronts.  8 independent LDS.128 per iteration.
__global__ void __launch_bounds__(1024, 1)
probe_lds_kernel(int32_t iters, unsigned int* __restrict__ sink)
{
    extern __shared__ __align__(16) unsigned char probe_smem[];
    uint4* s = reinterpret_cast<uint4*>(probe_smem);
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) s[i] = make_uint4(i, i + 1, i + 2, i + 3);
    __syncthreads();
    const uint32_t base = smem_u32(probe_smem);
    uint32_t off = (threadIdx.x & 31) * 16 + (threadIdx.x >> 5) * 2048;
    unsigned int acc = 0;
    for (int32_t it = 0; it < iters; ++it) {
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = lds128(base + ((off + u * 512) & 0xffffu));
#pragma unroll
        for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].w;
        off += 4096;
    }
    if (acc == 0x9e3779b9u) *sink = acc;
}

// 16 independent chains of setp.ge.and.f32 per iteration on register operands (one of which changes every
// iteration, so no compare is loop-invariant); 256 threads per block.
__global__ void __launch_bounds__(256)
probe_fsetp_kernel(int32_t iters, float a, float b, unsigned int* __restrict__ sink)
{
    const float x = a + threadIdx.x, y = b + threadIdx.x;
    unsigned int res;
    asm volatile(
        "{\n\t"
        ".reg .pred p<16>;\n\t"
        ".reg .pred q;\n\t"
        ".reg .s32 n;\n\t"
        ".reg .f32 fx, fy;\n\t"
        "mov.s32 n, %1;\n\t"
        "mov.f32 fx, %2;\n\t"
        "mov.f32 fy, %3;\n\t"
        "setp.ge.f32 p0, fx, fy;\n\t  setp.ge.f32 p1, fy, fx;\n\t  setp.ge.f32 p2, fx, fy;\n\t  setp.ge.f32 p3, fy, fx;\n\t"
        "setp.ge.f32 p4, fx, fy;\n\t  setp.ge.f32 p5, fy, fx;\n\t  setp.ge.f32 p6, fx, fy;\n\t  setp.ge.f32 p7, fy, fx;\n\t"
        "setp.ge.f32 p8, fx, fy;\n\t  setp.ge.f32 p9, fy, fx;\n\t  setp.ge.f32 p10, fx, fy;\n\t setp.ge.f32 p11, fy, fx;\n\t"
        "setp.ge.f32 p12, fx, fy;\n\t setp.ge.f32 p13, fy, fx;\n\t setp.ge.f32 p14, fx, fy;\n\t setp.ge.f32 p15, fy, fx;\n\t"
        "PROBE_FSETP_LOOP:\n\t"
        "setp.ge.and.f32 p0, fx, fy, p0;\n\t  setp.ge.and.f32 p1, fy, fx, p1;\n\t"
        "setp.ge.and.f32 p2, fx, fy, p2;\n\t  setp.ge.and.f32 p3, fy, fx, p3;\n\t"
        "setp.ge.and.f32 p4, fx, fy, p4;\n\t  setp.ge.and.f32 p5, fy, fx, p5;\n\t"
        "setp.ge.and.f32 p6, fx, fy, p6;\n\t  setp.ge.and.f32 p7, fy, fx, p7;\n\t"
        "setp.ge.and.f32 p8, fx, fy, p8;\n\t  setp.ge.and.f32 p9, fy, fx, p9;\n\t"
        "setp.ge.and.f32 p10, fx, fy, p10;\n\t setp.ge.and.f32 p11, fy, fx, p11;\n\t"
        "setp.ge.and.f32 p12, fx, fy, p12;\n\t setp.ge.and.f32 p13, fy, fx, p13;\n\t"
        "setp.ge.and.f32 p14, fx, fy, p14;\n\t setp.ge.and.f32 p15, fy, fx, p15;\n\t"
        "add.f32 fx, fx, 0f3F800000;\n\t"
        "sub.s32 n, n, 1;\n\t"
        "setp.gt.s32 q, n, 0;\n\t"
        "@q bra PROBE_FSETP_LOOP;\n\t"
        "and.pred p0, p0, p1;\n\t and.pred p2, p2, p3;\n\t and.pred p4, p4, p5;\n\t and.pred p6, p6, p7;\n\t"
        "and.pred p8, p8, p9;\n\t and.pred p10, p10, p11;\n\t and.pred p12, p12, p13;\n\t and.pred p14, p14, p15;\n\t"
        "and.pred p0, p0, p2;\n\t and.pred p4, p4, p6;\n\t and.pred p8, p8, p10;\n\t and.pred p12, p12, p14;\n\t"
        "and.pred p0, p0, p4;\n\t and.pred p8, p8, p12;\n\t and.pred p0, p0, p8;\n\t"
        "selp.u32 %0, 1, 0, p0;\n\t"
        "}"
        : "=r"(res)
        : "r"(iters), "f"(x), "f"(y));
    if (res != 0u) atomicAdd(sink, res);                        // data-dependent: the chains cannot be dropped
}

}  // namespace ebic
