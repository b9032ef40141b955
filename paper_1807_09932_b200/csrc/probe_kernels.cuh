// probe_kernels.cuh -- measurement utility, not a step of the path: the read bandwidth the SMs get from
// a buffer of a given size with plain coalesced 128-bit loads (8 independent LDG.128 per lane in flight,
// the same access shape as the PAIRBITS gather).  A buffer that fits the 126 MB L2 measures the L2 -> SM
// bandwidth, the roofline of the PAIRBITS kernel on matrices too wide for L1 residency;
// a buffer far larger than L2 measures HBM.  bench.py calls it through ebic_probe_read_bandwidth.
#pragma once
#include "ebic_device.cuh"

namespace ebic {

__global__ void __launch_bounds__(256)
probe_read_kernel(const uint4* __restrict__ buf, int64_t n_vec, int32_t reps, unsigned int* __restrict__ sink)
{
    const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
    const int64_t span = n_vec / (8 * stride) * (8 * stride);   // vectors every pass reads (host checks > 0)
    unsigned int acc = 0;
    for (int32_t r = 0; r < reps; ++r) {
        // a different rotation each pass, so no CTA re-reads the lines its L1 may still hold
        int64_t i = (static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x + static_cast<int64_t>(r) * 250112) % span;
        for (int64_t j = 0; j < span; j += 8 * stride) {
            uint4 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                int64_t a = i + j + u * stride;
                if (a >= span) a -= span;
                v[u] = __ldcg(buf + a);                        // L2 only: never allocates in L1
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
        }
    }
    if (acc == 0x9e3779b9u) *sink = acc;                        // keeps the loads alive
}

}  // namespace ebic
