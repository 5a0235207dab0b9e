// fp_probe.cuh -- read-bandwidth probes of the measurement harness ("L2 and L1 peaks come
// from a small read microbenchmark in the harness"; the paper's own metric is a cache-level access rate,
// PAPER.md:314, :351).  Not on the hot path: bench.py reports the projector's L2 and shared-memory rates
// against what these kernels reach on the same device.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace fpk {

// Streams `n4` float4 from `src` (grid-stride, `reps` passes) through L2 only (ld.global.cg bypasses L1).
// With a buffer that fits L2 this is the L2 -> SM read rate; with one that does not, the HBM read rate.
__global__ void __launch_bounds__(512)
fp_probe_read_kernel(const float4 *__restrict__ src, size_t n4, int reps, float *sink)
{
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        // four independent loads in flight per thread
        for (; i + 3 * stride < n4; i += 4 * stride) {
            const float4 a = __ldcg(src + i), b = __ldcg(src + i + stride), c = __ldcg(src + i + 2 * stride),
                         d = __ldcg(src + i + 3 * stride);
            acc.x += a.x + b.x + c.x + d.x;
            acc.y += a.y + b.y + c.y + d.y;
            acc.z += a.z + b.z + c.z + d.z;
            acc.w += a.w + b.w + c.w + d.w;
        }
        for (; i < n4; i += stride) {
            const float4 a = __ldcg(src + i);
            acc.x += a.x; acc.y += a.y; acc.z += a.z; acc.w += a.w;
        }
    }
    if (acc.x + acc.y + acc.z + acc.w == 123.456f) *sink = acc.x;      // never true: keeps the loads alive
}

// Conflict-free 32-bit shared-memory loads, the access the sampling kernels make (one wavefront per warp
// instruction, 128 B): every thread issues `iters` x 16 loads from a 32 KB tile.
__global__ void __launch_bounds__(1024)
fp_probe_shared_kernel(int iters, float *sink)
{
    __shared__ float tile[8192];
    for (int k = threadIdx.x; k < 8192; k += blockDim.x) tile[k] = (float)(k & 7);
    __syncthreads();
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    unsigned a = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            acc[u & 3] += tile[(a + 37u * u) & 8191u];     // consecutive lanes -> consecutive banks
        }
        a += 611u;
    }
    if (acc[0] + acc[1] + acc[2] + acc[3] == -1.0f) *sink = acc[0];
}

}  // namespace fpk
