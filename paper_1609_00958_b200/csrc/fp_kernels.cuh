// fp_kernels.cuh -- device kernels of libfp.so (sm_100a): sampling loop, ray-range export,
// volume permutation.  Citations are PAPER.md lines (arXiv 1609.00958).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "fp_setup.cuh"

namespace fpk {

// How the sampling kernel reads the slices of one driving axis m: element strides of the slice
// index i, the slow transverse axis and the fast transverse axis (sf == 1 in every layout the
// library builds itself; sf != 1 only when z-driven rays read the caller's z-fastest array).
struct AxisLayout {
    const float *base;
    long long si, ss, sf;
    int n_i, n_s, n_f;
    int pad_;
};

struct ProjDesc {
    double g[12];        // source, det origin, u, v (world units)
    int lane_v;          // 1: consecutive lanes of a warp run along v, 0: along u
    int pad_;
};

struct ProjectParams {
    GridDesc G;
    AxisLayout lay[3];                 // indexed by the driving axis m
    const ProjDesc *proj;              // [n_proj]
    const int *ids;                    // projections this launch handles (blockIdx.z -> projection), or null
    float *out;                        // [n_proj][nv][nu]
    unsigned long long *sample_count;  // may be null
    int nu, nv, n_proj;
    int interp;                        // 0 linear (Eq. 13), 1 spline (Eq. 14)
};

// Interpolation kernel weight of the FLOOR tap, w(d) (Eq. 7); the ceil tap gets
// 1 - w(d) (Eq. 8).  Linear: w = 1 - d (Eq. 13).  Spline: w = 1 - 3d^2 + 2d^3 (Eq. 14).
// We carry u = 1 - w (the weight of the ceil tap) because the lerp form uses it directly.
template <int INTERP>
__device__ __forceinline__ float ceil_weight(float d)
{
    if (INTERP == 1) return d * d * fmaf(-2.0f, d, 3.0f);
    return d;
}

constexpr int kTileLane = 32;   // pixels along the lane axis per block
constexpr int kTileRow = 8;     // pixels along the other detector axis per block
constexpr int kDirectThreads = kTileLane * kTileRow;
constexpr int kSegment = 64;    // slices per fp32 re-anchoring segment

__device__ __forceinline__ void block_count_samples(unsigned long long *counter, int n_mine)
{
    __shared__ unsigned int s_cnt;
    if (threadIdx.x == 0) s_cnt = 0u;
    __syncthreads();
    const unsigned int w = __reduce_add_sync(0xffffffffu, (unsigned int)n_mine);
    if ((threadIdx.x & 31) == 0 && w) atomicAdd(&s_cnt, w);
    __syncthreads();
    if (threadIdx.x == 0 && s_cnt) atomicAdd(counter, (unsigned long long)s_cnt);
}

// ------------------------------------------------------------------------------------------
// Direct sampling kernel: one thread per ray, taps read straight from global memory through
// the read-only path, index-masked (zero-extended volume, reading #2).
// Alg. 1 lines 6-20; Eq. 6 (:104) in the multiply form anchored at the
// middle slice of the ray; Eq. 15 (:165) tap selection; Eq. 11 (:142) product weights.
// ------------------------------------------------------------------------------------------
template <int INTERP>
__global__ void __launch_bounds__(kDirectThreads)
fp_direct_kernel(const __grid_constant__ ProjectParams P)
{
    const int proj = P.ids ? P.ids[blockIdx.z] : (int)blockIdx.z;
    const ProjDesc *pd = P.proj + proj;
    const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
    const bool lane_v = pd->lane_v != 0;
    const int a_lane = blockIdx.x * kTileLane + lane;
    const int a_row = blockIdx.y * kTileRow + row;
    const int iu = lane_v ? a_row : a_lane;
    const int iv = lane_v ? a_lane : a_row;
    const bool live = (iu < P.nu) && (iv < P.nv);
    // whole block outside the detector (grid is sized for either orientation)
    if ((lane_v ? blockIdx.y * kTileRow : blockIdx.x * kTileLane) >= P.nu ||
        (lane_v ? blockIdx.x * kTileLane : blockIdx.y * kTileRow) >= P.nv)
        return;

    int n_samples = 0;
    if (live) {
        const RaySetup R = ray_setup(pd->g, P.G, iu, iv);
        float acc = 0.0f;
        if (R.i_last >= R.i_first) {
            n_samples = R.i_last - R.i_first + 1;
            const AxisLayout &A = P.lay[R.m];
            const float r1 = (float)R.rt_a, r2 = (float)R.rt_b;
            const float *__restrict__ base = A.base;
            const long long si = A.si, ss = A.ss, sf = A.sf;
            const unsigned n_s = (unsigned)A.n_s, n_f = (unsigned)A.n_f;
            // Eq. 6 evaluated in fp32 per segment of kSegment slices: the anchor p_t(i_c) of the
            // segment's middle slice comes from fp64 and is split into an integer voxel index
            // and a fraction in [0,1), so |fp32 operand| <= kSegment/2 + 1 whatever the volume
            // size.
            for (int s0 = R.i_first; s0 <= R.i_last; s0 += kSegment) {
                const int s1 = min(s0 + kSegment - 1, R.i_last);
                const int ic = (s0 + s1) >> 1;
                const double pa = p_of_i(R.s_a, R.s_m, R.rt_a, ic), pb = p_of_i(R.s_b, R.s_m, R.rt_b, ic);
                const double fa = floor(pa), fb = floor(pb);
                const int ja = (int)fa, kb = (int)fb;
                const float a1 = (float)(pa - fa), a2 = (float)(pb - fb);
                const float *qseg = base + (long long)ja * ss + (long long)kb * sf;
                for (int i = s0; i <= s1; ++i) {
                    const float fi = (float)(i - ic);
                    const float p1 = fmaf(fi, r1, a1), p2 = fmaf(fi, r2, a2);
                    const float f1 = floorf(p1), f2 = floorf(p2);
                    const int jl = (int)f1, kl = (int)f2;
                    const int j = ja + jl, k = kb + kl;
                    const float u1 = ceil_weight<INTERP>(p1 - f1), u2 = ceil_weight<INTERP>(p2 - f2);
                    const bool j0 = (unsigned)j < n_s, j1 = (unsigned)(j + 1) < n_s;
                    const bool k0 = (unsigned)k < n_f, k1 = (unsigned)(k + 1) < n_f;
                    const float *q = qseg + (long long)i * si + (long long)jl * ss + (long long)kl * sf;
                    const float v00 = (j0 && k0) ? __ldg(q) : 0.0f;
                    const float v01 = (j0 && k1) ? __ldg(q + sf) : 0.0f;
                    const float v10 = (j1 && k0) ? __ldg(q + ss) : 0.0f;
                    const float v11 = (j1 && k1) ? __ldg(q + ss + sf) : 0.0f;
                    const float t0 = fmaf(u2, v01 - v00, v00);
                    const float t1 = fmaf(u2, v11 - v10, v10);
                    acc += fmaf(u1, t1 - t0, t0);
                }
            }
        }
        const float scale = (float)(P.G.delta * R.L);       // step length
        P.out[((size_t)proj * P.nv + iv) * P.nu + iu] = scale * acc;
    }
    if (P.sample_count) block_count_samples(P.sample_count, n_samples);
}

// Ray-range export (parity / debug): { m, i_first, i_last } per pixel.
__global__ void __launch_bounds__(256)
fp_ranges_kernel(GridDesc G, const ProjDesc *__restrict__ proj, int nu, int nv, int32_t *__restrict__ mfl)
{
    const int p = blockIdx.z;
    const int iu = blockIdx.x * 32 + (threadIdx.x & 31);
    const int iv = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (iu >= nu || iv >= nv) return;
    const RaySetup R = ray_setup(proj[p].g, G, iu, iv);
    int32_t *o = mfl + 3 * (((size_t)p * nv + iv) * nu + iu);
    o[0] = R.m;
    o[1] = R.i_first;
    o[2] = R.i_last;
}

// Volume layout stage (sec. 2.8): src [R][C] -> dst [C][R], used with
// R = nx*ny, C = nz to build the y-fastest copy [nz][nx][ny] read by z-driven rays.
__global__ void __launch_bounds__(256)
fp_transpose_kernel(const float *__restrict__ src, float *__restrict__ dst, long long R, long long C)
{
    __shared__ float tile[32][33];
    const long long r0 = (long long)blockIdx.x * 32, c0 = (long long)blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const long long r = r0 + ty + k, c = c0 + tx;
        if (r < R && c < C) tile[ty + k][tx] = src[r * C + c];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const long long c = c0 + ty + k, r = r0 + tx;
        if (r < R && c < C) dst[c * R + r] = tile[tx][ty + k];
    }
}

}  // namespace fpk
