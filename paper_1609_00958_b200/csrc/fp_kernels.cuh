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
// the read-only path.  Alg. 1 lines 6-20; Eq. 6 (:104) in the multiply form;
// Eq. 15 (:165) tap selection; Eq. 11 (:142) product weights.
//
// Eq. 6 is evaluated in fp32 per segment of kSegment slices: the anchor p_t(i_c) of the segment's
// middle slice comes from fp64 and is split into an integer voxel index and a fraction in [0,1),
// so |fp32 operand| <= kSegment/2 + 1 whatever the volume size.  Both transverse
// coordinates travel as one packed fp32x2 value (sm_100 FFMA2 / FADD2); floor is a round-down add
// of 1.5 * 2^23, whose low mantissa bits are the integer part.
//
// A ray's slices are split into an interior run, where all four taps of every sample are inside
// the volume (0.5 <= p_t <= N_t - 1.5 in fp64, far more margin than the fp32 error), sampled
// without masks, and the two edge runs before and after it, where taps are masked by index
// (zero-extended volume, reading #2).
// ------------------------------------------------------------------------------------------
template <int INTERP, bool MASKED>
__device__ __forceinline__ float direct_run(const RaySetup &R, const AxisLayout &A, int lo, int hi)
{
    float acc = 0.0f;
    const float2 r2 = make_float2((float)R.rt_a, (float)R.rt_b);
    const float *__restrict__ base = A.base;
    const long long si = A.si, ss = A.ss, sf = A.sf;
    const unsigned n_s = (unsigned)A.n_s, n_f = (unsigned)A.n_f;
    const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f), kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
    const float2 kNegOne2 = make_float2(-1.0f, -1.0f), kOne2 = make_float2(1.0f, 1.0f);
    for (int s0 = lo; s0 <= hi; s0 += kSegment) {
        const int s1 = min(s0 + kSegment - 1, hi);
        const int ic = (s0 + s1) >> 1;
        const double pa = p_of_i(R.s_a, R.s_m, R.rt_a, ic), pb = p_of_i(R.s_b, R.s_m, R.rt_b, ic);
        const double fa = floor(pa), fb = floor(pb);
        const int ja = (int)fa, kb = (int)fb;
        const float2 a2 = make_float2((float)(pa - fa), (float)(pb - fb));
        const float *qseg = base + (long long)ja * ss + (long long)kb * sf + (long long)s0 * si;
        float2 fi = make_float2((float)(s0 - ic), (float)(s0 - ic));
        for (int i = s0; i <= s1; ++i) {
            const float2 p = __ffma2_rn(fi, r2, a2);
            fi = __fadd2_rn(fi, kOne2);
            const float2 x = __fadd2_rd(p, kMagic2);              // bits = 0x4B400000 + floor(p)
            const float2 d = __ffma2_rn(__fadd2_rn(x, kNegMagic2), kNegOne2, p);
            const int jl = __float_as_int(x.x) - 0x4B400000, kl = __float_as_int(x.y) - 0x4B400000;
            const float u1 = ceil_weight<INTERP>(d.x), u2 = ceil_weight<INTERP>(d.y);
            const float *q = qseg + (long long)jl * ss + (long long)kl * sf;
            qseg += si;
            float v00, v01, v10, v11;
            if (MASKED) {
                const int j = ja + jl, k = kb + kl;
                const bool j0 = (unsigned)j < n_s, j1 = (unsigned)(j + 1) < n_s;
                const bool k0 = (unsigned)k < n_f, k1 = (unsigned)(k + 1) < n_f;
                v00 = (j0 && k0) ? __ldg(q) : 0.0f;
                v01 = (j0 && k1) ? __ldg(q + sf) : 0.0f;
                v10 = (j1 && k0) ? __ldg(q + ss) : 0.0f;
                v11 = (j1 && k1) ? __ldg(q + ss + sf) : 0.0f;
            } else {
                v00 = __ldg(q);
                v01 = __ldg(q + sf);
                v10 = __ldg(q + ss);
                v11 = __ldg(q + ss + sf);
            }
            // lerp along the fast axis for both rows at once, then along the slow axis
            const float2 lo2 = make_float2(v00, v10);
            const float2 t = __ffma2_rn(make_float2(u2, u2), __ffma2_rn(lo2, kNegOne2, make_float2(v01, v11)), lo2);
            acc += fmaf(u1, t.y - t.x, t.x);
        }
    }
    return acc;
}

// Slices of [lo, hi] on which lo_p <= s_t + (i - s_m) rt <= hi_p (fp64, one slice of slack inwards).
__device__ __forceinline__ void interior_clip(double s_t, double s_m, double rt, double lo_p, double hi_p, int &lo, int &hi)
{
    if (!(lo_p <= hi_p)) {            // fewer than two voxels along this axis: no interior
        hi = lo - 1;
        return;
    }
    if (rt == 0.0) {
        if (!(s_t >= lo_p && s_t <= hi_p)) hi = lo - 1;
        return;
    }
    const double x1 = s_m + (lo_p - s_t) / rt, x2 = s_m + (hi_p - s_t) / rt;
    const int a = clamp_to_int(ceil(fmin(x1, x2)) + 1.0, lo, hi + 1);
    const int b = clamp_to_int(floor(fmax(x1, x2)) - 1.0, lo - 1, hi);
    lo = max(lo, a);
    hi = min(hi, b);
}

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
            // interior run: every tap of every sample inside the volume
            int in_lo = R.i_first, in_hi = R.i_last;
            interior_clip(R.s_a, R.s_m, R.rt_a, 0.5, (double)A.n_s - 1.5, in_lo, in_hi);
            if (in_lo <= in_hi) interior_clip(R.s_b, R.s_m, R.rt_b, 0.5, (double)A.n_f - 1.5, in_lo, in_hi);
            if (in_lo <= in_hi) {
                acc = direct_run<INTERP, true>(R, A, R.i_first, in_lo - 1);
                acc += direct_run<INTERP, false>(R, A, in_lo, in_hi);
                acc += direct_run<INTERP, true>(R, A, in_hi + 1, R.i_last);
            } else {
                acc = direct_run<INTERP, true>(R, A, R.i_first, R.i_last);
            }
        }
        const float scale = (float)(P.G.delta * R.L);       // step length
        P.out[((size_t)proj * P.nv + iv) * P.nu + iu] = scale * acc;
    }
    if (P.sample_count) block_count_samples(P.sample_count, n_samples);
}

// ------------------------------------------------------------------------------------------
// Back-projection (the exact transpose of the sampling loop, PAPER.md:27,
// :308, :367): one thread per ray, same set-up, same slices, same four taps and product weights
// as fp_direct_kernel; instead of gathering vol[tap] * w it scatters delta ||r~|| w proj[ray]
// into vol_out[tap] with fp32 reductions in L2 (RED.ADD.F32).  Taps outside the volume belong to
// the zero extension (reading #2) and receive nothing.
// ------------------------------------------------------------------------------------------
struct BackprojectParams {
    GridDesc G;
    AxisLayout lay[3];                 // the OUTPUT volume [nx][ny][nz], indexed by the driving axis m
    const ProjDesc *proj;
    const int *ids;                    // [n_proj] projections this launch handles
    const float *in;                   // [all projections of the call][nv][nu]
    int nu, nv, n_proj;
};

template <int INTERP>
__global__ void __launch_bounds__(kDirectThreads)
fp_backproject_kernel(const __grid_constant__ BackprojectParams P)
{
    const int proj = P.ids[blockIdx.z];
    const ProjDesc *pd = P.proj + proj;
    const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
    const bool lane_v = pd->lane_v != 0;
    const int a_lane = blockIdx.x * kTileLane + lane;
    const int a_row = blockIdx.y * kTileRow + row;
    const int iu = lane_v ? a_row : a_lane;
    const int iv = lane_v ? a_lane : a_row;
    if (iu >= P.nu || iv >= P.nv) return;
    const RaySetup R = ray_setup(pd->g, P.G, iu, iv);
    if (R.i_last < R.i_first) return;
    const float y = P.in[((size_t)proj * P.nv + iv) * P.nu + iu] * (float)(P.G.delta * R.L);
    if (y == 0.0f) return;
    const AxisLayout &A = P.lay[R.m];
    float *__restrict__ base = const_cast<float *>(A.base);
    const long long si = A.si, ss = A.ss, sf = A.sf;
    const unsigned n_s = (unsigned)A.n_s, n_f = (unsigned)A.n_f;
    const float2 r2 = make_float2((float)R.rt_a, (float)R.rt_b);
    const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f), kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
    const float2 kNegOne2 = make_float2(-1.0f, -1.0f), kOne2 = make_float2(1.0f, 1.0f);
    for (int s0 = R.i_first; s0 <= R.i_last; s0 += kSegment) {
        const int s1 = min(s0 + kSegment - 1, R.i_last);
        const int ic = (s0 + s1) >> 1;
        const double pa = p_of_i(R.s_a, R.s_m, R.rt_a, ic), pb = p_of_i(R.s_b, R.s_m, R.rt_b, ic);
        const double fa = floor(pa), fb = floor(pb);
        const int ja = (int)fa, kb = (int)fb;
        const float2 a2 = make_float2((float)(pa - fa), (float)(pb - fb));
        float *qseg = base + (long long)ja * ss + (long long)kb * sf + (long long)s0 * si;
        float2 fi = make_float2((float)(s0 - ic), (float)(s0 - ic));
        for (int i = s0; i <= s1; ++i) {
            const float2 p = __ffma2_rn(fi, r2, a2);
            fi = __fadd2_rn(fi, kOne2);
            const float2 x = __fadd2_rd(p, kMagic2);
            const float2 d = __ffma2_rn(__fadd2_rn(x, kNegMagic2), kNegOne2, p);
            const int jl = __float_as_int(x.x) - 0x4B400000, kl = __float_as_int(x.y) - 0x4B400000;
            const float u1 = ceil_weight<INTERP>(d.x), u2 = ceil_weight<INTERP>(d.y);
            float *q = qseg + (long long)jl * ss + (long long)kl * sf;
            qseg += si;
            const int j = ja + jl, k = kb + kl;
            const bool j0 = (unsigned)j < n_s, j1 = (unsigned)(j + 1) < n_s;
            const bool k0 = (unsigned)k < n_f, k1 = (unsigned)(k + 1) < n_f;
            const float ya = y * (1.0f - u1), yb = y * u1;      // rows j, j + 1
            if (j0 && k0) atomicAdd(q, ya * (1.0f - u2));
            if (j0 && k1) atomicAdd(q + sf, ya * u2);
            if (j1 && k0) atomicAdd(q + ss, yb * (1.0f - u2));
            if (j1 && k1) atomicAdd(q + ss + sf, yb * u2);
        }
    }
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
