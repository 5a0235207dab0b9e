// fp_tex.cuh -- texture-pipe sampling kernel and its layout stage (any pose, all three driving axes).
//
// Layout stage (PAPER.md:290-294 sec. 2.8: "optimal memory layout"; :292 mentions Morton-like orders): for
// every driving axis m the volume is copied into a LAYERED 2-D CUDA array -- layer = slice index along m,
// row = slow transverse axis, column = fast transverse axis -- whose block-linear (brick-tiled) texel order
// keeps the 2 x 2 bilinear footprints of neighbouring rays in the same cache lines whatever the in-plane
// direction of the detector axes.  fp_fill_layers_kernel writes the arrays through surface stores.
//
// Sampling (Alg. 1 l.6-20): one thread per ray; per sample ONE tld4 (PTX tld4.r.a2d) returns
// the four taps of Eq. 15 (:165) -- texels (k, j), (k+1, j), (k, j+1), (k+1, j+1) of layer i -- and the
// product weights of Eq. 11 (:142) with w of Eq. 13 / 14 are applied in fp32, exactly as in the other
// kernels; texels outside the array read 0 (border mode = reading #2).  The texture pipe is a second data
// path beside the LSU / shared-memory pipe that bounds fp_tma_kernel: fp_project runs this kernel on part of
// a call's projections CONCURRENTLY with fp_tma_kernel.
//
// HW = true is the paper's GJP_hwlin (PAPER.md:215 sec. 2.6, :330 Table 1): one bilinear-FILTERED fetch at
// p(i) per sample.  Since p_m is an integer (:108) the tri-linear interpolation the paper describes reduces
// to the bi-linear one in the slice plane (:155 footnote), which a 2-D layered fetch evaluates; the hardware
// quantises the weights to 8 fractional bits, so this variant does NOT meet the tolerance and is never
// chosen by FP_KERNEL_AUTO (measured error: DESIGN.md).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "fp_setup.cuh"
#include "fp_kernels.cuh"

namespace fpk {

constexpr int kTexThreads = 128;          // most threads per block; a work unit is 32 lanes x (blockDim.x / 32) rows of detector pixels

struct TexParams {
    GridDesc G;
    unsigned long long tex[3];         // per driving axis: texture object of the layered array (point or linear filter)
    const ProjDesc *proj;              // all projections of the call
    const int *ids;                    // [n_sel] projections this launch handles
    float *out;                        // [n_proj][nv][nu]
    unsigned long long *sample_count;  // may be null
    int nu, nv, n_sel;
};

// layer = index along AXIS, row = slow transverse axis, column = fast transverse axis:
// AXIS 0: (x; y, z)   AXIS 1: (y; x, z)   AXIS 2: (z; x, y)
template <int AXIS>
__global__ void __launch_bounds__(256)
fp_fill_layers_kernel(const float *__restrict__ vol, cudaSurfaceObject_t surf, int nx, int ny, int nz)
{
    if (AXIS < 2) {
        // one block per (x, 8 values of y): threads run along z, the contiguous axis on both sides
        const int x = blockIdx.x, y0 = blockIdx.y * 8;
        for (int yy = threadIdx.x >> 5; yy < 8; yy += 8) {
            const int y = y0 + yy;
            if (y >= ny) continue;
            const float *src = vol + ((size_t)x * ny + y) * nz;
            for (int z = threadIdx.x & 31; z < nz; z += 32) {
                const float v = src[z];
                if (AXIS == 0) surf2DLayeredwrite(v, surf, z * 4, y, x);
                else surf2DLayeredwrite(v, surf, z * 4, x, y);
            }
        }
    } else {
        // fixed x, a 32 x 32 tile of (y, z): read along z, write along y
        __shared__ float tile[32][33];
        const int x = blockIdx.z, y0 = blockIdx.y * 32, z0 = blockIdx.x * 32;
        const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
        for (int k = 0; k < 32; k += 8) {
            const int y = y0 + ty + k, z = z0 + tx;
            if (y < ny && z < nz) tile[ty + k][tx] = vol[((size_t)x * ny + y) * nz + z];
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 32; k += 8) {
            const int z = z0 + ty + k, y = y0 + tx;
            if (y < ny && z < nz) surf2DLayeredwrite(tile[tx][ty + k], surf, y * 4, x, z);
        }
    }
}

// four taps of layer `layer` around the texel corner (x, y): .x = (k, j+1), .y = (k+1, j+1), .z = (k+1, j), .w = (k, j)
// for x = k + 1, y = j + 1 (texel k has its centre at k + 0.5)
__device__ __forceinline__ float4 tex_gather_layer(unsigned long long tex, int layer, float x, float y)
{
    float4 v;
    asm volatile("tld4.r.a2d.v4.f32.f32 {%0, %1, %2, %3}, [%4, {%5, %6, %7, %7}];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(tex), "r"(layer), "f"(x), "f"(y));
    return v;
}

// one bilinear-filtered fetch of layer `layer` at texel coordinates (x, y)
__device__ __forceinline__ float tex_filtered_layer(unsigned long long tex, int layer, float x, float y)
{
    float4 v;
    asm volatile("tex.a2d.v4.f32.f32 {%0, %1, %2, %3}, [%4, {%5, %6, %7, %7}];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(tex), "r"(layer), "f"(x), "f"(y));
    return v.x;
}

// N consecutive samples i .. i + N - 1 of one segment, all N tld4 in flight before the first is used.
template <int INTERP, int N>
__device__ __forceinline__ float tex_chunk(unsigned long long tex, int i, int ic, float2 r2, float2 a2, float2 o2)
{
    const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f), kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
    const float2 kNegOne2 = make_float2(-1.0f, -1.0f);
    float4 v[N];
    float2 d[N];
#pragma unroll
    for (int k = 0; k < N; ++k) {
        const float fi = (float)(i + k - ic);
        const float2 p = __ffma2_rn(make_float2(fi, fi), r2, a2);
        const float2 x = __fadd2_rd(p, kMagic2);
        const float2 f = __fadd2_rn(x, kNegMagic2);                       // floor(p)
        d[k] = __ffma2_rn(f, kNegOne2, p);                                // p - floor(p)
        const float2 c = __fadd2_rn(f, o2);
        v[k] = tex_gather_layer(tex, i + k, c.y, c.x);
    }
    float acc = 0.0f;
#pragma unroll
    for (int k = 0; k < N; ++k) {
        const float ua = ceil_weight<INTERP>(d[k].x), ub = ceil_weight<INTERP>(d[k].y);
        const float z0v = fmaf(ub, v[k].z - v[k].w, v[k].w);             // slow row j
        const float z1v = fmaf(ub, v[k].y - v[k].x, v[k].x);             // slow row j + 1
        acc += fmaf(ua, z1v - z0v, z0v);
    }
    return acc;
}

// Samples of slices [lo, hi] of one ray.  Eq. 6 in fp32 per segment of kSegment slices about an
// fp64 anchor split into integer voxel index + fraction (as fp_direct_kernel); U independent samples are in
// flight per thread.
template <int INTERP, bool HW, int U>
__device__ __forceinline__ float tex_run(const RaySetup &R, unsigned long long tex, int lo, int hi)
{
    float acc = 0.0f;
    const float2 r2 = make_float2((float)R.rt_a, (float)R.rt_b);
    for (int s0 = lo; s0 <= hi; s0 += kSegment) {
        const int s1 = min(s0 + kSegment - 1, hi);
        const int ic = (s0 + s1) >> 1;
        const double pa = p_of_i(R.s_a, R.s_m, R.rt_a, ic), pb = p_of_i(R.s_b, R.s_m, R.rt_b, ic);
        const double fa = floor(pa), fb = floor(pb);
        const float2 a2 = make_float2((float)(pa - fa), (float)(pb - fb));
        if (HW) {
            // filtered fetch at p + 0.5 (texel centres): coordinate = anchor integer + fp32 remainder
            const float2 o2 = make_float2((float)fa + 0.5f, (float)fb + 0.5f);
#pragma unroll 8
            for (int i = s0; i <= s1; ++i) {
                const float fi = (float)(i - ic);
                const float2 p = __ffma2_rn(make_float2(fi, fi), r2, a2);
                acc += tex_filtered_layer(tex, i, p.y + o2.y, p.x + o2.x);
            }
            continue;
        }
        const float2 o2 = make_float2((float)fa + 1.0f, (float)fb + 1.0f);     // + 1: corner between texels f and f + 1
        int i = s0;
        for (; i + U - 1 <= s1; i += U) acc += tex_chunk<INTERP, U>(tex, i, ic, r2, a2, o2);
        if (U > 4)
            for (; i + 3 <= s1; i += 4) acc += tex_chunk<INTERP, 4>(tex, i, ic, r2, a2, o2);
        for (; i <= s1; ++i) acc += tex_chunk<INTERP, 1>(tex, i, ic, r2, a2, o2);
    }
    return acc;
}

// Persistent grid: work unit = (projection, 32 x (blockDim.x / 32) pixel tile); units are handed out in order, so that
// concurrently running blocks work on neighbouring tiles of the same projection (shared texture-cache lines).
template <int INTERP, bool HW, int U>
__global__ void __launch_bounds__(kTexThreads, 1)
fp_tex_kernel(const __grid_constant__ TexParams P)
{
    const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
    const int rows = blockDim.x >> 5;
    const int tl = (max(P.nu, P.nv) + 31) / 32, tr = (max(P.nu, P.nv) + rows - 1) / rows;
    const long long per_proj = (long long)tl * tr, n_units = per_proj * P.n_sel;
    int n_samples = 0;
    for (long long unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
        const int sel = (int)(unit / per_proj);
        const int t = (int)(unit - (long long)sel * per_proj);
        const int bl = t % tl, br = t / tl;            // tiles along the lane axis are neighbours in time
        const int proj = P.ids[sel];
        const ProjDesc *pd = P.proj + proj;
        const bool lane_v = pd->lane_v != 0;
        const int a_lane = bl * 32 + lane, a_row = br * rows + row;
        const int iu = lane_v ? a_row : a_lane, iv = lane_v ? a_lane : a_row;
        if (iu >= P.nu || iv >= P.nv) continue;
        const RaySetup R = ray_setup(pd->g, P.G, iu, iv);
        float acc = 0.0f;
        if (R.i_last >= R.i_first) {
            n_samples += R.i_last - R.i_first + 1;
            // one call per driving axis: inside each the texture handle is a kernel parameter, hence provably
            // warp-uniform (a handle selected per lane would put a divergence loop around every tld4, and the
            // loop's back edge waits for the fetch it has just issued)
            if (R.m == 0) acc = tex_run<INTERP, HW, U>(R, P.tex[0], R.i_first, R.i_last);
            else if (R.m == 1) acc = tex_run<INTERP, HW, U>(R, P.tex[1], R.i_first, R.i_last);
            else acc = tex_run<INTERP, HW, U>(R, P.tex[2], R.i_first, R.i_last);
        }
        P.out[((size_t)proj * P.nv + iv) * P.nu + iu] = (float)(P.G.delta * R.L) * acc;   // step length
    }
    if (P.sample_count) block_count_samples(P.sample_count, n_samples);
}

}  // namespace fpk
