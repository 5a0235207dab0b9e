// fp_aligned.cuh -- sampling kernel for poses whose detector v axis is parallel to the volume's
// z axis (the fastest memory index) and whose u axis is perpendicular to it: every circular
// orbit about z (PAPER.md:294 sec. 2.8, :312 sec. 3.2 -- "rotational axis parallel to the
// fastest index").
//
// For such a pose r_x, r_y depend on the detector column iu only and r_z on the row iv only.
// With a driving axis m in {x, y} (the host checks that no ray is z-driven) this gives, for one
// column and one slice i (Eq. 6):
//     p_slow(i)     = s_slow + (i - s_m) r_slow / r_m          the same for every row
//     p_z(i, iv)    = s_z + ((i - s_m) / r_m) * r_z(iv)        affine in iv
// so the four-tap sample of Eq. 15 (:165) factors: one interpolation of two neighbouring
// z-lines along the slow axis per (column, slice) -- "phase A", vectorised float4, written to
// shared memory -- and one 2-tap interpolation along z per sample -- "phase B".  The product
// weights are those of Eq. 11 (:142) with w of Eq. 13 / Eq. 14 (:150-152).  Lines are staged
// as a zero-filled window, so taps outside the volume read 0 (reading #2) and no sample is
// masked; the exact (m, i_first, i_last) of fp_setup.cuh are needed only for the sample count.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "fp_setup.cuh"
#include "fp_kernels.cuh"

namespace fpk {

constexpr int kAlTU = 8;        // detector columns per block
constexpr int kAlSB = 4;        // slices per staging batch
constexpr int kAlNL = kAlTU * kAlSB;
constexpr int kAlTV = 256;      // detector rows per block = threads per block

struct AlignedParams {
    GridDesc G;
    const float *vol;                  // [nx][ny][nz]
    const ProjDesc *proj;              // all projections of the call
    const int *ids;                    // [n_sel] projections this launch handles
    float *out;                        // [n_proj][nv][nu]
    unsigned long long *sample_count;  // may be null
    unsigned int *err_flag;            // set to 1 if a staging window would overflow
    int nu, nv, n_sel;
};

struct AlColumn {          // per detector column, constant over the slice loop
    double s_m, inv_rm;    // source coordinate along m, 1 / r_m
    double s_s, rt_s;      // slow transverse axis: source coordinate, r~
    long long stride_m, stride_s;      // element strides of the slice index and of the slow axis
    int i_lo, i_hi;        // slices with -1 < p_slow < N_slow (exact, clip_axis)
    int n_s, m;
};

struct AlLine {            // per staged line (column, slice of the batch)
    const float *pa, *pb;  // rows j and j+1 at z = 0
    float u1;              // weight of row j+1
    int z0f;               // window origin (multiple of 4) | 1 (row j inside) | 2 (row j+1 inside)
    int pad_[2];
};

struct AlBatch {           // per (column, batch): z position of the window in ray-parameter form
    double t0;             // (i0 - s_m) / r_m at the batch's first slice
    double off;            // s_z - z0
};

struct AlShared {
    AlColumn col[kAlTU];
    AlLine line[2][kAlNL];
    AlBatch batch[2][kAlTU];
    double s_z, rho_first, rho_last;
    int n_batches;
    unsigned lines_bias;   // shared-window byte address of the staged lines minus (0x4B000000 << 2)
};

template <int W>
constexpr size_t aligned_smem_bytes() { return sizeof(AlShared) + sizeof(float) * (size_t)kAlNL * W; }

// r_z of detector row iv in grid units: d_z - s_z with D_z = (O_z + iu * 0) + iv V_z.
__device__ __forceinline__ double al_rho(const double *g, const GridDesc &G, int iv, double s_z)
{
    const double D = __dadd_rn(g[5], __dmul_rn((double)iv, g[11]));
    const double d = __ddiv_rn(__dsub_rn(D, G.origin[2]), G.delta);
    return __dsub_rn(d, s_z);
}

// 32-bit shared-memory load at a byte address (lets ptxas fold constant offsets into the LDS).
__device__ __forceinline__ float al_lds(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}

// Staging parameters of line l = (column c, slice s of batch b), written by one thread.
template <int INTERP, int W>
__device__ __forceinline__ void al_line_params(AlShared &S, const AlignedParams &P, int buf, int b, int l)
{
    const int c = l / kAlSB, s = l - c * kAlSB;
    const AlColumn &C = S.col[c];
    const int i0 = C.i_lo + b * kAlSB;
    const int i = i0 + s;
    // window origin of this (column, batch): the extreme rows at the first and at the last slice
    const double ta = __dmul_rn(__dsub_rn((double)i0, C.s_m), C.inv_rm);
    const double tb = __dmul_rn(__dsub_rn((double)(i0 + kAlSB - 1), C.s_m), C.inv_rm);
    const double z1 = ta * S.rho_first, z2 = ta * S.rho_last, z3 = tb * S.rho_first, z4 = tb * S.rho_last;
    const double zmin = S.s_z + fmin(fmin(z1, z2), fmin(z3, z4));
    const double zmax = S.s_z + fmax(fmax(z1, z2), fmax(z3, z4));
    const bool finite = (zmin > -1.0e9) && (zmax < 1.0e9);
    int z0 = finite ? (((int)floor(zmin) - 1) & ~3) : 0;
    // taps k, k+1 with k = floor(p_z - z0) in [1, W-3] (one spare on either side for fp32 rounding)
    const bool winok = finite && ((int)floor(zmax) + 3 - z0 <= W);
    const bool live = winok && (i <= C.i_hi);
    if (!winok && i <= C.i_hi) atomicOr(P.err_flag, 1u);
    AlLine L;
    L.pa = L.pb = P.vol;
    L.u1 = 0.0f;
    int flags = 0;
    if (live) {
        const double ps = p_of_i(C.s_s, C.s_m, C.rt_s, i);           // Eq. 6 along the slow axis
        const double jf = floor(ps);
        const int j = (int)jf;
        L.u1 = ceil_weight<INTERP>((float)(ps - jf));
        if (j >= 0 && j < C.n_s) flags |= 1;
        if (j + 1 >= 0 && j + 1 < C.n_s) flags |= 2;
        L.pa = P.vol + ((long long)i * C.stride_m + (long long)j * C.stride_s);
        L.pb = L.pa + C.stride_s;
    }
    L.z0f = (winok ? z0 : 0) | flags;
    L.pad_[0] = L.pad_[1] = 0;
    S.line[buf][l] = L;
    if (s == 0) {
        AlBatch B;
        // a window that does not fit is never sampled out of bounds: park every row at p = 4
        B.t0 = winok ? ta : 0.0;
        B.off = winok ? S.s_z - (double)z0 : 4.0;
        S.batch[buf][c] = B;
    }
}

// ------------------------------------------------------------------------------------------
// Block = kAlTU detector columns x kAlTV detector rows, one thread per row.  Loop over batches
// of kAlSB slices; per batch
//   phase A: for each (column, slice) blend the two volume rows j, j+1 (float4 loads along z,
//            zero-filled outside the volume) with the column's slow-axis weight and store the
//            W-voxel window of the blended line in shared memory;
//   phase B: every thread takes its row's sample from each staged line: position by one FMA
//            from a per-(column, batch) fp64 anchor, floor by a round-down add of 2^23, two
//            shared-memory taps, one lerp, one add (Alg. 1 l.7-18).
// Line parameters of batch b+1 are computed by warp 0 during phase A of batch b (double
// buffered), so a batch costs two block barriers.
// ------------------------------------------------------------------------------------------
template <int INTERP, int W>
__global__ void __launch_bounds__(kAlTV, 3)
fp_aligned_kernel(const __grid_constant__ AlignedParams P)
{
    extern __shared__ __align__(16) unsigned char al_smem_raw[];
    AlShared &S = *reinterpret_cast<AlShared *>(al_smem_raw);
    float *lines = reinterpret_cast<float *>(al_smem_raw + sizeof(AlShared));

    const int tid = threadIdx.x;
    const int proj = P.ids[blockIdx.z];
    const double *g = P.proj[proj].g;
    const int iu0 = blockIdx.x * kAlTU;
    const int row0 = blockIdx.y * kAlTV;
    const int iv = min(row0 + tid, P.nv - 1);

    // ---- column set-up (Eqs. 1-5, Alg. 1 l.1-5), one thread per column
    if (tid < kAlTU) {
        AlColumn C;
        const int iu = iu0 + tid;
        double s[3], r[2];
#pragma unroll
        for (int a = 0; a < 3; ++a) s[a] = __ddiv_rn(__dsub_rn(g[a], P.G.origin[a]), P.G.delta);
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const double D = __dadd_rn(g[3 + a], __dmul_rn((double)iu, g[6 + a]));   // + iv * 0 exactly
            const double d = __ddiv_rn(__dsub_rn(D, P.G.origin[a]), P.G.delta);
            r[a] = __dsub_rn(d, s[a]);
        }
        const int m = fabs(r[1]) > fabs(r[0]) ? 1 : 0;            // Eq. 2 (z excluded by the host plan)
        const double rm = m ? r[1] : r[0];
        const long long nz = P.G.n[2], ny = P.G.n[1];
        C.m = m;
        C.s_m = m ? s[1] : s[0];
        C.s_s = m ? s[0] : s[1];
        C.rt_s = __ddiv_rn(m ? r[0] : r[1], rm);                  // Eq. 4
        C.inv_rm = 1.0 / rm;
        C.stride_m = m ? nz : ny * nz;
        C.stride_s = m ? ny * nz : nz;
        C.n_s = m ? P.G.n[0] : P.G.n[1];
        int lo = 0, hi = (m ? P.G.n[1] : P.G.n[0]) - 1;
        if (iu < P.nu && rm != 0.0)
            clip_axis(C.s_s, C.s_m, C.rt_s, C.n_s, lo, hi);
        else {
            hi = -1;
            C.inv_rm = 0.0;
            C.rt_s = 0.0;
        }
        C.i_lo = lo;
        C.i_hi = hi;
        S.col[tid] = C;
        if (tid == 0) {
            S.s_z = s[2];
            S.rho_first = al_rho(g, P.G, row0, s[2]);
            S.rho_last = al_rho(g, P.G, min(row0 + kAlTV, P.nv) - 1, s[2]);
        }
    }
    __syncthreads();
    if (tid == 0) {
        int nb = 0;
#pragma unroll
        for (int c = 0; c < kAlTU; ++c) nb = max(nb, (S.col[c].i_hi - S.col[c].i_lo + 1 + kAlSB - 1) / kAlSB);
        S.n_batches = nb;
        S.lines_bias = (unsigned)__cvta_generic_to_shared(lines) - (0x4B000000u << 2);
    }
    if (tid < kAlNL) al_line_params<INTERP, W>(S, P, 0, 0, tid);

    // ---- per-thread constants: r_z of this row, per-column z increment per slice
    const double s_z = S.s_z;
    const double rho = al_rho(g, P.G, iv, s_z);
    float dz[kAlTU], acc[kAlTU];
#pragma unroll
    for (int c = 0; c < kAlTU; ++c) {
        dz[c] = (float)(rho * S.col[c].inv_rm);
        acc[c] = 0.0f;
    }
    __syncthreads();
    const int n_batches = S.n_batches;
    const int nz = P.G.n[2];
    const int warp = tid >> 5, lane = tid & 31;
    constexpr int QW = W / 4;
    constexpr int kWarps = kAlTV / 32;
    // shared-memory byte address of lines[0] minus the bias the 2^23 trick leaves in the float's bits
    // read back from shared memory so that neither compiler can split the bias into address + constant:
    // (bits << 2) + bias stays ONE add and the per-line constant folds into the load's immediate offset
    const unsigned lines_bias = *reinterpret_cast<volatile unsigned *>(&S.lines_bias);
    constexpr float kMagic = 8388608.0f;      // 2^23: x + 2^23 rounded down = floor(x) for 0 <= x < 2^22

    for (int b = 0; b < n_batches; ++b) {
        const int buf = b & 1;
        if (b) __syncthreads();               // parameters of batch b visible, phase B of b-1 done
        // ---------------- phase A
#pragma unroll
        for (int l = warp; l < kAlNL; l += kWarps) {
            const AlLine L = S.line[buf][l];
            const int z0 = L.z0f & ~3;
            float4 *dst = reinterpret_cast<float4 *>(lines + l * W);
#pragma unroll
            for (int q = lane; q < QW; q += 32) {
                const int z = z0 + 4 * q;
                const bool inz = (unsigned)z < (unsigned)nz;
                float4 va = make_float4(0.f, 0.f, 0.f, 0.f), vb = va;
                if (inz && (L.z0f & 1)) va = __ldg(reinterpret_cast<const float4 *>(L.pa + z));
                if (inz && (L.z0f & 2)) vb = __ldg(reinterpret_cast<const float4 *>(L.pb + z));
                float4 o;
                o.x = fmaf(L.u1, vb.x - va.x, va.x);
                o.y = fmaf(L.u1, vb.y - va.y, va.y);
                o.z = fmaf(L.u1, vb.z - va.z, va.z);
                o.w = fmaf(L.u1, vb.w - va.w, va.w);
                dst[q] = o;
            }
        }
        if (tid < kAlNL && b + 1 < n_batches) al_line_params<INTERP, W>(S, P, buf ^ 1, b + 1, tid);
        __syncthreads();
        // ---------------- phase B
#pragma unroll
        for (int c = 0; c < kAlTU; ++c) {
            const AlBatch B = S.batch[buf][c];
            const float a = (float)fma(B.t0, rho, B.off);
#pragma unroll
            for (int s = 0; s < kAlSB; ++s) {
                const float p = fmaf((float)s, dz[c], a);
                const float x = __fadd_rd(p, kMagic);             // bits = 0x4B000000 + floor(p)
                const float d = p - (x - kMagic);
                const unsigned addr = (__float_as_uint(x) << 2) + lines_bias + (unsigned)((c * kAlSB + s) * W * 4);
                const float v0 = al_lds(addr), v1 = al_lds(addr + 4u);
                acc[c] += fmaf(ceil_weight<INTERP>(d), v1 - v0, v0);
            }
        }
    }

    // ---- weight by the step length Delta * ||r~|| and store
    const bool live = (row0 + tid) < P.nv;
    int n_samples = 0;
    if (live) {
        float o[kAlTU];
#pragma unroll
        for (int c = 0; c < kAlTU; ++c) {
            const double rz = rho * S.col[c].inv_rm, rs = S.col[c].rt_s;
            // same summation order as the definition: x^2 + y^2 + z^2 with r~_m = 1
            const double a0 = S.col[c].m ? rs * rs : 1.0, a1 = S.col[c].m ? 1.0 : rs * rs;
            const double L = sqrt((a0 + a1) + rz * rz);
            o[c] = (float)(P.G.delta * L) * acc[c];
        }
        float *dst = P.out + ((size_t)proj * P.nv + iv) * P.nu + iu0;
        if ((P.nu & 3) == 0 && iu0 + kAlTU <= P.nu) {
            reinterpret_cast<float4 *>(dst)[0] = make_float4(o[0], o[1], o[2], o[3]);
            reinterpret_cast<float4 *>(dst)[1] = make_float4(o[4], o[5], o[6], o[7]);
        } else {
#pragma unroll
            for (int c = 0; c < kAlTU; ++c)
                if (iu0 + c < P.nu) dst[c] = o[c];
        }
        if (P.sample_count) {
            for (int c = 0; c < kAlTU; ++c)
                if (iu0 + c < P.nu) {
                    const RaySetup R = ray_setup(g, P.G, iu0 + c, iv);
                    n_samples += max(R.i_last - R.i_first + 1, 0);
                }
        }
    }
    if (P.sample_count) block_count_samples(P.sample_count, n_samples);
}

}  // namespace fpk
