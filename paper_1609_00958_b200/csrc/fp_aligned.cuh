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
    int fov;                           // 1: the volume is zero outside the inscribed cylinder about z (FP_OPT_FOV_CYLINDER)
    int out_vec;                       // 1: out is 16-byte aligned and nu % 4 == 0 (vector stores allowed)
    int group;                         // projections whose blocks are interleaved in launch order (>= 1), as in fp_tma.cuh
};

struct AlColumn {          // per detector column, constant over the slice loop
    double s_m, inv_rm;    // source coordinate along m, 1 / r_m
    double s_s, rt_s;      // slow transverse axis: source coordinate, r~
    long long stride_m, stride_s;      // element strides of the slice index and of the slow axis
    int i_lo, i_hi;        // slices with -1 < p_slow < N_slow (exact, clip_axis)
    int n_s, m;
    int i_start, dir;      // slice of batch 0, step +1 / -1: slices are visited in order of ascending ray
                           // parameter t = (i - s_m) / r_m, all columns of a block starting at the same t
};

struct __align__(16) AlLine {   // per staged line (column, slice of the batch)
    const float *pa, *pb;  // rows j and j+1 at z = 0
    float u1;              // weight of row j+1
    int flags;             // 1 (row j inside the volume) | 2 (row j+1 inside)
    int pad_[2];
};

struct __align__(16) AlBatch {  // per batch: the common z window of all its lines
    double off;            // s_z - (z0 + zc): positions are taken relative to the window's centre
    int z0, nq;            // window origin (multiple of 4), float4 quads to stage
    int zc, pad_;          // centre of the window relative to z0
};

struct __align__(16) AlShared {
    AlColumn col[kAlTU];
    AlLine line[2][kAlNL];
    double t0[2][kAlTU];   // per (buffer, column): (i0 - s_m) / r_m at the batch's first slice
    AlBatch batch[2];
    double s_z, rho_first, rho_last;
    int n_batches;
    unsigned lines_bias;   // shared-window byte address of the staged lines minus (0x4B400000 << 2)
};

static_assert(sizeof(AlShared) % 16 == 0 && sizeof(AlLine) == 32 && sizeof(AlBatch) == 32, "shared layout");

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

__device__ __forceinline__ int al_to_int(double x)      // saturating double -> int
{
    return (int)fmin(fmax(x, -1.0e9), 1.0e9);
}

// Staging parameters of batch b, computed by warp 0: lane l = (column c, slice s) writes its line;
// the z window is common to the whole batch (min / max over the 32 lines by warp reductions).
template <int INTERP, int W, bool PREFETCH>
__device__ __forceinline__ void al_batch_params(AlShared &S, const AlignedParams &P, int buf, int b, int l)
{
    const int c = l / kAlSB, s = l - c * kAlSB;
    const AlColumn &C = S.col[c];
    const int i0 = C.i_start + C.dir * (b * kAlSB);
    const int i = i0 + C.dir * s;
    // z range of this line over the block's rows: p_z = s_z + t * r_z is monotone in the row
    const double t0 = __dmul_rn(__dsub_rn((double)i0, C.s_m), C.inv_rm);
    const double t = __dmul_rn(__dsub_rn((double)i, C.s_m), C.inv_rm);
    const double za = S.s_z + t * S.rho_first, zb = S.s_z + t * S.rho_last;
    const int zlo = __reduce_min_sync(0xffffffffu, al_to_int(floor(fmin(za, zb))));
    const int zhi = __reduce_max_sync(0xffffffffu, al_to_int(floor(fmax(za, zb))));
    // taps k, k+1 with k = floor(p_z - z0) in [1, W-3] (one spare on either side for fp32 rounding)
    const int z0 = (zlo - 1) & ~3;
    const int need = zhi + 3 - z0;
    const bool winok = (zlo > -1000000000) && (zhi < 1000000000) && (need <= W);
    const bool live = winok && (i >= C.i_lo) && (i <= C.i_hi);
    AlLine L;
    L.pa = L.pb = P.vol;
    L.u1 = 0.0f;
    L.flags = 0;
    if (live) {
        const double ps = p_of_i(C.s_s, C.s_m, C.rt_s, i);           // Eq. 6 along the slow axis
        const double jf = floor(ps);
        const int j = (int)jf;
        L.u1 = ceil_weight<INTERP>((float)(ps - jf));
        if (j >= 0 && j < C.n_s) L.flags |= 1;
        if (j + 1 >= 0 && j + 1 < C.n_s) L.flags |= 2;
        L.pa = P.vol + ((long long)i * C.stride_m + (long long)j * C.stride_s);
        L.pb = L.pa + C.stride_s;
    }
    L.pad_[0] = L.pad_[1] = 0;
    S.line[buf][l] = L;
    if (PREFETCH && live) {
        // pull the two volume rows of this line towards L2 one batch ahead of phase A (128 B per request)
        const int nzv = P.G.n[2];
        const int ze = min(z0 + need, nzv);
        for (int z = max(z0, 0) & ~31; z < ze; z += 32) {
            if (L.flags & 1) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.pa + z));
            if (L.flags & 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(L.pb + z));
        }
    }
    // a window that does not fit is never sampled out of bounds: park every row at p = 4
    if (s == 0) S.t0[buf][c] = winok ? t0 : 0.0;
    if (l == 0) {
        if (!winok) atomicOr(P.err_flag, 1u);
        AlBatch B;
        B.zc = winok ? need >> 1 : 0;
        B.pad_ = 0;
        B.off = winok ? S.s_z - (double)(z0 + B.zc) : 4.0;
        B.z0 = winok ? z0 : 0;
        B.nq = winok ? (need + 3) >> 2 : 0;
        S.batch[buf] = B;
    }
}

// ------------------------------------------------------------------------------------------
// Block = kAlTU detector columns x kAlTV detector rows, one thread per row.  Loop over batches
// of kAlSB slices; per batch
//   phase A: for each (column, slice) blend the two volume rows j, j+1 (float4 loads along z,
//            zero-filled outside the volume) with the column's slow-axis weight and store the
//            needed part of the W-voxel window of the blended line in shared memory;
//   phase B: every thread takes its row's sample from each staged line: position by one FMA
//            from a per-(column, batch) fp64 anchor, floor by a round-down add of 2^23, two
//            shared-memory taps, one lerp, one add (Alg. 1 l.7-18), two
//            slices at a time in packed fp32x2 arithmetic (sm_100 FFMA2 / FADD2).
// Parameters of batch b+1 are computed by warp 0 during phase A of batch b (double buffered),
// so a batch costs two block barriers.
// ------------------------------------------------------------------------------------------
template <int INTERP, int W>
__global__ void __launch_bounds__(kAlTV, 4)
fp_aligned_kernel(const __grid_constant__ AlignedParams P)
{
    extern __shared__ __align__(16) unsigned char al_smem_raw[];
    AlShared &S = *reinterpret_cast<AlShared *>(al_smem_raw);
    float *lines = reinterpret_cast<float *>(al_smem_raw + sizeof(AlShared));

    const int tid = threadIdx.x;
    // blockIdx.x = (detector tile) * group + (projection within the group): neighbouring poses sweep the volume
    // in step and share its rows through L2 (fp_tma.cuh)
    const int sel = blockIdx.z * P.group + (int)(blockIdx.x % (unsigned)P.group);
    if (sel >= P.n_sel) return;                            // the whole block (the last group may be short)
    const int proj = P.ids[sel];
    const double *g = P.proj[proj].g;
    const int iu0 = (int)(blockIdx.x / (unsigned)P.group) * kAlTU;
    const int row0 = blockIdx.y * kAlTV;
    const int iv = min(row0 + tid, P.nv - 1);

    // ---- column set-up (Eqs. 1-5, Alg. 1 l.1-5), one thread per column; columns past the detector
    //      edge reuse the last column's geometry with an empty slice range
    if (tid < kAlTU) {
        AlColumn C;
        const int iu = min(iu0 + tid, P.nu - 1);
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
        C.rt_s = rm != 0.0 ? __ddiv_rn(m ? r[0] : r[1], rm) : 0.0;   // Eq. 4
        C.inv_rm = rm != 0.0 ? 1.0 / rm : 0.0;
        C.stride_m = m ? nz : ny * nz;
        C.stride_s = m ? ny * nz : nz;
        C.n_s = m ? P.G.n[0] : P.G.n[1];
        int lo = 0, hi = (m ? P.G.n[1] : P.G.n[0]) - 1;
        if (iu0 + tid < P.nu && rm != 0.0) {
            clip_axis(C.s_s, C.s_m, C.rt_s, C.n_s, lo, hi);
            if (P.fov && lo <= hi) {
                // samples whose taps (p_s +- 1) all lie outside the cylinder read zeros: skip those slices
                const double cx = 0.5 * (P.G.n[0] - 1), cy = 0.5 * (P.G.n[1] - 1), rad = 0.5 * min(P.G.n[0], P.G.n[1]) + 1.5;
                clip_circle(C.s_s, C.s_m, C.rt_s, m ? cy : cx, m ? cx : cy, rad, lo, hi);
            }
        } else {
            hi = -1;
        }
        if (lo > hi) { lo = 0; hi = -1; }
        C.i_lo = lo;
        C.i_hi = hi;
        S.col[tid] = C;
        if (tid == 0) {
            S.s_z = s[2];
            S.rho_first = al_rho(g, P.G, row0, s[2]);
            S.rho_last = al_rho(g, P.G, min(row0 + kAlTV, P.nv) - 1, s[2]);
            S.lines_bias = (unsigned)__cvta_generic_to_shared(lines) - (0x4B400000u << 2);
        }
    }
    __syncthreads();
    // common start: the smallest ray parameter t = (i_lo - s_m) / r_m among the block's columns; every
    // column starts at the slice where its own t reaches it, so that the columns advance through the
    // volume together and one z window serves the whole batch (matters where the driving axis switches
    // inside the block and where neighbouring columns enter through a side face)
    if (tid < kAlTU) {
        double t_ref = 1.0e300;
#pragma unroll
        for (int c = 0; c < kAlTU; ++c) {
            const AlColumn &C = S.col[c];
            const int i_first = C.inv_rm < 0.0 ? C.i_hi : C.i_lo;
            if (C.i_hi >= C.i_lo) t_ref = fmin(t_ref, ((double)i_first - C.s_m) * C.inv_rm);
        }
        AlColumn &C = S.col[tid];
        const int dir = C.inv_rm < 0.0 ? -1 : 1;
        int i_start = dir > 0 ? C.i_lo : C.i_hi;
        if (t_ref < 1.0e299 && C.inv_rm != 0.0) {
            // slice of this column at t_ref, never inside its own range; a column without slices just
            // follows the others (its lines are never live)
            const double x = C.s_m + t_ref / C.inv_rm;
            if (C.i_hi < C.i_lo)
                i_start = min(max(al_to_int(floor(x)), -65536), 65536 + C.n_s);
            else if (dir > 0)
                i_start = min(C.i_lo, max(al_to_int(floor(x)), C.i_lo - 65536));
            else
                i_start = max(C.i_hi, min(al_to_int(ceil(x)), C.i_hi + 65536));
        }
        C.i_start = i_start;
        C.dir = dir;
    }
    __syncthreads();
    if (tid == 0) {
        int nb = 0;
#pragma unroll
        for (int c = 0; c < kAlTU; ++c) {
            const AlColumn &C = S.col[c];
            if (C.i_hi >= C.i_lo) nb = max(nb, ((C.dir > 0 ? C.i_hi - C.i_start : C.i_start - C.i_lo) + kAlSB) / kAlSB);
        }
        S.n_batches = nb;
    }
    __syncthreads();
    if (tid < kAlNL) al_batch_params<INTERP, W, false>(S, P, 0, 0, tid);

    // ---- per-thread constants: r_z of this row, per-column z increment per slice
    const double rho = al_rho(g, P.G, iv, S.s_z);
    float dz[kAlTU];
    float2 acc[kAlTU];
#pragma unroll
    for (int c = 0; c < kAlTU; ++c) {
        dz[c] = (float)(rho * S.col[c].inv_rm * (double)S.col[c].dir);
        acc[c] = make_float2(0.0f, 0.0f);
    }
    __syncthreads();
    const int n_batches = S.n_batches;
    // read back from shared memory so that neither compiler can split the bias into address + constant:
    // (bits << 2) + bias stays ONE add and the per-line constant folds into the load's immediate offset
    const unsigned lines_bias = *reinterpret_cast<volatile unsigned *>(&S.lines_bias);
    const int nz = P.G.n[2];
    const int warp = tid >> 5, lane = tid & 31;
    constexpr int kWarps = kAlTV / 32;
    const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f);    // 1.5 * 2^23 (positions may be negative)
    const float2 kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
    const float2 kNegOne2 = make_float2(-1.0f, -1.0f);

    for (int b = 0; b < n_batches; ++b) {
        const int buf = b & 1;
        if (b) __syncthreads();               // parameters of batch b visible, phase B of b-1 done
        const AlBatch B = S.batch[buf];
        // ---------------- phase A
#pragma unroll
        for (int l = warp; l < kAlNL; l += kWarps) {
            const AlLine L = S.line[buf][l];
            const float2 u2 = make_float2(L.u1, L.u1);
            float4 *dst = reinterpret_cast<float4 *>(lines + l * W);
            // all loads of the line first (predicated, no branches: they overlap), then the blends
            float4 va[W / 128], vb[W / 128];
#pragma unroll
            for (int k = 0; k < W / 128; ++k) {
                const int q = lane + 32 * k;
                const int z = B.z0 + 4 * q;
                const bool ok = (q < B.nq) && ((unsigned)z < (unsigned)nz);
                va[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                vb[k] = va[k];
                if (ok && (L.flags & 1)) va[k] = __ldg(reinterpret_cast<const float4 *>(L.pa + z));
                if (ok && (L.flags & 2)) vb[k] = __ldg(reinterpret_cast<const float4 *>(L.pb + z));
            }
#pragma unroll
            for (int k = 0; k < W / 128; ++k) {
                const int q = lane + 32 * k;
                // va + u (vb - va), two voxels per instruction
                const float2 d0 = __ffma2_rn(make_float2(va[k].x, va[k].y), kNegOne2, make_float2(vb[k].x, vb[k].y));
                const float2 d1 = __ffma2_rn(make_float2(va[k].z, va[k].w), kNegOne2, make_float2(vb[k].z, vb[k].w));
                const float2 o0 = __ffma2_rn(u2, d0, make_float2(va[k].x, va[k].y));
                const float2 o1 = __ffma2_rn(u2, d1, make_float2(va[k].z, va[k].w));
                if (q < B.nq) dst[q] = make_float4(o0.x, o0.y, o1.x, o1.y);
            }
        }
        if (tid < kAlNL && b + 1 < n_batches) al_batch_params<INTERP, W, true>(S, P, buf ^ 1, b + 1, tid);
        __syncthreads();
        // ---------------- phase B
        // positions relative to the CENTRE of the window (|p| <= W / 2: one more bit of fp32 precision)
        const unsigned bias_b = lines_bias + (unsigned)(B.zc * 4);
#pragma unroll
        for (int c = 0; c < kAlTU; ++c) {
            const float a = (float)fma(S.t0[buf][c], rho, B.off);
#pragma unroll
            for (int s = 0; s < kAlSB; s += 2) {
                const float2 p = __ffma2_rn(make_float2((float)s, (float)(s + 1)), make_float2(dz[c], dz[c]), make_float2(a, a));
                const float2 x = __fadd2_rd(p, kMagic2);                  // bits = 0x4B400000 + floor(p)
                const float2 f = __fadd2_rn(x, kNegMagic2);
                const float2 d = __ffma2_rn(f, kNegOne2, p);              // p - floor(p)
                const unsigned a0 = (__float_as_uint(x.x) << 2) + bias_b + (unsigned)((c * kAlSB + s) * W * 4);
                const unsigned a1 = (__float_as_uint(x.y) << 2) + bias_b + (unsigned)((c * kAlSB + s + 1) * W * 4);
                const float2 v0 = make_float2(al_lds(a0), al_lds(a1));
                const float2 v1 = make_float2(al_lds(a0 + 4u), al_lds(a1 + 4u));
                const float2 wz = make_float2(ceil_weight<INTERP>(d.x), ceil_weight<INTERP>(d.y));
                const float2 df = __ffma2_rn(v0, kNegOne2, v1);           // v1 - v0
                acc[c] = __fadd2_rn(acc[c], __ffma2_rn(wz, df, v0));
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
            o[c] = (float)(P.G.delta * L) * (acc[c].x + acc[c].y);
        }
        float *dst = P.out + ((size_t)proj * P.nv + iv) * P.nu + iu0;
        if (P.out_vec && iu0 + kAlTU <= P.nu) {
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
