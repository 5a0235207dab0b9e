// fp_bp.cuh -- back-projection for the poses of fp_tma.cuh (detector v parallel to the volume's z axis, u
// perpendicular to it, no z-driven ray): the transpose of fp_tma_kernel, sample by sample.
//
// vol_out = A^T proj.  A block owns the same 8 detector columns x
// 256 rows as fp_tma_kernel, a producer warp plans the same batches of four slices in fp64 (Eqs. 4-6,
// volume row j and weight u of every column on every slice, the centre of the batch's z window),
// and the consumer threads compute, per column and slice, the SAME fp32 z positions, floors and weights as the
// forward kernel (two detector rows per thread as one packed fp32x2 value).  Where the forward kernel reads four
// taps and accumulates w * vol[tap], this one adds w * Delta ||r~|| * proj[ray] to the four taps with fp32
// reductions in L2 (RED.ADD.F32).  The lanes of a warp are neighbouring detector rows, i.e. neighbouring z: one
// reduction instruction covers about 22 consecutive voxels of one volume row (3-4 sectors), where the ray-driven
// scatter of fp_backproject_kernel (fp_kernels.cuh) touched 8.6 sectors and spent 101 instructions per warp-sample.
// Nothing is staged in shared memory, so no window or row limit applies: every pose the host plan calls aligned
// takes this kernel.  Taps outside the volume belong to the zero extension (reading #2) and receive nothing.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "fp_setup.cuh"
#include "fp_kernels.cuh"
#include "fp_aligned.cuh"
#include "fp_tma.cuh"

namespace fpk {

constexpr int kBpRows = 256;                       // detector rows per block, two per consumer thread
constexpr int kBpConsumers = kBpRows / 2;
constexpr int kBpThreads = kBpConsumers + 32;      // + one planning warp

struct __align__(64) BpParams {
    TmaParams T;                       // geometry, grid, detector size, projection ids (maps, out, counters unused)
    const float *in;                   // [n_proj][nv][nu]
    float *vol;                        // [nx][ny][nz], cleared by the caller
};

struct __align__(16) BpShared {
    TmShared S;
    // per (stage, column): element index of (row j, window centre) and of (row j + 1, window centre) in the volume
    // (0xFFFFFFFF: that row is outside the volume or the column has no sample on the slice), weight bits of u
    // .w = 1: neighbouring detector rows are more than half a voxel apart in z on this slice, so at most two
    // neighbouring lanes share a word and the warp merges them before the reduction (see the kernel)
    uint4 tap[kTmSB][kTmTU];
    int zbase[2];                      // per batch parity: z of the window centre
    double drho;                       // |r_z(row + 1) - r_z(row)|, grid units
};

// Predicated fp32 reduction in L2 (no branch around it).
__device__ __forceinline__ void bp_red(float *p, float v, bool on)
{
    asm volatile(
        "{\n"
        ".reg .pred q;\n"
        "setp.ne.b32 q, %2, 0;\n"
        "@q red.global.add.f32 [%0], %1;\n"
        "}\n" ::"l"(p),
        "f"(v), "r"((int)on)
        : "memory");
}

// Planning warp, one batch: lane = (slice s of the batch) * 8 + column c.  The same fp64 plan as tm_produce_batch
// (fp_tma.cuh) -- volume row j = floor(p_slow) and weight u per (slice, column), centre of the batch's z window --
// published as volume element indices instead of tile addresses; no copy is issued.
template <int INTERP>
__device__ __forceinline__ void bp_plan_batch(BpShared &B, const BpParams &P, int pass, int b, unsigned gb, int lane)
{
    TmShared &S = B.S;
    const int c = lane & (kTmTU - 1), s = lane >> 3;
    const TmColumn C = S.col[c];
    const int i0 = S.i_begin + S.dir * (b * kTmSB), i = i0 + S.dir * s;
    const bool live = (C.i_lo <= i) && (i <= C.i_hi);
    // Eq. 6 along the slow axis, floor / weight as in Alg. 1 l.9-14
    const double ps = p_of_i(S.s_s, S.s_m, C.rt_s, i);
    const int j = __double2int_rd(ps);
    const float u = ceil_weight<INTERP>((float)(ps - (double)j));
    // z window of the batch: p_z = s_z + t r_z is monotone in the row, so the extremes sit at the block's end rows
    const double t = __dmul_rn(__dsub_rn((double)i, S.s_m), C.inv_rm);
    const double za = S.s[2] + t * S.rho_first, zb = S.s[2] + t * S.rho_last;
    const int zlo = __reduce_min_sync(0xffffffffu, __double2int_rd(fmin(za, zb)));
    const int zhi = __reduce_max_sync(0xffffffffu, __double2int_rd(fmax(za, zb)));
    const bool winok = (zlo > -1000000000) && (zhi < 1000000000);
    if (!winok && lane == 0) atomicOr(P.T.err_flag, 1u);
    // positions are taken relative to the centre of the window, like the forward kernel's
    const int zbase = winok ? zlo + ((zhi - zlo) >> 1) : 0;
    const int bp = gb & 1;
    if (s == 0) S.t0[bp][c] = winok ? __dmul_rn(__dsub_rn((double)i0, S.s_m), C.inv_rm) : 0.0;
    // element index of the start of volume row (slice i, slow index j): m = x: (i, j, 0), m = y: (j, i, 0)
    const long long ny = P.T.G.n[1], nz = P.T.G.n[2];
    const bool r0 = live && winok && j >= 0 && j < S.n_s, r1 = live && winok && j + 1 >= 0 && j + 1 < S.n_s;
    const long long e0 = pass == 0 ? ((long long)i * ny + j) * nz : ((long long)j * ny + i) * nz;
    const long long estep = pass == 0 ? nz : ny * nz;
    const unsigned merge = fabs(t) * B.drho > 0.505 ? 1u : 0u;
    const uint4 tap = make_uint4(r0 ? (unsigned)e0 : 0xFFFFFFFFu, r1 ? (unsigned)(e0 + estep) : 0xFFFFFFFFu, __float_as_uint(u), merge);
#pragma unroll
    for (int ss = 0; ss < kTmSB; ++ss) {
        if (gb > 0) tm_mbar_wait(&S.empty[ss], (gb - 1) & 1);
        if (ss == 0 && lane == 0) {
            S.off[bp] = winok ? S.s[2] - (double)zbase : 4.0;
            B.zbase[bp] = zbase;
        }
        if (s == ss) B.tap[ss][c] = tap;
        __syncwarp();
        if (lane == 0) tm_mbar_arrive(&S.full[ss]);
    }
}

template <int INTERP>
__global__ void __launch_bounds__(kBpThreads, 5)
fp_bp_aligned_kernel(const __grid_constant__ BpParams P)
{
    __shared__ BpShared B;
    TmShared &S = B.S;
    const TmaParams &T = P.T;

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const bool producer = warp == kBpConsumers / 32;
    // blockIdx.x = (detector tile) * group + (projection within the group), as in fp_tma_kernel
    const int sel = blockIdx.z * T.group + (int)(blockIdx.x % (unsigned)T.group);
    if (sel >= T.n_sel) return;
    const int proj = T.ids[sel];
    const double *g = T.proj[proj].g;
    const int iu0 = (int)(blockIdx.x / (unsigned)T.group) * kTmTU;
    const int row0 = blockIdx.y * kBpRows;
    // consumer thread t carries detector rows row0 + t and row0 + 128 + t
    const int ct = min(tid, kBpConsumers - 1);
    const int iv0 = row0 + ct, iv1 = row0 + kBpConsumers + ct;

    // ---- geometry ingest (Eq. 1): source and per-column r_x, r_y in grid units; barriers
    if (tid < kTmTU) {
        const int iu = min(iu0 + tid, T.nu - 1);
        double s[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) s[a] = __ddiv_rn(__dsub_rn(g[a], T.G.origin[a]), T.G.delta);
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const double D = __dadd_rn(g[3 + a], __dmul_rn((double)iu, g[6 + a]));   // + iv * 0 exactly
            const double d = __ddiv_rn(__dsub_rn(D, T.G.origin[a]), T.G.delta);
            S.rxy[tid][a] = __dsub_rn(d, s[a]);
        }
        if (tid == 0) {
            S.s[0] = s[0];
            S.s[1] = s[1];
            S.s[2] = s[2];
            S.rho_first = al_rho(g, T.G, row0, s[2]);
            S.rho_last = al_rho(g, T.G, min(row0 + kBpRows, T.nv) - 1, s[2]);
            B.drho = fabs(g[11]) / T.G.delta;
#pragma unroll
            for (int k = 0; k < kTmSB; ++k) {
                tm_mbar_init(&S.full[k], 1);
                tm_mbar_init(&S.empty[k], kBpConsumers / 32);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    __syncthreads();

    if (producer) {
        unsigned gb = 0;
        for (int pass = 0; pass < 2; ++pass) {
            __syncthreads();                               // every warp is done with the previous pass
            tm_pass_setup(S, T, pass, iu0, lane);
            __syncthreads();
            if (!S.any) continue;
            const int n_batches = S.n_batches;
            for (int b = 0; b < n_batches; ++b, ++gb) bp_plan_batch<INTERP>(B, P, pass, b, gb, lane);
        }
    } else {
        const double rho0 = al_rho(g, T.G, min(iv0, T.nv - 1), S.s[2]), rho1 = al_rho(g, T.G, min(iv1, T.nv - 1), S.s[2]);
        const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f);    // 1.5 * 2^23
        const float2 kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
        const float2 kNegOne2 = make_float2(-1.0f, -1.0f);
        // what each of the thread's 16 rays carries back: Delta ||r~|| proj[ray]
        float2 yb[kTmTU];
        bool any0 = false, any1 = false;
#pragma unroll
        for (int c = 0; c < kTmTU; ++c) {
            float y0 = 0.0f, y1 = 0.0f;
            if (iu0 + c < T.nu) {
                if (iv0 < T.nv) y0 = __ldg(P.in + ((size_t)proj * T.nv + iv0) * T.nu + iu0 + c) * tm_step_length(S, T, c, rho0);
                if (iv1 < T.nv) y1 = __ldg(P.in + ((size_t)proj * T.nv + iv1) * T.nu + iu0 + c) * tm_step_length(S, T, c, rho1);
            }
            yb[c] = make_float2(y0, y1);
            any0 |= y0 != 0.0f;
            any1 |= y1 != 0.0f;
        }
        // a row past the detector edge (or with nothing to add) never passes the z test below
        const int dead0 = any0 ? 0 : 0x40000000, dead1 = any1 ? 0 : 0x40000000;
        const unsigned nz = (unsigned)T.G.n[2];
        float *__restrict__ vol = P.vol;
        unsigned gb = 0;                                   // batches consumed so far
        for (int pass = 0; pass < 2; ++pass) {
            __syncthreads();
            __syncthreads();
            if (!S.any) continue;
            const int n_batches = S.n_batches;
            float2 dz[kTmTU];                              // z increment per slice of the two rows, per column
#pragma unroll
            for (int c = 0; c < kTmTU; ++c) {
                const double st = fabs(S.col[c].inv_rm);
                dz[c] = make_float2((float)(rho0 * st), (float)(rho1 * st));
            }
            for (int b = 0; b < n_batches; ++b, ++gb) {
                const unsigned par = gb & 1;
                tm_mbar_wait(&S.full[0], par);
                // Eq. 6 for z per (column, row), relative to the centre of the batch's window (fp_tma.cuh)
                float2 a[kTmTU];
                const double off = S.off[par];
                const int zb0 = B.zbase[par] - 0x4B400000 + dead0, zb1 = B.zbase[par] - 0x4B400000 + dead1;
#pragma unroll
                for (int c = 0; c < kTmTU; ++c) {
                    const double t0 = S.t0[par][c];
                    a[c] = make_float2((float)fma(t0, rho0, off), (float)fma(t0, rho1, off));
                }
                // not unrolled: the body (8 columns x 16 reductions) already fills the instruction cache
#pragma unroll 1
                for (int s = 0; s < kTmSB; ++s) {
                    if (s) tm_mbar_wait(&S.full[s], par);
                    const float2 fs = make_float2((float)s, (float)s);
#pragma unroll
                    for (int c = 0; c < kTmTU; ++c) {
                        const uint4 tp = B.tap[s][c];
                        const float2 p = __ffma2_rn(fs, dz[c], a[c]);
                        const float2 x = __fadd2_rd(p, kMagic2);                  // bits = 0x4B400000 + floor(p)
                        const float2 f = __fadd2_rn(x, kNegMagic2);
                        const float2 d = __ffma2_rn(f, kNegOne2, p);              // p - floor(p)
                        const float2 wz = make_float2(ceil_weight<INTERP>(d.x), ceil_weight<INTERP>(d.y));
                        const float uy = __uint_as_float(tp.z);
                        // rows j + 1 and j of the volume, then taps k + 1 and k of each (the weights of Eq. 11, :142)
                        const float2 hi = __fmul2_rn(yb[c], make_float2(uy, uy));
                        const float2 lo = __ffma2_rn(hi, kNegOne2, yb[c]);
                        const float2 t01 = __fmul2_rn(lo, wz), t11 = __fmul2_rn(hi, wz);
                        float2 t00 = __ffma2_rn(t01, kNegOne2, lo), t10 = __ffma2_rn(t11, kNegOne2, hi);
                        float2 t01m = t01, t11m = t11;
                        int k0 = (int)__float_as_uint(x.x) + zb0, k1 = (int)__float_as_uint(x.y) + zb1;   // z of the lower tap
                        if (tp.w) {
                            // lanes are neighbouring detector rows, z is monotone in the row, rows are more than half a
                            // voxel apart: a word is shared by at most two neighbouring lanes.  The first of them adds
                            // the second one's values to its own and the second one drops out: every reduction
                            // instruction then carries each word once (half the L2 reduction operations).
                            const unsigned full = 0xffffffffu;
                            const int k0n = __shfl_down_sync(full, k0, 1), k0p = __shfl_up_sync(full, k0, 1);
                            const int k1n = __shfl_down_sync(full, k1, 1), k1p = __shfl_up_sync(full, k1, 1);
                            const bool take0 = lane < 31 && k0n == k0, take1 = lane < 31 && k1n == k1;
                            const float a00 = __shfl_down_sync(full, t00.x, 1), a01 = __shfl_down_sync(full, t01m.x, 1);
                            const float a10 = __shfl_down_sync(full, t10.x, 1), a11 = __shfl_down_sync(full, t11m.x, 1);
                            const float b00 = __shfl_down_sync(full, t00.y, 1), b01 = __shfl_down_sync(full, t01m.y, 1);
                            const float b10 = __shfl_down_sync(full, t10.y, 1), b11 = __shfl_down_sync(full, t11m.y, 1);
                            if (take0) { t00.x += a00; t01m.x += a01; t10.x += a10; t11m.x += a11; }
                            if (take1) { t00.y += b00; t01m.y += b01; t10.y += b10; t11m.y += b11; }
                            if (lane > 0 && k0p == k0) k0 = 0x40000000;
                            if (lane > 0 && k1p == k1) k1 = 0x40000000;
                        }
                        const bool a0 = (unsigned)k0 < nz, a1 = (unsigned)(k0 + 1) < nz;
                        const bool b0 = (unsigned)k1 < nz, b1 = (unsigned)(k1 + 1) < nz;
                        const bool r0 = tp.x != 0xFFFFFFFFu, r1 = tp.y != 0xFFFFFFFFu;
                        // one branch per detector row: a lane that dropped out in the merge (or whose row is past the
                        // detector edge) skips its eight reductions together; the interior case runs them unguarded
                        if (a0 || a1) {
                            float *q0 = vol + ((long long)tp.x + k0), *q1 = vol + ((long long)tp.y + k0);
                            if (a0 && a1 && r0 && r1) {
                                atomicAdd(q0, t00.x);
                                atomicAdd(q0 + 1, t01m.x);
                                atomicAdd(q1, t10.x);
                                atomicAdd(q1 + 1, t11m.x);
                            } else {
                                bp_red(q0, t00.x, r0 && a0);
                                bp_red(q0 + 1, t01m.x, r0 && a1);
                                bp_red(q1, t10.x, r1 && a0);
                                bp_red(q1 + 1, t11m.x, r1 && a1);
                            }
                        }
                        if (b0 || b1) {
                            float *q0 = vol + ((long long)tp.x + k1), *q1 = vol + ((long long)tp.y + k1);
                            if (b0 && b1 && r0 && r1) {
                                atomicAdd(q0, t00.y);
                                atomicAdd(q0 + 1, t01m.y);
                                atomicAdd(q1, t10.y);
                                atomicAdd(q1 + 1, t11m.y);
                            } else {
                                bp_red(q0, t00.y, r0 && b0);
                                bp_red(q0 + 1, t01m.y, r0 && b1);
                                bp_red(q1, t10.y, r1 && b0);
                                bp_red(q1 + 1, t11m.y, r1 && b1);
                            }
                        }
                    }
                    // the plan of this stage has been read
                    __syncwarp();
                    if (lane == 0) tm_mbar_arrive(&S.empty[s]);
                }
            }
        }
    }
}

}  // namespace fpk
