// fp_tma.cuh -- TMA-fed sampling kernel for the same class of poses as fp_aligned.cuh (detector v
// parallel to the volume's z axis, u perpendicular to it, no z-driven ray): circular orbits about
// the fastest memory index (PAPER.md:294 sec. 2.8, :312 sec. 3.2).
//
// A block owns 8 detector columns x 256 rows.  All its columns share the driving axis m (a block
// where the axis switches runs two passes), so at slice i they cut the same plane and need only the
// volume rows j_min .. j_min + R - 1 (R <= 12) along the slow transverse axis, over the z window the
// block's rows span.  A producer warp plans each batch of 4 slices in fp64 (Eqs. 4-6)
// and has the TMA engine copy that rows x window tile of every slice straight from the caller's
// volume into shared memory (cp.async.bulk.tensor, zero fill outside the volume = reading #2), four
// slices in flight behind mbarriers.  The consumer warps read the four taps of Eq. 15 (:165) of every
// sample from the tile and apply the product weights of Eq. 11 (:142); each thread carries two
// detector rows as one packed fp32x2 value.  No staging pass, no block-wide barrier in the loop.
//
// Projections are processed in groups of `group` (TmaParams): the blocks of the same detector tile of
// the group's projections are neighbours in launch order, so they start together and sweep the volume
// in step -- neighbouring orbit poses cut nearly the same volume rows on every slice, and whichever
// block comes second finds them in L2.  This takes the DRAM traffic below one volume pass per projection.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>
#include "fp_setup.cuh"
#include "fp_kernels.cuh"
#include "fp_aligned.cuh"

namespace fpk {

constexpr int kTmTU = 8;                 // detector columns per block
constexpr int kTmSB = 4;                 // slices per batch = pipeline stages
constexpr int kTmRows = 256;             // detector rows per block, two per consumer thread ...
constexpr int kTmRowsNarrow = 192;       // ... or 192 where the z window of 256 rows does not fit the largest box (wide cones)
__host__ __device__ constexpr int tm_threads(int rows) { return rows / 2 + 32; }   // consumers + one producer warp
constexpr int kTmW = 256;                // largest z window (voxels) = largest inner TMA box size
constexpr int kTmWBoxes = 4;             // inner box sizes 160, 192, 224, 256: the tile's row pitch follows the box
constexpr int kTmWMin = 160, kTmWStep = 32;
constexpr int kTmNR = 12;                // most volume rows per tile (largest box)
constexpr int kTmMaps = 5;               // tensor maps per pass: boxes of 4, 6, 8, 10, 12 rows
constexpr int kTmStageFloats = kTmNR * kTmW;
constexpr unsigned kTmTileBytes = kTmSB * kTmStageFloats * 4u;   // 48 KB of tiles; the zero region follows
constexpr int kTmZeroFloats = 3 * kTmW;  // zeros for columns without a sample: window positions -128 .. 128, rows j and j + 1

struct __align__(64) TmaParams {
    CUtensorMap map[2][kTmWBoxes][kTmMaps];   // [pass = driving axis x / y][box width][box of 4, 6, 8, 10 or 12 rows]
    GridDesc G;
    const ProjDesc *proj;              // all projections of the call
    const int *ids;                    // [n_sel] projections this launch handles
    float *out;                        // [n_proj][nv][nu]
    unsigned long long *sample_count;  // may be null
    unsigned int *err_flag;
    int nu, nv, n_sel;
    int fov;                           // 1: the volume is zero outside the inscribed cylinder about z (FP_OPT_FOV_CYLINDER)
    int out_vec;                       // 1: out is 16-byte aligned and nu % 4 == 0 (vector stores allowed)
    int group;                         // projections whose blocks are interleaved in launch order (>= 1)
};

struct TmColumn {          // per detector column and pass, all parametrised along the pass axis
    double inv_rm;         // 1 / r_m (of the nearest column of this pass if the column is not in it)
    double rt_s;           // r~ along the slow transverse axis
    int i_lo, i_hi;        // slices with -1 < p_slow < N_slow; empty if the column is not in this pass
};

struct __align__(16) TmShared {
    unsigned long long full[kTmSB], empty[kTmSB];      // mbarriers
    uint2 stage_col[kTmSB][kTmTU];     // per (stage, column): byte offset of its lower row in the tiles, weight bits
    double t0[2][kTmTU];               // per (batch parity, column): (i0 - s_m) / r_m
    double off[2];                     // per batch parity: s_z - z0
    unsigned pitch[2];                 // per batch parity: byte pitch of the tile rows (= box width * 4)
    TmColumn col[kTmTU];
    double s[3];                       // source, grid units
    double rxy[kTmTU][2];              // r_x, r_y per column
    double rho_first, rho_last;
    double s_m, s_s;                   // per pass
    int n_s, n_m, i_begin, dir, n_batches, any;
};

__device__ __forceinline__ unsigned tm_smem(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tm_mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(tm_smem(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void tm_mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tm_smem(bar)) : "memory");
}
__device__ __forceinline__ void tm_mbar_arrive_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tm_smem(bar)), "r"(bytes) : "memory");
}
// The suspend-time hint lets the warp sleep in hardware until the phase completes instead of spinning
// through issue slots that the other warps of the scheduler need.
__device__ __forceinline__ void tm_mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(tm_smem(bar)),
        "r"(parity), "r"(0x989680u)
        : "memory");
}
// Orders this thread's earlier generic-proxy accesses to shared memory (the tap loads) before later async-proxy
// accesses (the TMA engine's next write into the same stage) -- issued by every consumer thread before its warp
// releases a stage.
__device__ __forceinline__ void tm_fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tm_load_3d(const CUtensorMap *map, unsigned dst, unsigned long long *bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(tm_smem(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}

// Per pass (driving axis m = pass): Eqs. 2-5 for the block's columns, all
// parametrised along axis `pass`.  A column whose own driving axis is the other one (or that lies
// past the detector edge) gets an empty slice range -- it reads the tile's zero rows -- and
// borrows r_m from the nearest column of the pass so that its z positions stay inside the window.
// Executed by the producer warp.
__device__ __forceinline__ void tm_pass_setup(TmShared &S, const TmaParams &P, int pass, int iu0, int lane)
{
    const int c = lane & (kTmTU - 1);
    const double rm = S.rxy[c][pass], rs = S.rxy[c][1 - pass];
    const int true_m = fabs(S.rxy[c][1]) > fabs(S.rxy[c][0]) ? 1 : 0;        // Eq. 2 (z excluded by the host plan)
    const bool active = (true_m == pass) && (iu0 + c < P.nu) && (rm != 0.0);
    const double s_m = S.s[pass], s_s = S.s[1 - pass];
    const int n_m = P.G.n[pass], n_s = P.G.n[1 - pass];
    double inv = active ? 1.0 / rm : 0.0;
    const double rt = active ? __ddiv_rn(rs, rm) : 0.0;                      // Eq. 4
    int lo = 0, hi = -1;
    if (active) {
        hi = n_m - 1;
        clip_axis(s_s, s_m, rt, n_s, lo, hi);
        if (P.fov && lo <= hi) {
            const double cx = 0.5 * (P.G.n[0] - 1), cy = 0.5 * (P.G.n[1] - 1), rad = 0.5 * min(P.G.n[0], P.G.n[1]) + 1.5;
            clip_circle(s_s, s_m, rt, pass ? cy : cx, pass ? cx : cy, rad, lo, hi);
        }
        if (lo > hi) { lo = 0; hi = -1; }
    }
    const unsigned act = __ballot_sync(0xffffffffu, active) & 0xffu;
    int src = c;
    if (!active && act) {
        for (int d = 1; d < kTmTU; ++d) {
            if (c - d >= 0 && ((act >> (c - d)) & 1u)) { src = c - d; break; }
            if (c + d < kTmTU && ((act >> (c + d)) & 1u)) { src = c + d; break; }
        }
    }
    inv = __shfl_sync(0xffffffffu, inv, src);
    const int first = act ? __ffs(act) - 1 : 0;
    const int dir = __shfl_sync(0xffffffffu, inv, first) < 0.0 ? -1 : 1;
    const bool has = hi >= lo;
    const int glo = __reduce_min_sync(0xffffffffu, has ? lo : 0x7fffffff);
    const int ghi = __reduce_max_sync(0xffffffffu, has ? hi : -1);
    // spread of the slow-axis positions over the pass's columns, in rows, at either end of the slice range
    double rt_min = has ? rt : 1.0e300, rt_max = has ? rt : -1.0e300;
#pragma unroll
    for (int k = 1; k < kTmTU; k <<= 1) {
        rt_min = fmin(rt_min, __shfl_xor_sync(0xffffffffu, rt_min, k));
        rt_max = fmax(rt_max, __shfl_xor_sync(0xffffffffu, rt_max, k));
    }
    if (lane < kTmTU) {
        TmColumn C;
        C.inv_rm = inv;
        C.rt_s = rt;
        C.i_lo = lo;
        C.i_hi = hi;
        S.col[c] = C;
    }
    if (lane == 0) {
        const bool any = ghi >= glo;
        S.any = any;
        S.dir = dir;
        S.i_begin = any ? (dir > 0 ? glo : ghi) : 0;
        S.n_batches = any ? (ghi - glo + kTmSB) / kTmSB : 0;
        S.s_m = s_m;
        S.s_s = s_s;
        S.n_s = n_s;
        S.n_m = n_m;
        double spread = 0.0;
        if (any) spread = fmax(fabs((double)glo - s_m), fabs((double)(ghi + kTmSB) - s_m)) * (rt_max - rt_min);
        if ((int)fmin(spread, 1.0e6) + 3 > kTmNR) atomicOr(P.err_flag, 2u);
    }
}

// Producer warp, one batch: lane = (slice s of the batch) * 8 + column c.  Plans the four slices in
// fp64, then per slice waits until the consumers have released the stage, publishes the per-column
// tile row / weight and launches the TMA copy of the slice's rows x window tile.
template <int INTERP>
__device__ __forceinline__ void tm_produce_batch(TmShared &S, const TmaParams &P, unsigned tiles_smem, int pass, int b,
                                                 unsigned gb, int lane)
{
    const int c = lane & (kTmTU - 1), s = lane >> 3;
    const TmColumn C = S.col[c];
    const int i0 = S.i_begin + S.dir * (b * kTmSB), i = i0 + S.dir * s;
    const bool live = (C.i_lo <= i) && (i <= C.i_hi);
    // Eq. 6 along the slow axis, floor / weight as in Alg. 1 l.9-14
    const double ps = p_of_i(S.s_s, S.s_m, C.rt_s, i);
    const int j = __double2int_rd(ps);                       // floor, saturating
    const float u = ceil_weight<INTERP>((float)(ps - (double)j));
    const unsigned grp = 0xffu << (8 * s);
    const int jmin = __reduce_min_sync(grp, live ? j : 0x7fffffff);
    const int jmax = __reduce_max_sync(grp, live ? j : -0x7fffffff);
    const bool anylive = jmin != 0x7fffffff;
    // smallest box (4, 6, ..., 12 rows) that holds rows j_min .. j_max + 1
    const int mi = anylive ? min(max((jmax - jmin + 3) / 2 - 2, 0), (kTmNR - 4) / 2) : 0;
    const int box_rows = 4 + 2 * mi;
    const bool fits = live && (j - jmin + 2 <= box_rows);
    if (live && !fits) atomicOr(P.err_flag, 2u);
    // z window of the batch: p_z = s_z + t r_z is monotone in the row, so the extremes sit at the block's end rows
    const double t = __dmul_rn(__dsub_rn((double)i, S.s_m), C.inv_rm);
    const double za = S.s[2] + t * S.rho_first, zb = S.s[2] + t * S.rho_last;
    const int zlo = __reduce_min_sync(0xffffffffu, __double2int_rd(fmin(za, zb)));
    const int zhi = __reduce_max_sync(0xffffffffu, __double2int_rd(fmax(za, zb)));
    // taps k, k+1 with k = floor(p_z - z0) in [1, W-3] (one spare on either side for fp32 rounding)
    const int z0 = (zlo - 1) & ~3;
    const int need = zhi + 3 - z0;
    const bool winok = (zlo > -1000000000) && (zhi < 1000000000) && (need <= kTmW);
    // narrowest box that holds the window: less HBM / L2 / shared-memory traffic than always copying 256 voxels
    const int wi = winok ? min(max((need - kTmWMin + kTmWStep - 1) / kTmWStep, 0), kTmWBoxes - 1) : kTmWBoxes - 1;
    const int pitch = kTmWMin + kTmWStep * wi;
    if (!winok && lane == 0) atomicOr(P.err_flag, 1u);
    const int bp = gb & 1;
    if (s == 0) S.t0[bp][c] = winok ? __dmul_rn(__dsub_rn((double)i0, S.s_m), C.inv_rm) : 0.0;
    // positions are taken relative to the centre of the window (|p| <= 128: one more bit of fp32 precision than
    // relative to its start); a window that does not fit is never sampled out of bounds: every row is parked at p = 4
    const int zc = winok ? (need >> 1) : 0;
    if (lane == 0) {
        S.off[bp] = winok ? S.s[2] - (double)(z0 + zc) : 4.0;
        S.pitch[bp] = (unsigned)(pitch * 4);
    }
    const bool use = fits && winok;
    const unsigned row_off = (unsigned)((j - jmin) * pitch * 4);
    const unsigned wbits = use ? __float_as_uint(u) : 0u;
    // per slice: does it copy a tile, and how large a box (bit 0 = some column live, bits 1.. = box index)
    const int info = (anylive && winok) ? (1 | (mi << 1)) : 0;
#pragma unroll
    for (int ss = 0; ss < kTmSB; ++ss) {
        const int info_s = __shfl_sync(0xffffffffu, info, 8 * ss);
        const int jmin_s = __shfl_sync(0xffffffffu, jmin, 8 * ss);
        const int i_s = i0 + S.dir * ss;
        const int mi_s = info_s >> 1;
        const unsigned bytes = (info_s & 1) ? (unsigned)((4 + 2 * mi_s) * pitch * 4) : 0u;
        if (gb > 0) tm_mbar_wait(&S.empty[ss], (gb - 1) & 1);
        const unsigned phys = (unsigned)(ss * kTmStageFloats * 4);
        // published: the shared-window address of the word at window position p = 0 of the column's lower row, minus
        // (0x4B400000 << 2) -- the consumers add (bits of p + 1.5 * 2^23) << 2.  A column without a sample on this slice
        // reads the zero region behind the tiles (from its position 128 on: p may be negative).
        const unsigned addr0 = tiles_smem - (0x4B400000u << 2) + (use ? phys + row_off + (unsigned)(zc * 4) : kTmTileBytes + (unsigned)(kTmW / 2) * 4u);
        if (s == ss) S.stage_col[ss][c] = make_uint2(addr0, wbits);
        __syncwarp();
        if (lane == 0) {
            tm_fence_proxy_async();
            if (bytes) {
                tm_mbar_arrive_tx(&S.full[ss], bytes);
                const CUtensorMap *map = &P.map[pass][wi][mi_s];
                // tensor dimensions are (z, y, x); the slow axis is y for m = x and x for m = y
                if (pass == 0)
                    tm_load_3d(map, tiles_smem + phys, &S.full[ss], z0, jmin_s, i_s);
                else
                    tm_load_3d(map, tiles_smem + phys, &S.full[ss], z0, i_s, jmin_s);
            } else {
                tm_mbar_arrive(&S.full[ss]);
            }
        }
    }
}

// Step length Delta * ||r~|| of the ray of column c and a row with r_z = rho, fp64.
__device__ __forceinline__ float tm_step_length(const TmShared &S, const TmaParams &P, int c, double rho)
{
    const double rx = S.rxy[c][0], ry = S.rxy[c][1];
    const double rm = fabs(ry) > fabs(rx) ? ry : rx;
    double L = 0.0;
    if (rm != 0.0) {
        // r~ = r / r_m, summed x^2 + y^2 + z^2 like the definition
        const double tx = rx / rm, ty = ry / rm, tz = rho / rm;
        L = sqrt((tx * tx + ty * ty) + tz * tz);
    }
    return (float)(P.G.delta * L);
}

template <int INTERP, int ROWS>
__global__ void __launch_bounds__(tm_threads(ROWS), 4)
fp_tma_kernel(const __grid_constant__ TmaParams P)
{
    constexpr int kTmConsumers = ROWS / 2;
    static_assert(ROWS % 64 == 0 && ROWS <= 256, "whole consumer warps of two rows per thread");
    extern __shared__ __align__(128) unsigned char tm_smem_raw[];
    float *tiles = reinterpret_cast<float *>(tm_smem_raw);                   // kTmSB stages, then the zero region; 128-byte aligned
    TmShared &S = *reinterpret_cast<TmShared *>(tm_smem_raw + kTmTileBytes + sizeof(float) * kTmZeroFloats);

    const int tid = threadIdx.x, lane = tid & 31;
    // the shuffle tells the compiler that the warp index (and with it the role) is warp-uniform
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const bool producer = warp == kTmConsumers / 32;
    // blockIdx.x = (detector tile) * group + (projection within the group): see the header
    const int sel = blockIdx.z * P.group + (int)(blockIdx.x % (unsigned)P.group);
    if (sel >= P.n_sel) return;                            // the whole block (the last group may be short)
    const int proj = P.ids[sel];
    const double *g = P.proj[proj].g;
    const int iu0 = (int)(blockIdx.x / (unsigned)P.group) * kTmTU;
    const int row0 = blockIdx.y * ROWS;
    // consumer thread t carries detector rows row0 + t and row0 + ROWS / 2 + t
    const int ct = min(tid, kTmConsumers - 1);
    const int iv0 = min(row0 + ct, P.nv - 1), iv1 = min(row0 + kTmConsumers + ct, P.nv - 1);

    // ---- geometry ingest (Eq. 1): source and per-column r_x, r_y in grid units; barriers; zero rows
    if (tid < kTmTU) {
        const int iu = min(iu0 + tid, P.nu - 1);
        double s[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) s[a] = __ddiv_rn(__dsub_rn(g[a], P.G.origin[a]), P.G.delta);
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const double D = __dadd_rn(g[3 + a], __dmul_rn((double)iu, g[6 + a]));   // + iv * 0 exactly
            const double d = __ddiv_rn(__dsub_rn(D, P.G.origin[a]), P.G.delta);
            S.rxy[tid][a] = __dsub_rn(d, s[a]);
        }
        if (tid == 0) {
            S.s[0] = s[0];
            S.s[1] = s[1];
            S.s[2] = s[2];
            S.rho_first = al_rho(g, P.G, row0, s[2]);
            S.rho_last = al_rho(g, P.G, min(row0 + ROWS, P.nv) - 1, s[2]);
#pragma unroll
            for (int k = 0; k < kTmSB; ++k) {
                tm_mbar_init(&S.full[k], 1);
                tm_mbar_init(&S.empty[k], kTmConsumers / 32);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    for (int k = tid; k < kTmZeroFloats; k += blockDim.x) tiles[kTmSB * kTmStageFloats + k] = 0.0f;
    __syncthreads();

    // Two roles, one code region each (so that no role carries another role's registers); every warp
    // passes the same two block barriers per pass.
    int n_samples = 0;
    if (producer) {
        unsigned gb = 0;                                   // batches issued so far (consumers count alike)
        const unsigned tiles_smem = tm_smem(tiles);
        for (int pass = 0; pass < 2; ++pass) {
            __syncthreads();                               // every warp is done with the previous pass
            tm_pass_setup(S, P, pass, iu0, lane);
            __syncthreads();
            if (!S.any) continue;
            const int n_batches = S.n_batches;
            for (int b = 0; b < n_batches; ++b, ++gb) tm_produce_batch<INTERP>(S, P, tiles_smem, pass, b, gb, lane);
        }
    } else {
        const double rho0 = al_rho(g, P.G, iv0, S.s[2]), rho1 = al_rho(g, P.G, iv1, S.s[2]);
        const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f);    // 1.5 * 2^23
        const float2 kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
        const float2 kNegOne2 = make_float2(-1.0f, -1.0f);
        float2 acc[kTmTU];
#pragma unroll
        for (int c = 0; c < kTmTU; ++c) acc[c] = make_float2(0.0f, 0.0f);
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
                // Eq. 6 for z per (column, row), relative to the CENTRE of the batch's window: p = a + s dz
                // with |p| <= 128, i.e. fp32 positions good to 4e-6 voxel
                float2 a[kTmTU];
                unsigned pitchB;
                {
                    const double off = S.off[par];
                    pitchB = S.pitch[par];
#pragma unroll
                    for (int c = 0; c < kTmTU; ++c) {
                        const double t0 = S.t0[par][c];
                        a[c] = make_float2((float)fma(t0, rho0, off), (float)fma(t0, rho1, off));
                    }
                }
#pragma unroll
                for (int s = 0; s < kTmSB; ++s) {
                    if (s) {
                        tm_mbar_wait(&S.full[s], par);
                        // release the PREVIOUS stage here, where its loads have long returned: the proxy fence (generic
                        // reads before the next async-proxy write into the stage) then has nothing to wait for
                        __syncwarp();
                        if (lane == 0) tm_mbar_arrive(&S.empty[s - 1]);
                    }
                    const float2 fs = make_float2((float)s, (float)s);
                    uint4 pq2 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                    for (int c = 0; c < kTmTU; ++c) {
                        // one 16-byte broadcast load serves two columns
                        if ((c & 1) == 0) pq2 = *reinterpret_cast<const uint4 *>(&S.stage_col[s][c]);
                        const uint2 pc = (c & 1) ? make_uint2(pq2.z, pq2.w) : make_uint2(pq2.x, pq2.y);
                        const float2 p = __ffma2_rn(fs, dz[c], a[c]);
                        const float2 x = __fadd2_rd(p, kMagic2);                  // bits = 0x4B400000 + floor(p)
                        const float2 f = __fadd2_rn(x, kNegMagic2);
                        const float2 d = __ffma2_rn(f, kNegOne2, p);              // p - floor(p)
                        // pc.x = shared-window address of word 0 of the column's lower row minus (0x4B400000 << 2)
                        const unsigned a0 = (__float_as_uint(x.x) << 2) + pc.x, a1 = (__float_as_uint(x.y) << 2) + pc.x;
                        const float2 v00 = make_float2(al_lds(a0), al_lds(a1));
                        const float2 v01 = make_float2(al_lds(a0 + 4u), al_lds(a1 + 4u));
                        const unsigned b0 = a0 + pitchB, b1 = a1 + pitchB;        // row j + 1
                        const float2 v10 = make_float2(al_lds(b0), al_lds(b1));
                        const float2 v11 = make_float2(al_lds(b0 + 4u), al_lds(b1 + 4u));
                        const float2 wz = make_float2(ceil_weight<INTERP>(d.x), ceil_weight<INTERP>(d.y));
                        const float uy = __uint_as_float(pc.y);
                        const float2 t0 = __ffma2_rn(wz, __ffma2_rn(v00, kNegOne2, v01), v00);   // row j
                        const float2 t1 = __ffma2_rn(wz, __ffma2_rn(v10, kNegOne2, v11), v10);   // row j + 1
                        acc[c] = __fadd2_rn(acc[c], __ffma2_rn(make_float2(uy, uy), __ffma2_rn(t0, kNegOne2, t1), t0));
                    }
                    if (s == kTmSB - 1) {
                        __syncwarp();
                        if (lane == 0) tm_mbar_arrive(&S.empty[s]);
                    }
                }
            }
        }
        // ---- weight by the step length Delta * ||r~|| and store
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int iv = row0 + h * kTmConsumers + tid;
            if (iv >= P.nv) continue;
            const double rho = h ? rho1 : rho0;
            float o[kTmTU];
#pragma unroll
            for (int c = 0; c < kTmTU; ++c) o[c] = tm_step_length(S, P, c, rho) * (h ? acc[c].y : acc[c].x);
            float *dst = P.out + ((size_t)proj * P.nv + iv) * P.nu + iu0;
            if (P.out_vec && iu0 + kTmTU <= P.nu) {
                reinterpret_cast<float4 *>(dst)[0] = make_float4(o[0], o[1], o[2], o[3]);
                reinterpret_cast<float4 *>(dst)[1] = make_float4(o[4], o[5], o[6], o[7]);
            } else {
#pragma unroll
                for (int c = 0; c < kTmTU; ++c)
                    if (iu0 + c < P.nu) dst[c] = o[c];
            }
            if (P.sample_count) {
                for (int c = 0; c < kTmTU; ++c)
                    if (iu0 + c < P.nu) {
                        const RaySetup R = ray_setup(g, P.G, iu0 + c, iv);
                        n_samples += max(R.i_last - R.i_first + 1, 0);
                    }
            }
        }
    }
    if (P.sample_count) block_count_samples(P.sample_count, n_samples);
}

constexpr size_t tma_smem_bytes() { return kTmTileBytes + sizeof(float) * kTmZeroFloats + sizeof(TmShared); }

}  // namespace fpk
