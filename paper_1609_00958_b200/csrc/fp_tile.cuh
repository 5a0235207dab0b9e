// fp_tile.cuh -- TMA-staged sampling kernel for GENERAL poses (any source / detector orientation, all three
// driving axes): the same Alg. 1 as fp_direct_kernel, but the four taps of Eq. 15 (:165) come
// from shared memory instead of four uncoalesced global loads per sample.
//
// A block owns a 32 x 16 tile of detector pixels (512 rays, two per consumer thread as one packed fp32x2
// value).  If its four corner rays share the driving axis m (Eq. 2, :81) -- then every ray of the tile does,
// the set { r : m(r) = m } being a convex cone -- the rays cut slice i of axis m inside the quadrilateral spanned by
// the corner rays' intersection points (the map pixel -> intersection point is projective).  A producer warp
// evaluates those four points per slice in fp64 (Eq. 6, :104) and has the TMA engine copy the bounding box of the
// quadrilateral (rows x cols voxels of the slice plane, zero-filled outside the volume = reading #2; the fast
// in-plane axis is the contiguous one: the caller's array for m = x, y, the y-fastest copy of the layout stage,
// PAPER.md:290-294, for m = z) into a ring of shared-memory stages behind full / empty mbarriers.  The consumers
// step through the block's slices together: position by one packed FMA per in-plane axis from an fp64 anchor
// that is renewed every 64 slices (integer + fraction split, so the fp32 operands stay below 33 whatever the
// volume size), floor by a round-down add, four shared-memory taps, product weights of Eq. 11 (:142).  A ray
// outside its own slice range [i_first, i_last] has a transverse coordinate outside (-1, N_t), so all its taps
// lie in the zero fill: no masks, no per-ray loop bounds.
//
// Three blocks per SM (72 registers): the fp64 parameters of a thread's two rays are parked in shared memory
// during the loop (read back once per segment), and the loop walks the barrier / origin arrays with one running
// byte address, so its stage bookkeeping runs on the uniform datapath (45 instructions per warp and slice).
//
// Tiles whose corner rays have different driving axes (about 4 % of C4's tiles), whose box would not fit the
// largest stage, or whose rays all miss run the direct path (fp_kernels.cuh) inside the same launch.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>
#include "fp_setup.cuh"
#include "fp_kernels.cuh"
#include "fp_tma.cuh"

namespace fpk {

constexpr int kTlU = 32, kTlV = 16;              // detector pixels per block along u and v
constexpr int kTlConsumers = kTlU * kTlV / 2;    // two rays per consumer thread
constexpr int kTlThreads = kTlConsumers + 32;    // + one producer warp
constexpr int kTlSizes = 5;                      // box classes per dimension: a block takes the smallest rows x cols box that holds its quadrilaterals
__host__ __device__ constexpr int tl_rows(int k) { return k == 0 ? 20 : (k == 1 ? 28 : (k == 2 ? 36 : (k == 3 ? 44 : 60))); }
__host__ __device__ constexpr int tl_cols(int k) { return k == 0 ? 28 : (k == 1 ? 36 : (k == 2 ? 44 : (k == 3 ? 52 : 68))); }
constexpr int kTlStagesMax = 12;                 // slices in flight: as many stages as fit the 48 KB of tiles, at most 12
constexpr unsigned kTlTileBytes = 49152u;
// a stage is the box rounded up to 128 B (TMA destination alignment)
__host__ __device__ constexpr unsigned tl_stage_stride(int rows, int cols) { return ((unsigned)(rows * cols * 4) + 127u) & ~127u; }

struct __align__(64) TileParams {
    CUtensorMap map[3][kTlSizes][kTlSizes];   // [driving axis][rows class][cols class]
    GridDesc G;
    AxisLayout lay[3];                 // for the direct path of tiles that do not qualify
    const ProjDesc *proj;              // all projections of the call
    const int *ids;                    // [n_sel] projections this launch handles
    float *out;                        // [n_proj][nv][nu]
    unsigned long long *sample_count;  // may be null
    int nu, nv, n_sel;
    int z_staged;                      // 1: map[2] covers the y-fastest copy of the layout stage; 0: z-driven tiles run the direct path
};

struct TlCorner {                      // one corner ray, parametrised along the tile's driving axis
    double s_m, s_a, s_b, rt_a, rt_b;
};

struct TlPass {                        // one pass = the tile's rays whose driving axis is m
    int lo, hi;                        // union of their slice ranges; hi < lo: no such ray
    int size_r, size_c, staged;        // box classes; staged = 1: staged pass, 0: those rays take the direct path
    int pad_;
};

struct __align__(16) TlShared {
    // the consumers walk these three arrays with ONE running byte address (stage * 8): keep them 8 bytes per stage
    // and in this order (kTlEmptyOff, kTlOrgOff below)
    unsigned long long full[kTlStagesMax], empty[kTlStagesMax];
    uint2 org[kTlStagesMax];           // .x per stage: byte address of tile word (0, 0) minus (js0 * pitch + kf0) * 4 terms, see below
    unsigned long long sink;           // barrier nobody waits on: takes the release of "the stage before the first"
    TlCorner corner[3][4];             // per pass (= driving axis m): the four corner rays parametrised along m
    double cr[4][3];                   // the corner rays' directions r (Eq. 1), grid units
    double cs[3];                      // the source, grid units
    TlPass pass[3];
};

constexpr unsigned kTlEmptyOff = 8u * kTlStagesMax, kTlOrgOff = 16u * kTlStagesMax, kTlSinkOff = 24u * kTlStagesMax;
static_assert(offsetof(TlShared, empty) == kTlEmptyOff && offsetof(TlShared, org) == kTlOrgOff && offsetof(TlShared, sink) == kTlSinkOff,
              "TlShared layout");
// fp64 parameters of the two rays of every consumer thread, parked in shared memory while the sampling loop runs (they
// are needed once per segment only; in registers they would cost a third of the occupancy): [4][kTlConsumers] double2
// plus one slot per pass holding a corner ray's parameters: what a ray reads in a pass that is not its own
constexpr int kTlRaySlots = kTlConsumers + 4;
constexpr unsigned kTlRayBytes = 4u * kTlRaySlots * 16u;

__device__ __forceinline__ void tl_wait_addr(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity), "r"(0x989680u)
        : "memory");
}
__device__ __forceinline__ void tl_arrive_addr(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// Direct path for one ray (the body of fp_direct_kernel).
template <int INTERP>
__device__ __forceinline__ float tl_direct_ray(const RaySetup &R, const AxisLayout *lay)
{
    float acc = 0.0f;
    if (R.i_last >= R.i_first) {
        const AxisLayout &A = lay[R.m];
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
    return acc;
}

// Direct path for one pixel, set-up included (kept out of line: only tiles whose box does not fit a stage, or whose
// z-driven rays have no y-fastest copy to be staged from, come here).
template <int INTERP>
__device__ __noinline__ float tl_direct_pixel(const double *g, const GridDesc &G, const AxisLayout *lay, int iu, int iv)
{
    const RaySetup R = ray_setup(g, G, iu, iv);
    return (float)(G.delta * R.L) * tl_direct_ray<INTERP>(R, lay);
}

__device__ __forceinline__ void tl_mbar_inval(unsigned long long *bar)
{
    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(tm_smem(bar)) : "memory");
}

template <int INTERP>
__global__ void __launch_bounds__(kTlThreads, 3)
fp_tile_kernel(const __grid_constant__ TileParams P)
{
    extern __shared__ __align__(128) unsigned char tl_smem_raw[];
    TlShared &S = *reinterpret_cast<TlShared *>(tl_smem_raw + kTlTileBytes);
    const unsigned tiles_smem = tm_smem(tl_smem_raw);

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const bool producer = warp == kTlConsumers / 32;
    const int proj = P.ids[blockIdx.z];
    const ProjDesc *pd = P.proj + proj;
    const double *g = pd->g;
    const int tu0 = blockIdx.x * kTlU, tv0 = blockIdx.y * kTlV;

    // ---- corner rays (Eq. 1, the operations of ray_setup): the tile's rectangle, also where it sticks out past the
    //      detector edge
    if (tid < 4) {
        const int iu = tu0 + ((tid & 1) ? kTlU - 1 : 0), iv = tv0 + ((tid & 2) ? kTlV - 1 : 0);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double D = __dadd_rn(__dadd_rn(g[3 + a], __dmul_rn((double)iu, g[6 + a])), __dmul_rn((double)iv, g[9 + a]));
            const double s = __ddiv_rn(__dsub_rn(g[a], P.G.origin[a]), P.G.delta);
            const double d = __ddiv_rn(__dsub_rn(D, P.G.origin[a]), P.G.delta);
            S.cr[tid][a] = __dsub_rn(d, s);
            if (tid == 0) S.cs[a] = s;
        }
    }
    if (tid == 0) {
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            S.pass[m].lo = 0x7fffffff;
            S.pass[m].hi = -1;
            S.pass[m].staged = 0;
        }
#pragma unroll
        for (int k = 0; k < kTlStagesMax; ++k) {
            tm_mbar_init(&S.full[k], 1);
            tm_mbar_init(&S.empty[k], kTlConsumers / 32);
        }
        tm_mbar_init(&S.sink, kTlConsumers / 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ---- per-ray exact set-up (fp64, Eqs. 1-6 and the exact slice range); lanes run along the detector axis that
    //      maps onto the contiguous in-plane axis of the first corner's driving axis (neighbouring lanes ->
    //      neighbouring words)
    bool lanes_v;
    {
        const double r0 = fabs(S.cr[0][0]), r1 = fabs(S.cr[0][1]), r2 = fabs(S.cr[0][2]);
        const int m0 = (r2 > r1 && r2 > r0) ? 2 : (r1 > r0 ? 1 : 0);
        const int fa = m0 == 2 ? 1 : 2;                       // fast in-plane axis: z, or y on the permuted copy
        lanes_v = fabs(g[9 + fa]) > fabs(g[6 + fa]);
    }
    int iuA = 0, ivA = 0, iuB = 0, ivB = 0;
    if (!producer) {
        // A warp's 32 rays of one tap load form a 4 x 8 pixel patch, 4 along the detector axis that maps onto the
        // contiguous in-plane axis: about 3 x 7 voxels of the slice plane, 8 tile rows of 4 words each.  With the
        // tile pitches of the box classes (28, 36, 44, 52, 68 words = 4, 12 or 20 modulo 32 up to sign) consecutive tile
        // rows are 4 banks apart, so the patch's words fall into distinct banks: 1.3-1.5 shared-memory wavefronts
        // per load where a line of 32 pixels, which crosses tile rows at a stride the pitch does not match, needs 2.1.
        const int w = tid >> 5, la = lane & 3, lb = lane >> 2;
        if (!lanes_v) {                                       // patch: 4 along u x 8 along v; rays A, B: the two halves in v
            iuA = iuB = tu0 + 4 * w + la;
            ivA = tv0 + lb;
            ivB = tv0 + lb + 8;
        } else {                                              // patch: 4 along v x 8 along u; rays A, B: neighbouring patches in u
            ivA = ivB = tv0 + 4 * (w & 3) + la;
            iuA = tu0 + 16 * (w >> 2) + lb;
            iuB = iuA + 8;
        }
    }
    const bool liveA = !producer && iuA < P.nu && ivA < P.nv, liveB = !producer && iuB < P.nu && ivB < P.nv;
    // a thread's state across the passes: driving axis of its two rays (3: the ray misses the volume), the scales
    // Delta ||r~||; the fp64 parameters go to shared memory (read back once per segment)
    int mA = 3, mB = 3, n_samples = 0;
    float scA = 0.0f, scB = 0.0f;
    double2 *rayp = reinterpret_cast<double2 *>(tl_smem_raw + kTlTileBytes + sizeof(TlShared));
    if (!producer) {
        const double src[3] = {S.cs[0], S.cs[1], S.cs[2]};       // the source in grid units, computed once per block
        const RaySetup RA = ray_setup_from(g, P.G, src, min(iuA, P.nu - 1), min(ivA, P.nv - 1));
        const RaySetup RB = ray_setup_from(g, P.G, src, min(iuB, P.nu - 1), min(ivB, P.nv - 1));
        if (RA.i_last >= RA.i_first) { mA = RA.m; scA = (float)(P.G.delta * RA.L); }
        if (RB.i_last >= RB.i_first) { mB = RB.m; scB = (float)(P.G.delta * RB.L); }
        rayp[0 * kTlRaySlots + tid] = make_double2(RA.s_a, RA.rt_a);
        rayp[1 * kTlRaySlots + tid] = make_double2(RA.s_b, RA.rt_b);
        rayp[2 * kTlRaySlots + tid] = make_double2(RB.s_a, RB.rt_a);
        rayp[3 * kTlRaySlots + tid] = make_double2(RB.s_b, RB.rt_b);
        if (liveA) n_samples += max(RA.i_last - RA.i_first + 1, 0);
        if (liveB) n_samples += max(RB.i_last - RB.i_first + 1, 0);
        // slice range of every pass: the union over its rays
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            int lo = 0x7fffffff, hi = -1;
            if (mA == m) { lo = RA.i_first; hi = RA.i_last; }
            if (mB == m) { lo = min(lo, RB.i_first); hi = max(hi, RB.i_last); }
            lo = __reduce_min_sync(0xffffffffu, lo);
            hi = __reduce_max_sync(0xffffffffu, hi);
            if (lane == 0 && hi >= lo) {
                atomicMin(&S.pass[m].lo, lo);
                atomicMax(&S.pass[m].hi, hi);
            }
        }
        // a ray that misses the volume (or the degenerate ray) writes +0.0
        if (liveA && mA == 3) P.out[((size_t)proj * P.nv + ivA) * P.nu + iuA] = 0.0f;
        if (liveB && mB == 3) P.out[((size_t)proj * P.nv + ivB) * P.nu + iuB] = 0.0f;
    }
    __syncthreads();
    // ---- plan of the passes (thread m plans pass m).  In pass m EVERY ray of the tile is parametrised along axis m
    //      (r~ = r / r_m, Eq. 4): if r_m has one sign at the four corners it has that sign on the whole tile (r is
    //      affine in the pixel), the map pixel -> intersection point with slice i is projective, and all rays cut the
    //      slice inside the quadrilateral of the corner rays' points.  The pass copies the bounding box of that
    //      quadrilateral; the rays whose driving axis IS m (Eq. 2) sample it, the others go through the motions with
    //      the first corner's parameters and drop the result.  Box classes from both ends of the slice range (every
    //      corner point is affine in the slice index, so the extents are largest at one of the ends).
    if (tid < 3 && S.pass[tid].hi >= S.pass[tid].lo) {
        const int m = tid, ta = axis_slow(m), tb = axis_fast(m);
        TlPass &Q = S.pass[m];
        const double r0 = S.cr[0][m], r1 = S.cr[1][m], r2 = S.cr[2][m], r3 = S.cr[3][m];
        const bool one_sign = (r0 > 0.0 && r1 > 0.0 && r2 > 0.0 && r3 > 0.0) || (r0 < 0.0 && r1 < 0.0 && r2 < 0.0 && r3 < 0.0);
        int size_r = -1, size_c = -1;
        if (one_sign && (m != 2 || P.z_staged)) {
            for (int c = 0; c < 4; ++c) {
                TlCorner C;
                C.s_m = S.cs[m];
                C.s_a = S.cs[ta];
                C.s_b = S.cs[tb];
                C.rt_a = __ddiv_rn(S.cr[c][ta], S.cr[c][m]);
                C.rt_b = __ddiv_rn(S.cr[c][tb], S.cr[c][m]);
                S.corner[m][c] = C;
            }
            int rows = 0, cols = 0;
            for (int e = 0; e < 2; ++e) {
                const int i = e ? Q.hi : Q.lo;
                double smin = 1e300, smax = -1e300, fmin_ = 1e300, fmax_ = -1e300;
                for (int c = 0; c < 4; ++c) {
                    const TlCorner &C = S.corner[m][c];
                    const double ps = p_of_i(C.s_a, C.s_m, C.rt_a, i), pf = p_of_i(C.s_b, C.s_m, C.rt_b, i);
                    smin = fmin(smin, ps); smax = fmax(smax, ps);
                    fmin_ = fmin(fmin_, pf); fmax_ = fmax(fmax_, pf);
                }
                // extent e of the positions: floor(max) - floor(min) <= floor(e) + 1 on any slice in between; rows
                // floor(min) - 1 .. floor(max) + 2 are copied (one spare on either side of the taps)
                rows = max(rows, (int)fmin(smax - smin, 1.0e6) + 5);
                cols = max(cols, (int)fmin(fmax_ - fmin_, 1.0e6) + 8);     // + 3: the box starts on a 16-byte boundary
            }
            for (int k = kTlSizes - 1; k >= 0; --k) {
                if (rows <= tl_rows(k)) size_r = k;
                if (cols <= tl_cols(k)) size_c = k;
            }
            // the slot a ray reads in a pass that is not its own: the first corner's parameters
            const TlCorner &C0 = S.corner[m][0];
#pragma unroll
            for (int q = 0; q < 4; ++q)
                rayp[q * kTlRaySlots + kTlConsumers + m] = (q & 1) ? make_double2(C0.s_b, C0.rt_b) : make_double2(C0.s_a, C0.rt_a);
        }
        Q.size_r = max(size_r, 0);
        Q.size_c = max(size_c, 0);
        Q.staged = size_r >= 0 && size_c >= 0;
    }
    __syncthreads();

    bool ring_used = false;
    for (int m = 0; m < 3; ++m) {
        const int lo = S.pass[m].lo, hi = S.pass[m].hi;
        if (hi < lo) continue;                                           // no ray of the tile has this driving axis
        if (!S.pass[m].staged) {
            // ---- direct path for the rays of this axis (oversized box, no staged copy for z, r_m changing sign)
            if (liveA && mA == m) P.out[((size_t)proj * P.nv + ivA) * P.nu + iuA] = tl_direct_pixel<INTERP>(g, P.G, P.lay, iuA, ivA);
            if (liveB && mB == m) P.out[((size_t)proj * P.nv + ivB) * P.nu + iuB] = tl_direct_pixel<INTERP>(g, P.G, P.lay, iuB, ivB);
            continue;
        }
        if (ring_used) {
            // a second staged pass (about 4 % of C4's tiles): the ring starts over with its own stage size
            __syncthreads();
            if (tid == 0) {
                for (int k = 0; k < kTlStagesMax; ++k) {
                    tl_mbar_inval(&S.full[k]);
                    tl_mbar_inval(&S.empty[k]);
                    tm_mbar_init(&S.full[k], 1);
                    tm_mbar_init(&S.empty[k], kTlConsumers / 32);
                }
                asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            }
            __syncthreads();
        }
        ring_used = true;
        const int n_slices = hi - lo + 1;
        const int size_r = S.pass[m].size_r, size_c = S.pass[m].size_c;
        const int rows = tl_rows(size_r), cols = tl_cols(size_c);
        const unsigned pitchB = (unsigned)cols * 4u, boxB = (unsigned)(rows * cols * 4), stageB = tl_stage_stride(rows, cols);
        const int nst = min(kTlStagesMax, (int)(kTlTileBytes / stageB));   // stages in flight
        if (producer) {
            // lane = slice-in-batch * 8 + corner * 2 + coordinate; batches of four slices
            const int sb = lane >> 3, cc = (lane >> 1) & 3, co = lane & 1;
            const TlCorner C = S.corner[m][cc];
            const double s_t = co ? C.s_b : C.s_a, rt_t = co ? C.rt_b : C.rt_a;
            const CUtensorMap *map = &P.map[m][size_r][size_c];
            int st = 0;
            unsigned ph = 0;                                             // parity of the empty phase to wait for (from the second round on)
            for (int n0 = 0; n0 < n_slices; n0 += 4) {
                const int i = lo + n0 + sb;
                const double p = p_of_i(s_t, C.s_m, rt_t, min(i, hi));
                double pmin = p;
                pmin = fmin(pmin, __shfl_xor_sync(0xffffffffu, pmin, 2));
                pmin = fmin(pmin, __shfl_xor_sync(0xffffffffu, pmin, 4));
                // first row / column of the box: one spare on the low side for fp32 rounding of the consumers' positions;
                // the first column on a 16-byte boundary of the volume's rows (the TMA engine traps otherwise)
                const int o_t = co ? ((__double2int_rd(pmin) - 1) & ~3) : (__double2int_rd(pmin) - 1);
                const int js0_l = __shfl_sync(0xffffffffu, o_t, 8 * sb), kf0_l = __shfl_sync(0xffffffffu, o_t, 8 * sb + 1);
                // the part of the published origin that depends on the box position, once per batch on all lanes
                const unsigned rel_l = (0x4B400000u + (unsigned)js0_l) * pitchB + ((0x4B400000u + (unsigned)kf0_l) << 2);
                for (int q = 0; q < 4 && n0 + q < n_slices; ++q) {
                    const int n = n0 + q;
                    // slice q of the batch is issued by the lane that already holds its box position (lane 8 q): no
                    // broadcast of the position per slice
                    const int js0 = js0_l, kf0 = kf0_l;
                    const unsigned rel = rel_l;
                    if (n >= nst) tm_mbar_wait(&S.empty[st], ph);
                    if (lane == 8 * q) {
                        // the consumers' reads of this stage (generic proxy, ordered before this point by their
                        // arrival on empty[]) before the copy below (async proxy)
                        tm_fence_proxy_async();
                        // consumers add bits(row) * pitch + bits(col) * 4 with bits = 0x4B400000 + index (mod 2^32)
                        const unsigned dst = tiles_smem + st * stageB;
                        S.org[st].x = dst - rel;
                        tm_mbar_arrive_tx(&S.full[st], boxB);
                        const int ii = lo + n;
                        // tensor dimensions, fastest first: m = x: (z, y, x); m = y: (z, y, x) with the slow axis x;
                        // m = z: the y-fastest copy (y, x, z)
                        tm_load_3d(map, dst, &S.full[st], kf0, m == 1 ? ii : js0, m == 1 ? js0 : ii);
                    }
                    __syncwarp();
                    if (++st == nst) {
                        st = 0;
                        if (n >= nst) ph ^= 1u;
                    }
                }
            }
        } else {
            const float2 kMagic2 = make_float2(12582912.0f, 12582912.0f), kNegMagic2 = make_float2(-12582912.0f, -12582912.0f);
            const float2 kNegOne2 = make_float2(-1.0f, -1.0f), kOne2 = make_float2(1.0f, 1.0f);
            const double s_m = S.cs[m];                                  // the source's coordinate along m: the same for every ray
            // a ray of another driving axis reads the pass's corner slot instead of its own
            const double2 *rpA = rayp + (mA == m ? tid : kTlConsumers + m), *rpB = rayp + (mB == m ? tid : kTlConsumers + m);

            float2 acc = make_float2(0.0f, 0.0f);
            // one running address walks full[], empty[] (+ kTlEmptyOff) and org[] (+ kTlOrgOff)
            const unsigned bar0 = tm_smem(&S.full[0]), bar_end = bar0 + 8u * (unsigned)nst;
            unsigned bar = bar0, prev = bar0 + (kTlSinkOff - kTlEmptyOff);
            unsigned ph = 0;                                             // parity of the full phase to wait for
            for (int s0 = lo; s0 <= hi; s0 += kSegment) {
                const int s1 = min(s0 + kSegment - 1, hi), ic = (s0 + s1) >> 1;
                // fp64 anchors at the segment's middle slice, split into integer voxel index + fraction
                const double2 qa = rpA[0 * kTlRaySlots], qb = rpA[1 * kTlRaySlots];
                const double2 qc = rpB[2 * kTlRaySlots], qd = rpB[3 * kTlRaySlots];
                const double paA = p_of_i(qa.x, s_m, qa.y, ic), pbA = p_of_i(qb.x, s_m, qb.y, ic);
                const double paB = p_of_i(qc.x, s_m, qc.y, ic), pbB = p_of_i(qd.x, s_m, qd.y, ic);
                // increments along the two in-plane axes of both rays (packed: .x = ray A, .y = ray B)
                const float2 rs2 = make_float2((float)qa.y, (float)qc.y), rf2 = make_float2((float)qb.y, (float)qd.y);
                const double faA = floor(paA), fbA = floor(pbA), faB = floor(paB), fbB = floor(pbB);
                const float2 as2 = make_float2((float)(paA - faA), (float)(paB - faB));
                const float2 af2 = make_float2((float)(pbA - fbA), (float)(pbB - fbB));
                // per-ray address constant: (integer anchor row) * pitch + (integer anchor column) * 4
                unsigned kA = (unsigned)__double2int_rd(faA) * pitchB + ((unsigned)__double2int_rd(fbA) << 2);
                unsigned kB = (unsigned)__double2int_rd(faB) * pitchB + ((unsigned)__double2int_rd(fbB) << 2);
                asm volatile("" : "+r"(kA), "+r"(kB));                  // one constant per ray: keep the sum out of the loop
                float2 fi = make_float2((float)(s0 - ic), (float)(s0 - ic));
                for (int i = s0; i <= s1; ++i) {
                    tl_wait_addr(bar, ph);
                    // release the PREVIOUS stage here, where its loads have returned (the producer orders the
                    // consumers' generic-proxy reads before its next async-proxy copy with a proxy fence)
                    __syncwarp();
                    if (lane == 0) tl_arrive_addr(prev + kTlEmptyOff);
                    prev = bar;
                    const unsigned org = __float_as_uint(al_lds(bar + kTlOrgOff));
                    const float2 ps = __ffma2_rn(fi, rs2, as2), pf = __ffma2_rn(fi, rf2, af2);
                    fi = __fadd2_rn(fi, kOne2);
                    const float2 xs = __fadd2_rd(ps, kMagic2), xf = __fadd2_rd(pf, kMagic2);     // bits = 0x4B400000 + floor
                    const float2 ds = __ffma2_rn(__fadd2_rn(xs, kNegMagic2), kNegOne2, ps);
                    const float2 df = __ffma2_rn(__fadd2_rn(xf, kNegMagic2), kNegOne2, pf);
                    const unsigned a0 = __float_as_uint(xs.x) * pitchB + (__float_as_uint(xf.x) << 2) + (kA + org);
                    const unsigned b0 = __float_as_uint(xs.y) * pitchB + (__float_as_uint(xf.y) << 2) + (kB + org);
                    const float2 v00 = make_float2(al_lds(a0), al_lds(b0));
                    const float2 v01 = make_float2(al_lds(a0 + 4u), al_lds(b0 + 4u));
                    const unsigned a1 = a0 + pitchB, b1 = b0 + pitchB;
                    const float2 v10 = make_float2(al_lds(a1), al_lds(b1));
                    const float2 v11 = make_float2(al_lds(a1 + 4u), al_lds(b1 + 4u));
                    const float2 wf = make_float2(ceil_weight<INTERP>(df.x), ceil_weight<INTERP>(df.y));
                    const float2 ws = make_float2(ceil_weight<INTERP>(ds.x), ceil_weight<INTERP>(ds.y));
                    const float2 t0 = __ffma2_rn(wf, __ffma2_rn(v00, kNegOne2, v01), v00);       // row j
                    const float2 t1 = __ffma2_rn(wf, __ffma2_rn(v10, kNegOne2, v11), v10);       // row j + 1
                    acc = __fadd2_rn(acc, __ffma2_rn(ws, __ffma2_rn(t0, kNegOne2, t1), t0));
                    bar += 8u;
                    if (bar == bar_end) {
                        bar = bar0;
                        ph ^= 1u;
                    }
                }
            }
            if (liveA && mA == m) P.out[((size_t)proj * P.nv + ivA) * P.nu + iuA] = scA * acc.x + 0.0f;
            if (liveB && mB == m) P.out[((size_t)proj * P.nv + ivB) * P.nu + iuB] = scB * acc.y + 0.0f;
        }
    }
    if (P.sample_count) block_count_samples(P.sample_count, n_samples);
}

constexpr size_t tile_smem_bytes() { return kTlTileBytes + sizeof(TlShared) + kTlRayBytes; }

}  // namespace fpk
