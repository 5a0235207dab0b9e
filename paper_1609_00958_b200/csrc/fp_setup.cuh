// fp_setup.cuh -- per-ray set-up of the Generalized Joseph Projector on the device.
//
// PAPER.md:71-106 sec. 2.1 Eqs. 1-6 and Alg. 1 lines 1-5 (:220-228): ray r = d - s, driving
// axis m = argmax|r_a|, increment r~ = r / r_m, offset o = -s_m; sec. 2.6: the
// in-volume test of Alg. 1 line 8 "becomes obsolete when entry and exit points are calculated
// exactly" -- which is what ray_setup() does.
//
// Every DECISION (m, i_first, i_last) is taken in IEEE fp64 with a fixed operation order and
// explicit round-to-nearest intrinsics (__dadd_rn, __dmul_rn, __ddiv_rn are never contracted
// into FMAs), DESIGN.md "Index-parity rule".  The slice interval is first SOLVED by a division
// and then FIXED UP by evaluating the defining predicate  -1 < p_t(i) < N_t  at the candidate
// and its neighbours, so the result is the exact extreme slice of the predicate whatever the
// rounding of the division was.  No branch depends on the driving axis.
#pragma once
#include <cstdint>

namespace fpk {

struct GridDesc {
    int n[3];            // nx, ny, nz
    int pad_;
    double delta;        // voxel pitch, world units
    double origin[3];    // world position of the centre of voxel (0,0,0)
};

struct RaySetup {
    int m;               // driving axis (0 = x, 1 = y, 2 = z)
    int i_first, i_last; // first / last slice with -1 < p_t < N_t for both transverse axes; (0,-1) = miss
    double s_m;          // source coordinate along m (grid units)
    double s_a, s_b;     // source coordinates along the kernel's transverse axes (slow, fast)
    double rt_a, rt_b;   // r~ along them
    double L;            // ||r~||_2, 1 <= L <= sqrt(3)
};

__device__ __forceinline__ double sel3(int k, double a0, double a1, double a2)
{
    return k == 0 ? a0 : (k == 1 ? a1 : a2);
}
__device__ __forceinline__ int sel3i(int k, int a0, int a1, int a2)
{
    return k == 0 ? a0 : (k == 1 ? a1 : a2);
}

// Transverse coordinate of sample i:  p_t(i) = s_t + (i - s_m) r~_t   (Eqs. 5-6, Alg. 1 l.3, l.7).
__device__ __forceinline__ double p_of_i(double s_t, double s_m, double rt_t, int i)
{
    return __dadd_rn(s_t, __dmul_rn(__dsub_rn((double)i, s_m), rt_t));
}

__device__ __forceinline__ bool inside_t(double s_t, double s_m, double rt_t, double n_t, int i)
{
    const double p = p_of_i(s_t, s_m, rt_t, i);
    return (-1.0 < p) && (p < n_t);
}

// Clamp a real-valued slice estimate into [lo, hi] (as doubles) before the int conversion, so
// that huge or non-finite quotients cannot overflow.  fmax/fmin drop a NaN operand.
__device__ __forceinline__ int clamp_to_int(double x, int lo, int hi)
{
    return (int)fmin(fmax(x, (double)lo), (double)hi);
}

// Intersect [lo, hi] with { i : -1 < p_t(i) < N_t }.  Each of the two inequalities is monotone
// in i (every rounded operation in p_of_i is monotone), so each holds on a half line whose end
// is found by estimate + fix-up against the predicate itself.
__device__ __forceinline__ void clip_axis(double s_t, double s_m, double rt_t, int n_t, int &lo, int &hi)
{
    const double nt = (double)n_t;
    if (rt_t == 0.0) {                       // p_t is the same for every slice
        const double p = p_of_i(s_t, s_m, rt_t, 0);
        if (!((-1.0 < p) && (p < nt))) hi = lo - 1;
        return;
    }
    // real-valued slice positions where p_t = -1 and p_t = N_t.  They are ESTIMATES only -- the fix-up below
    // evaluates the defining predicate and ends on its exact extreme slice whatever the estimate was -- so an fp32
    // reciprocal (|rt_t| <= 1: no overflow; a denormal rt_t gives inf / NaN, which clamp_to_int absorbs) replaces
    // the two fp64 divisions: four of the ten divisions of a ray's set-up
    const double inv = (double)__frcp_rn((float)rt_t);
    const double x_m1 = __dadd_rn(s_m, __dmul_rn(__dsub_rn(-1.0, s_t), inv));
    const double x_nt = __dadd_rn(s_m, __dmul_rn(__dsub_rn(nt, s_t), inv));
    const bool up = rt_t > 0.0;
    // "enter": inequality false -> true with growing i; "leave": true -> false
    const double x_enter = up ? x_m1 : x_nt;
    const double x_leave = up ? x_nt : x_m1;
    const int lo0 = lo, hi0 = hi;

    // least i in [lo0, hi0 + 1] with the entering inequality true
    int a = clamp_to_int(ceil(x_enter), lo0, hi0 + 1);
    // greatest i in [lo0 - 1, hi0] with the leaving inequality true
    int b = clamp_to_int(floor(x_leave), lo0 - 1, hi0);
    if (up) {
        while (a > lo0 && (-1.0 < p_of_i(s_t, s_m, rt_t, a - 1))) --a;
        while (a <= hi0 && !(-1.0 < p_of_i(s_t, s_m, rt_t, a))) ++a;
        while (b < hi0 && (p_of_i(s_t, s_m, rt_t, b + 1) < nt)) ++b;
        while (b >= lo0 && !(p_of_i(s_t, s_m, rt_t, b) < nt)) --b;
    } else {
        while (a > lo0 && (p_of_i(s_t, s_m, rt_t, a - 1) < nt)) --a;
        while (a <= hi0 && !(p_of_i(s_t, s_m, rt_t, a) < nt)) ++a;
        while (b < hi0 && (-1.0 < p_of_i(s_t, s_m, rt_t, b + 1))) ++b;
        while (b >= lo0 && !(-1.0 < p_of_i(s_t, s_m, rt_t, b))) --b;
    }
    lo = a > lo ? a : lo;
    hi = b < hi ? b : hi;
}

// Field-of-view clip (FP_OPT_FOV_CYLINDER; Fig. 9: "projections of a cylindric volume within a
// cubic bounding box"): intersect [lo, hi] with the slices whose sample point (i, p_s(i)) in the (driving axis,
// in-plane transverse axis) plane lies within radius rm of the centre (c_m, c_s).  rm already holds the margin
// that keeps every tap of a dropped sample outside the cylinder; the quadratic is solved in fp64 and the range
// widened by one slice on either side, so the clip is conservative.
__device__ __forceinline__ void clip_circle(double s_s, double s_m, double rt_s, double c_m, double c_s, double rm,
                                            int &lo, int &hi)
{
    const double q = s_s - s_m * rt_s - c_s;                 // p_s(i) - c_s = q + i rt_s
    const double A = 1.0 + rt_s * rt_s, B = q * rt_s - c_m, C = c_m * c_m + q * q - rm * rm;   // A i^2 + 2 B i + C <= 0
    const double disc = B * B - A * C;
    if (!(disc >= 0.0)) {
        hi = lo - 1;
        return;
    }
    const double sq = sqrt(disc);
    const int a = clamp_to_int(floor((-B - sq) / A) - 1.0, lo, hi + 1);
    const int b = clamp_to_int(ceil((-B + sq) / A) + 1.0, lo - 1, hi);
    lo = max(lo, a);
    hi = min(hi, b);
}

// Transverse axes as the sampling kernels order them: (slow, fast) = (y,z), (x,z), (x,y) for
// m = x, y, z.  The fast one is contiguous in memory for the layout the kernel reads.
__device__ __forceinline__ int axis_slow(int m) { return m == 0 ? 1 : 0; }
__device__ __forceinline__ int axis_fast(int m) { return m == 2 ? 1 : 2; }

// g = { S xyz, O xyz, U xyz, V xyz } in world units; pixel centre D = (O + iu U) + iv V.
// s = the source in grid units, (g[a] - origin[a]) / delta per axis in exactly these operations: the same for every
// ray of a pose, so a block may compute it once (ray_setup below computes it per call).
// x / delta (Eq. 1's world -> grid map).  Where delta is a power of two -- every BASELINE configuration -- the
// product with the exactly representable 1 / delta is the same correctly rounded value as the quotient (the two
// real numbers are equal), so the division is skipped; the test is uniform over the launch.
struct GridScale {
    double inv;          // 1 / delta if delta is a power of two with a representable reciprocal, else 0
};
__device__ __forceinline__ GridScale grid_scale(double delta)
{
    const long long b = __double_as_longlong(delta);
    const long long e = (b >> 52) & 0x7ffLL;
    GridScale K;
    K.inv = (b > 0 && (b & 0x000fffffffffffffLL) == 0 && e >= 2 && e <= 2044) ? __longlong_as_double((2046LL - e) << 52) : 0.0;
    return K;
}
__device__ __forceinline__ double to_grid(double x, double delta, const GridScale &K)
{
    return K.inv != 0.0 ? __dmul_rn(x, K.inv) : __ddiv_rn(x, delta);
}

__device__ __forceinline__ RaySetup ray_setup_from(const double *__restrict__ g, const GridDesc &G, const double s[3], int iu, int iv)
{
    const GridScale K = grid_scale(G.delta);
    double r[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double D = __dadd_rn(__dadd_rn(g[3 + a], __dmul_rn((double)iu, g[6 + a])),
                                   __dmul_rn((double)iv, g[9 + a]));
        const double d = to_grid(__dsub_rn(D, G.origin[a]), G.delta, K);
        r[a] = __dsub_rn(d, s[a]);                                   // Eq. 1
    }
    RaySetup R;
    R.i_first = 0;
    R.i_last = -1;
    R.m = 0;
    R.L = 0.0;
    R.s_m = R.s_a = R.s_b = R.rt_a = R.rt_b = 0.0;
    if (r[0] == 0.0 && r[1] == 0.0 && r[2] == 0.0) return R;         // degenerate ray

    int m = 0;                                                       // Eq. 2, ties -> lowest axis
    double rm = r[0];
    if (fabs(r[1]) > fabs(rm)) { m = 1; rm = r[1]; }
    if (fabs(r[2]) > fabs(rm)) { m = 2; rm = r[2]; }
    const int ta = axis_slow(m), tb = axis_fast(m);
    // Eq. 4: two divisions, r~_m := 1 (reading #9)
    const double rta = __ddiv_rn(sel3(ta, r[0], r[1], r[2]), rm), rtb = __ddiv_rn(sel3(tb, r[0], r[1], r[2]), rm);
    const double rt0 = m == 0 ? 1.0 : rta;                           // ta = x unless m = x
    const double rt1 = m == 1 ? 1.0 : (m == 0 ? rta : rtb);          // y is the slow axis for m = x, the fast one for m = z
    const double rt2 = m == 2 ? 1.0 : rtb;                           // tb = z unless m = z
    R.L = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(rt0, rt0), __dmul_rn(rt1, rt1)), __dmul_rn(rt2, rt2)));
    R.m = m;
    R.s_m = sel3(m, s[0], s[1], s[2]);
    R.s_a = sel3(ta, s[0], s[1], s[2]);
    R.s_b = sel3(tb, s[0], s[1], s[2]);
    R.rt_a = rta;
    R.rt_b = rtb;
    int lo = 0, hi = sel3i(m, G.n[0], G.n[1], G.n[2]) - 1;
    clip_axis(R.s_a, R.s_m, R.rt_a, sel3i(ta, G.n[0], G.n[1], G.n[2]), lo, hi);
    if (lo <= hi) clip_axis(R.s_b, R.s_m, R.rt_b, sel3i(tb, G.n[0], G.n[1], G.n[2]), lo, hi);
    if (lo <= hi) { R.i_first = lo; R.i_last = hi; }
    return R;
}

__device__ __forceinline__ RaySetup ray_setup(const double *__restrict__ g, const GridDesc &G, int iu, int iv)
{
    double s[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) s[a] = __ddiv_rn(__dsub_rn(g[a], G.origin[a]), G.delta);
    return ray_setup_from(g, G, s, iu, iv);
}

}  // namespace fpk
