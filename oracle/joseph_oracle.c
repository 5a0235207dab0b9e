/*
 * joseph_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded fp64 CPU implementation of the "Generalized Joseph
 * Projector" (GJP) of arXiv 1609.00958 (J. Dittmann), written from the paper
 * and SURVEY.md section 8(c).  It shares no code, header,
 * table or helper with the CUDA path in paper_1609_00958_b200/csrc and must
 * never be imported, linked or executed by the product path.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC  (see oracle/build.py).
 * -ffp-contract=off matters: the set-up decisions (driving axis, entry/exit slice)
 * are defined as IEEE fp64 expressions in a FIXED operation order without FMA.
 *
 * Parity status: every function here is pinned by tests/test_oracle_pins.py
 * (closed forms, invariants, a library trilinear routine, brute force on tiny
 * inputs, a hand-worked example; the back-projection voxel by voxel against the pinned
 * forward projection of unit volumes) -- nothing is "parity unpinned".
 *
 * What is computed (PAPER.md line numbers; section / equation in brackets):
 *   r = d - s                                   :77  [sec 2.1, Eq. 1]
 *   m = argmax_a |r_a|                          :81  [Eq. 2]   (ties -> lowest axis, reading #8)
 *   r~ = r / r_m                                :92  [Eq. 4]
 *   o = -s_m                                    :98  [Eq. 5]
 *   p(i) = (s + o r~) + i r~,  p_m(i) = i       :104 [Eq. 6], :243 [Alg. 1 l.10]
 *   2x2 taps floor/ceil in the two non-driving axes  :165 [Eq. 15], :237-240 [Alg. 1 l.9-10]
 *   weights w(d), 1 - w(d), product over axes   :131 [Eq. 8], :142 [Eq. 11], :150-152 [Eqs. 13, 14]
 *   a += volume[tap] * ||r~|| * w * w           :258-264 [Alg. 1 l.15-18], :211
 * Readings where the paper is silent or garbled are numbered as in DESIGN.md
 * ("Readings of the paper"): voxel k sits at grid coordinate k (#1); the volume
 * is zero outside 0..N-1 and a sample counts when -1 < p_t < N_t for both
 * transverse axes (#2); i runs over 0..N_m-1 (#3); the ray is the infinite line
 * through s and d (#10); every visited slice carries the full ||r~|| (#11).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define JO_KERNEL_LIN 0   /* w_lin(d) = 1 - d            PAPER.md:150 Eq. 13 */
#define JO_KERNEL_SPL 1   /* w_spl(d) = 1 - 3d^2 + 2d^3  PAPER.md:152 Eq. 14 */

/* Interpolation kernel w(d), d in [0,1)  (PAPER.md:126 Eq. 7, :150-152). */
static double jo_w(int kernel, double d)
{
    if (kernel == JO_KERNEL_SPL)
        return 1.0 - 3.0 * d * d + 2.0 * d * d * d;
    return 1.0 - d;
}

/* Zero-extended voxel read: vol0[ix][iy][iz], C order, z fastest (reading #2, #13). */
static double jo_vox(const float *vol, const int n[3], long ix, long iy, long iz)
{
    if (ix < 0 || iy < 0 || iz < 0 || ix >= n[0] || iy >= n[1] || iz >= n[2])
        return 0.0;
    return (double)vol[((size_t)ix * (size_t)n[1] + (size_t)iy) * (size_t)n[2] + (size_t)iz];
}

/* Per-ray set-up, steps 2-4 of SURVEY.md 8(c): r, m, r~, L = ||r~||_2.
 * Returns 0 for the degenerate ray r = 0, else 1. */
static int jo_setup(const double s[3], const double d[3], int *m_out, double rt[3], double *L)
{
    double r[3];
    int a, m;
    for (a = 0; a < 3; ++a)
        r[a] = d[a] - s[a];                              /* Eq. 1 */
    if (r[0] == 0.0 && r[1] == 0.0 && r[2] == 0.0)
        return 0;
    m = 0;                                               /* Eq. 2, strict '>' */
    if (fabs(r[1]) > fabs(r[m])) m = 1;
    if (fabs(r[2]) > fabs(r[m])) m = 2;
    for (a = 0; a < 3; ++a)
        rt[a] = r[a] / r[m];                             /* Eq. 4 */
    rt[m] = 1.0;
    *L = sqrt(rt[0] * rt[0] + rt[1] * rt[1] + rt[2] * rt[2]);
    *m_out = m;
    return 1;
}

/* Transverse coordinate of sample i: p_t(i) = s_t + (i - s_m) r~_t  (Eqs. 5-6, Alg. 1 l.3, l.7). */
static double jo_pt(const double s[3], const double rt[3], int m, int t, int i)
{
    return s[t] + ((double)i - s[m]) * rt[t];
}

/*
 * jo_ray_grid: one ray given in GRID coordinates (units of the voxel pitch, voxel
 * (0,0,0) at the origin).  Step-by-step form, SURVEY.md 8(c) steps 2-8.
 *   value_grid = ||r~|| * sum_i sample(i)   (multiply by the voxel pitch for world units)
 *   mfl        = { m, i_first, i_last }     ((m,0,-1) for a miss, (0,0,-1) for r = 0)
 *   L          = ||r~||_2
 *   margins    = { relative gap between the two largest |r_a|,
 *                  smallest distance of p_t(i) from -1 / N_t over i in
 *                  {i_first-1, i_first, i_last, i_last+1} (or over all i for a miss) }
 */
void jo_ray_grid(const float *vol, const int n[3], const double s[3], const double d[3],
                 int kernel, double *value_grid, int32_t mfl[3], double *L_out, double margins[2])
{
    double rt[3], L = 0.0, acc = 0.0;
    int m = 0, t1, t2, i, i_first = 0, i_last = -1, found = 0;

    *value_grid = 0.0;
    mfl[0] = 0; mfl[1] = 0; mfl[2] = -1;
    if (L_out) *L_out = 0.0;
    if (margins) { margins[0] = 0.0; margins[1] = 0.0; }
    if (!jo_setup(s, d, &m, rt, &L))
        return;
    t1 = (m + 1) % 3;
    t2 = (m + 2) % 3;
    mfl[0] = m;
    if (L_out) *L_out = L;

    /* step 6: brute-force the in-volume predicate over every slice */
    for (i = 0; i < n[m]; ++i) {
        double p1 = jo_pt(s, rt, m, t1, i), p2 = jo_pt(s, rt, m, t2, i);
        int inside = (-1.0 < p1) && (p1 < (double)n[t1]) && (-1.0 < p2) && (p2 < (double)n[t2]);
        if (inside) {
            if (!found) { i_first = i; found = 1; }
            i_last = i;
        }
    }
    if (margins) {
        double r[3], big = 0.0, second = 0.0, mi = 1e300;
        int a;
        for (a = 0; a < 3; ++a) r[a] = fabs(d[a] - s[a]);
        for (a = 0; a < 3; ++a) { if (a == m) big = r[a]; else if (r[a] > second) second = r[a]; }
        margins[0] = (big - second) / big;
        for (i = 0; i < n[m]; ++i) {
            int near = found ? (i == i_first - 1 || i == i_first || i == i_last || i == i_last + 1) : 1;
            if (near) {
                double p1 = jo_pt(s, rt, m, t1, i), p2 = jo_pt(s, rt, m, t2, i), q;
                q = fabs(p1 + 1.0); if (q < mi) mi = q;
                q = fabs(p1 - (double)n[t1]); if (q < mi) mi = q;
                q = fabs(p2 + 1.0); if (q < mi) mi = q;
                q = fabs(p2 - (double)n[t2]); if (q < mi) mi = q;
            }
        }
        margins[1] = mi;
    }
    if (!found)
        return;
    mfl[1] = i_first;
    mfl[2] = i_last;

    /* steps 7-8: 2x2 taps per slice, ascending i */
    for (i = i_first; i <= i_last; ++i) {
        double p[3], f[3], w0[3], w1[3];
        long fl[3];
        int a, b;
        p[m] = (double)i;
        p[t1] = jo_pt(s, rt, m, t1, i);
        p[t2] = jo_pt(s, rt, m, t2, i);
        for (a = 0; a < 3; ++a) {
            f[a] = floor(p[a]);                            /* Alg. 1 l.9 */
            fl[a] = (long)f[a];
            w0[a] = jo_w(kernel, p[a] - f[a]);             /* Alg. 1 l.12: w_fl = w(p - p_fl) */
            w1[a] = 1.0 - w0[a];                           /* l.13 */
        }
        w0[m] = 1.0;                                       /* l.14: driving axis */
        w1[m] = 1.0;
        /* The four (floor, floor+1) combinations in the (t1, t2) plane.  floor+1 instead of
         * ceil: when p_t is an integer the second tap's weight is exactly 0. */
        for (a = 0; a < 2; ++a)
            for (b = 0; b < 2; ++b) {
                long idx[3];
                idx[m] = fl[m];
                idx[t1] = fl[t1] + a;
                idx[t2] = fl[t2] + b;
                acc += jo_vox(vol, n, idx[0], idx[1], idx[2])
                       * (a ? w1[t1] : w0[t1]) * (b ? w1[t2] : w0[t2]);
            }
    }
    *value_grid = L * acc;                                 /* weighted by the sampling interval, :211 */
}

/*
 * jo_ray_definition: the plain definition, no floor, no clipping, no index
 * ranges -- O(N^3) per ray, tiny inputs only:
 *   value_grid = ||r~|| * sum_{i,j,k} vol[m:i, t1:j, t2:k] * H(p_t1(i) - j) * H(p_t2(i) - k)
 * with H(x) = w(|x|) for |x| < 1, else 0: the hat for w_lin (PAPER.md:131-133 Eq. 8-9, :150).
 */
void jo_ray_definition(const float *vol, const int n[3], const double s[3], const double d[3],
                       int kernel, double *value_grid)
{
    double rt[3], L, acc = 0.0;
    int m, t1, t2, idx[3];
    *value_grid = 0.0;
    if (!jo_setup(s, d, &m, rt, &L))
        return;
    t1 = (m + 1) % 3;
    t2 = (m + 2) % 3;
    for (idx[0] = 0; idx[0] < n[0]; ++idx[0])
        for (idx[1] = 0; idx[1] < n[1]; ++idx[1])
            for (idx[2] = 0; idx[2] < n[2]; ++idx[2]) {
                int i = idx[m];
                double x1 = fabs(jo_pt(s, rt, m, t1, i) - (double)idx[t1]);
                double x2 = fabs(jo_pt(s, rt, m, t2, i) - (double)idx[t2]);
                double h1 = x1 < 1.0 ? jo_w(kernel, x1) : 0.0;
                double h2 = x2 < 1.0 ? jo_w(kernel, x2) : 0.0;
                acc += jo_vox(vol, n, idx[0], idx[1], idx[2]) * h1 * h2;
            }
    *value_grid = L * acc;
}

/* Step 1 of SURVEY.md 8(c): world -> grid.  D = (O + iu*U) + iv*V; s = (S - origin)/delta;
 * d = (D - origin)/delta, in this operation order (PAPER.md:57 Fig. 1, :63). */
static void jo_pixel_to_grid(const double geom[12], double delta, const double origin[3],
                             int iu, int iv, double s[3], double d[3])
{
    int a;
    for (a = 0; a < 3; ++a) {
        double D = (geom[3 + a] + (double)iu * geom[6 + a]) + (double)iv * geom[9 + a];
        s[a] = (geom[a] - origin[a]) / delta;
        d[a] = (D - origin[a]) / delta;
    }
}

/*
 * jo_project_rays: world-unit ray sums for a list of detector pixels.
 *   geom     [n_proj][12]  = source xyz, det_origin xyz, u xyz, v xyz
 *   ray_ids  [n_rays][3]   = (projection, iv, iu)
 *   values   [n_rays]        delta * ||r~|| * sum (fp64)
 *   mfl      [n_rays][3]     m, i_first, i_last            (may be NULL)
 *   pathlen  [n_rays]        delta * ||r~|| * (i_last - i_first + 1)   (may be NULL)
 *   margins  [n_rays][2]                                  (may be NULL)
 */
void jo_project_rays(const float *vol, const int n[3], double delta, const double origin[3],
                     const double *geom, int kernel, long n_rays, const int32_t *ray_ids,
                     double *values, int32_t *mfl, double *pathlen, double *margins)
{
    long q;
    for (q = 0; q < n_rays; ++q) {
        double s[3], d[3], v, L, mg[2];
        int32_t t[3];
        const double *g = geom + 12 * (size_t)ray_ids[3 * q];
        jo_pixel_to_grid(g, delta, origin, ray_ids[3 * q + 2], ray_ids[3 * q + 1], s, d);
        jo_ray_grid(vol, n, s, d, kernel, &v, t, &L, mg);
        values[q] = delta * v;
        if (mfl) { mfl[3 * q] = t[0]; mfl[3 * q + 1] = t[1]; mfl[3 * q + 2] = t[2]; }
        if (pathlen) pathlen[q] = delta * L * (double)(t[2] - t[1] + 1);
        if (margins) { margins[2 * q] = mg[0]; margins[2 * q + 1] = mg[1]; }
    }
}

/*
 * jo_project_block: the pixel rectangle [iv0, iv1) x [iu0, iu1) of ONE projection,
 * outputs indexed [(iv - iv0)][(iu - iu0)], u fastest (reading #14).
 */
void jo_project_block(const float *vol, const int n[3], double delta, const double origin[3],
                      const double geom[12], int kernel, int iu0, int iu1, int iv0, int iv1,
                      double *values, int32_t *mfl, double *pathlen, double *margins)
{
    int iu, iv;
    size_t q = 0;
    for (iv = iv0; iv < iv1; ++iv)
        for (iu = iu0; iu < iu1; ++iu, ++q) {
            double s[3], d[3], v, L, mg[2];
            int32_t t[3];
            jo_pixel_to_grid(geom, delta, origin, iu, iv, s, d);
            jo_ray_grid(vol, n, s, d, kernel, &v, t, &L, mg);
            values[q] = delta * v;
            if (mfl) { mfl[3 * q] = t[0]; mfl[3 * q + 1] = t[1]; mfl[3 * q + 2] = t[2]; }
            if (pathlen) pathlen[q] = delta * L * (double)(t[2] - t[1] + 1);
            if (margins) { margins[2 * q] = mg[0]; margins[2 * q + 1] = mg[1]; }
        }
}

/*
 * jo_backproject: the exact transpose of jo_project_block over whole projections
 * (SURVEY.md 8(f) #2; PAPER.md:27, :308, :367 -- iterative methods pair the projector with
 * its back-projection).  With A the linear map volume -> projections defined by
 * jo_ray_grid (same set-up, same in-volume predicate, same taps and weights, times the voxel
 * pitch), this accumulates  vol_out += A^T proj :  every tap (voxel) of every sample of every
 * ray receives  delta * ||r~|| * w * w * proj[ray].  Taps outside 0..N-1 belong to the zero
 * extension (reading #2) and receive nothing.
 *   proj     [n_proj][nv][nu]  fp64, u fastest
 *   vol_out  [nx][ny][nz]      fp64, z fastest; NOT cleared here
 */
void jo_backproject(const double *proj, const int n[3], double delta, const double origin[3],
                    const double *geom, int kernel, int n_proj, int nu, int nv, double *vol_out)
{
    int p, iu, iv;
    for (p = 0; p < n_proj; ++p)
        for (iv = 0; iv < nv; ++iv)
            for (iu = 0; iu < nu; ++iu) {
                double s[3], d[3], rt[3], L = 0.0;
                int m = 0, t1, t2, i;
                const double y = proj[((size_t)p * (size_t)nv + (size_t)iv) * (size_t)nu + (size_t)iu];
                jo_pixel_to_grid(geom + 12 * (size_t)p, delta, origin, iu, iv, s, d);
                if (!jo_setup(s, d, &m, rt, &L))
                    continue;
                t1 = (m + 1) % 3;
                t2 = (m + 2) % 3;
                for (i = 0; i < n[m]; ++i) {
                    double pc[3], w0[3], w1[3];
                    long fl[3];
                    int a, b;
                    pc[m] = (double)i;
                    pc[t1] = jo_pt(s, rt, m, t1, i);
                    pc[t2] = jo_pt(s, rt, m, t2, i);
                    /* the predicate of step 6; a sample outside it has no tap inside the volume anyway */
                    if (!((-1.0 < pc[t1]) && (pc[t1] < (double)n[t1]) && (-1.0 < pc[t2]) && (pc[t2] < (double)n[t2])))
                        continue;
                    for (a = 0; a < 3; ++a) {
                        double f = floor(pc[a]);
                        fl[a] = (long)f;
                        w0[a] = jo_w(kernel, pc[a] - f);
                        w1[a] = 1.0 - w0[a];
                    }
                    for (a = 0; a < 2; ++a)
                        for (b = 0; b < 2; ++b) {
                            long idx[3];
                            idx[m] = fl[m];
                            idx[t1] = fl[t1] + a;
                            idx[t2] = fl[t2] + b;
                            if (idx[0] < 0 || idx[1] < 0 || idx[2] < 0 || idx[0] >= n[0] || idx[1] >= n[1] || idx[2] >= n[2])
                                continue;
                            vol_out[((size_t)idx[0] * (size_t)n[1] + (size_t)idx[1]) * (size_t)n[2] + (size_t)idx[2]] +=
                                delta * L * (a ? w1[t1] : w0[t1]) * (b ? w1[t2] : w0[t2]) * y;
                        }
                }
            }
}

/*
 * jo_ray_grid_axis: the step-by-step form of jo_ray_grid with the driving axis GIVEN instead of
 * chosen by Eq. 2.  The paper is silent on exact ties |r_a| = |r_b| (DESIGN.md
 * reading #8): both axes give a valid Joseph sum, and they differ.  The parity harness uses this
 * routine only for rays whose two largest |r_a| agree to within 1e-9 relative and for which the
 * GPU took the other axis: the GPU value must then match the sum along ITS axis.  Same formulas as
 * jo_ray_grid (Eqs. 4-6, Alg. 1 l.6-20) with m := m_forced; r_m must be non-zero.
 *   mfl = { m_forced, i_first, i_last }
 */
void jo_ray_grid_axis(const float *vol, const int n[3], const double s[3], const double d[3],
                      int kernel, int m_forced, double *value_grid, int32_t mfl[3], double *L_out)
{
    double r[3], rt[3], L, acc = 0.0;
    int a, m = m_forced, t1, t2, i, i_first = 0, i_last = -1, found = 0;
    *value_grid = 0.0;
    mfl[0] = m; mfl[1] = 0; mfl[2] = -1;
    if (L_out) *L_out = 0.0;
    if (m < 0 || m > 2) return;
    for (a = 0; a < 3; ++a) r[a] = d[a] - s[a];            /* Eq. 1 */
    if (r[m] == 0.0) return;
    for (a = 0; a < 3; ++a) rt[a] = r[a] / r[m];           /* Eq. 4 with the given axis */
    rt[m] = 1.0;
    L = sqrt(rt[0] * rt[0] + rt[1] * rt[1] + rt[2] * rt[2]);
    if (L_out) *L_out = L;
    t1 = (m + 1) % 3;
    t2 = (m + 2) % 3;
    for (i = 0; i < n[m]; ++i) {                           /* step 6 */
        double p1 = jo_pt(s, rt, m, t1, i), p2 = jo_pt(s, rt, m, t2, i);
        if ((-1.0 < p1) && (p1 < (double)n[t1]) && (-1.0 < p2) && (p2 < (double)n[t2])) {
            if (!found) { i_first = i; found = 1; }
            i_last = i;
        }
    }
    if (!found) return;
    mfl[1] = i_first;
    mfl[2] = i_last;
    for (i = i_first; i <= i_last; ++i) {                  /* steps 7-8 */
        double p[3], w0[3], w1[3];
        long fl[3];
        int b;
        p[m] = (double)i;
        p[t1] = jo_pt(s, rt, m, t1, i);
        p[t2] = jo_pt(s, rt, m, t2, i);
        for (a = 0; a < 3; ++a) {
            double f = floor(p[a]);
            fl[a] = (long)f;
            w0[a] = jo_w(kernel, p[a] - f);
            w1[a] = 1.0 - w0[a];
        }
        for (a = 0; a < 2; ++a)
            for (b = 0; b < 2; ++b) {
                long idx[3];
                idx[m] = fl[m];
                idx[t1] = fl[t1] + a;
                idx[t2] = fl[t2] + b;
                acc += jo_vox(vol, n, idx[0], idx[1], idx[2]) * (a ? w1[t1] : w0[t1]) * (b ? w1[t2] : w0[t2]);
            }
    }
    *value_grid = L * acc;
}

/* jo_project_rays_axis: jo_project_rays with a driving axis given per ray (axis[q] in 0..2). */
void jo_project_rays_axis(const float *vol, const int n[3], double delta, const double origin[3],
                          const double *geom, int kernel, long n_rays, const int32_t *ray_ids,
                          const int32_t *axis, double *values, int32_t *mfl, double *pathlen)
{
    long q;
    for (q = 0; q < n_rays; ++q) {
        double s[3], d[3], v, L;
        int32_t t[3];
        const double *g = geom + 12 * (size_t)ray_ids[3 * q];
        jo_pixel_to_grid(g, delta, origin, ray_ids[3 * q + 2], ray_ids[3 * q + 1], s, d);
        jo_ray_grid_axis(vol, n, s, d, kernel, axis[q], &v, t, &L);
        values[q] = delta * v;
        if (mfl) { mfl[3 * q] = t[0]; mfl[3 * q + 1] = t[1]; mfl[3 * q + 2] = t[2]; }
        if (pathlen) pathlen[q] = delta * L * (double)(t[2] - t[1] + 1);
    }
}

/*
 * jo_backproject_voxels: (A^T proj)[v] for a LIST of voxels, by the definition of the transpose,
 * (A^T y)[v] = sum_rays y[ray] * (A e_v)[ray].
 * With e_v the unit volume at voxel v = (ix, iy, iz), a ray sees it on exactly one slice, i = v_m,
 * with the weight  delta * ||r~|| * H(p_t1(i) - v_t1) * H(p_t2(i) - v_t2),  H the hat of
 * jo_ray_definition -- no floor, no tap list.  Only the pixels within `halfwin` of the voxel
 * centre's projection onto the detector are visited (every other ray passes more than one voxel
 * away from v on slice v_m and has weight zero; the caller chooses halfwin and the tests check it
 * against the full jo_backproject).
 *   vox   [n_vox][3] = ix, iy, iz;     out [n_vox]  (overwritten)
 */
void jo_backproject_voxels(const double *proj, const int n[3], double delta, const double origin[3],
                           const double *geom, int kernel, int n_proj, int nu, int nv, int halfwin,
                           long n_vox, const int32_t *vox, double *out)
{
    long q;
    int p;
    for (q = 0; q < n_vox; ++q) {
        const int32_t *v = vox + 3 * q;
        double acc = 0.0;
        out[q] = 0.0;
        if (v[0] < 0 || v[1] < 0 || v[2] < 0 || v[0] >= n[0] || v[1] >= n[1] || v[2] >= n[2])
            continue;
        for (p = 0; p < n_proj; ++p) {
            const double *g = geom + 12 * (size_t)p;
            double x[3], e[3], nrm[3], uu = 0.0, vv = 0.0, uv = 0.0, den = 0.0, num = 0.0, lam, h[3], bu = 0.0, bv = 0.0, det;
            int a, iu, iv, cu, cv;
            /* voxel centre in world units; intersect the line source -> centre with the detector plane */
            for (a = 0; a < 3; ++a) x[a] = origin[a] + delta * (double)v[a];
            nrm[0] = g[7] * g[11] - g[8] * g[10];
            nrm[1] = g[8] * g[9] - g[6] * g[11];
            nrm[2] = g[6] * g[10] - g[7] * g[9];
            for (a = 0; a < 3; ++a) { e[a] = x[a] - g[a]; den += nrm[a] * e[a]; num += nrm[a] * (g[3 + a] - g[a]); }
            if (den == 0.0) continue;
            lam = num / den;
            if (!(lam > 0.0)) continue;
            for (a = 0; a < 3; ++a) h[a] = g[a] + lam * e[a] - g[3 + a];     /* hit point relative to det_origin */
            for (a = 0; a < 3; ++a) { uu += g[6 + a] * g[6 + a]; vv += g[9 + a] * g[9 + a]; uv += g[6 + a] * g[9 + a];
                                      bu += g[6 + a] * h[a]; bv += g[9 + a] * h[a]; }
            det = uu * vv - uv * uv;
            if (det == 0.0) continue;
            cu = (int)floor((bu * vv - bv * uv) / det + 0.5);
            cv = (int)floor((bv * uu - bu * uv) / det + 0.5);
            for (iv = cv - halfwin; iv <= cv + halfwin; ++iv)
                for (iu = cu - halfwin; iu <= cu + halfwin; ++iu) {
                    double s[3], d[3], rt[3], L, x1, x2, h1, h2;
                    int m, t1, t2, i;
                    if (iu < 0 || iv < 0 || iu >= nu || iv >= nv) continue;
                    jo_pixel_to_grid(g, delta, origin, iu, iv, s, d);
                    if (!jo_setup(s, d, &m, rt, &L)) continue;
                    t1 = (m + 1) % 3;
                    t2 = (m + 2) % 3;
                    i = v[m];
                    x1 = fabs(jo_pt(s, rt, m, t1, i) - (double)v[t1]);
                    x2 = fabs(jo_pt(s, rt, m, t2, i) - (double)v[t2]);
                    h1 = x1 < 1.0 ? jo_w(kernel, x1) : 0.0;
                    h2 = x2 < 1.0 ? jo_w(kernel, x2) : 0.0;
                    acc += delta * L * h1 * h2
                           * proj[((size_t)p * (size_t)nv + (size_t)iv) * (size_t)nu + (size_t)iu];
                }
        }
        out[q] = acc;
    }
}
