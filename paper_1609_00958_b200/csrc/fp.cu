// fp.cu -- host side of libfp.so: the C ABI declared in include/fp.h.
// Argument validation, per-projection planning on the host, workspace ownership, launches.
// No arithmetic of the method lives here except the host planning heuristics (which kernel,
// which warp orientation); every step of the hot path runs in the kernels of fp_kernels.cuh.
#include <cmath>
#include <mutex>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/fp.h"
#include "fp_kernels.cuh"
#include "fp_aligned.cuh"
#include "fp_tma.cuh"
#include "fp_tex.cuh"
#include "fp_tile.cuh"
#include "fp_bp.cuh"
#include "fp_probe.cuh"

using namespace fpk;

struct fp_ctx {
    GridDesc G;
    // options
    int opt_kernel = FP_KERNEL_AUTO;
    int opt_volatile = 1;
    int opt_interp = FP_INTERP_LINEAR;
    int opt_permuted = 1;
    int opt_count = 0;
    int opt_fov = 0;
    int opt_group = 8;                         // projections per launch-order group of the aligned / TMA kernels
    int opt_force_tma = 0;                     // test hook: every aligned pose goes to fp_tma_kernel whether it fits or not
    // layout stage: y-fastest copy [nz][nx][ny] for z-driven rays
    float *vol_perm = nullptr;
    const float *perm_src = nullptr;
    bool perm_valid = false;
    // per-call workspaces
    ProjDesc *proj_dev = nullptr;
    int proj_cap = 0;
    unsigned long long *count_dev = nullptr;   // [0] sample count, [1] (low word) staging-window error flag
    int *ids_dev = nullptr;                    // [4 * ids_cap]: aligned ids, direct ids, TMA ids, texture-kernel ids
    int ids_cap = 0;
    bool aligned_attr_set = false;
    // tensor maps of the TMA kernel: valid for one volume pointer
    CUtensorMap tmap[2][kTmWBoxes][kTmMaps];
    const float *tmap_vol = nullptr;
    // tensor maps of the tile kernel: [driving axis][box size]; axis 2 covers the y-fastest copy
    CUtensorMap tlmap[3][kTlSizes][kTlSizes];
    const float *tlmap_vol = nullptr, *tlmap_perm = nullptr;
    // layout stage of fp_tex_kernel: one layered 2-D array per driving axis (layer = slice), its surface (fill
    // kernel) and two texture objects over it (point sampling for tld4, linear filtering for GJP_hwlin)
    cudaArray_t arr[3] = {nullptr, nullptr, nullptr};
    cudaSurfaceObject_t surf[3] = {0, 0, 0};
    cudaTextureObject_t atex[3][2] = {{0, 0}, {0, 0}, {0, 0}};
    const float *arr_src[3] = {nullptr, nullptr, nullptr};
    bool arr_valid[3] = {false, false, false};
    int n_sm = 0;
    cudaStream_t last_stream = nullptr;
    cudaEvent_t ev_last = nullptr;                   // end of the most recent call: a call on another stream waits for it
    bool ev_valid = false;
    bool counted = false;
    int last_launches = 0;
    // fp_project_host workspaces
    float *hvol_dev = nullptr;
    float *hout_dev[2] = {nullptr, nullptr};
    size_t hout_cap = 0;
    cudaStream_t hstream[2] = {nullptr, nullptr};
    cudaEvent_t hevent[2] = {nullptr, nullptr};      // batch sampled (compute stream)
    cudaEvent_t hcopied[2] = {nullptr, nullptr};     // batch copied to the host (copy stream)
    bool keep_count = false;                         // fp_project_host: batches add to one sample count
    // host plan of the most recent fp_project call (which kernel takes which projection): reused when the next call
    // brings the same geometry, detector, options and volume alignment -- the calls of an iterative reconstruction
    // -- instead of being worked out again (C3: about 30 microseconds per pose)
    struct PlanCache {
        std::vector<double> geom;
        int nu = 0, nv = 0, opt_kernel = -1, opt_force_tma = -1;
        unsigned vol_align = ~0u;
        std::vector<int> ids_al, ids_di, ids_tm, ids_tn, ids_tx;
        int w_al = 0;
    } plan;
    std::string err;
};

static fp_status fail(fp_ctx *c, fp_status s, const std::string &msg)
{
    if (c) c->err = msg;
    return s;
}

static fp_status cuda_fail(fp_ctx *c, cudaError_t e, const char *what)
{
    char buf[512];
    snprintf(buf, sizeof buf, "%s: %s (%s)", what, cudaGetErrorString(e), cudaGetErrorName(e));
    cudaGetLastError();   // clear the sticky flag of non-fatal errors
    return fail(c, e == cudaErrorMemoryAllocation ? FP_ERR_OOM : FP_ERR_CUDA, buf);
}

#define FP_CUDA(ctx, call)                                             \
    do {                                                               \
        cudaError_t e_ = (call);                                       \
        if (e_ != cudaSuccess) return cuda_fail((ctx), e_, #call);     \
    } while (0)

// The per-context workspaces (geometry rows, projection ids, counters) are rewritten by every call in stream
// order.  A call on another stream than the previous one first waits for that call's end, so that two streams
// never race on them (the calls are then serialised: use one context per stream for concurrency).
static fp_status enter_stream(fp_ctx *c, cudaStream_t st)
{
    if (c->ev_valid && st != c->last_stream) FP_CUDA(c, cudaStreamWaitEvent(st, c->ev_last, 0));
    if (!c->count_dev) {
        FP_CUDA(c, cudaMalloc(&c->count_dev, 2 * sizeof(unsigned long long)));
        FP_CUDA(c, cudaMemsetAsync(c->count_dev, 0, 2 * sizeof(unsigned long long), st));
    }
    return FP_OK;
}

static fp_status leave_stream(fp_ctx *c, cudaStream_t st)
{
    if (!c->ev_last) FP_CUDA(c, cudaEventCreateWithFlags(&c->ev_last, cudaEventDisableTiming));
    FP_CUDA(c, cudaEventRecord(c->ev_last, st));
    c->ev_valid = true;
    c->last_stream = st;
    return FP_OK;
}

// Synchronises the stream of the most recent call and reads { sample count, error flag }; a raised flag (a
// staging window or row tile of the aligned / TMA kernels did not fit: the host plan was too small and the
// affected rays hold wrong values) is cleared by the read.
static fp_status read_counters(fp_ctx *c, unsigned long long h[2])
{
    h[0] = h[1] = 0;
    if (!c->count_dev) return FP_OK;
    FP_CUDA(c, cudaStreamSynchronize(c->last_stream));
    FP_CUDA(c, cudaMemcpy(h, c->count_dev, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    if (h[1] != 0) FP_CUDA(c, cudaMemset(c->count_dev + 1, 0, sizeof(unsigned long long)));
    return FP_OK;
}

static const char *kPlanError =
    "a staging window or row tile of the aligned / TMA kernel did not fit (host plan too small): the projections "
    "written since the last check are invalid; repeat the call with FP_OPT_KERNEL = FP_KERNEL_DIRECT";

static size_t n_voxels(const fp_ctx *c) { return (size_t)c->G.n[0] * c->G.n[1] * c->G.n[2]; }

extern "C" const char *fp_version(void) { return "libfp 0.1 (sm_100a)"; }

extern "C" const char *fp_status_string(fp_status s)
{
    switch (s) {
    case FP_OK: return "FP_OK";
    case FP_ERR_INVALID_ARG: return "FP_ERR_INVALID_ARG";
    case FP_ERR_CUDA: return "FP_ERR_CUDA";
    case FP_ERR_OOM: return "FP_ERR_OOM";
    case FP_ERR_UNSUPPORTED: return "FP_ERR_UNSUPPORTED";
    }
    return "FP_ERR_?";
}

extern "C" const char *fp_last_error(fp_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

extern "C" fp_status fp_create(int nx, int ny, int nz, double voxel_size, const double origin[3], fp_ctx **out)
{
    if (!out) return FP_ERR_INVALID_ARG;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1 || !origin) return FP_ERR_INVALID_ARG;
    if (!(voxel_size > 0.0) || !std::isfinite(voxel_size)) return FP_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a)
        if (!std::isfinite(origin[a])) return FP_ERR_INVALID_ARG;
    if ((double)nx * ny * nz >= 1099511627776.0) return FP_ERR_INVALID_ARG;
    fp_ctx *c = new (std::nothrow) fp_ctx;
    if (!c) return FP_ERR_OOM;
    c->G.n[0] = nx;
    c->G.n[1] = ny;
    c->G.n[2] = nz;
    c->G.pad_ = 0;
    c->G.delta = voxel_size;
    for (int a = 0; a < 3; ++a) c->G.origin[a] = origin[a];
    *out = c;
    return FP_OK;
}

extern "C" fp_status fp_destroy(fp_ctx *c)
{
    if (!c) return FP_ERR_INVALID_ARG;
    cudaDeviceSynchronize();
    cudaFree(c->vol_perm);
    cudaFree(c->proj_dev);
    cudaFree(c->count_dev);
    if (c->ev_last) cudaEventDestroy(c->ev_last);
    cudaFree(c->ids_dev);
    cudaFree(c->hvol_dev);
    for (int a = 0; a < 3; ++a) {
        for (int f = 0; f < 2; ++f)
            if (c->atex[a][f]) cudaDestroyTextureObject(c->atex[a][f]);
        if (c->surf[a]) cudaDestroySurfaceObject(c->surf[a]);
        if (c->arr[a]) cudaFreeArray(c->arr[a]);
    }
    for (int k = 0; k < 2; ++k) {
        cudaFree(c->hout_dev[k]);
        if (c->hstream[k]) cudaStreamDestroy(c->hstream[k]);
        if (c->hevent[k]) cudaEventDestroy(c->hevent[k]);
        if (c->hcopied[k]) cudaEventDestroy(c->hcopied[k]);
    }
    cudaGetLastError();
    delete c;
    return FP_OK;
}

extern "C" fp_status fp_set_option(fp_ctx *c, int key, int value)
{
    if (!c) return FP_ERR_INVALID_ARG;
    switch (key) {
    case FP_OPT_KERNEL:
        if (value < FP_KERNEL_AUTO || value > FP_KERNEL_TILE) return fail(c, FP_ERR_INVALID_ARG, "bad kernel variant");
        c->opt_kernel = value;
        return FP_OK;
    case FP_OPT_VOLATILE: c->opt_volatile = value != 0; return FP_OK;
    case FP_OPT_INTERP:
        if (value != FP_INTERP_LINEAR && value != FP_INTERP_SPLINE) return fail(c, FP_ERR_INVALID_ARG, "bad interpolation kernel");
        c->opt_interp = value;
        return FP_OK;
    case FP_OPT_PERMUTED_COPY:
        c->opt_permuted = value != 0;
        c->perm_valid = false;
        return FP_OK;
    case FP_OPT_COUNT_SAMPLES: c->opt_count = value != 0; return FP_OK;
    case FP_OPT_FOV_CYLINDER: c->opt_fov = value != 0; return FP_OK;
    case FP_OPT_GROUP:
        if (value < 1 || value > 64) return fail(c, FP_ERR_INVALID_ARG, "FP_OPT_GROUP must be 1 .. 64");
        c->opt_group = value;
        return FP_OK;
    case FP_OPT_TEST_FORCE_TMA: c->opt_force_tma = value != 0; return FP_OK;
    }
    return fail(c, FP_ERR_INVALID_ARG, "unknown option key");
}

extern "C" fp_status fp_get_option(fp_ctx *c, int key, int *value)
{
    if (!c || !value) return FP_ERR_INVALID_ARG;
    switch (key) {
    case FP_OPT_KERNEL: *value = c->opt_kernel; return FP_OK;
    case FP_OPT_VOLATILE: *value = c->opt_volatile; return FP_OK;
    case FP_OPT_INTERP: *value = c->opt_interp; return FP_OK;
    case FP_OPT_PERMUTED_COPY: *value = c->opt_permuted; return FP_OK;
    case FP_OPT_COUNT_SAMPLES: *value = c->opt_count; return FP_OK;
    case FP_OPT_FOV_CYLINDER: *value = c->opt_fov; return FP_OK;
    case FP_OPT_GROUP: *value = c->opt_group; return FP_OK;
    case FP_OPT_TEST_FORCE_TMA: *value = c->opt_force_tma; return FP_OK;
    }
    return fail(c, FP_ERR_INVALID_ARG, "unknown option key");
}

// ---------------------------------------------------------------------------- host planning

// Does the open detector rectangle contain directions whose largest component is z?  The ray
// direction is affine in (iu, iv), so { r : |r_z| > |r_x|, |r_z| > |r_y| } cuts the detector
// plane in two convex polygons (one per sign of r_z): clip the rectangle against the four half
// planes of each.  Conservative (closed half planes); only decides whether the permuted copy
// is worth building -- the kernels are correct either way.
static bool has_axis_driven(const double *g, int nu, int nv, int axis);
static bool has_z_driven(const double *g, int nu, int nv) { return has_axis_driven(g, nu, nv, 2); }

// The same for any axis: does some ray of the pose have `axis` as its largest direction component?
static bool has_axis_driven(const double *g, int nu, int nv, int axis)
{
    const int o1 = (axis + 1) % 3, o2 = (axis + 2) % 3;
    const double c0[3] = {g[3] - g[0], g[4] - g[1], g[5] - g[2]};   // r at (0,0)
    for (int sign = -1; sign <= 1; sign += 2) {
        // polygon in (iu, iv)
        std::vector<std::pair<double, double>> poly = {
            {-0.5, -0.5}, {nu - 0.5, -0.5}, {nu - 0.5, nv - 0.5}, {-0.5, nv - 0.5}};
        for (int k = 0; k < 4 && !poly.empty(); ++k) {
            const int ax = (k >> 1) ? o2 : o1;           // the two other axes
            const double sg = (k & 1) ? 1.0 : -1.0;      // sign*r_axis -/+ r_ax >= 0
            const double A = sign * c0[axis] + sg * c0[ax];
            const double B = sign * g[6 + axis] + sg * g[6 + ax];
            const double C = sign * g[9 + axis] + sg * g[9 + ax];
            std::vector<std::pair<double, double>> nxt;
            const size_t n = poly.size();
            for (size_t q = 0; q < n; ++q) {
                const auto &a = poly[q], &b = poly[(q + 1) % n];
                const double fa = A + B * a.first + C * a.second, fb = A + B * b.first + C * b.second;
                if (fa >= 0) nxt.push_back(a);
                if ((fa >= 0) != (fb >= 0)) {
                    const double t = fa / (fa - fb);
                    nxt.push_back({a.first + t * (b.first - a.first), a.second + t * (b.second - a.second)});
                }
            }
            poly.swap(nxt);
        }
        if (poly.size() >= 3) {
            double area = 0;
            for (size_t q = 0; q < poly.size(); ++q) {
                const auto &a = poly[q], &b = poly[(q + 1) % poly.size()];
                area += a.first * b.second - a.second * b.first;
            }
            if (std::fabs(area) > 1e-9) return true;
        }
    }
    return false;
}

// Warp orientation: lanes run along the detector vector with the larger component along the
// axis that is contiguous for the central ray's driving axis (adjacent rays
// should read consecutive addresses).
static int plan_lane_v(const double *g, int nu, int nv, bool permuted)
{
    double r[3];
    for (int a = 0; a < 3; ++a)
        r[a] = g[3 + a] + 0.5 * (nu - 1) * g[6 + a] + 0.5 * (nv - 1) * g[9 + a] - g[a];
    int m = 0;
    if (std::fabs(r[1]) > std::fabs(r[m])) m = 1;
    if (std::fabs(r[2]) > std::fabs(r[m])) m = 2;
    const int fast = (m == 2 && permuted) ? 1 : 2;
    if (m == 2 && !permuted) return std::fabs(g[9 + 1]) > std::fabs(g[6 + 1]);
    return std::fabs(g[9 + fast]) > std::fabs(g[6 + fast]);
}

// Can fp_aligned_kernel take this pose, and how wide a staging window (voxels along z) does it
// need?  Conditions: u perpendicular to z, v parallel to z (exact zeros, so that r_x, r_y depend
// on the column only and r_z on the row only), no z-driven ray, nz a multiple of 4 and a
// 16-byte aligned volume (float4 loads along z).  The window bound is conservative: the largest
// ray parameter |t| = |(i - s_m) / r_m| over all slices a batch can touch, times the r_z spread
// of the rows of one block, plus the drift inside a batch, alignment and tap margins.
static int plan_aligned(const fp_ctx *c, const float *vol, const double *g, int nu, int nv, int *tile_rows = nullptr,
                        int block_rows = kAlTV)
{
    if (tile_rows) *tile_rows = 1 << 30;
    for (int k = 0; k < 12; ++k)
        if (!std::isfinite(g[k])) return 0;
    if (g[8] != 0.0 || g[9] != 0.0 || g[10] != 0.0 || g[11] == 0.0) return 0;
    if ((c->G.n[2] & 3) != 0 || ((uintptr_t)vol & 15) != 0) return 0;
    const double dl = c->G.delta;
    double s[3];
    for (int a = 0; a < 3; ++a) s[a] = (g[a] - c->G.origin[a]) / dl;
    auto rho = [&](int iv) { return ((g[5] + iv * g[11]) - c->G.origin[2]) / dl - s[2]; };
    const double rz_max = std::max(std::fabs(rho(0)), std::fabs(rho(nv - 1)));
    // per column: the slices whose slow-axis position can lie inside (-1, N_s) (one slice of slack on
    // either side), widened by one batch; the ray parameter t = (i - s_m) / r_m over them
    double rm_min = INFINITY, t_lo = INFINITY, t_hi = -INFINITY;
    struct ColInfo { int m; double rt, dmax; };
    std::vector<ColInfo> cols((size_t)nu, ColInfo{-1, 0.0, 0.0});
    for (int iu = 0; iu < nu; ++iu) {
        double r[2];
        for (int a = 0; a < 2; ++a) r[a] = ((g[3 + a] + iu * g[6 + a]) - c->G.origin[a]) / dl - s[a];
        const int m = std::fabs(r[1]) > std::fabs(r[0]) ? 1 : 0;
        const double rm = r[m], rs = r[1 - m];
        rm_min = std::min(rm_min, std::fabs(rm));
        if (rm == 0.0) return 0;
        double i_a = 0.0, i_b = (double)(c->G.n[m] - 1);
        const double rt = rs / rm, ss = s[1 - m], ns = (double)c->G.n[1 - m];
        if (rt != 0.0) {
            const double x1 = s[m] + (-1.0 - ss) / rt, x2 = s[m] + (ns - ss) / rt;
            i_a = std::max(i_a, std::floor(std::min(x1, x2)) - 1.0);
            i_b = std::min(i_b, std::ceil(std::max(x1, x2)) + 1.0);
        } else if (!(ss > -1.0 && ss < ns)) {
            continue;
        }
        if (i_a > i_b) continue;
        i_b += kAlSB;
        cols[iu] = ColInfo{m, rt, std::max(std::fabs(i_a - s[m]), std::fabs(i_b - s[m]))};
        const double t_a = (i_a - s[m]) / rm, t_b = (i_b - s[m]) / rm;
        t_lo = std::min(t_lo, std::min(t_a, t_b));
        t_hi = std::max(t_hi, std::max(t_a, t_b));
    }
    if (!(rz_max <= rm_min * (1.0 - 1e-9))) return 0;            // a z-driven (or tied) ray somewhere
    if (!(t_lo <= t_hi)) return 16;                              // every column misses: any window will do
    const double t_max = std::max(std::fabs(t_lo), std::fabs(t_hi));
    const int rows = std::min(nv, block_rows);
    // rows of one block at one t, the drift inside a batch, and the difference in t between the columns
    // of a block, which share one window: their first slices differ (entry through a side face) and
    // their r_m differ by at most kAlTU detector steps
    const double du = std::max(std::fabs(g[6]), std::fabs(g[7])) / dl;
    const double dt_cols = t_max * (kAlTU * du / rm_min) + 4.0 / rm_min;
    const double span = t_max * (rows - 1) * std::fabs(g[11] / dl) + (kAlSB - 1) * (rz_max / rm_min) + dt_cols * rz_max;
    if (!(span < 1.0e6)) return 0;
    if (tile_rows) {
        // volume rows one block of fp_tma_kernel needs per slice: the columns of a block that share a driving
        // axis spread over |i - s_m| (max r~_s - min r~_s) rows of the slice plane, plus the two taps
        int rows = 0;
        for (int iu0 = 0; iu0 < nu; iu0 += kTmTU)
            for (int m = 0; m < 2; ++m) {
                double lo = INFINITY, hi = -INFINITY, d = 0.0;
                for (int iu = iu0; iu < std::min(nu, iu0 + kTmTU); ++iu)
                    if (cols[iu].m == m) {
                        lo = std::min(lo, cols[iu].rt);
                        hi = std::max(hi, cols[iu].rt);
                        d = std::max(d, cols[iu].dmax);
                    }
                if (lo <= hi) rows = std::max(rows, (int)std::min(d * (hi - lo), 1.0e6) + 3);
            }
        *tile_rows = rows;
    }
    return (int)std::ceil(span) + 10;
}

static fp_status ensure_ids(fp_ctx *c, int n_proj)
{
    if (n_proj <= c->ids_cap) return FP_OK;
    if (c->ids_dev) {
        FP_CUDA(c, cudaDeviceSynchronize());
        cudaFree(c->ids_dev);
        c->ids_dev = nullptr;
        c->ids_cap = 0;
    }
    const int cap = n_proj + 64;
    FP_CUDA(c, cudaMalloc(&c->ids_dev, sizeof(int) * 5 * (size_t)cap));
    c->ids_cap = cap;
    return FP_OK;
}

template <int INTERP, int W>
static fp_status launch_aligned_w(fp_ctx *c, const AlignedParams &A, dim3 grid, cudaStream_t st)
{
    constexpr size_t smem = aligned_smem_bytes<W>();
    // the attribute is per device; setting it on every launch is cheap
    FP_CUDA(c, cudaFuncSetAttribute(fp_aligned_kernel<INTERP, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    fp_aligned_kernel<INTERP, W><<<grid, kAlTV, smem, st>>>(A);
    FP_CUDA(c, cudaGetLastError());
    return FP_OK;
}

template <int INTERP>
static fp_status launch_aligned(fp_ctx *c, const AlignedParams &A, int w, dim3 grid, cudaStream_t st)
{
    if (w <= 128) return launch_aligned_w<INTERP, 128>(c, A, grid, st);
    if (w <= 256) return launch_aligned_w<INTERP, 256>(c, A, grid, st);
    if (w <= 384) return launch_aligned_w<INTERP, 384>(c, A, grid, st);
    return launch_aligned_w<INTERP, 512>(c, A, grid, st);
}

constexpr int kAlignedMaxW = 512;

// Tensor maps of fp_tma_kernel over the caller's volume, dimensions (z, y, x): a box is kTmW voxels along z
// and 8 or 12 rows along the slow transverse axis of the pass (y for m = x, x for m = y) of one slice.
typedef CUresult (*tensor_map_encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                         const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                         CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static tensor_map_encode_fn g_encode = nullptr;

static fp_status get_encoder(fp_ctx *c)
{
    if (!g_encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        FP_CUDA(c, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) return fail(c, FP_ERR_UNSUPPORTED, "cuTensorMapEncodeTiled not available");
        g_encode = (tensor_map_encode_fn)fn;
    }
    return FP_OK;
}

// Tensor maps of fp_tile_kernel: per driving axis a rows x cols box of one slice plane, fast in-plane axis innermost.
// m = x, y: the caller's volume, dimensions (z, y, x); m = z: the y-fastest copy [nz][nx][ny], dimensions (y, x, z).
static fp_status build_tile_maps(fp_ctx *c, const float *vol, const float *perm)
{
    if (c->tlmap_vol == vol && c->tlmap_perm == perm) return FP_OK;
    fp_status s = get_encoder(c);
    if (s != FP_OK) return s;
    const cuuint32_t estr[3] = {1, 1, 1};
    for (int m = 0; m < 3; ++m) {
        if (m == 2 && !perm) continue;
        const cuuint64_t nx = c->G.n[0], ny = c->G.n[1], nz = c->G.n[2];
        const cuuint64_t dims[3] = {m == 2 ? ny : nz, m == 2 ? nx : ny, m == 2 ? nz : nx};
        const cuuint64_t strides[2] = {dims[0] * 4, dims[0] * dims[1] * 4};
        for (int k = 0; k < kTlSizes * kTlSizes; ++k) {
            const cuuint32_t rows = (cuuint32_t)tl_rows(k / kTlSizes), cols = (cuuint32_t)tl_cols(k % kTlSizes);
            const cuuint32_t box[3] = {cols, m == 1 ? 1u : rows, m == 1 ? rows : 1u};
            const CUresult r = g_encode(&c->tlmap[m][k / kTlSizes][k % kTlSizes], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)(m == 2 ? perm : vol), dims,
                                        strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) {
                char buf[96];
                snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled (tile kernel) failed (%d)", (int)r);
                return fail(c, FP_ERR_CUDA, buf);
            }
        }
    }
    c->tlmap_vol = vol;
    c->tlmap_perm = perm;
    return FP_OK;
}

static fp_status build_tensor_maps(fp_ctx *c, const float *vol)
{
    if (c->tmap_vol == vol) return FP_OK;
    fp_status es = get_encoder(c);
    if (es != FP_OK) return es;
    tensor_map_encode_fn encode = g_encode;
    const cuuint64_t dims[3] = {(cuuint64_t)c->G.n[2], (cuuint64_t)c->G.n[1], (cuuint64_t)c->G.n[0]};
    const cuuint64_t strides[2] = {(cuuint64_t)c->G.n[2] * 4, (cuuint64_t)c->G.n[2] * c->G.n[1] * 4};
    const cuuint32_t estr[3] = {1, 1, 1};
    for (int pass = 0; pass < 2; ++pass)
        for (int wi = 0; wi < kTmWBoxes; ++wi)
            for (int big = 0; big < kTmMaps; ++big) {
                const cuuint32_t rows = 4 + 2 * big, width = kTmWMin + kTmWStep * wi;
                const cuuint32_t box[3] = {width, pass == 0 ? rows : 1u, pass == 0 ? 1u : rows};
                const CUresult r = encode(&c->tmap[pass][wi][big], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)vol, dims,
                                          strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                          CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                if (r != CUDA_SUCCESS) {
                    char buf[96];
                    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (%d)", (int)r);
                    return fail(c, FP_ERR_CUDA, buf);
                }
            }
    c->tmap_vol = vol;
    return FP_OK;
}

// Does a pose with this z window and these volume rows per slice fit fp_tma_kernel's tiles?
static bool fits_tma(int window, int rows) { return window > 0 && window <= kTmW && rows <= kTmNR; }

template <int INTERP, int ROWS>
static fp_status launch_tma(fp_ctx *c, const TmaParams &T, dim3 grid, cudaStream_t st)
{
    // per device and cheap: set on every launch
    const size_t smem = tma_smem_bytes();
    FP_CUDA(c, cudaFuncSetAttribute(fp_tma_kernel<INTERP, ROWS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    fp_tma_kernel<INTERP, ROWS><<<grid, tm_threads(ROWS), smem, st>>>(T);
    FP_CUDA(c, cudaGetLastError());
    return FP_OK;
}

// Which fp_tma_kernel takes an aligned pose: 256 detector rows per block, 192 where only their narrower z window
// fits the largest TMA box, 0 = neither.  w256 / tile_rows: plan_aligned() of the pose for 256-row blocks.
static int tma_block_rows(const fp_ctx *c, const float *vol, const double *g, int nu, int nv, int w256, int tile_rows,
                          int *window = nullptr)
{
    if (window) *window = w256;
    if (fits_tma(w256, tile_rows)) return kTmRows;
    if (w256 <= 0 || tile_rows > kTmNR) return 0;
    const int w = plan_aligned(c, vol, g, nu, nv, nullptr, kTmRowsNarrow);
    if (!fits_tma(w, tile_rows)) return 0;
    if (window) *window = w;
    return kTmRowsNarrow;
}


// Layout stage of fp_tex_kernel (sec. 2.8): the layered array of driving axis `axis`
// (layer = slice, row = slow transverse axis, column = fast transverse axis), filled from the caller's volume
// on `st`.  Arrays, surfaces and texture objects are created once per context.
static fp_status ensure_layers(fp_ctx *c, const float *vol, int axis, cudaStream_t st)
{
    const int nx = c->G.n[0], ny = c->G.n[1], nz = c->G.n[2];
    const int n_layer = c->G.n[axis];
    const int n_row = axis == 0 ? ny : nx, n_col = axis == 2 ? ny : nz;
    if (!c->arr[axis]) {
        int dev = 0, lim[3] = {0, 0, 0};
        FP_CUDA(c, cudaGetDevice(&dev));
        FP_CUDA(c, cudaDeviceGetAttribute(&lim[0], cudaDevAttrMaxTexture2DLayeredWidth, dev));
        FP_CUDA(c, cudaDeviceGetAttribute(&lim[1], cudaDevAttrMaxTexture2DLayeredHeight, dev));
        FP_CUDA(c, cudaDeviceGetAttribute(&lim[2], cudaDevAttrMaxTexture2DLayeredLayers, dev));
        if (n_col > lim[0] || n_row > lim[1] || n_layer > lim[2])
            return fail(c, FP_ERR_UNSUPPORTED, "volume too large for a layered texture array on this device");
        cudaChannelFormatDesc cd = cudaCreateChannelDesc<float>();
        FP_CUDA(c, cudaMalloc3DArray(&c->arr[axis], &cd, make_cudaExtent((size_t)n_col, (size_t)n_row, (size_t)n_layer),
                                     cudaArrayLayered | cudaArraySurfaceLoadStore));
        cudaResourceDesc rd;
        memset(&rd, 0, sizeof rd);
        rd.resType = cudaResourceTypeArray;
        rd.res.array.array = c->arr[axis];
        FP_CUDA(c, cudaCreateSurfaceObject(&c->surf[axis], &rd));
        for (int f = 0; f < 2; ++f) {
            cudaTextureDesc td;
            memset(&td, 0, sizeof td);
            td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeBorder;   // outside: 0 (reading #2)
            td.filterMode = f ? cudaFilterModeLinear : cudaFilterModePoint;
            td.readMode = cudaReadModeElementType;
            td.normalizedCoords = 0;
            FP_CUDA(c, cudaCreateTextureObject(&c->atex[axis][f], &rd, &td, nullptr));
        }
    }
    if (axis < 2) {
        dim3 grid((unsigned)nx, (unsigned)((ny + 7) / 8));
        if (axis == 0) fp_fill_layers_kernel<0><<<grid, 256, 0, st>>>(vol, c->surf[0], nx, ny, nz);
        else fp_fill_layers_kernel<1><<<grid, 256, 0, st>>>(vol, c->surf[1], nx, ny, nz);
    } else {
        dim3 grid((unsigned)((nz + 31) / 32), (unsigned)((ny + 31) / 32), (unsigned)nx);
        fp_fill_layers_kernel<2><<<grid, 256, 0, st>>>(vol, c->surf[2], nx, ny, nz);
    }
    FP_CUDA(c, cudaGetLastError());
    c->arr_src[axis] = vol;
    c->arr_valid[axis] = true;
    c->last_launches += 1;
    return FP_OK;
}

// fp_tex_kernel: a persistent grid of as many blocks as fit.
template <int INTERP, bool HW, int U>
static fp_status launch_tex_u(fp_ctx *c, const TexParams &T, cudaStream_t st)
{
    int occ = 0;
    FP_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fp_tex_kernel<INTERP, HW, U>, kTexThreads, 0));
    fp_tex_kernel<INTERP, HW, U><<<(unsigned)(c->n_sm * std::max(occ, 1)), kTexThreads, 0, st>>>(T);
    FP_CUDA(c, cudaGetLastError());
    return FP_OK;
}

static fp_status launch_tex(fp_ctx *c, const TexParams &T, bool hw, cudaStream_t st)
{
    if (!c->n_sm) {
        int dev = 0;
        FP_CUDA(c, cudaGetDevice(&dev));
        FP_CUDA(c, cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev));
    }
    const bool spl = c->opt_interp == FP_INTERP_SPLINE;
    if (hw) return launch_tex_u<0, true, 1>(c, T, st);
    return spl ? launch_tex_u<1, false, 8>(c, T, st) : launch_tex_u<0, false, 8>(c, T, st);
}

static fp_status ensure_proj(fp_ctx *c, int n_proj)
{
    if (n_proj <= c->proj_cap) return FP_OK;
    if (c->proj_dev) {
        // an earlier call may still be reading the old buffer
        FP_CUDA(c, cudaDeviceSynchronize());
        cudaFree(c->proj_dev);
        c->proj_dev = nullptr;
        c->proj_cap = 0;
    }
    const int cap = n_proj + 64;
    FP_CUDA(c, cudaMalloc(&c->proj_dev, sizeof(ProjDesc) * (size_t)cap));
    c->proj_cap = cap;
    return FP_OK;
}

static fp_status upload_geometry(fp_ctx *c, int n_proj, const double *geom, int nu, int nv, bool permuted,
                                 cudaStream_t st)
{
    fp_status s = ensure_proj(c, n_proj);
    if (s != FP_OK) return s;
    std::vector<ProjDesc> h((size_t)n_proj);
    for (int p = 0; p < n_proj; ++p) {
        memcpy(h[p].g, geom + 12 * (size_t)p, sizeof(double) * 12);
        h[p].lane_v = plan_lane_v(h[p].g, nu, nv, permuted);
        h[p].pad_ = 0;
    }
    // pageable source: the runtime stages the bytes before returning, so `h` may die here
    FP_CUDA(c, cudaMemcpyAsync(c->proj_dev, h.data(), sizeof(ProjDesc) * (size_t)n_proj, cudaMemcpyHostToDevice, st));
    return FP_OK;
}

static fp_status build_permuted(fp_ctx *c, const float *vol_dev, cudaStream_t st)
{
    const size_t nvox = n_voxels(c);
    if (!c->vol_perm) FP_CUDA(c, cudaMalloc(&c->vol_perm, nvox * sizeof(float)));
    const long long R = (long long)c->G.n[0] * c->G.n[1], C = c->G.n[2];
    dim3 grid((unsigned)((R + 31) / 32), (unsigned)((C + 31) / 32));
    fp_transpose_kernel<<<grid, 256, 0, st>>>(vol_dev, c->vol_perm, R, C);
    FP_CUDA(c, cudaGetLastError());
    c->perm_src = vol_dev;
    c->perm_valid = true;
    c->last_launches += 1;
    return FP_OK;
}

extern "C" fp_status fp_prepare(fp_ctx *c, const float *vol_dev, fp_stream stream)
{
    if (!c || !vol_dev) return fail(c, FP_ERR_INVALID_ARG, "fp_prepare: null argument");
    c->last_launches = 0;
    if (!c->opt_permuted) return FP_OK;
    return build_permuted(c, vol_dev, (cudaStream_t)stream);
}

static void fill_layouts(const fp_ctx *c, const float *vol, bool use_perm, AxisLayout lay[3])
{
    const long long nx = c->G.n[0], ny = c->G.n[1], nz = c->G.n[2];
    // m = x: slices [x], slow y, fast z
    lay[0] = AxisLayout{vol, ny * nz, nz, 1, (int)nx, (int)ny, (int)nz, 0};
    // m = y: slices [y], slow x, fast z
    lay[1] = AxisLayout{vol, nz, ny * nz, 1, (int)ny, (int)nx, (int)nz, 0};
    // m = z: slow x, fast y; permuted copy [nz][nx][ny] when built
    if (use_perm)
        lay[2] = AxisLayout{c->vol_perm, nx * ny, ny, 1, (int)nz, (int)nx, (int)ny, 0};
    else
        lay[2] = AxisLayout{vol, 1, ny * nz, nz, (int)nz, (int)nx, (int)ny, 0};
}

static fp_status check_project_args(fp_ctx *c, const void *vol, int n_proj, const double *geom, int nu, int nv,
                                    const void *out)
{
    if (!c) return FP_ERR_INVALID_ARG;
    if (n_proj < 0) return fail(c, FP_ERR_INVALID_ARG, "n_proj < 0");
    if (nu < 1 || nv < 1) return fail(c, FP_ERR_INVALID_ARG, "nu, nv must be >= 1");
    if (n_proj > 0 && (!vol || !geom || !out)) return fail(c, FP_ERR_INVALID_ARG, "null pointer");
    if (n_proj > 65535) return fail(c, FP_ERR_UNSUPPORTED, "n_proj > 65535 per call: split the call");
    return FP_OK;
}

extern "C" fp_status fp_project(fp_ctx *c, const float *vol_dev, int n_proj, const double *geom, int nu, int nv,
                                float *out_dev, fp_stream stream)
{
    fp_status s = check_project_args(c, vol_dev, n_proj, geom, nu, nv, out_dev);
    if (s != FP_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_launches = 0;
    c->counted = false;
    if (n_proj == 0) return FP_OK;
    s = enter_stream(c, st);
    if (s != FP_OK) return s;

    // plan: which kernel takes which projection
    fp_ctx::PlanCache &pc = c->plan;
    std::vector<int> &ids_al = pc.ids_al, &ids_di = pc.ids_di, &ids_tm = pc.ids_tm, &ids_tn = pc.ids_tn, &ids_tx = pc.ids_tx;
    int &w_al = pc.w_al;
    const bool all_tex = c->opt_kernel == FP_KERNEL_TEX || c->opt_kernel == FP_KERNEL_HWLIN;
    const size_t n_geom = 12 * (size_t)n_proj;
    const bool plan_hit = pc.geom.size() == n_geom && pc.nu == nu && pc.nv == nv && pc.opt_kernel == c->opt_kernel &&
                          pc.opt_force_tma == c->opt_force_tma && pc.vol_align == (unsigned)((uintptr_t)vol_dev & 15) &&
                          memcmp(pc.geom.data(), geom, sizeof(double) * n_geom) == 0;
    if (!plan_hit) {
        pc.geom.clear();                               // no valid plan while it is being rebuilt
        ids_al.clear(); ids_di.clear(); ids_tm.clear(); ids_tn.clear(); ids_tx.clear();
        w_al = 0;
    }
    for (int p = 0; p < n_proj && !plan_hit; ++p) {
        if (all_tex) {
            ids_tx.push_back(p);
            continue;
        }
        int rows = 0;
        const int w = c->opt_kernel == FP_KERNEL_DIRECT ? 0 : plan_aligned(c, vol_dev, geom + 12 * (size_t)p, nu, nv, &rows);
        const int tm_rows = c->opt_kernel == FP_KERNEL_ALIGNED ? 0
                            : (c->opt_force_tma && w > 0) ? kTmRows
                                                          : tma_block_rows(c, vol_dev, geom + 12 * (size_t)p, nu, nv, w, rows);
        if (tm_rows == kTmRows) {
            ids_tm.push_back(p);                       // fits the TMA-fed kernel's tile
        } else if (tm_rows == kTmRowsNarrow) {
            ids_tn.push_back(p);                       // ... with 192 detector rows per block
        } else if (w > 0 && w <= kAlignedMaxW) {
            ids_al.push_back(p);
            w_al = std::max(w_al, w);
        } else {
            ids_di.push_back(p);
        }
    }
    if (!plan_hit) {
        pc.geom.assign(geom, geom + n_geom);
        pc.nu = nu;
        pc.nv = nv;
        pc.opt_kernel = c->opt_kernel;
        pc.opt_force_tma = c->opt_force_tma;
        pc.vol_align = (unsigned)((uintptr_t)vol_dev & 15);
    }
    // layout stage: only when some projection of the direct kernel has z-driven rays
    bool want_perm = false;
    if (c->opt_permuted)
        for (size_t q = 0; q < ids_di.size() && !want_perm; ++q)
            want_perm = has_z_driven(geom + 12 * (size_t)ids_di[q], nu, nv);
    if (want_perm && (!c->perm_valid || c->perm_src != vol_dev || c->opt_volatile)) {
        s = build_permuted(c, vol_dev, st);
        if (s != FP_OK) return s;
    }
    const bool use_perm = want_perm && c->perm_valid;
    // layout stage of the texture kernel: the layered array of every driving axis its projections have
    for (int a = 0; a < 3 && !ids_tx.empty(); ++a) {
        bool want = false;
        for (size_t q = 0; q < ids_tx.size() && !want; ++q) want = has_axis_driven(geom + 12 * (size_t)ids_tx[q], nu, nv, a);
        if (want && (!c->arr_valid[a] || c->arr_src[a] != vol_dev || c->opt_volatile)) {
            s = ensure_layers(c, vol_dev, a, st);
            if (s != FP_OK) return s;
        }
    }

    s = upload_geometry(c, n_proj, geom, nu, nv, use_perm, st);
    if (s != FP_OK) return s;
    s = ensure_ids(c, n_proj);
    if (s != FP_OK) return s;
    if (!ids_al.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev, ids_al.data(), sizeof(int) * ids_al.size(), cudaMemcpyHostToDevice, st));
    if (!ids_di.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev + c->ids_cap, ids_di.data(), sizeof(int) * ids_di.size(),
                                   cudaMemcpyHostToDevice, st));
    if (!ids_tm.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev + 2 * c->ids_cap, ids_tm.data(), sizeof(int) * ids_tm.size(),
                                   cudaMemcpyHostToDevice, st));
    if (!ids_tn.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev + 4 * c->ids_cap, ids_tn.data(), sizeof(int) * ids_tn.size(), cudaMemcpyHostToDevice, st));
    if (!ids_tx.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev + 3 * c->ids_cap, ids_tx.data(), sizeof(int) * ids_tx.size(),
                                   cudaMemcpyHostToDevice, st));

    // the sample count restarts with every call; the error flag stays up until it is read (fp_check)
    if (!c->keep_count) FP_CUDA(c, cudaMemsetAsync(c->count_dev, 0, sizeof(unsigned long long), st));
    c->counted = c->opt_count != 0;

    if (!ids_tx.empty()) {
        TexParams X;
        X.G = c->G;
        const int filt = c->opt_kernel == FP_KERNEL_HWLIN ? 1 : 0;
        for (int a = 0; a < 3; ++a) X.tex[a] = (unsigned long long)c->atex[a][filt];
        X.proj = c->proj_dev;
        X.ids = c->ids_dev + 3 * c->ids_cap;
        X.out = out_dev;
        X.sample_count = c->opt_count ? c->count_dev : nullptr;
        X.nu = nu;
        X.nv = nv;
        X.n_sel = (int)ids_tx.size();
        s = launch_tex(c, X, filt != 0, st);
        if (s != FP_OK) return s;
        c->last_launches += 1;
    }
    for (int narrow = 0; narrow < 2; ++narrow) {
        const std::vector<int> &ids = narrow ? ids_tn : ids_tm;
        if (ids.empty()) continue;
        const int block_rows = narrow ? kTmRowsNarrow : kTmRows;
        s = build_tensor_maps(c, vol_dev);
        if (s != FP_OK) return s;
        TmaParams T;
        memcpy(T.map, c->tmap, sizeof T.map);
        T.G = c->G;
        T.proj = c->proj_dev;
        T.ids = c->ids_dev + (narrow ? 4 : 2) * c->ids_cap;
        T.out = out_dev;
        T.sample_count = c->opt_count ? c->count_dev : nullptr;
        T.err_flag = reinterpret_cast<unsigned int *>(c->count_dev + 1);
        T.nu = nu;
        T.nv = nv;
        T.n_sel = (int)ids.size();
        T.fov = c->opt_fov;
        T.out_vec = ((uintptr_t)out_dev & 15) == 0 && (nu & 3) == 0;
        // groups of neighbouring poses share their volume rows through L2 (fp_tma.cuh)
        T.group = std::max(1, std::min(c->opt_group, (int)ids.size()));
        dim3 grid((unsigned)((nu + kTmTU - 1) / kTmTU * T.group), (unsigned)((nv + block_rows - 1) / block_rows),
                  (unsigned)((ids.size() + T.group - 1) / T.group));
        if (narrow)
            s = c->opt_interp == FP_INTERP_SPLINE ? launch_tma<1, kTmRowsNarrow>(c, T, grid, st) : launch_tma<0, kTmRowsNarrow>(c, T, grid, st);
        else
            s = c->opt_interp == FP_INTERP_SPLINE ? launch_tma<1, kTmRows>(c, T, grid, st) : launch_tma<0, kTmRows>(c, T, grid, st);
        if (s != FP_OK) return s;
        c->last_launches += 1;
    }
    if (!ids_al.empty()) {
        AlignedParams A;
        A.G = c->G;
        A.vol = vol_dev;
        A.proj = c->proj_dev;
        A.ids = c->ids_dev;
        A.out = out_dev;
        A.sample_count = c->opt_count ? c->count_dev : nullptr;
        A.err_flag = reinterpret_cast<unsigned int *>(c->count_dev + 1);
        A.nu = nu;
        A.nv = nv;
        A.n_sel = (int)ids_al.size();
        A.fov = c->opt_fov;
        A.out_vec = ((uintptr_t)out_dev & 15) == 0 && (nu & 3) == 0;
        A.group = std::max(1, std::min(c->opt_group, (int)ids_al.size()));
        dim3 grid((unsigned)((nu + kAlTU - 1) / kAlTU * A.group), (unsigned)((nv + kAlTV - 1) / kAlTV),
                  (unsigned)((ids_al.size() + A.group - 1) / A.group));
        s = c->opt_interp == FP_INTERP_SPLINE ? launch_aligned<1>(c, A, w_al, grid, st)
                                              : launch_aligned<0>(c, A, w_al, grid, st);
        if (s != FP_OK) return s;
        c->last_launches += 1;
    }

    // general poses: the TMA-staged tile kernel when the volume can be addressed by tensor maps (16-byte aligned
    // base, row lengths that are multiples of 4 voxels), else -- or with FP_KERNEL_DIRECT -- the direct kernel
    const bool tile_ok = c->opt_kernel != FP_KERNEL_DIRECT && ((uintptr_t)vol_dev & 15) == 0 && (c->G.n[2] & 3) == 0 &&
                         (!use_perm || (c->G.n[1] & 3) == 0);
    if (!ids_di.empty() && tile_ok) {
        s = build_tile_maps(c, vol_dev, use_perm ? c->vol_perm : nullptr);
        if (s != FP_OK) return s;
        TileParams T;
        memcpy(T.map, c->tlmap, sizeof T.map);
        T.G = c->G;
        fill_layouts(c, vol_dev, use_perm, T.lay);
        T.proj = c->proj_dev;
        T.ids = c->ids_dev + c->ids_cap;
        T.out = out_dev;
        T.sample_count = c->opt_count ? c->count_dev : nullptr;
        T.nu = nu;
        T.nv = nv;
        T.n_sel = (int)ids_di.size();
        T.z_staged = use_perm ? 1 : 0;
        dim3 grid((unsigned)((nu + kTlU - 1) / kTlU), (unsigned)((nv + kTlV - 1) / kTlV), (unsigned)ids_di.size());
        const size_t smem = tile_smem_bytes();
        if (c->opt_interp == FP_INTERP_SPLINE) {
            FP_CUDA(c, cudaFuncSetAttribute(fp_tile_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            fp_tile_kernel<1><<<grid, kTlThreads, smem, st>>>(T);
        } else {
            FP_CUDA(c, cudaFuncSetAttribute(fp_tile_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            fp_tile_kernel<0><<<grid, kTlThreads, smem, st>>>(T);
        }
        FP_CUDA(c, cudaGetLastError());
        c->last_launches += 1;
    } else if (!ids_di.empty()) {
        ProjectParams P;
        P.G = c->G;
        fill_layouts(c, vol_dev, use_perm, P.lay);
        P.proj = c->proj_dev;
        P.ids = c->ids_dev + c->ids_cap;
        P.out = out_dev;
        P.sample_count = c->opt_count ? c->count_dev : nullptr;
        P.nu = nu;
        P.nv = nv;
        P.n_proj = (int)ids_di.size();
        P.interp = c->opt_interp;
        const unsigned gl = (unsigned)((std::max(nu, nv) + kTileLane - 1) / kTileLane);
        const unsigned gr = (unsigned)((std::max(nu, nv) + kTileRow - 1) / kTileRow);
        dim3 grid(gl, gr, (unsigned)ids_di.size());
        if (c->opt_interp == FP_INTERP_SPLINE)
            fp_direct_kernel<1><<<grid, kDirectThreads, 0, st>>>(P);
        else
            fp_direct_kernel<0><<<grid, kDirectThreads, 0, st>>>(P);
        FP_CUDA(c, cudaGetLastError());
        c->last_launches += 1;
    }
    return leave_stream(c, st);
}

extern "C" fp_status fp_backproject(fp_ctx *c, const float *proj_dev, int n_proj, const double *geom, int nu, int nv,
                                    float *vol_out_dev, fp_stream stream)
{
    fp_status s = check_project_args(c, proj_dev, n_proj, geom, nu, nv, vol_out_dev);
    if (s != FP_OK) return s;
    if (!vol_out_dev) return fail(c, FP_ERR_INVALID_ARG, "null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    c->last_launches = 0;
    c->counted = false;
    s = enter_stream(c, st);
    if (s != FP_OK) return s;
    FP_CUDA(c, cudaMemsetAsync(vol_out_dev, 0, n_voxels(c) * sizeof(float), st));
    if (n_proj == 0) return leave_stream(c, st);
    s = upload_geometry(c, n_proj, geom, nu, nv, false, st);
    if (s != FP_OK) return s;
    // plan: poses of the aligned class (fp_tma.cuh) take the transpose of the TMA-fed kernel, everything else --
    // and everything with FP_KERNEL_DIRECT -- the ray-driven scatter.  The aligned kernel addresses the volume
    // with 32-bit element indices.
    std::vector<int> ids_al, ids_di;
    const bool small = n_voxels(c) < 0xFFFFFFF0ull;
    for (int p = 0; p < n_proj; ++p) {
        const bool al = small && c->opt_kernel != FP_KERNEL_DIRECT && c->opt_kernel != FP_KERNEL_TEX &&
                        c->opt_kernel != FP_KERNEL_HWLIN && plan_aligned(c, nullptr, geom + 12 * (size_t)p, nu, nv) > 0;
        (al ? ids_al : ids_di).push_back(p);
    }
    s = ensure_ids(c, n_proj);
    if (s != FP_OK) return s;
    if (!ids_al.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev, ids_al.data(), sizeof(int) * ids_al.size(), cudaMemcpyHostToDevice, st));
    if (!ids_di.empty())
        FP_CUDA(c, cudaMemcpyAsync(c->ids_dev + c->ids_cap, ids_di.data(), sizeof(int) * ids_di.size(), cudaMemcpyHostToDevice, st));
    if (!ids_al.empty()) {
        BpParams B;
        memset(&B, 0, sizeof B);
        B.T.G = c->G;
        B.T.proj = c->proj_dev;
        B.T.ids = c->ids_dev;
        B.T.err_flag = reinterpret_cast<unsigned int *>(c->count_dev + 1);
        B.T.nu = nu;
        B.T.nv = nv;
        B.T.n_sel = (int)ids_al.size();
        B.T.group = std::max(1, std::min(c->opt_group, (int)ids_al.size()));
        B.in = proj_dev;
        B.vol = vol_out_dev;
        dim3 grid((unsigned)((nu + kTmTU - 1) / kTmTU * B.T.group), (unsigned)((nv + kBpRows - 1) / kBpRows),
                  (unsigned)((ids_al.size() + B.T.group - 1) / B.T.group));
        if (c->opt_interp == FP_INTERP_SPLINE)
            fp_bp_aligned_kernel<1><<<grid, kBpThreads, 0, st>>>(B);
        else
            fp_bp_aligned_kernel<0><<<grid, kBpThreads, 0, st>>>(B);
        FP_CUDA(c, cudaGetLastError());
        c->last_launches += 1;
    }
    if (!ids_di.empty()) {
        BackprojectParams B;
        B.G = c->G;
        fill_layouts(c, vol_out_dev, false, B.lay);
        B.proj = c->proj_dev;
        B.ids = c->ids_dev + c->ids_cap;
        B.in = proj_dev;
        B.nu = nu;
        B.nv = nv;
        B.n_proj = (int)ids_di.size();
        const unsigned gl = (unsigned)((std::max(nu, nv) + kTileLane - 1) / kTileLane);
        const unsigned gr = (unsigned)((std::max(nu, nv) + kTileRow - 1) / kTileRow);
        dim3 grid(gl, gr, (unsigned)ids_di.size());
        if (c->opt_interp == FP_INTERP_SPLINE)
            fp_backproject_kernel<1><<<grid, kDirectThreads, 0, st>>>(B);
        else
            fp_backproject_kernel<0><<<grid, kDirectThreads, 0, st>>>(B);
        FP_CUDA(c, cudaGetLastError());
        c->last_launches += 1;
    }
    return leave_stream(c, st);
}

extern "C" fp_status fp_ray_ranges(fp_ctx *c, int n_proj, const double *geom, int nu, int nv, int32_t *mfl_dev,
                                   fp_stream stream)
{
    fp_status s = check_project_args(c, mfl_dev, n_proj, geom, nu, nv, mfl_dev);
    if (s != FP_OK) return s;
    if (n_proj == 0) return FP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    s = enter_stream(c, st);
    if (s != FP_OK) return s;
    s = upload_geometry(c, n_proj, geom, nu, nv, false, st);
    if (s != FP_OK) return s;
    dim3 grid((unsigned)((nu + 31) / 32), (unsigned)((nv + 7) / 8), (unsigned)n_proj);
    fp_ranges_kernel<<<grid, 256, 0, st>>>(c->G, c->proj_dev, nu, nv, mfl_dev);
    FP_CUDA(c, cudaGetLastError());
    return leave_stream(c, st);
}

extern "C" fp_status fp_last_sample_count(fp_ctx *c, unsigned long long *n)
{
    if (!c || !n) return FP_ERR_INVALID_ARG;
    *n = 0;
    unsigned long long h[2];
    fp_status s = read_counters(c, h);
    if (s != FP_OK) return s;
    if (h[1] != 0) return fail(c, FP_ERR_UNSUPPORTED, kPlanError);
    if (!c->counted || !c->count_dev) return fail(c, FP_ERR_INVALID_ARG, "no counted fp_project call to report");
    *n = h[0];
    return FP_OK;
}

extern "C" fp_status fp_check(fp_ctx *c)
{
    if (!c) return FP_ERR_INVALID_ARG;
    unsigned long long h[2];
    fp_status s = read_counters(c, h);
    if (s != FP_OK) return s;
    if (h[1] != 0) return fail(c, FP_ERR_UNSUPPORTED, kPlanError);
    return FP_OK;
}

extern "C" fp_status fp_plan(fp_ctx *c, const double *geom, int nu, int nv, int *kernel, int *window, int *z_driven)
{
    if (!c || !geom || !kernel || !window || !z_driven) return fail(c, FP_ERR_INVALID_ARG, "fp_plan: null argument");
    if (nu < 1 || nv < 1) return fail(c, FP_ERR_INVALID_ARG, "nu, nv must be >= 1");
    int rows = 0;
    const int w = c->opt_kernel == FP_KERNEL_DIRECT ? 0 : plan_aligned(c, nullptr, geom, nu, nv, &rows);
    const bool al = w > 0 && w <= kAlignedMaxW;
    *kernel = al ? FP_KERNEL_ALIGNED : ((c->opt_kernel != FP_KERNEL_DIRECT && (c->G.n[2] & 3) == 0) ? FP_KERNEL_TILE : FP_KERNEL_DIRECT);
    *window = al ? w : 0;
    // the TMA-fed kernel reports the window of its own blocks (256 or 192 detector rows)
    if (al && c->opt_kernel != FP_KERNEL_ALIGNED && tma_block_rows(c, nullptr, geom, nu, nv, w, rows, window) != 0) *kernel = FP_KERNEL_TMA;
    if (c->opt_kernel == FP_KERNEL_TEX || c->opt_kernel == FP_KERNEL_HWLIN) {
        *kernel = c->opt_kernel;                           // every pose goes through the texture pipe
        *window = 0;
    }
    *z_driven = has_z_driven(geom, nu, nv) ? 1 : 0;
    return FP_OK;
}

extern "C" fp_status fp_last_launch_count(fp_ctx *c, int *n)
{
    if (!c || !n) return FP_ERR_INVALID_ARG;
    *n = c->last_launches;
    return FP_OK;
}

// End-to-end entry point: host volume in, host projections out.  The volume goes up once; the
// projections are computed in batches on two streams so that the device-to-host copy of one
// batch overlaps the kernels of the next.
extern "C" fp_status fp_project_host(fp_ctx *c, const float *vol_host, int n_proj, const double *geom, int nu,
                                     int nv, float *out_host)
{
    fp_status s = check_project_args(c, vol_host, n_proj, geom, nu, nv, out_host);
    if (s != FP_OK) return s;
    if (n_proj == 0) return FP_OK;
    const size_t nvox = n_voxels(c);
    const size_t per_proj = (size_t)nu * nv;
    int batch = (int)std::max<size_t>(1, std::min<size_t>((size_t)n_proj, ((size_t)256 << 20) / (per_proj * sizeof(float))));
    for (int k = 0; k < 2; ++k) {
        if (!c->hstream[k]) FP_CUDA(c, cudaStreamCreateWithFlags(&c->hstream[k], cudaStreamNonBlocking));
        if (!c->hevent[k]) FP_CUDA(c, cudaEventCreateWithFlags(&c->hevent[k], cudaEventDisableTiming));
    }
    if (!c->hvol_dev) FP_CUDA(c, cudaMalloc(&c->hvol_dev, nvox * sizeof(float)));
    if (c->hout_cap < (size_t)batch * per_proj) {
        for (int k = 0; k < 2; ++k) {
            cudaFree(c->hout_dev[k]);
            c->hout_dev[k] = nullptr;
            FP_CUDA(c, cudaMalloc(&c->hout_dev[k], (size_t)batch * per_proj * sizeof(float)));
        }
        c->hout_cap = (size_t)batch * per_proj;
    }
    for (int k = 0; k < 2; ++k)
        if (!c->hcopied[k]) FP_CUDA(c, cudaEventCreateWithFlags(&c->hcopied[k], cudaEventDisableTiming));
    // stream 0 carries the volume upload and every kernel, stream 1 the device-to-host copies: the copy of
    // batch k overlaps the kernels of batch k+1, and the host plans batch k+1 while batch k runs (no host
    // synchronisation inside the loop; the shared geometry buffer is safe because all kernels are in one stream)
    cudaStream_t compute = c->hstream[0], copy = c->hstream[1];
    FP_CUDA(c, cudaMemcpyAsync(c->hvol_dev, vol_host, nvox * sizeof(float), cudaMemcpyHostToDevice, compute));
    s = enter_stream(c, compute);
    if (s != FP_OK) return s;
    FP_CUDA(c, cudaMemsetAsync(c->count_dev, 0, sizeof(unsigned long long), compute));
    // the layout copy (if any) is made once, then kept for all batches
    const int was_volatile = c->opt_volatile;
    int launches = 0;
    c->keep_count = true;
    for (int p0 = 0, b = 0; p0 < n_proj; p0 += batch, ++b) {
        const int k = b & 1;
        const int np = std::min(batch, n_proj - p0);
        if (b > 0) c->opt_volatile = 0;
        cudaError_t e = b >= 2 ? cudaStreamWaitEvent(compute, c->hcopied[k], 0) : cudaSuccess;   // output buffer k is free
        s = e == cudaSuccess ? fp_project(c, c->hvol_dev, np, geom + 12 * (size_t)p0, nu, nv, c->hout_dev[k], compute)
                             : cuda_fail(c, e, "cudaStreamWaitEvent");
        c->opt_volatile = was_volatile;
        if (s == FP_OK) {
            launches += c->last_launches;
            e = cudaEventRecord(c->hevent[k], compute);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(copy, c->hevent[k], 0);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(out_host + (size_t)p0 * per_proj, c->hout_dev[k], (size_t)np * per_proj * sizeof(float),
                                    cudaMemcpyDeviceToHost, copy);
            if (e == cudaSuccess) e = cudaEventRecord(c->hcopied[k], copy);
            if (e != cudaSuccess) s = cuda_fail(c, e, "fp_project_host: copy pipeline");
        }
        if (s != FP_OK) {
            c->keep_count = false;
            cudaStreamSynchronize(compute);
            cudaStreamSynchronize(copy);
            return s;
        }
    }
    c->keep_count = false;
    FP_CUDA(c, cudaStreamSynchronize(compute));
    FP_CUDA(c, cudaStreamSynchronize(copy));
    c->last_launches = launches;
    c->last_stream = compute;
    c->counted = c->opt_count != 0;
    // a window or row tile that did not fit (the host plan was too small): the call is repeated with the
    // general-pose kernel, which has no such limit, instead of returning wrong numbers
    unsigned long long h[2];
    s = read_counters(c, h);
    if (s != FP_OK) return s;
    if (h[1] != 0 && c->opt_kernel != FP_KERNEL_DIRECT) {
        const int was_kernel = c->opt_kernel;
        c->opt_kernel = FP_KERNEL_DIRECT;
        s = fp_project_host(c, vol_host, n_proj, geom, nu, nv, out_host);
        c->opt_kernel = was_kernel;
        return s;
    }
    if (h[1] != 0) return fail(c, FP_ERR_UNSUPPORTED, kPlanError);
    return FP_OK;
}

// Read-bandwidth probes of the measurement harness (fp_probe.cuh): best of five timed runs, CUDA events.
extern "C" fp_status fp_probe_bandwidth(int what, double *gbs)
{
    if (!gbs) return FP_ERR_INVALID_ARG;
    *gbs = 0.0;
    if (what != FP_PROBE_HBM_READ && what != FP_PROBE_L2_READ && what != FP_PROBE_SHARED_READ) return FP_ERR_INVALID_ARG;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return FP_ERR_CUDA;
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float *buf = nullptr, *sink = nullptr;
    fp_status st = FP_OK;
    double best = 0.0;
    // HBM: 2 GiB streamed once per run; L2: 48 MiB (well inside the 126 MB L2) streamed 64 times per run
    const size_t bytes = what == FP_PROBE_HBM_READ ? ((size_t)2 << 30) : ((size_t)48 << 20);
    const int reps = what == FP_PROBE_HBM_READ ? 1 : 64, iters = 4096;
    do {
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess ||
            cudaMalloc(&sink, sizeof(float)) != cudaSuccess) { st = FP_ERR_CUDA; break; }
        if (what != FP_PROBE_SHARED_READ) {
            if (cudaMalloc(&buf, bytes) != cudaSuccess) { st = FP_ERR_OOM; break; }
            if (cudaMemset(buf, 0, bytes) != cudaSuccess) { st = FP_ERR_CUDA; break; }
        }
        for (int run = 0; run < 6 && st == FP_OK; ++run) {          // run 0 warms up
            cudaEventRecord(e0, 0);
            double moved = 0.0;
            if (what == FP_PROBE_SHARED_READ) {
                fp_probe_shared_kernel<<<n_sm * 2, 1024>>>(iters, sink);
                moved = (double)n_sm * 2 * 1024 * (double)iters * 16 * 4;
            } else {
                fp_probe_read_kernel<<<n_sm * 4, 512>>>(reinterpret_cast<const float4 *>(buf), bytes / 16, reps, sink);
                moved = (double)bytes * reps;
            }
            cudaEventRecord(e1, 0);
            if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { st = FP_ERR_CUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (run > 0 && ms > 0.f) best = std::max(best, moved / (ms * 1e-3) / 1e9);
        }
    } while (false);
    cudaFree(buf);
    cudaFree(sink);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaGetLastError();
    *gbs = best;
    return st;
}

// ------------------------------------------------------------------------------------------
// fp_project_static (include/fp.h): the forward projector for callers that may not allocate.
// fp_direct_kernel with its scratch -- the per-projection descriptor table the kernel reads and the
// sample counter it adds to -- in a file-scope device array instead of the context's cudaMalloc'ed
// workspaces.  No context, no cudaMalloc / cudaFree, no host heap.
// ------------------------------------------------------------------------------------------
namespace {

constexpr size_t kStaticCounterBytes = 256;      // [0, 8): the sample counter; the rest keeps the table 256-byte aligned
constexpr size_t kStaticBytes = kStaticCounterBytes + sizeof(ProjDesc) * (size_t)FP_STATIC_MAX_PROJ;

// Every device that loads the library holds these kStaticBytes (about 52 KB) until exit.  In host code this name is a
// host-side stand-in, not a device address: the address a kernel may use comes from cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

constexpr int kStaticMaxDevices = 64;
unsigned char *g_static_ptr[kStaticMaxDevices];  // per device: device address of g_static_scratch, null = not asked yet
std::mutex g_static_mu;

fp_status static_fail(fp_status s, char *err, size_t err_len, const char *msg)
{
    if (err && err_len) snprintf(err, err_len, "%s", msg);
    return s;
}

// Once per device, with that device current: the device address of the scratch array.
fp_status static_scratch(unsigned char **ptr, char *err, size_t err_len)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(FP_ERR_CUDA, err, err_len, cudaGetErrorString(e));
    if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(FP_ERR_UNSUPPORTED, err, err_len, "fp_project_static: device ordinal >= 64");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            char buf[192];
            snprintf(buf, sizeof buf, "fp_project_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return static_fail(FP_ERR_CUDA, err, err_len, buf);
        }
        g_static_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *ptr = g_static_ptr[dev];
    return FP_OK;
}

}  // namespace

extern "C" fp_status fp_project_static(int nx, int ny, int nz, double voxel_size, const double origin[3],
                                       const float *vol_dev, int n_proj, const double *geom, int nu, int nv, int interp,
                                       float *out_dev, unsigned long long *n_samples_dev, fp_stream stream, char *err,
                                       size_t err_len)
{
    if (err && err_len) err[0] = '\0';
    if (nx < 1 || ny < 1 || nz < 1 || !origin || !(voxel_size > 0.0) || !std::isfinite(voxel_size))
        return static_fail(FP_ERR_INVALID_ARG, err, err_len, "fp_project_static: bad grid");
    for (int a = 0; a < 3; ++a)
        if (!std::isfinite(origin[a])) return static_fail(FP_ERR_INVALID_ARG, err, err_len, "fp_project_static: bad origin");
    if ((double)nx * ny * nz >= 1099511627776.0) return static_fail(FP_ERR_INVALID_ARG, err, err_len, "fp_project_static: grid too large");
    if (n_proj < 0 || nu < 1 || nv < 1) return static_fail(FP_ERR_INVALID_ARG, err, err_len, "fp_project_static: n_proj < 0 or nu, nv < 1");
    if (interp != FP_INTERP_LINEAR && interp != FP_INTERP_SPLINE)
        return static_fail(FP_ERR_INVALID_ARG, err, err_len, "fp_project_static: interp must be FP_INTERP_LINEAR or FP_INTERP_SPLINE");
    if (n_proj > FP_STATIC_MAX_PROJ) {
        char buf[192];
        snprintf(buf, sizeof buf, "fp_project_static: n_proj = %d exceeds FP_STATIC_MAX_PROJ = %d (the static scratch holds that many "
                 "projection descriptors): split the call", n_proj, FP_STATIC_MAX_PROJ);
        return static_fail(FP_ERR_UNSUPPORTED, err, err_len, buf);
    }
    if (n_proj > 0 && (!vol_dev || !geom || !out_dev)) return static_fail(FP_ERR_INVALID_ARG, err, err_len, "fp_project_static: null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *scratch = nullptr;
    fp_status s = static_scratch(&scratch, err, err_len);
    if (s != FP_OK) return s;
    unsigned long long *count = reinterpret_cast<unsigned long long *>(scratch);
    ProjDesc *table = reinterpret_cast<ProjDesc *>(scratch + kStaticCounterBytes);
    cudaError_t e;
#define FP_STATIC_CUDA(call)                                                                         \
    do {                                                                                             \
        e = (call);                                                                                  \
        if (e != cudaSuccess) {                                                                      \
            char buf_[192];                                                                          \
            snprintf(buf_, sizeof buf_, "fp_project_static: %s: %s", #call, cudaGetErrorString(e)); \
            cudaGetLastError();                                                                      \
            return static_fail(FP_ERR_CUDA, err, err_len, buf_);                                     \
        }                                                                                            \
    } while (0)
    // the array keeps the last call's contents: the counter must start at zero, the table is overwritten
    FP_STATIC_CUDA(cudaMemsetAsync(count, 0, sizeof(unsigned long long), st));
    if (n_proj > 0) {
        ProjDesc h[FP_STATIC_MAX_PROJ];                 // on the stack: no host heap either
        for (int p = 0; p < n_proj; ++p) {
            memcpy(h[p].g, geom + 12 * (size_t)p, sizeof(double) * 12);
            h[p].lane_v = plan_lane_v(h[p].g, nu, nv, false);
            h[p].pad_ = 0;
        }
        // pageable source: the runtime stages the bytes before returning, so `h` may die here
        FP_STATIC_CUDA(cudaMemcpyAsync(table, h, sizeof(ProjDesc) * (size_t)n_proj, cudaMemcpyHostToDevice, st));
        ProjectParams P;
        P.G.n[0] = nx;
        P.G.n[1] = ny;
        P.G.n[2] = nz;
        P.G.pad_ = 0;
        P.G.delta = voxel_size;
        for (int a = 0; a < 3; ++a) P.G.origin[a] = origin[a];
        const long long lx = nx, ly = ny, lz = nz;
        P.lay[0] = AxisLayout{vol_dev, ly * lz, lz, 1, (int)lx, (int)ly, (int)lz, 0};       // m = x: slow y, fast z
        P.lay[1] = AxisLayout{vol_dev, lz, ly * lz, 1, (int)ly, (int)lx, (int)lz, 0};       // m = y: slow x, fast z
        P.lay[2] = AxisLayout{vol_dev, 1, ly * lz, lz, (int)lz, (int)lx, (int)ly, 0};       // m = z: slow x, fast y (strided)
        P.proj = table;
        P.ids = nullptr;
        P.out = out_dev;
        P.sample_count = count;
        P.nu = nu;
        P.nv = nv;
        P.n_proj = n_proj;
        P.interp = interp;
        const unsigned gl = (unsigned)((std::max(nu, nv) + kTileLane - 1) / kTileLane);
        const unsigned gr = (unsigned)((std::max(nu, nv) + kTileRow - 1) / kTileRow);
        dim3 grid(gl, gr, (unsigned)n_proj);
        if (interp == FP_INTERP_SPLINE)
            fp_direct_kernel<1><<<grid, kDirectThreads, 0, st>>>(P);
        else
            fp_direct_kernel<0><<<grid, kDirectThreads, 0, st>>>(P);
        FP_STATIC_CUDA(cudaGetLastError());
    }
    if (n_samples_dev)
        FP_STATIC_CUDA(cudaMemcpyAsync(n_samples_dev, count, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, st));
#undef FP_STATIC_CUDA
    return FP_OK;
}
