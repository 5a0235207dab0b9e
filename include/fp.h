/*
 * fp.h -- C ABI of libfp.so: the B200 (sm_100a) Generalized Joseph forward projector.
 *
 * The operation is the linear-kernel "Generalized Joseph Projector" (GJP_lin) of
 * arXiv 1609.00958 (J. Dittmann).  Citations are /root/reference/PAPER.md line numbers with
 * the section / equation / algorithm they fall in; "reading #k" refers to the table
 * "Readings of the paper" in DESIGN.md.
 *
 * For every detector pixel the library forms the ray r = d - s from the source s to the
 * pixel centre d (sec. 2.1 Eq. 1), picks the driving axis m = argmax_a |r_a|
 * (:81 Eq. 2), steps once per voxel slice along m with the increment r~ = r / r_m (:92 Eq. 4,
 * :104 Eq. 6), interpolates the volume bilinearly in the two transverse axes at the ray's
 * intersection with each slice plane (:165 Eq. 15, :150 Eq. 13, :142 Eq. 11) and returns
 *
 *     out(ray) = voxel_size * ||r~||_2 * sum_{i = i_first}^{i_last} sample(i)      (:211, Alg. 1 :217-269)
 *
 * where [i_first, i_last] is the exact set of slices whose intersection point lies in the
 * zero-padded transverse extent -1 < p_t < N_t (:213 sec. 2.6 "entry and exit points are
 * calculated exactly"; reading #2).
 *
 * Conventions (all entry points):
 *   - Coordinates: world units.  Voxel (ix, iy, iz) has its CENTRE at
 *     origin + voxel_size * (ix, iy, iz).  Grid coordinate g = (world - origin) / voxel_size
 *     (PAPER.md:57 Fig. 1, :63: units normalised to the grid spacing; reading #1).
 *   - Volume: fp32, C order [nx][ny][nz], z FASTEST (PAPER.md:294 sec. 2.8, :312: the rotation
 *     axis is parallel to the fastest index).  DEVICE pointer unless the name says _host.
 *   - Geometry: HOST pointer to n_proj rows of 12 doubles
 *         { source xyz, det_origin xyz, u-pitch vector xyz, v-pitch vector xyz },
 *     the centre of pixel (iu, iv) is det_origin + iu * u + iv * v.  The rows are read during
 *     the call; the caller may reuse the buffer as soon as the call returns.
 *   - Output: fp32, [n_proj][nv][nu], u fastest (reading #14).  Rays that miss the volume
 *     (and the degenerate ray r = 0) write +0.0f.
 *   - Streams: every kernel and copy is enqueued on the given stream; fp_project does not
 *     synchronise the host with the device.  Outputs are valid once the stream reaches that point.
 *     A context owns one set of workspaces: a call on another stream than the context's previous call
 *     first waits (on the device) for that call to end, so calls on one context never overlap.  Use one
 *     context per stream for concurrent projections.
 *   - Ownership: the caller owns the volume, the geometry and the outputs.  The library owns
 *     the context, its internal volume copies and workspaces (freed by fp_destroy).
 *   - Errors: status codes only, nothing is thrown.  fp_last_error(ctx) holds the text of the
 *     most recent failure on that context.  A context is not thread-safe; different contexts
 *     are independent.  Non-finite geometry gives unspecified output values but never a fault.
 *   - There is NO CPU fallback: without a CUDA device every compute entry point returns
 *     FP_ERR_CUDA.
 */
#ifndef FP_H_
#define FP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fp_ctx fp_ctx;                 /* opaque, library-owned */
typedef struct CUstream_st *fp_stream;        /* a cudaStream_t (0 = the legacy default stream) */

typedef enum {
    FP_OK = 0,
    FP_ERR_INVALID_ARG = 1,
    FP_ERR_CUDA = 2,
    FP_ERR_OOM = 3,
    FP_ERR_UNSUPPORTED = 4
} fp_status;

/* fp_set_option keys.  Options are explicit; no environment variable changes behaviour. */
enum {
    /* Sampling-kernel variant.  Poses whose v vector is parallel to the volume's z axis, whose u vector is
     * perpendicular to it and that have no z-driven ray (every circular orbit about z)
     * are "aligned"; all other poses use FP_KERNEL_TILE (32 x 16 pixel tiles whose slice footprints the TMA engine
     * copies to shared memory; needs nz % 4 == 0 and a 16-byte aligned volume) or, failing that or when forced,
     * FP_KERNEL_DIRECT (one thread per ray, four global taps per sample).  For each aligned pose (one launch per
     * kernel and call):
     *   FP_KERNEL_AUTO     FP_KERNEL_TMA if the pose fits a 256-voxel z window and 12 volume rows per block
     *                      and slice, else FP_KERNEL_ALIGNED;
     *   FP_KERNEL_TMA      the same as AUTO (tiles of the caller's volume copied to shared memory by
     *                      cp.async.bulk.tensor, four taps per sample read from the tile);
     *   FP_KERNEL_ALIGNED  always the line-staging kernel (two volume rows blended into shared memory per
     *                      column and slice, two taps per sample);
     *   FP_KERNEL_DIRECT   the direct kernel for every pose;
     *   FP_KERNEL_TILE     the same as AUTO;
     *   FP_KERNEL_TEX      every pose (aligned or not) through the texture pipe: the layout stage copies the
     *                      volume into one layered 2-D array per driving axis in use (brick-tiled texel order,
     *                      PAPER.md:290-294), one tld4 per sample returns the four taps, explicit fp32 weights;
     *   FP_KERNEL_HWLIN    the paper's GJP_hwlin (Table 1): one hardware-filtered bilinear
     *                      fetch per sample from the same arrays.  The hardware quantises the interpolation
     *                      weights to 8 fractional bits: the result is OUTSIDE the library's tolerance
     *                      (DESIGN.md records the measured error); never chosen by FP_KERNEL_AUTO. */
    FP_OPT_KERNEL = 1,
    /* 1 (default): the volume contents may have changed since the last call, internal copies
     * are rebuilt by every fp_project that needs them.  0: internal copies made by fp_prepare
     * (or the first fp_project) stay valid until the next fp_prepare. */
    FP_OPT_VOLATILE = 2,
    /* Interpolation kernel w(d): FP_INTERP_LINEAR (Eq. 13) or
     * FP_INTERP_SPLINE (:152 Eq. 14). */
    FP_OPT_INTERP = 3,
    /* 1 (default): a y-fastest permuted copy of the volume is built when a projection has
     * z-driven rays, so that their in-plane taps are contiguous (sec. 2.8).
     * 0: z-driven rays read the caller's layout with strided taps. */
    FP_OPT_PERMUTED_COPY = 4,
    /* 1: fp_project accumulates the number of samples sum(i_last - i_first + 1) for
     * fp_last_sample_count (default 0: the count costs one exact fp64 ray set-up per ray that the
     * aligned / TMA sampling kernels do not otherwise need). */
    FP_OPT_COUNT_SAMPLES = 5,
    /* 1: the caller promises that the volume is ZERO outside the cylinder about the z axis through the grid
     * centre ((nx-1)/2, (ny-1)/2) with diameter min(nx, ny) voxels (the paper's benchmark object: "a cylindric
     * volume within a cubic bounding box", Fig. 9).  The aligned / TMA kernels then skip
     * the slices of a ray on which every tap lies outside that cylinder; for such a volume the result is the
     * same sum.  The direct kernel ignores the option; fp_last_sample_count keeps counting the box samples.
     * Default 0. */
    FP_OPT_FOV_CYLINDER = 6,
    /* Projections per launch-order group of the aligned / TMA kernels (1 .. 64, default 8): the thread blocks of
     * the same detector tile of `group` consecutive poses of a call start together and sweep the volume in step,
     * so that neighbouring poses of an orbit read the volume rows they share from L2 instead of DRAM.  A tuning
     * knob only: results do not depend on it. */
    FP_OPT_GROUP = 7,
    /* TEST HOOK, not for production: 1 sends every aligned pose to FP_KERNEL_TMA whether the host plan says its
     * tiles fit or not, so that the kernel's own bound checks (fp_check) can be exercised. */
    FP_OPT_TEST_FORCE_TMA = 100
};

enum { FP_KERNEL_AUTO = 0, FP_KERNEL_DIRECT = 1, FP_KERNEL_ALIGNED = 2, FP_KERNEL_TMA = 3, FP_KERNEL_TEX = 4, FP_KERNEL_HWLIN = 5,
       FP_KERNEL_TILE = 6 };
enum { FP_INTERP_LINEAR = 0, FP_INTERP_SPLINE = 1 };

/*
 * fp_create: describe the voxel grid (PAPER.md:57 Fig. 1, :63 sec. 2).
 *   nx, ny, nz  >= 1, nx*ny*nz < 2^40;   voxel_size > 0 and finite;
 *   origin[3]   host pointer, world position of the centre of voxel (0,0,0), finite.
 * Allocates nothing on the device.  Returns FP_ERR_INVALID_ARG on bad arguments.
 */
fp_status fp_create(int nx, int ny, int nz, double voxel_size, const double origin[3], fp_ctx **out);

/* fp_destroy: frees the context and every device allocation it owns (synchronises the device). */
fp_status fp_destroy(fp_ctx *ctx);

fp_status fp_set_option(fp_ctx *ctx, int key, int value);
fp_status fp_get_option(fp_ctx *ctx, int key, int *value);

/*
 * fp_prepare: volume-layout stage (sec. 2.8) run now, on `stream`: builds the
 * internal copies of vol_dev that the configured kernels want.  Optional: fp_project runs
 * the stage itself when it needs a copy that is missing or (FP_OPT_VOLATILE = 1) stale.
 */
fp_status fp_prepare(fp_ctx *ctx, const float *vol_dev, fp_stream stream);

/*
 * fp_project: the forward projection (Alg. 1) of n_proj poses.
 *   vol_dev    device, fp32 [nx][ny][nz]
 *   n_proj     >= 0 (0 is a no-op)
 *   geom_host  host, double [n_proj][12]
 *   nu, nv     >= 1 detector pixels along u and v
 *   out_dev    device, fp32 [n_proj][nv][nu], fully overwritten
 * geom_host is read before the call returns (the caller may reuse the array).  The context keeps the host plan of its
 * most recent fp_project call -- which kernel takes which pose -- together with a copy of that call's geometry, and
 * reuses the plan when the next call brings bit-identical geometry, the same nu, nv, kernel option and volume
 * alignment (the calls of an iterative reconstruction); anything else re-plans.  The results do
 * not depend on whether the plan was reused.
 */
fp_status fp_project(fp_ctx *ctx, const float *vol_dev, int n_proj, const double *geom_host,
                     int nu, int nv, float *out_dev, fp_stream stream);

/*
 * fp_project_host: the same with HOST volume and HOST output; the library copies the volume to
 * the device, projects in batches and copies the result back.  Synchronises before returning.
 * This is the end-to-end entry point (bench.py "e2e").
 *   vol_host   host, fp32 [nx][ny][nz]     out_host   host, fp32 [n_proj][nv][nu]
 */
fp_status fp_project_host(fp_ctx *ctx, const float *vol_host, int n_proj, const double *geom_host,
                          int nu, int nv, float *out_host);

/*
 * fp_backproject: the exact transpose of fp_project (SURVEY.md section 8(f) #2; PAPER.md:27, :308, :367:
 * iterative reconstruction pairs the projector with its back-projection).  With A the linear map
 * volume -> projections that fp_project computes for these poses, writes vol_out = A^T proj: every tap of
 * every sample of every ray receives voxel_size * ||r~|| * w * w * proj[ray] (same set-up, slices, taps and
 * weights; FP_OPT_INTERP applies).  fp32 reductions (RED.ADD.F32.FTZ: denormal contributions are flushed to
 * zero) in arbitrary order: results are reproducible only to
 * fp32 rounding of the sum.  Poses of the aligned class (the ones fp_plan gives FP_KERNEL_TMA / FP_KERNEL_ALIGNED)
 * take fp_bp_aligned_kernel, the transpose of the TMA-fed forward kernel with the same fp32 positions and weights;
 * all others -- and every pose with FP_OPT_KERNEL = FP_KERNEL_DIRECT -- the ray-driven scatter
 * fp_backproject_kernel.  FP_OPT_FOV_CYLINDER is ignored (it would change the operator).
 *   proj_dev     device, fp32 [n_proj][nv][nu]
 *   vol_out_dev  device, fp32 [nx][ny][nz], fully overwritten (cleared first, also for n_proj = 0)
 */
fp_status fp_backproject(fp_ctx *ctx, const float *proj_dev, int n_proj, const double *geom_host,
                         int nu, int nv, float *vol_out_dev, fp_stream stream);

/*
 * fp_ray_ranges: per-ray set-up only (PAPER.md:71-106 Eqs. 1-6, Alg. 1 l.1-5, :213): writes
 * { m, i_first, i_last } per pixel; a miss is { m, 0, -1 }, the degenerate ray { 0, 0, -1 }.
 * The decisions are taken in IEEE fp64 in the operation order DESIGN.md fixes, so they are
 * bit-identical to the oracle's.
 *   mfl_dev    device, int32 [n_proj][nv][nu][3]
 */
fp_status fp_ray_ranges(fp_ctx *ctx, int n_proj, const double *geom_host, int nu, int nv,
                        int32_t *mfl_dev, fp_stream stream);

/*
 * fp_last_sample_count: number of samples (visited slices summed over rays) of the most recent
 * fp_project / fp_project_host on this context; synchronises the stream that call used.
 * This is the unit of the paper's "memory access rate" = 16 B x samples / time.
 * Returns FP_ERR_UNSUPPORTED if fp_check would (and clears that flag), FP_ERR_INVALID_ARG if the most recent
 * call did not count (FP_OPT_COUNT_SAMPLES = 0).
 */
fp_status fp_last_sample_count(fp_ctx *ctx, unsigned long long *n);

/*
 * fp_check: synchronises the stream of the most recent call on this context and reports whether any sampling
 * kernel since the last fp_check / fp_last_sample_count found that the host plan had under-sized a staging
 * window or a row tile of the aligned / TMA kernels (the plan bounds them by geometry; the kernels verify the
 * bound and raise a flag instead of reading out of bounds).  FP_OK: every projection written since the last
 * check is valid.  FP_ERR_UNSUPPORTED: some are not -- repeat those calls with FP_OPT_KERNEL = FP_KERNEL_DIRECT
 * (fp_project_host does this by itself).  The flag is cleared by the call.  fp_project cannot report this
 * itself because it never synchronises.
 */
fp_status fp_check(fp_ctx *ctx);

/*
 * fp_plan: the host-side plan fp_project makes for ONE pose (no device needed, nothing is launched):
 *   *kernel    FP_KERNEL_ALIGNED, FP_KERNEL_TMA, FP_KERNEL_TILE, FP_KERNEL_DIRECT (or FP_KERNEL_TEX / FP_KERNEL_HWLIN when one
 *              of those is forced): the sampling kernel this pose gets under the current FP_OPT_KERNEL
 *   *window    staging window of the aligned kernel in voxels along z (0 for the direct kernel)
 *   *z_driven  1 if some ray of the pose has z as its driving axis (Eq. 2), which is
 *              what makes fp_project build the permuted copy of the layout stage
 * Assumes a 16-byte aligned volume pointer.  geom_host: host, double [12].
 */
fp_status fp_plan(fp_ctx *ctx, const double *geom_host, int nu, int nv, int *kernel, int *window, int *z_driven);

/* fp_last_launch_count: how many kernels of this library the most recent fp_project enqueued. */
fp_status fp_last_launch_count(fp_ctx *ctx, int *n);

/*
 * fp_probe_bandwidth: read-bandwidth probes of the measurement harness (the L2 and
 * L1 / shared-memory peaks come from a read microbenchmark in the harness, no published figure is relied on;
 * the paper's own metric is a cache-level access rate).  Runs a small kernel on the current
 * device's default stream, synchronises, and returns the best of five runs in GB/s (1e9 bytes per second):
 *   FP_PROBE_HBM_READ     a 2 GiB buffer streamed once through L2 only (ld.global.cg)
 *   FP_PROBE_L2_READ      a 48 MiB buffer (resident in L2) streamed 64 times the same way
 *   FP_PROBE_SHARED_READ  conflict-free 32-bit shared-memory loads, the access the sampling kernels make
 * Needs no context.  FP_ERR_OOM if the buffer cannot be allocated.
 */
enum { FP_PROBE_HBM_READ = 0, FP_PROBE_L2_READ = 1, FP_PROBE_SHARED_READ = 2 };
fp_status fp_probe_bandwidth(int what, double *gbs);

/*
 * fp_project_static: fp_project for callers that may not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc).  Same operation and output as fp_project with FP_OPT_KERNEL =
 * FP_KERNEL_DIRECT (Alg. 1, any pose, no preconditions on the volume), but the kernel's scratch --
 * the per-projection descriptor table it reads and the sample counter it adds to -- lives in a file-scope
 * `static __device__` array of 256 + 104 * FP_STATIC_MAX_PROJ bytes (about 52 KB) that every GPU which loads the
 * library holds until exit.  Needs no context; calls no cudaMalloc, cudaFree or other allocating routine, on the
 * device or the host; enqueues on `stream` and returns without synchronising.
 *   nx, ny, nz, voxel_size, origin   the grid, as for fp_create
 *   vol_dev        device, fp32 [nx][ny][nz], read only
 *   n_proj         0 .. FP_STATIC_MAX_PROJ; more is rejected with FP_ERR_UNSUPPORTED (split the call)
 *   geom_host      host, double [n_proj][12], as for fp_project; may be reused when the call returns
 *   interp         FP_INTERP_LINEAR or FP_INTERP_SPLINE
 *   out_dev        device, fp32 [n_proj][nv][nu], fully overwritten
 *   n_samples_dev  device, one unsigned 64-bit word: receives the number of samples taken; may be null
 *   err, err_len   host buffer for the message of a failed call (always NUL-terminated); may be null / 0
 * Every call on a device shares the one array, which keeps the last call's contents: the call clears the counter and
 * overwrites the table itself, in stream order.  Calls that OVERLAP on the GPU (different streams without an event
 * between them, or two host threads) race on it and give undefined projections; calls on one stream are safe.
 * z-driven rays read the caller's array with a stride (no permuted copy is built): this is the slow, always
 * available path -- use fp_project where allocation is allowed.
 */
#define FP_STATIC_MAX_PROJ 512
fp_status fp_project_static(int nx, int ny, int nz, double voxel_size, const double origin[3], const float *vol_dev,
                            int n_proj, const double *geom_host, int nu, int nv, int interp, float *out_dev,
                            unsigned long long *n_samples_dev, fp_stream stream, char *err, size_t err_len);

const char *fp_status_string(fp_status s);
const char *fp_last_error(fp_ctx *ctx);
const char *fp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FP_H_ */
