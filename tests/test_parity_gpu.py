"""GPU parity: libfp.so (through the C ABI binding) against the fp64 oracle, element by element,
on the same seeded inputs.  Tolerance (BASELINE.json north_star): per ray
|gpu - oracle| <= 2e-5 |oracle| + 1e-6 * path length * max|voxel|; (m, i_first, i_last) exact."""
import math

import numpy as np
import pytest

from parity_util import assert_parity, make_recompute

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def fp():
    from paper_1609_00958_b200 import fp as m
    m.load()
    return m


@pytest.fixture(scope="module")
def synth():
    from paper_1609_00958_b200 import synth as s
    return s


def all_ids(n_proj, nv, nu, projs=None):
    projs = range(n_proj) if projs is None else projs
    p, v, u = np.meshgrid(np.array(list(projs)), np.arange(nv), np.arange(nu), indexing="ij")
    return np.stack([p.ravel(), v.ravel(), u.ravel()], axis=1).astype(np.int32)


def run_gpu(torch, fp, vol_np, delta, origin, geom, nu, nv, options=()):
    vol = torch.from_numpy(np.ascontiguousarray(vol_np, dtype=np.float32)).cuda()
    with fp.Projector(*vol_np.shape, delta, origin) as P:
        P.set_option(fp.OPT_COUNT_SAMPLES, 1)
        for k, v in options:
            P.set_option(k, v)
        out = P.project(vol, geom, nu, nv)
        mfl = P.ray_ranges(geom, nu, nv)
        torch.cuda.synchronize()
        n = P.last_sample_count()
        return out.cpu().numpy(), mfl.cpu().numpy(), n


def compare_full(torch, fp, oracle, vol_np, delta, origin, geom, nu, nv, options=(), kernel=0, what=""):
    geom = np.asarray(geom, dtype=np.float64).reshape(-1, 12)
    out, mfl, n = run_gpu(torch, fp, vol_np, delta, origin, geom, nu, nv, options)
    ids = all_ids(geom.shape[0], nv, nu)
    ov, om, pl, mg = oracle.project_rays(vol_np, delta, origin, geom, ids, kernel=kernel, threads=oracle.host_cores())
    worst = assert_parity(out.ravel(), mfl.reshape(-1, 3), ov, om, pl, mg, float(np.abs(vol_np).max()), what,
                          recompute=make_recompute(oracle, vol_np, delta, origin, geom, ids, kernel))
    assert n == int(np.maximum(om[:, 2] - om[:, 1] + 1, 0).sum()), "sample count"
    return worst, out, om


# ----------------------------------------------------------------------------- BASELINE configs

def test_c1_tiny_cone_beam_full(torch, fp, synth, oracle):
    cfg = synth.CONFIGS["C1"]
    vol = synth.make_volume(cfg).numpy()
    geom = synth.make_geometry(cfg)
    worst, out, om = compare_full(torch, fp, oracle, vol, cfg.voxel_size, cfg.origin, geom, cfg.nu, cfg.nv, what="C1")
    assert out.shape == (16, 48, 48) and worst < 1.0
    assert set(np.unique(om[:, 0])) == {0, 1}


def test_c2_128_cube_full_orbit(torch, fp, synth, oracle):
    cfg = synth.CONFIGS["C2"]
    vol = synth.make_volume(cfg).numpy()
    geom = synth.make_geometry(cfg)
    out, mfl, n = run_gpu(torch, fp, vol, cfg.voxel_size, cfg.origin, geom, cfg.nu, cfg.nv)
    # every ray of 12 projections (including the driving-axis switches at 45 deg + k 90 deg) ...
    projs = [0, 22, 23, 44, 45, 67, 68, 90, 113, 135, 158, 179]
    ids = all_ids(cfg.n_proj, cfg.nv, cfg.nu, projs)
    # ... plus 2^18 random rays over the whole orbit
    ids = np.concatenate([ids, synth.sample_rays(cfg, 1 << 18)])
    ov, om, pl, mg = oracle.project_rays(vol, cfg.voxel_size, cfg.origin, geom, ids, threads=oracle.host_cores())
    g = out[ids[:, 0], ids[:, 1], ids[:, 2]]
    gm = mfl[ids[:, 0], ids[:, 1], ids[:, 2]]
    assert assert_parity(g, gm, ov, om, pl, mg, float(np.abs(vol).max()), "C2",
                         recompute=make_recompute(oracle, vol, cfg.voxel_size, cfg.origin, geom, ids)) < 1.0
    assert n == int(np.maximum(mfl[..., 2] - mfl[..., 1] + 1, 0).sum())


def test_c1_and_c2_through_the_direct_kernel(torch, fp, synth, oracle):
    """FP_OPT_KERNEL = FP_KERNEL_DIRECT: the general-pose kernel on the circular-orbit configs (the
    default plan would pick the aligned kernel for all of them)."""
    cfg = synth.CONFIGS["C1"]
    worst, _, _ = compare_full(torch, fp, oracle, synth.make_volume(cfg).numpy(), cfg.voxel_size, cfg.origin,
                               synth.make_geometry(cfg), cfg.nu, cfg.nv,
                               options=[(fp.OPT_KERNEL, fp.KERNEL_DIRECT)], what="C1 direct")
    assert worst < 1.0
    cfg = synth.CONFIGS["C2"]
    vol = synth.make_volume(cfg).numpy()
    geom = synth.make_geometry(cfg)[[0, 22, 23, 45, 90, 113, 158]]
    worst, _, _ = compare_full(torch, fp, oracle, vol, cfg.voxel_size, cfg.origin, geom, cfg.nu, cfg.nv,
                               options=[(fp.OPT_KERNEL, fp.KERNEL_DIRECT)], what="C2 direct")
    assert worst < 1.0


def _big_config_subset(torch, fp, synth, oracle, name, projs, n_random, batch=None, options=()):
    """Full-size volume on the device, the launch configuration bench.py times (whole batches
    through fp_project), compared on sampled rays the oracle computes one by one."""
    cfg = synth.CONFIGS[name]
    vol_t = synth.make_volume(cfg, device="cuda")
    vol = vol_t.cpu().numpy()
    geom = synth.make_geometry(cfg)
    sub = geom[projs]
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_COUNT_SAMPLES, 1)
        for k, v in options:
            P.set_option(k, v)
        out = P.project(vol_t, sub, cfg.nu, cfg.nv)
        mfl = P.ray_ranges(sub, cfg.nu, cfg.nv)
        torch.cuda.synchronize()
        n = P.last_sample_count()
        out, mfl = out.cpu().numpy(), mfl.cpu().numpy()
    rng = np.random.default_rng(cfg.seed + 77)
    ids = np.stack([rng.integers(0, len(projs), n_random), rng.integers(0, cfg.nv, n_random),
                    rng.integers(0, cfg.nu, n_random)], axis=1).astype(np.int32)
    # one full detector row and column per projection as well (tile edges, ragged tails)
    extra = []
    for p in range(len(projs)):
        extra += [(p, cfg.nv // 3, u) for u in range(cfg.nu)] + [(p, v, cfg.nu - 1) for v in range(cfg.nv)]
    ids = np.concatenate([ids, np.array(extra, dtype=np.int32)])
    ov, om, pl, mg = oracle.project_rays(vol, cfg.voxel_size, cfg.origin, sub, ids, threads=oracle.host_cores())
    g = out[ids[:, 0], ids[:, 1], ids[:, 2]]
    gm = mfl[ids[:, 0], ids[:, 1], ids[:, 2]]
    worst = assert_parity(g, gm, ov, om, pl, mg, float(np.abs(vol).max()), name,
                          recompute=make_recompute(oracle, vol, cfg.voxel_size, cfg.origin, sub, ids))
    assert n == int(np.maximum(mfl[..., 2] - mfl[..., 1] + 1, 0).sum())
    return worst, om


def test_c3_paper_scale_sampled(torch, fp, synth, oracle):
    worst, om = _big_config_subset(torch, fp, synth, oracle, "C3", [0, 44, 45, 46, 90, 135, 201, 359], 60000)
    assert worst < 1.0 and set(np.unique(om[:, 0])) == {0, 1}


def test_c4_wide_cone_general_poses_sampled(torch, fp, synth, oracle):
    worst, om = _big_config_subset(torch, fp, synth, oracle, "C4", [0, 1, 2, 3, 100, 255], 60000)
    assert worst < 1.0
    assert set(np.unique(om[:, 0])) == {0, 1, 2}          # all three driving axes
    assert (om[:, 2] < om[:, 1]).mean() > 0.05            # and a fair share of misses


def test_c5_large_volume_sampled(torch, fp, synth, oracle):
    worst, om = _big_config_subset(torch, fp, synth, oracle, "C5", [0, 89, 90, 91, 400, 719], 40000)
    assert worst < 1.0


def test_p1_paper_shaped_sampled(torch, fp, synth, oracle):
    """The paper-shaped workload at full size (512^3 cylinder -> 512^2, 10 degree cone, grid matched by Eq. 17;
    PAPER.md:312-314, :326) with FP_OPT_FOV_CYLINDER, default plan (the 384-voxel instantiation of
    fp_aligned_kernel with the circle clip), poses around the driving-axis switch included."""
    worst, om = _big_config_subset(torch, fp, synth, oracle, "P1", [0, 44, 45, 46, 90, 135, 201, 359], 60000,
                                   options=[(fp.OPT_FOV_CYLINDER, 1)])
    assert worst < 1.0 and set(np.unique(om[:, 0])) == {0, 1}


# ----------------------------------------------------------------------------- edge cases

def small_problem(rng, shape=(19, 13, 23), delta=0.7):
    vol = rng.uniform(-1.0, 2.0, size=shape).astype(np.float32)
    origin = tuple(-(n - 1) / 2.0 * delta + 0.3 * k for k, n in enumerate(shape))
    return vol, delta, origin


def pose(src, look_at, nu, nv, pitch, sdd, roll=0.0):
    src = np.asarray(src, float)
    n = np.asarray(look_at, float) - src
    n /= np.linalg.norm(n)
    ax = np.zeros(3)
    ax[int(np.argmin(np.abs(n)))] = 1.0
    e1 = np.cross(n, ax)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(n, e1)
    U = pitch * (math.cos(roll) * e1 + math.sin(roll) * e2)
    V = pitch * (-math.sin(roll) * e1 + math.cos(roll) * e2)
    C = src + sdd * n
    O = C - (nu - 1) / 2.0 * U - (nv - 1) / 2.0 * V
    return np.concatenate([src, O, U, V])


@pytest.mark.parametrize("nu,nv", [(1, 1), (37, 53), (33, 9), (8, 65)])
def test_ragged_detectors_and_anisotropic_grid_all_axes(torch, fp, oracle, nu, nv):
    rng = np.random.default_rng(100 + nu)
    vol, delta, origin = small_problem(rng)
    geom = np.stack([pose(s, (0.2, -0.1, 0.3), nu, nv, 0.5, 60.0, roll)
                     for s, roll in [((-30, 2, 1), 0.0), ((1, 28, -3), 0.4), ((2, -1, 31), 1.1),
                                     ((-14, -15, 16), 2.0), ((20, 3, -19), 0.7)]])
    for perm in (1, 0):
        worst, _, om = compare_full(torch, fp, oracle, vol, delta, origin, geom, nu, nv,
                                    options=[(fp.OPT_PERMUTED_COPY, perm)], what="ragged %dx%d perm=%d" % (nu, nv, perm))
        assert worst < 1.0
    if nu * nv > 100:
        assert set(np.unique(om[:, 0])) == {0, 1, 2}


def test_spline_kernel(torch, fp, oracle):
    rng = np.random.default_rng(5)
    vol, delta, origin = small_problem(rng)
    geom = np.stack([pose((-30, 4, 2), (0, 0, 0), 40, 24, 0.45, 60.0, 0.3), pose((3, 4, 29), (0, 0, 0), 40, 24, 0.45, 55.0, 0.0)])
    worst, _, _ = compare_full(torch, fp, oracle, vol, delta, origin, geom, 40, 24,
                               options=[(fp.OPT_INTERP, fp.INTERP_SPLINE)], kernel=1, what="spline")
    assert worst < 1.0


def test_all_rays_miss_and_n_proj_zero(torch, fp, oracle):
    rng = np.random.default_rng(6)
    vol, delta, origin = small_problem(rng)
    geom = pose((-30, 200, 2), (0, 400, 0), 16, 16, 0.5, 60.0)[None]       # looks away from the volume
    worst, out, om = compare_full(torch, fp, oracle, vol, delta, origin, geom, 16, 16, what="miss")
    assert np.all(out == 0.0) and np.all(om[:, 2] < om[:, 1])
    volt = torch.from_numpy(vol).cuda()
    with fp.Projector(*vol.shape, delta, origin) as P:
        out = P.project(volt, np.zeros((0, 12)), 16, 16)
        assert out.shape == (0, 16, 16)


def test_axis_parallel_rays_ties_and_degenerate_ray(torch, fp, oracle):
    """Rays exactly parallel to an axis (r~_t = 0), exact |r| ties (lowest axis wins, reading #8),
    integer sample positions (second tap weight 0) and a pixel that coincides with the
    source (r = 0 -> output 0)."""
    vol = np.arange(6 * 5 * 4, dtype=np.float32).reshape(6, 5, 4) / 8.0
    delta, origin = 1.0, (0.0, 0.0, 0.0)
    rows = []
    # parallel-ish fan: source far on -x, detector plane x = 10, pixel centres on integer (y, z)
    rows.append(np.array([-1e6, 2.0, 1.0, 10.0, 0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0]))
    # source on the x axis: the central pixel's ray is exactly axis-parallel
    rows.append(np.array([-20.0, 2.0, 1.0, 10.0, 0.0, -1.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0]))
    # exact ties |r_x| = |r_y| on the diagonal pixels
    rows.append(np.array([-8.0, -8.0, 1.5, -6.0, -6.0, 1.5, 0.0, 1.0, 0.0, 1.0, 0.0, 0.0]))
    # detector plane through the source: pixel (2,1) is the source itself
    rows.append(np.array([3.0, 2.0, 9.0, 1.0, 1.0, 9.0, 1.0, 0.0, 0.0, 0.0, 1.0, 0.0]))
    geom = np.stack(rows)
    worst, out, om = compare_full(torch, fp, oracle, vol, delta, origin, geom, 6, 5, what="axis-parallel")
    assert worst < 1.0
    assert out[3, 1, 2] == 0.0


def test_single_slice_and_single_voxel_volumes(torch, fp, oracle):
    rng = np.random.default_rng(8)
    for shape in [(1, 9, 7), (9, 1, 7), (9, 7, 1), (1, 1, 1)]:
        vol = rng.uniform(0.5, 1.5, size=shape).astype(np.float32)
        origin = tuple(-(n - 1) / 2.0 for n in shape)
        geom = np.stack([pose((-25, 1, 2), (0, 0, 0), 24, 20, 0.6, 50.0), pose((2, 1, 25), (0, 0, 0), 24, 20, 0.6, 50.0),
                         pose((1, -25, 2), (0, 0, 0), 24, 20, 0.6, 50.0)])
        worst, _, _ = compare_full(torch, fp, oracle, vol, 1.0, origin, geom, 24, 20, what=str(shape))
        assert worst < 1.0


def test_constant_volume_chord_property_at_full_size(torch, fp):
    """A property that holds at any size (no oracle needed): for a constant volume every ray that
    enters and leaves through the driving-axis faces returns c * delta * ||r~|| * N_m."""
    n = 512
    vol = torch.full((n, n, n), 0.5, device="cuda", dtype=torch.float32)
    from paper_1609_00958_b200 import synth
    cfg = synth.CONFIGS["C3"]
    geom = synth.make_geometry(cfg)[[10]]
    with fp.Projector(n, n, n, 1.0, cfg.origin) as P:
        out = P.project(vol, geom, cfg.nu, cfg.nv).cpu().numpy()[0]
        mfl = P.ray_ranges(geom, cfg.nu, cfg.nv).cpu().numpy()[0]
    full = (mfl[..., 1] == 0) & (mfl[..., 2] == n - 1)
    assert full.mean() > 0.3
    # ||r~|| recomputed here from the geometry
    g = geom[0]
    iv, iu = np.meshgrid(np.arange(cfg.nv), np.arange(cfg.nu), indexing="ij")
    D = g[3:6][None, None] + iu[..., None] * g[6:9] + iv[..., None] * g[9:12]
    r = D - g[0:3]
    L = np.linalg.norm(r, axis=-1) / np.abs(r).max(axis=-1)
    # interior rays only (all four taps inside on every slice): compare where the value is the chord
    expect = 0.5 * L * n
    inner = full & (np.abs(out - expect) <= 2e-5 * expect + 1e-6 * L * n * 0.5)
    # rays whose transverse range touches the zero padding have smaller values; all others must match
    assert np.all(out[full] <= expect[full] * (1 + 3e-5))
    assert inner.sum() > 0.25 * full.size


def test_project_host_matches_device_path(torch, fp, synth):
    cfg = synth.CONFIGS["C1"]
    vol = synth.make_volume(cfg)
    geom = synth.make_geometry(cfg)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_COUNT_SAMPLES, 1)
        a = P.project(vol.cuda(), geom, cfg.nu, cfg.nv).cpu()
        n1 = P.last_sample_count()
        b = P.project_host(vol.pin_memory(), geom, cfg.nu, cfg.nv)
        n2 = P.last_sample_count()
    assert torch.equal(a, b) and n1 == n2


def test_reuse_context_changed_volume_and_streams(torch, fp, synth, oracle):
    """The volume changes between calls (iterative reconstruction): with the default
    FP_OPT_VOLATILE = 1 the z-driven layout copy is rebuilt; work runs on a caller's stream."""
    rng = np.random.default_rng(9)
    vol, delta, origin = small_problem(rng)
    geom = np.stack([pose((2, -1, 31), (0, 0, 0), 32, 32, 0.5, 60.0, 0.2)])
    ids = all_ids(1, 32, 32)
    s = torch.cuda.Stream()
    with fp.Projector(*vol.shape, delta, origin) as P:
        for scale in (1.0, -2.0):
            v = (vol * scale).astype(np.float32)
            vt = torch.from_numpy(v).cuda()
            torch.cuda.synchronize()
            with torch.cuda.stream(s):
                out = P.project(vt, geom, 32, 32, stream=s)
            s.synchronize()
            ov, om, pl, mg = oracle.project_rays(v, delta, origin, geom, ids)
            gm = P.ray_ranges(geom, 32, 32).cpu().numpy()
            assert assert_parity(out.cpu().numpy().ravel(), gm.reshape(-1, 3), ov, om, pl, mg, float(np.abs(v).max())) < 1.0


def test_host_plan_is_reused_only_for_the_same_geometry_and_options(torch, fp, synth):
    """fp_project keeps the host plan of its last call (libfp's PlanCache, fp.cu) and reuses it when the next call
    brings the same geometry, detector, options and volume alignment.  One context is driven through aligned poses,
    general poses of the same count, the aligned poses again (a hit), then the same poses with another kernel
    option (must re-plan): every result equals the one a fresh context gives, bit for bit."""
    cfg = synth.CONFIGS["C2"]
    vol = synth.make_volume(cfg, device="cuda")
    nu = nv = 96
    g_al = synth.make_geometry(cfg)[[0, 44, 45, 46, 90, 133]].copy()
    for g in g_al:                                    # same orbit, smaller detector: keep it centred
        g[3:6] += (cfg.nu - nu) / 2 * g[6:9] + (cfg.nv - nv) / 2 * g[9:12]
    g_ge = synth.make_geometry(synth.CONFIGS["C4"])[:6].copy()
    g_ge[:, :6] *= 128.0 / 512.0                      # C4's general poses, scaled to the 128^3 grid
    g_ge[:, 6:] *= 3.0

    def fresh(geom, options=()):
        with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as Q:
            for k, v in options:
                Q.set_option(k, v)
            o = Q.project(vol, geom, nu, nv)
            torch.cuda.synchronize()
            return o.cpu().numpy()

    ref_al, ref_ge = fresh(g_al), fresh(g_ge)
    ref_di = fresh(g_al, [(fp.OPT_KERNEL, fp.KERNEL_DIRECT)])
    assert np.abs(ref_al).max() > 0 and np.abs(ref_ge).max() > 0
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        seq = [(g_al, ref_al), (g_al, ref_al), (g_ge, ref_ge), (g_al, ref_al), (g_ge, ref_ge), (g_ge, ref_ge)]
        for k, (g, ref) in enumerate(seq):
            o = P.project(vol, g, nu, nv)
            torch.cuda.synchronize()
            assert np.array_equal(o.cpu().numpy(), ref), "call %d" % k
        P.check()
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_DIRECT)  # same geometry as the last aligned call, other plan
        for g, ref in ((g_al, ref_di), (g_al, ref_di)):
            o = P.project(vol, g, nu, nv)
            torch.cuda.synchronize()
            assert np.array_equal(o.cpu().numpy(), ref)
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_AUTO)
        o = P.project(vol, g_al, nu, nv)
        torch.cuda.synchronize()
        assert np.array_equal(o.cpu().numpy(), ref_al)
        # a volume view that is only 4-byte aligned: the aligned-class kernels need 16 bytes, so the plan changes
        flat = torch.zeros(vol.numel() + 4, device="cuda", dtype=torch.float32)
        v1 = flat[1:1 + vol.numel()].view(vol.shape)
        v1.copy_(vol)
        o = P.project(v1, g_al, nu, nv)
        torch.cuda.synchronize()
        o = o.cpu().numpy()
        P.check()
        assert np.allclose(o, ref_al, rtol=1e-4, atol=1e-4 * float(np.abs(ref_al).max()))
        o = P.project(vol, g_al, nu, nv)
        torch.cuda.synchronize()
        assert np.array_equal(o.cpu().numpy(), ref_al)


# ----------------------------------------------------------------------------- aligned kernel edge cases

def aligned_pose(theta, sid, sdd, nu, nv, pitch, src_z=0.0, det_shift=(0.0, 0.0), flip_u=False, flip_v=False):
    """v parallel to z, u perpendicular to z: the geometry class fp_aligned_kernel takes."""
    c, s = math.cos(theta), math.sin(theta)
    S = np.array([sid * c, sid * s, src_z])
    C = S - sdd * np.array([c, s, 0.0])
    U = pitch * np.array([-s, c, 0.0]) * (-1.0 if flip_u else 1.0)
    V = pitch * np.array([0.0, 0.0, 1.0]) * (-1.0 if flip_v else 1.0)
    O = C - ((nu - 1) / 2 + det_shift[0]) * U - ((nv - 1) / 2 + det_shift[1]) * V
    return np.concatenate([S, O, U, V])


@pytest.mark.parametrize("nu,nv,interp", [(37, 300, 0), (8, 5, 0), (66, 40, 1)])
def test_aligned_kernel_edge_cases(torch, fp, oracle, nu, nv, interp):
    """Ragged detectors (nu not a multiple of 8 or 4, more than one 256-row block), exact |r_x| = |r_y|
    ties and the axis switch inside a block (45 degrees), both senses of u and v, a source off the
    mid-plane, a detector shifted so far that some columns and rows miss, rays parallel to an axis."""
    rng = np.random.default_rng(300 + nu)
    shape = (21, 18, 24)                                    # nz a multiple of 4
    vol = rng.uniform(-1.0, 2.0, size=shape).astype(np.float32)
    delta = 0.8
    origin = tuple(-(n - 1) / 2.0 * delta + 0.17 * k for k, n in enumerate(shape))
    pitch = 0.9 * 24 * delta * 2.2 / nv if nv > 100 else 0.55
    poses = []
    for k, th in enumerate([0.0, math.pi / 4, 0.7853, 1.1, math.pi / 2, 2.5, math.pi, 3.9269908, 4.4, 5.9]):
        poses.append(aligned_pose(th, 40.0, 90.0, nu, nv, pitch, src_z=(k % 3 - 1) * 3.0,
                                  det_shift=((k % 4) * 2.5, -(k % 2) * 3.0), flip_u=bool(k & 1), flip_v=bool(k & 2)))
    geom = np.stack(poses)
    with fp.Projector(*shape, delta, origin) as P:
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_ALIGNED)
        assert all(P.plan(g, nu, nv)[0] == fp.KERNEL_ALIGNED for g in geom)
    worst, out, om = compare_full(torch, fp, oracle, vol, delta, origin, geom, nu, nv,
                                  options=[(fp.OPT_KERNEL, fp.KERNEL_ALIGNED), (fp.OPT_INTERP, interp)], kernel=interp,
                                  what="aligned %dx%d" % (nu, nv))
    assert worst < 1.0
    assert set(np.unique(om[:, 0])) <= {0, 1}
    if nv > 100:
        assert (om[:, 2] < om[:, 1]).any() and (om[:, 2] >= om[:, 1]).any()     # some rays miss, most hit


def test_aligned_kernel_window_sizes_and_direct_kernel_agree(torch, fp):
    """The aligned kernel (whatever staging window the plan picks) and the direct kernel are two
    implementations of the same sum: on the same inputs they agree to fp32 rounding (a property that
    needs no oracle, so it runs at a size the oracle would not finish)."""
    from paper_1609_00958_b200 import synth
    cfg = synth.CONFIGS["C2"]
    vol = synth.make_volume(cfg, device="cuda")
    windows = set()
    for pitch, nv in [(0.7, 64), (1.5, 192), (2.0, 256), (2.5, 270)]:
        geom = np.stack([aligned_pose(th, cfg.sid, cfg.sdd, 96, nv, pitch) for th in (0.2, 0.8, 2.0, 4.0)])
        with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
            P.set_option(fp.OPT_KERNEL, fp.KERNEL_ALIGNED)
            plans = [P.plan(g, 96, nv) for g in geom]
            assert all(k == fp.KERNEL_ALIGNED for k, _, _ in plans), plans
            windows.add((max(w for _, w, _ in plans) + 127) // 128)
            a = P.project(vol, geom, 96, nv).cpu().numpy().astype(np.float64)
            P.set_option(fp.OPT_KERNEL, fp.KERNEL_DIRECT)
            b = P.project(vol, geom, 96, nv).cpu().numpy().astype(np.float64)
        scale = np.abs(b).max()
        assert np.abs(a - b).max() <= 2e-5 * scale, (pitch, nv, np.abs(a - b).max(), scale)
    assert len(windows) >= 3                                # several of the 128 / 256 / 384 / 512 instantiations ran


# ----------------------------------------------------------------------------- TMA-fed kernel (FP_KERNEL_TMA)

def test_tma_kernel_parity(torch, fp, synth, oracle):
    """fp_tma_kernel against the oracle: C1 in full, C2 on the poses whose row tile fits, the ragged /
    mixed-axis / flipped / off-plane edge poses of the aligned kernel, spline weights."""
    opt = [(fp.OPT_KERNEL, fp.KERNEL_TMA)]
    cfg = synth.CONFIGS["C1"]
    geom = synth.make_geometry(cfg)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_TMA)
        assert all(P.plan(g, cfg.nu, cfg.nv)[0] == fp.KERNEL_TMA for g in geom)
    worst, _, _ = compare_full(torch, fp, oracle, synth.make_volume(cfg).numpy(), cfg.voxel_size, cfg.origin, geom,
                               cfg.nu, cfg.nv, options=opt, what="C1 tma")
    assert worst < 1.0
    cfg = synth.CONFIGS["C2"]
    geom = synth.make_geometry(cfg)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_TMA)
        sel = [p for p in range(cfg.n_proj) if P.plan(geom[p], cfg.nu, cfg.nv)[0] == fp.KERNEL_TMA]
    assert len(sel) > 20
    sel = sel[:: max(1, len(sel) // 8)]
    worst, _, _ = compare_full(torch, fp, oracle, synth.make_volume(cfg).numpy(), cfg.voxel_size, cfg.origin, geom[sel],
                               cfg.nu, cfg.nv, options=opt, what="C2 tma")
    assert worst < 1.0
    for nu, nv, interp in [(37, 300, 0), (66, 40, 1)]:
        rng = np.random.default_rng(400 + nu)
        shape = (21, 18, 24)
        vol = rng.uniform(-1.0, 2.0, size=shape).astype(np.float32)
        delta = 0.8
        origin = tuple(-(n - 1) / 2.0 * delta + 0.17 * k for k, n in enumerate(shape))
        pitch = 0.9 * 24 * delta * 2.2 / nv if nv > 100 else 0.55
        geom = np.stack([aligned_pose(th, 40.0, 90.0, nu, nv, pitch, src_z=(k % 3 - 1) * 3.0,
                                      det_shift=((k % 4) * 2.5, -(k % 2) * 3.0), flip_u=bool(k & 1), flip_v=bool(k & 2))
                         for k, th in enumerate([0.0, math.pi / 4, 0.7853, 1.1, math.pi / 2, 2.5, math.pi, 3.9269908, 4.4, 5.9])])
        with fp.Projector(*shape, delta, origin) as P:
            P.set_option(fp.OPT_KERNEL, fp.KERNEL_TMA)
            assert all(P.plan(g, nu, nv)[0] == fp.KERNEL_TMA for g in geom)
        worst, _, _ = compare_full(torch, fp, oracle, vol, delta, origin, geom, nu, nv,
                                   options=opt + [(fp.OPT_INTERP, interp)], kernel=interp, what="tma %dx%d" % (nu, nv))
        assert worst < 1.0


def test_tma_kernel_c3_sampled_and_fallback(torch, fp, synth, oracle):
    cfg = synth.CONFIGS["C3"]
    vol_t = synth.make_volume(cfg, device="cuda")
    geom = synth.make_geometry(cfg)[[0, 44, 45, 46, 90, 135, 201, 359]]
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_TMA)
        assert all(P.plan(g, cfg.nu, cfg.nv)[0] == fp.KERNEL_TMA for g in geom)
        out = P.project(vol_t, geom, cfg.nu, cfg.nv)
        torch.cuda.synchronize()
        P.check()                              # raises if a window or row tile overflowed
        out = out.cpu().numpy()
        # a pose that does not fit the tile (coarse detector columns) silently uses the aligned kernel
        coarse = aligned_pose(0.8, cfg.sid, cfg.sdd, 96, 64, 3.0)
        assert P.plan(coarse, 96, 64)[0] == fp.KERNEL_ALIGNED
        P.project(vol_t, coarse[None], 96, 64)
        torch.cuda.synchronize()
        P.check()
    vol = vol_t.cpu().numpy()
    rng = np.random.default_rng(99)
    n = 30000
    ids = np.stack([rng.integers(0, len(geom), n), rng.integers(0, cfg.nv, n), rng.integers(0, cfg.nu, n)], axis=1).astype(np.int32)
    ov, om, pl, mg = oracle.project_rays(vol, cfg.voxel_size, cfg.origin, geom, ids, threads=oracle.host_cores())
    g = out[ids[:, 0], ids[:, 1], ids[:, 2]]
    tol = 2e-5 * np.abs(ov) + 1e-6 * pl * float(np.abs(vol).max())
    assert np.all(np.abs(g - ov) <= tol), float(np.max(np.abs(g - ov) / np.maximum(tol, 1e-300)))


# ----------------------------------------------------------------------------- back-projection

def bp_tolerance(oracle, proj, shape, delta, origin, geom, kernel):
    """|gpu - oracle| <= 2e-5 * (A^T |y|)[v] + 1e-6 * max_v (A^T 1) * max|y|: the forward tolerance transposed.
    The relative term is taken against the sum of the magnitudes a voxel receives; the absolute term is the
    forward's 1e-6 * path length * max|input| with the path length replaced by the largest total weight any
    voxel receives (a voxel at the rim receives many samples with tiny weights, each carrying the same
    absolute fp32 weight error as an interior one)."""
    absy = oracle.backproject(np.abs(proj), shape, delta, origin, geom, kernel=kernel, threads=oracle.host_cores())
    wsum = oracle.backproject(np.ones_like(proj), shape, delta, origin, geom, kernel=kernel, threads=oracle.host_cores())
    return 2e-5 * absy + 1e-6 * float(wsum.max()) * float(np.abs(proj).max())


@pytest.mark.parametrize("interp", [0, 1])
def test_backprojection_parity_small_all_axes(torch, fp, oracle, interp):
    rng = np.random.default_rng(500 + interp)
    vol, delta, origin = small_problem(rng)
    shape = vol.shape
    nu, nv = 37, 29
    geom = np.stack([pose(s, (0.2, -0.1, 0.3), nu, nv, 0.5, 60.0, roll)
                     for s, roll in [((-30, 2, 1), 0.0), ((1, 28, -3), 0.4), ((2, -1, 31), 1.1),
                                     ((-14, -15, 16), 2.0), ((20, 3, -19), 0.7)]]
                    + [aligned_pose(0.8, 40.0, 90.0, nu, nv, 0.5), pose((-30, 200, 2), (0, 400, 0), nu, nv, 0.5, 60.0)])
    y = rng.uniform(-1.0, 2.0, size=(len(geom), nv, nu)).astype(np.float32)
    with fp.Projector(*shape, delta, origin) as P:
        P.set_option(fp.OPT_INTERP, interp)
        out = P.backproject(torch.from_numpy(y).cuda(), geom, nu, nv)
        torch.cuda.synchronize()
        g = out.cpu().numpy().astype(np.float64)
        # n_proj = 0 clears the volume
        z = P.backproject(torch.zeros((0, nv, nu), device="cuda"), np.zeros((0, 12)), nu, nv, out=out)
        assert float(z.abs().max()) == 0.0
    ref = oracle.backproject(y.astype(np.float64), shape, delta, origin, geom, kernel=interp, threads=oracle.host_cores())
    tol = bp_tolerance(oracle, y.astype(np.float64), shape, delta, origin, geom, interp)
    err = np.abs(g - ref)
    assert np.all(err <= tol), float(np.max(err / np.maximum(tol, 1e-300)))
    assert np.abs(ref).max() > 1.0


def test_backprojection_c1_parity_and_adjoint_identity_at_c3_size(torch, fp, synth, oracle):
    cfg = synth.CONFIGS["C1"]
    geom = synth.make_geometry(cfg)
    rng = np.random.default_rng(61)
    y = rng.uniform(0.0, 1.0, size=(cfg.n_proj, cfg.nv, cfg.nu)).astype(np.float32)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        g = P.backproject(torch.from_numpy(y).cuda(), geom, cfg.nu, cfg.nv).cpu().numpy().astype(np.float64)
    ref = oracle.backproject(y.astype(np.float64), cfg.n, cfg.voxel_size, cfg.origin, geom, threads=oracle.host_cores())
    tol = bp_tolerance(oracle, y.astype(np.float64), cfg.n, cfg.voxel_size, cfg.origin, geom, 0)
    assert np.all(np.abs(g - ref) <= tol)
    # a property that holds at any size: <A x, y> = <x, A^T y> with the (oracle-checked) forward kernel,
    # on the full 512^3 volume and four C3 poses
    cfg = synth.CONFIGS["C3"]
    geom = synth.make_geometry(cfg)[[3, 47, 200, 311]]
    x = synth.make_volume(cfg, device="cuda")
    gen = torch.Generator(device="cuda").manual_seed(5)
    yy = torch.rand((len(geom), cfg.nv, cfg.nu), device="cuda", generator=gen)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        ax = P.project(x, geom, cfg.nu, cfg.nv)
        aty = P.backproject(yy, geom, cfg.nu, cfg.nv)
        torch.cuda.synchronize()
    lhs = float((ax.double() * yy.double()).sum())
    rhs = float((x.double() * aty.double()).sum())
    assert abs(lhs - rhs) <= 2e-5 * abs(lhs), (lhs, rhs)


@pytest.mark.parametrize("interp", [0, 1])
def test_backprojection_aligned_kernel_and_ray_driven_kernel_against_the_oracle(torch, fp, synth, oracle, interp):
    """Circular-orbit poses take fp_bp_aligned_kernel (the transpose of the TMA-fed kernel), FP_KERNEL_DIRECT forces
    the ray-driven scatter: both against the oracle on C2 (192 detector rows = a ragged row block, 11 poses = a
    short last group, both driving axes and blocks where the axis switches)."""
    cfg = synth.CONFIGS["C2"]
    geom = synth.make_geometry(cfg)[np.r_[0:180:17]]
    rng = np.random.default_rng(77 + interp)
    y = rng.uniform(-1.0, 2.0, size=(len(geom), cfg.nv, cfg.nu)).astype(np.float32)
    yd = torch.from_numpy(y).cuda()
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_INTERP, interp)
        assert all(P.plan(g, cfg.nu, cfg.nv)[0] in (fp.KERNEL_TMA, fp.KERNEL_ALIGNED) for g in geom)
        g2 = P.backproject(yd, geom, cfg.nu, cfg.nv).cpu().numpy().astype(np.float64)
        assert P.last_launch_count() == 1
        P.check()
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_DIRECT)
        g1 = P.backproject(yd, geom, cfg.nu, cfg.nv).cpu().numpy().astype(np.float64)
    ref = oracle.backproject(y.astype(np.float64), cfg.n, cfg.voxel_size, cfg.origin, geom, kernel=interp, threads=oracle.host_cores())
    tol = bp_tolerance(oracle, y.astype(np.float64), cfg.n, cfg.voxel_size, cfg.origin, geom, interp)
    for name, g in (("aligned", g2), ("ray-driven", g1)):
        err = np.abs(g - ref)
        assert np.all(err <= tol), (name, float(np.max(err / np.maximum(tol, 1e-300))))
    assert np.abs(ref).max() > 1.0


def test_backprojection_c3_size_sampled_voxels(torch, fp, synth, oracle):
    """Element by element at full size: fp_backproject on the 512^3 grid of C3 (four poses, both driving axes),
    compared on 2^18 seeded voxels plus the volume's corners and centre,
    with (A^T y)[v] computed voxel by voxel from the definition of the transpose (oracle.backproject_voxels).
    Tolerance as in bp_tolerance, with max_v (A^T 1) taken over the sampled voxels only (never larger)."""
    cfg = synth.CONFIGS["C3"]
    geom = synth.make_geometry(cfg)[[3, 47, 200, 311]]
    gen = torch.Generator(device="cuda").manual_seed(6)
    yy = torch.rand((len(geom), cfg.nv, cfg.nu), device="cuda", generator=gen) * 2.0 - 0.5
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        aty = P.backproject(yy, geom, cfg.nu, cfg.nv)
        torch.cuda.synchronize()
    rng = np.random.default_rng(cfg.seed + 99)
    nx, ny, nz = cfg.n
    vox = np.stack([rng.integers(0, nx, 1 << 18), rng.integers(0, ny, 1 << 18), rng.integers(0, nz, 1 << 18)], axis=1)
    special = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (nx - 1, 0, 0), (0, ny - 1, nz - 1), (nx // 2, ny // 2, nz // 2),
               (nx - 1, ny // 2, 3), (nx // 2 + 1, 0, 0)]
    vox = np.concatenate([vox, np.array(special)]).astype(np.int32)
    idx = torch.from_numpy(vox.astype(np.int64)).cuda()
    g = aty[idx[:, 0], idx[:, 1], idx[:, 2]].cpu().numpy().astype(np.float64)
    y = yy.cpu().numpy().astype(np.float64)
    th = oracle.host_cores()
    # the hat footprint of a voxel is +-1 voxel = +-(SDD / (SID - half diagonal)) = +-2.4 pixels here
    ref = oracle.backproject_voxels(y, cfg.n, cfg.voxel_size, cfg.origin, geom, vox, halfwin=4, threads=th)
    absy = oracle.backproject_voxels(np.abs(y), cfg.n, cfg.voxel_size, cfg.origin, geom, vox, halfwin=4, threads=th)
    wsum = oracle.backproject_voxels(np.ones_like(y), cfg.n, cfg.voxel_size, cfg.origin, geom, vox, halfwin=4, threads=th)
    tol = 2e-5 * absy + 1e-6 * float(wsum.max()) * float(np.abs(y).max())
    err = np.abs(g - ref)
    assert np.abs(ref).max() > 1.0 and (ref != 0).mean() > 0.5
    assert np.all(err <= tol), (float(np.max(err / np.maximum(tol, 1e-300))), vox[int(np.argmax(err - tol))])


def test_tma_kernel_follows_the_volume_pointer_and_contents(torch, fp, oracle):
    """The tensor maps of the TMA-fed kernel are cached per volume pointer: a second volume at another address
    and new contents at the same address must both be projected from the data as it is at call time."""
    rng = np.random.default_rng(77)
    shape, delta = (24, 20, 32), 0.9
    origin = tuple(-(n - 1) / 2.0 * delta for n in shape)
    nu, nv = 40, 36
    geom = np.stack([aligned_pose(th, 50.0, 110.0, nu, nv, 0.8) for th in (0.3, 1.9, 4.0)])
    ids = all_ids(len(geom), nv, nu)
    va = rng.uniform(0.0, 1.0, size=shape).astype(np.float32)
    vb = rng.uniform(-1.0, 1.0, size=shape).astype(np.float32)
    ta, tb = torch.from_numpy(va).cuda(), torch.from_numpy(vb).cuda()
    with fp.Projector(*shape, delta, origin) as P:
        assert all(P.plan(g, nu, nv)[0] == fp.KERNEL_TMA for g in geom)
        outs = [P.project(ta, geom, nu, nv).cpu().numpy(), P.project(tb, geom, nu, nv).cpu().numpy()]
        ta.copy_(tb)                                       # same pointer, new contents
        outs.append(P.project(ta, geom, nu, nv).cpu().numpy())
        mfl = P.ray_ranges(geom, nu, nv).cpu().numpy()
    for out, v in zip(outs, (va, vb, vb)):
        ov, om, pl, mg = oracle.project_rays(v, delta, origin, geom, ids)
        assert assert_parity(out.ravel(), mfl.reshape(-1, 3), ov, om, pl, mg, float(np.abs(v).max())) < 1.0
    assert np.array_equal(outs[1], outs[2])


@pytest.mark.parametrize("kernel_opt", ["tma", "aligned"])
def test_aligned_class_kernels_on_degenerate_grids_and_detectors(torch, fp, oracle, kernel_opt):
    """One-voxel-thick volumes along x or y, the smallest z extent the float4 / TMA paths take (nz = 4),
    1 x 1 and 1 x n detectors, poses on the axes and on the diagonals."""
    rng = np.random.default_rng(88)
    opt = fp.KERNEL_TMA if kernel_opt == "tma" else fp.KERNEL_ALIGNED
    for shape in [(1, 9, 8), (9, 1, 8), (5, 6, 4), (2, 2, 12)]:
        vol = rng.uniform(0.5, 1.5, size=shape).astype(np.float32)
        origin = tuple(-(n - 1) / 2.0 for n in shape)
        for nu, nv in [(1, 1), (1, 7), (9, 1), (12, 10)]:
            geom = np.stack([aligned_pose(th, 30.0, 60.0, nu, nv, 0.7, src_z=0.4)
                             for th in (0.0, math.pi / 4, math.pi / 2, 2.2, math.pi, 5.4977871)])
            with fp.Projector(*shape, 1.0, origin) as P:
                P.set_option(fp.OPT_KERNEL, opt)
                assert all(P.plan(g, nu, nv)[0] == opt for g in geom), (shape, nu, nv)
            worst, _, _ = compare_full(torch, fp, oracle, vol, 1.0, origin, geom, nu, nv,
                                       options=[(fp.OPT_KERNEL, opt)], what="%s %s %dx%d" % (kernel_opt, shape, nu, nv))
            assert worst < 1.0


@pytest.mark.parametrize("kernel_opt", ["tma", "aligned"])
def test_cylinder_field_of_view_option(torch, fp, oracle, kernel_opt):
    """FP_OPT_FOV_CYLINDER: for a volume that is zero outside the inscribed cylinder about z the clipped slice
    ranges give the same sums (only exact zeros are dropped; the batches start on other slices, so the fp32
    rounding of positions and the summation order differ) and match the oracle."""
    rng = np.random.default_rng(91)
    opt = fp.KERNEL_TMA if kernel_opt == "tma" else fp.KERNEL_ALIGNED
    shape, delta = (30, 26, 16), 1.0
    origin = tuple(-(n - 1) / 2.0 for n in shape)
    vol = rng.uniform(0.5, 1.5, size=shape).astype(np.float32)
    ix = np.arange(shape[0])[:, None, None] - 0.5 * (shape[0] - 1)
    iy = np.arange(shape[1])[None, :, None] - 0.5 * (shape[1] - 1)
    vol *= ((ix * ix + iy * iy) <= (0.5 * min(shape[0], shape[1])) ** 2)
    assert (vol == 0).mean() > 0.2
    nu, nv = 64, 20
    geom = np.stack([aligned_pose(th, 60.0, 120.0, nu, nv, 1.1, src_z=1.0, det_shift=(1.5, 0.0))
                     for th in np.linspace(0.0, 2 * math.pi, 13)[:-1]])
    volt = torch.from_numpy(vol).cuda()
    with fp.Projector(*shape, delta, origin) as P:
        P.set_option(fp.OPT_KERNEL, opt)
        assert all(P.plan(g, nu, nv)[0] == opt for g in geom)
        box = P.project(volt, geom, nu, nv).cpu().numpy()
        P.set_option(fp.OPT_FOV_CYLINDER, 1)
        assert P.get_option(fp.OPT_FOV_CYLINDER) == 1
        cyl = P.project(volt, geom, nu, nv).cpu().numpy()
        mfl = P.ray_ranges(geom, nu, nv).cpu().numpy()
    assert np.abs(box - cyl).max() <= 1e-5 * np.abs(box).max()
    assert np.array_equal(box == 0, cyl == 0)
    ids = all_ids(len(geom), nv, nu)
    ov, om, pl, mg = oracle.project_rays(vol, delta, origin, geom, ids, threads=oracle.host_cores())
    assert assert_parity(cyl.ravel(), mfl.reshape(-1, 3), ov, om, pl, mg, float(np.abs(vol).max())) < 1.0


# ----------------------------------------------------------------------------- host plan against the kernels' own checks

def aligned_pose2(theta, sid, sdd, nu, nv, pitch_u, pitch_v, src_z=0.0, det_shift=(0.0, 0.0), flip_u=False, flip_v=False):
    """aligned_pose with separate pixel pitches along u and v."""
    c, s = math.cos(theta), math.sin(theta)
    S = np.array([sid * c, sid * s, src_z])
    C = S - sdd * np.array([c, s, 0.0])
    U = pitch_u * np.array([-s, c, 0.0]) * (-1.0 if flip_u else 1.0)
    V = pitch_v * np.array([0.0, 0.0, 1.0]) * (-1.0 if flip_v else 1.0)
    O = C - ((nu - 1) / 2 + det_shift[0]) * U - ((nv - 1) / 2 + det_shift[1]) * V
    return np.concatenate([S, O, U, V])


def test_plan_overflow_is_reported_and_project_host_recovers(torch, fp, oracle):
    """A pose whose tiles do not fit fp_tma_kernel, sent there by the test hook: the kernel's bound check raises
    the flag, fp_check / fp_last_sample_count return FP_ERR_UNSUPPORTED (once: the read clears it), and
    fp_project_host repeats the call with the general-pose kernel and returns the right projections."""
    rng = np.random.default_rng(910)
    shape = (40, 36, 64)
    vol = rng.uniform(0.0, 1.0, size=shape).astype(np.float32)
    delta = 1.0
    origin = tuple(-(n - 1) / 2.0 * delta for n in shape)
    nu, nv = 16, 64
    # wide pixels along u: the eight columns of a block fan out over more than the 12 volume rows a tile holds
    geom = np.stack([aligned_pose2(0.6, 60.0, 120.0, nu, nv, 3.0, 1.0), aligned_pose2(0.75, 60.0, 120.0, nu, nv, 3.0, 1.0)])
    with fp.Projector(*shape, delta, origin) as P:
        assert all(P.plan(g, nu, nv)[0] == fp.KERNEL_ALIGNED for g in geom)
        vt = torch.from_numpy(vol).cuda()
        P.project(vt, geom, nu, nv)
        P.check()                                            # the default plan: nothing to report
        P.set_option(fp.OPT_TEST_FORCE_TMA, 1)
        P.project(vt, geom, nu, nv)
        with pytest.raises(fp.FpError) as e:
            P.check()
        assert e.value.status == 4                           # FP_ERR_UNSUPPORTED
        P.check()                                            # cleared by the read
        P.set_option(fp.OPT_COUNT_SAMPLES, 0)
        P.project(vt, geom, nu, nv)
        with pytest.raises(fp.FpError) as e:
            P.last_sample_count()                            # reported even when the call did not count
        assert e.value.status == 4
        # the end-to-end entry point notices and repeats the call with the direct kernel
        out = P.project_host(vol, geom, nu, nv)
        P.check()
    ids = all_ids(len(geom), nv, nu)
    ov, om, pl, mg = oracle.project_rays(vol, delta, origin, geom, ids, threads=oracle.host_cores())
    tol = 2e-5 * np.abs(ov) + 1e-6 * pl * float(np.abs(vol).max())
    assert np.all(np.abs(out.numpy().ravel().astype(np.float64) - ov) <= tol)


def phantom_like_volume(rng, shape):
    """The BASELINE recipe in miniature: a few overlapping random boxes with values in [0, 1] plus Gaussian noise
    of sigma 0.01 (flat regions, unit edges) -- unlike the uniform-noise volumes of the edge-case tests, whose
    voxel-to-voxel jumps are as large as max|voxel| everywhere."""
    v = rng.normal(0.0, 0.01, size=shape)
    for _ in range(6):
        lo = [int(rng.integers(0, n - 2)) for n in shape]
        hi = [int(rng.integers(l + 2, n + 1)) for l, n in zip(lo, shape)]
        v[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] += rng.uniform(0.0, 1.0)
    return v.astype(np.float32)


def test_random_aligned_poses_never_trip_the_kernels_bound_checks(torch, fp, oracle):
    """2400 random poses of the aligned class (source distance, magnification, pixel pitches, detector size and
    shifts, source height, both flips, volume shapes) through the default plan: the kernels' own window / row-tile
    checks must never fire (fp_check), every pose the plan gives to the TMA or aligned kernel included, and a
    sample of them is compared with the oracle ray by ray."""
    rng = np.random.default_rng(911)
    shapes = [(48, 40, 32), (33, 57, 64), (64, 64, 96), (20, 90, 44)]
    kernels_seen = set()
    n_checked = 0
    for si, shape in enumerate(shapes):
        vol = phantom_like_volume(rng, shape)
        delta = float(rng.uniform(0.4, 1.6))
        origin = tuple(-(n - 1) / 2.0 * delta + rng.uniform(-0.3, 0.3) for n in shape)
        vt = torch.from_numpy(vol).cuda()
        half = 0.5 * delta * math.hypot(shape[0], shape[1])
        with fp.Projector(*shape, delta, origin) as P:
            for q in range(600):
                nu, nv = int(rng.integers(1, 70)), int(rng.integers(1, 600))
                sid = half * float(rng.uniform(1.05, 12.0))
                sdd = sid * float(rng.uniform(1.05, 3.0))
                zext = shape[2] * delta
                pitch_v = zext * (sdd / sid) * float(rng.uniform(0.3, 2.5)) / nv
                pitch_u = 2 * half * (sdd / sid) * float(rng.uniform(0.2, 1.5)) / max(nu, 8)
                g = aligned_pose2(float(rng.uniform(0, 2 * math.pi)), sid, sdd, nu, nv, pitch_u, pitch_v,
                                  src_z=float(rng.uniform(-0.6, 0.6)) * zext,
                                  det_shift=(float(rng.uniform(-0.3, 0.3)) * nu, float(rng.uniform(-0.3, 0.3)) * nv),
                                  flip_u=bool(rng.integers(0, 2)), flip_v=bool(rng.integers(0, 2)))
                kernels_seen.add(P.plan(g, nu, nv)[0])
                out = P.project(vt, g[None], nu, nv)
                if q % 40 == 0:
                    P.check()
                    ids = all_ids(1, nv, nu)
                    ov, om, pl, mg = oracle.project_rays(vol, delta, origin, g[None], ids, threads=oracle.host_cores())
                    gm = P.ray_ranges(g[None], nu, nv).cpu().numpy().reshape(-1, 3)
                    worst = assert_parity(out.cpu().numpy().ravel(), gm, ov, om, pl, mg, float(np.abs(vol).max()),
                                          "random aligned pose %d/%d" % (si, q),
                                          recompute=make_recompute(oracle, vol, delta, origin, g[None], ids))
                    assert worst < 1.0
                    n_checked += 1
            P.check()
    assert fp.KERNEL_TMA in kernels_seen and fp.KERNEL_ALIGNED in kernels_seen
    assert n_checked >= 60


def test_output_pointer_that_is_only_four_byte_aligned(torch, fp, oracle):
    """out_dev one float past a 16-byte boundary: the aligned / TMA kernels must fall back to scalar stores
    (a float4 store there would fault)."""
    rng = np.random.default_rng(912)
    shape = (24, 20, 32)
    vol = rng.uniform(0.0, 1.0, size=shape).astype(np.float32)
    delta, nu, nv = 1.0, 16, 40
    origin = tuple(-(n - 1) / 2.0 * delta for n in shape)
    geom = np.stack([aligned_pose(t, 80.0, 160.0, nu, nv, 1.5) for t in (0.1, 0.8, 2.0)])
    vt = torch.from_numpy(vol).cuda()
    buf = torch.zeros(len(geom) * nv * nu + 1, device="cuda", dtype=torch.float32)
    view = buf[1:].view(len(geom), nv, nu)
    assert view.data_ptr() % 16 == 4
    with fp.Projector(*shape, delta, origin) as P:
        for kern in (fp.KERNEL_AUTO, fp.KERNEL_ALIGNED):
            P.set_option(fp.OPT_KERNEL, kern)
            ref = P.project(vt, geom, nu, nv)
            got = P.project(vt, geom, nu, nv, out=view)
            torch.cuda.synchronize()
            assert torch.equal(ref, got)
            P.check()
    assert float(buf[0]) == 0.0


# ----------------------------------------------------------------------------- texture pipe: explicit weights and GJP_hwlin

def test_texture_kernel_parity_all_axes(torch, fp, synth, oracle):
    """FP_KERNEL_TEX: one tld4 per sample from the layered arrays of the layout stage, explicit fp32 weights --
    the same sums as every other kernel, inside the tolerance, on C1 and on general poses with all three axes."""
    cfg = synth.CONFIGS["C1"]
    worst, _, _ = compare_full(torch, fp, oracle, synth.make_volume(cfg).numpy(), cfg.voxel_size, cfg.origin,
                               synth.make_geometry(cfg), cfg.nu, cfg.nv, options=[(fp.OPT_KERNEL, fp.KERNEL_TEX)], what="C1 tex")
    assert worst < 1.0
    rng = np.random.default_rng(701)
    vol, delta, origin = small_problem(rng)
    nu, nv = 37, 29
    geom = np.stack([pose(s, (0.2, -0.1, 0.3), nu, nv, 0.5, 60.0, roll)
                     for s, roll in [((-30, 2, 1), 0.0), ((1, 28, -3), 0.4), ((2, -1, 31), 1.1), ((-14, -15, 16), 2.0)]])
    worst, _, om = compare_full(torch, fp, oracle, vol, delta, origin, geom, nu, nv,
                                options=[(fp.OPT_KERNEL, fp.KERNEL_TEX)], what="tex general")
    assert worst < 1.0 and set(np.unique(om[:, 0])) == {0, 1, 2}


def test_hwlin_hardware_filtering_error_is_recorded(torch, fp, synth, oracle, capsys):
    """GJP_hwlin (PAPER.md:215 sec. 2.6, :330 Table 1): one hardware-filtered fetch per sample.  The texture unit
    interpolates with 8-bit fixed-point weights, so the result is NOT expected inside the 2e-5 tolerance: the
    test measures the error against the oracle on C1 and C2, prints it (DESIGN.md quotes it), and checks only
    that it is the size 8-bit weights give -- well above the tolerance, well below 1 % of the largest ray sum."""
    report = {}
    for name, projs in (("C1", None), ("C2", [0, 23, 45, 90, 158])):
        cfg = synth.CONFIGS[name]
        vol = synth.make_volume(cfg).numpy()
        geom = synth.make_geometry(cfg)
        if projs is not None:
            geom = geom[projs]
        out, mfl, _ = run_gpu(torch, fp, vol, cfg.voxel_size, cfg.origin, geom, cfg.nu, cfg.nv,
                              options=[(fp.OPT_KERNEL, fp.KERNEL_HWLIN)])
        ids = all_ids(len(geom), cfg.nv, cfg.nu)
        ov, om, pl, mg = oracle.project_rays(vol, cfg.voxel_size, cfg.origin, geom, ids, threads=oracle.host_cores())
        assert np.array_equal(mfl.reshape(-1, 3), om)                  # the set-up is the exact one
        g = out.ravel().astype(np.float64)
        assert np.all(np.isfinite(g))
        tol = 2e-5 * np.abs(ov) + 1e-6 * pl * float(np.abs(vol).max())
        hit = om[:, 2] >= om[:, 1]
        ratio = float(np.max(np.abs(g - ov)[hit] / tol[hit]))
        rel = float(np.max(np.abs(g - ov)[hit]) / np.abs(ov).max())     # against the largest ray sum
        report[name] = (ratio, rel)
        assert np.all(g[~hit] == 0.0)
        assert 1.0 < ratio < 1e4 and rel < 1e-2, (name, ratio, rel)
    with capsys.disabled():
        print("\nGJP_hwlin error vs oracle: " + ", ".join(
            "%s worst err/tol %.1f (worst error / largest ray sum %.2e)" % (k, v[0], v[1]) for k, v in report.items()))


# ----------------------------------------------------------------------------- SART with the matched pair

def test_sart_ten_iterations_residual_falls_and_matches_the_oracle_loop(torch, fp, synth, oracle):
    """"10 SART iterations".  Simulated projections of the C1 phantom, x_0 = 0, lambda = 1: the
    weighted residual falls monotonically, the reconstruction approaches the phantom, and the whole loop agrees
    with the same ten updates run on the fp64 oracle (forward and back-projection oracles, numpy for the rest)."""
    from paper_1609_00958_b200 import sart
    cfg = synth.CONFIGS["C1"]
    x_true = synth.make_volume(cfg)
    geom = synth.make_geometry(cfg)
    th = oracle.host_cores()
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        y = P.project(x_true.cuda(), geom, cfg.nu, cfg.nv)
        x, res = sart.sart(P, y, geom, cfg.nu, cfg.nv, n_iter=10, lam=1.0)
        P.check()
    assert len(res) == 11 and all(b < a for a, b in zip(res, res[1:])), res
    assert res[-1] < 0.2 * res[0]
    err0 = float(x_true.norm())
    assert float((x.cpu() - x_true).norm()) < 0.6 * err0
    # the same loop on the oracle
    yo = y.cpu().numpy().astype(np.float64)
    ones_v = np.ones(cfg.n, dtype=np.float32)
    row, _, _ = oracle.project(ones_v, cfg.voxel_size, cfg.origin, geom, cfg.nu, cfg.nv, threads=th)
    col = oracle.backproject(np.ones_like(yo), cfg.n, cfg.voxel_size, cfg.origin, geom, threads=th)
    inv_row = np.where(row > 1e-6, 1.0 / np.maximum(row, 1e-6), 0.0)
    inv_col = np.where(col > 1e-6, 1.0 / np.maximum(col, 1e-6), 0.0)
    xo = np.zeros(cfg.n, dtype=np.float64)
    res_o = []
    for _ in range(10):
        ax, _, _ = oracle.project(xo.astype(np.float32), cfg.voxel_size, cfg.origin, geom, cfg.nu, cfg.nv, threads=th)
        r = yo - ax
        res_o.append(math.sqrt(float((r ** 2 * inv_row).sum())))
        xo += oracle.backproject(r * inv_row, cfg.n, cfg.voxel_size, cfg.origin, geom, threads=th) * inv_col
    assert np.allclose(res[:10], res_o, rtol=2e-4)
    assert float(np.abs(x.cpu().numpy() - xo).max()) < 2e-4 * float(np.abs(xo).max())
