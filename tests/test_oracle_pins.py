"""Pins of the fp64 oracle against what the paper and the mathematics fix.

No printed worked example exists in the paper, so the oracle is
pinned by closed forms, invariants, an independent library routine (scipy's
trilinear interpolation), brute force of the plain definition on tiny inputs and a
hand-worked example (tests/golden/hand_example.txt).  Each test names the passage
it checks and the kind of mistake it would catch.
"""
import itertools
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def rand_vol(rng, shape=(7, 6, 5)):
    return rng.uniform(-1.0, 2.0, size=shape).astype(np.float32)


def rays_through(rng, shape, n, spread=1.6, axis=None):
    """Random source/detector pairs (grid coordinates) aimed at a box around the volume;
    ``spread`` > 1 produces grazing and missing rays as well."""
    N = np.array(shape, dtype=np.float64)
    c = (N - 1) / 2.0
    out = []
    for _ in range(n):
        a = rng.integers(0, 3) if axis is None else axis
        tgt0 = c + (rng.uniform(-0.5, 0.5, 3) * spread) * (N + 1)
        tgt1 = c + (rng.uniform(-0.5, 0.5, 3) * spread) * (N + 1)
        s = tgt0.copy()
        d = tgt1.copy()
        s[a] = -rng.uniform(3.0, 40.0)
        d[a] = N[a] + rng.uniform(3.0, 40.0)
        if rng.random() < 0.5:
            s, d = d, s
        out.append((s, d))
    return out


# ---------------------------------------------------------------- whole operator

@pytest.mark.parametrize("kernel", [0, 1])
def test_stepwise_equals_plain_definition(oracle, kernel):
    """step-by-step form == triple-sum definition (no floor / clipping / ranges).
    Catches: wrong tap offsets, swapped weights, wrong in-volume predicate, lost boundary taps."""
    rng = np.random.default_rng(11)
    vol = rand_vol(rng)
    seen_axes, n_miss, n_graze = set(), 0, 0
    for s, d in rays_through(rng, vol.shape, 400):
        r = oracle.ray_grid(vol, s, d, kernel)
        ref = oracle.ray_definition(vol, s, d, kernel)
        assert abs(r["value"] - ref) <= 1e-13 * max(1.0, abs(ref))
        seen_axes.add(r["m"])
        n_miss += r["i_last"] < r["i_first"]
        n_graze += 0 <= (r["i_last"] - r["i_first"]) < 3
    assert seen_axes == {0, 1, 2} and n_miss > 10 and n_graze > 5


def test_hand_worked_example(oracle):
    """tests/golden/hand_example.txt: a 3x2x2 volume and one ray worked by hand from
    Eqs. 1-6, 13.  Catches a wrong step weight or offset o."""
    kv = {}
    with open(os.path.join(GOLDEN, "hand_example.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                kv[k.strip()] = v.strip()
    nx, ny, nz = (int(x) for x in kv["shape"].split())
    vol = np.zeros((nx, ny, nz), dtype=np.float32)
    for i, j, k in itertools.product(range(nx), range(ny), range(nz)):
        vol[i, j, k] = 1 + i + 10 * j + 100 * k
    s = [float(x) for x in kv["s"].split()]
    d = [float(x) for x in kv["d"].split()]
    expect = float(kv["sum_of_samples"]) * math.sqrt(float(kv["L_squared"]))
    r = oracle.ray_grid(vol, s, d)
    assert (r["m"], r["i_first"], r["i_last"]) == (0, 0, 2)
    assert abs(r["L"] - math.sqrt(17.0) / 4.0) < 1e-15
    assert abs(r["value"] - expect) < 1e-12
    # same ray through the world-unit entry point with voxel pitch 2 and a shifted origin
    delta, origin = 2.0, np.array([5.0, -3.0, 7.0])
    S = np.array(s) * delta + origin
    D = np.array(d) * delta + origin
    geom = np.concatenate([S, D, [0, 0.1, 0], [0, 0, 0.1]])[None, :]
    val, mfl, pl, _ = oracle.project_rays(vol, delta, origin, geom, np.array([[0, 0, 0]], dtype=np.int32))
    assert abs(val[0] - delta * expect) < 1e-11
    assert abs(pl[0] - delta * math.sqrt(17.0) / 4.0 * 3) < 1e-12


# ------------------------------------------------------ north_star (a): tap / weight logic

def test_axis_aligned_rays_through_voxel_centres_bit_exact(oracle):
    """north_star (a): an axis-aligned ray through voxel centres returns exactly the
    pitch-weighted sum of the voxels on the line (integer data => bit exact)."""
    rng = np.random.default_rng(5)
    shape = (6, 5, 4)
    vol = rng.integers(-8, 9, size=shape).astype(np.float32)
    for m in range(3):
        t1, t2 = (m + 1) % 3, (m + 2) % 3
        for j in range(shape[t1]):
            for k in range(shape[t2]):
                for sign in (+1, -1):
                    s = np.zeros(3)
                    d = np.zeros(3)
                    s[t1] = d[t1] = j
                    s[t2] = d[t2] = k
                    s[m], d[m] = (-9.0, 20.0) if sign > 0 else (20.0, -9.0)
                    r = oracle.ray_grid(vol, s, d)
                    line = np.take(np.take(vol, j, axis=t1), k, axis=t2 - 1 if t2 > t1 else t2)
                    assert r["value"] == float(line.astype(np.float64).sum())
                    assert (r["m"], r["i_first"], r["i_last"], r["L"]) == (m, 0, shape[m] - 1, 1.0)


# ------------------------------------------- north_star (b): step weight and slice count

def test_constant_volume_gives_chord_length(oracle):
    """north_star (b): constant volume c, ray entering and leaving through the m-faces with
    every sample at 0 <= p_t <= N_t-1  =>  c * delta * ||r~|| * N_m = c * chord through the
    slab [-1/2, N_m - 1/2] (samples every ||r~||; reading #11)."""
    rng = np.random.default_rng(6)
    shape = (9, 8, 10)
    c = 0.75
    vol = np.full(shape, c, dtype=np.float32)
    N = np.array(shape, float)
    for m in range(3):
        t1, t2 = (m + 1) % 3, (m + 2) % 3
        for _ in range(50):
            # choose entry / exit points on slices 0 and N_m-1 well inside the transverse range
            a = np.zeros(3)
            b = np.zeros(3)
            a[m], b[m] = 0.0, N[m] - 1
            for t in (t1, t2):
                a[t] = rng.uniform(0, N[t] - 1)
                b[t] = rng.uniform(max(0, a[t] - (N[m] - 1) * 0.99), min(N[t] - 1, a[t] + (N[m] - 1) * 0.99))
            dirv = b - a
            s = a - 3.7 * dirv
            d = b + 2.2 * dirv
            r = oracle.ray_grid(vol, s, d)
            assert r["m"] == m and (r["i_first"], r["i_last"]) == (0, shape[m] - 1)
            # geometric chord of the line through the slab, computed independently
            unit = dirv / np.linalg.norm(dirv)
            chord = N[m] / abs(unit[m])
            assert abs(r["value"] - c * chord) < 1e-10
            assert 1.0 <= r["L"] <= math.sqrt(3.0) + 1e-15
            delta = 0.4
            origin = np.array([1.0, 2.0, 3.0])
            geom = np.concatenate([s * delta + origin, d * delta + origin, [0.1, 0, 0], [0, 0.1, 0]])[None]
            val, _, pl, _ = oracle.project_rays(vol, delta, origin, geom, np.zeros((1, 3), np.int32))
            assert abs(val[0] - c * delta * chord) < 1e-10 and abs(pl[0] - delta * chord) < 1e-10


def test_side_face_clipping_within_boundary_half_voxel(oracle):
    """north_star (b), second half ("up to the boundary half-voxel"): with zero padding (reading #2)
    the per-sample weight of a constant volume lies between the indicators of the transverse boxes
    [0, N_t-1] and (-1, N_t), i.e. half a voxel inside / outside the geometric faces at -1/2 and
    N_t-1/2.  Hence  L (l_in - 1) <= value <= L (l_out + 1)  with l the chord, in driving-axis
    units, of the line through slab_m [-1/2, N_m-1/2] x that transverse box."""
    rng = np.random.default_rng(7)
    shape = (12, 11, 10)
    vol = np.ones(shape, dtype=np.float32)
    N = np.array(shape, float)
    n_side = 0

    def chord_in_m_units(s, r, m, lo, hi):
        with np.errstate(divide="ignore", invalid="ignore"):
            ta, tb = (lo - s) / r, (hi - s) / r
        ta, tb = np.where(r == 0, np.where((s >= lo) & (s <= hi), -np.inf, np.inf), ta), \
            np.where(r == 0, np.where((s >= lo) & (s <= hi), np.inf, -np.inf), tb)
        t0, t1 = np.max(np.minimum(ta, tb)), np.min(np.maximum(ta, tb))
        return max(0.0, t1 - t0) * abs(r[m])

    for s, d in rays_through(rng, shape, 600, spread=2.4):
        g = oracle.ray_grid(vol, s, d)
        r = d - s
        m = int(np.argmax(np.abs(r)))
        lo_in, hi_in = np.zeros(3), N - 1.0
        lo_out, hi_out = -np.ones(3), N.copy()
        for b in (lo_in, lo_out):
            b[m] = -0.5
        for b in (hi_in, hi_out):
            b[m] = N[m] - 0.5
        l_in = chord_in_m_units(s, r, m, lo_in, hi_in)
        l_out = chord_in_m_units(s, r, m, lo_out, hi_out)
        L = np.linalg.norm(r / r[m])
        assert L * (l_in - 1.0) - 1e-9 <= g["value"] <= L * (l_out + 1.0) + 1e-9
        hit = g["i_last"] >= g["i_first"]
        n_side += hit and (g["i_first"] > 0 or g["i_last"] < shape[m] - 1)
        if hit:   # number of visited slices agrees with the outer chord to within one per end
            assert abs((g["i_last"] - g["i_first"] + 1) - l_out) <= 1.0 + 1e-9
    assert n_side > 30


# ------------------------------------------------------------------ interpolation closed form

@pytest.mark.parametrize("m", [0, 1, 2])
def test_bilinear_closed_form(oracle, m):
    """vol = h(i) (a + b j + c k + e j k) is reproduced exactly by bilinear interpolation, so an
    interior ray gives ||r~|| sum_i h(i) (a + b p1 + c p2 + e p1 p2) with p_t(i) from Eq. 6
    (PAPER.md:104, :150).  Catches wrong fractional weights and transposed taps.  All
    coefficients are dyadic so the fp32 volume holds the function exactly."""
    rng = np.random.default_rng(20 + m)
    t1, t2 = (m + 1) % 3, (m + 2) % 3
    shape = [0, 0, 0]
    shape[m], shape[t1], shape[t2] = 8, 30, 28
    h = rng.integers(4, 13, size=shape[m]) / 8.0
    a, b, c, e = 0.25, -0.125, 0.0625, 1.0 / 64
    idx = np.indices(shape)
    vol = h[idx[m]] * (a + b * idx[t1] + c * idx[t2] + e * idx[t1] * idx[t2])
    vol32 = vol.astype(np.float32)
    assert np.array_equal(vol32.astype(np.float64), vol)
    for _ in range(40):
        s = np.zeros(3)
        d = np.zeros(3)
        s[m], d[m] = -rng.uniform(5, 30), shape[m] + rng.uniform(5, 30)
        for t in (t1, t2):
            s[t] = rng.uniform(10, 17)
            d[t] = s[t] + rng.uniform(-0.15, 0.15) * (d[m] - s[m])
        if rng.random() < 0.5:
            s, d = d, s
        r = d - s
        rt = r / r[m]
        L = np.linalg.norm(rt)
        i = np.arange(shape[m], dtype=np.float64)
        p1 = s[t1] + (i - s[m]) * rt[t1]
        p2 = s[t2] + (i - s[m]) * rt[t2]
        # samples stay strictly inside [1, N_t - 2]: no zero padding is touched
        assert p1.min() > 1 and p1.max() < shape[t1] - 2 and p2.min() > 1 and p2.max() < shape[t2] - 2
        expect = L * np.sum(h * (a + b * p1 + c * p2 + e * p1 * p2))
        got = oracle.ray_grid(vol32, s, d)
        assert got["m"] == m and (got["i_first"], got["i_last"]) == (0, shape[m] - 1)
        assert abs(got["value"] - expect) < 1e-12 * abs(expect)


def test_single_voxel_footprint(oracle):
    """A unit impulse at voxel (a,b,c) projects to ||r~|| * hat(p_t1(a_m) - b) * hat(p_t2(a_m) - c):
    the box (x) box footprint of PAPER.md:187 convolved to the hat of Eq. 13."""
    rng = np.random.default_rng(8)
    shape = (7, 6, 5)
    for _ in range(300):
        pos = [int(rng.integers(0, n)) for n in shape]
        vol = np.zeros(shape, dtype=np.float32)
        vol[tuple(pos)] = 1.0
        (s, d), = rays_through(rng, shape, 1, spread=1.0)
        r = oracle.ray_grid(vol, s, d)
        m = r["m"]
        rr = d - s
        rt = rr / rr[m]
        val = np.linalg.norm(rt)
        for t in ((m + 1) % 3, (m + 2) % 3):
            p = s[t] + (pos[m] - s[m]) * rt[t]
            val *= max(0.0, 1.0 - abs(p - pos[t]))
        assert abs(r["value"] - val) < 1e-14
        # spline kernel: H(x) = 1 - 3x^2 + 2|x|^3  (Eq. 14)
        vs = np.linalg.norm(rt)
        for t in ((m + 1) % 3, (m + 2) % 3):
            x = abs(s[t] + (pos[m] - s[m]) * rt[t] - pos[t])
            vs *= (1 - 3 * x * x + 2 * x ** 3) if x < 1 else 0.0
        assert abs(oracle.ray_grid(vol, s, d, 1)["value"] - vs) < 1e-14


# ------------------------------------------------------------------- invariants (c), (d), (e)

def test_linearity(oracle):
    """north_star (c): P(alpha A + beta B) = alpha P(A) + beta P(B)."""
    rng = np.random.default_rng(9)
    A = rng.integers(-4, 5, size=(7, 6, 5)).astype(np.float32)
    B = rng.integers(-4, 5, size=(7, 6, 5)).astype(np.float32)
    al, be = 3.0, -2.0                       # exact in fp32
    C = (al * A + be * B).astype(np.float32)
    for s, d in rays_through(rng, A.shape, 100):
        pa, pb, pc = (oracle.ray_grid(v, s, d)["value"] for v in (A, B, C))
        assert abs(pc - (al * pa + be * pb)) < 1e-12 * (1 + abs(pa) + abs(pb))


def test_axis_permutation_and_mirror_symmetry(oracle):
    """north_star (d): the algorithm is driving-axis agnostic: permuting the
    volume axes together with the geometry components, or mirroring one axis (voxel j -> N-1-j,
    coordinate y -> N-1-y), leaves every ray sum unchanged.  Catches per-axis stride/index slips."""
    rng = np.random.default_rng(10)
    vol = rand_vol(rng, (7, 6, 5))
    rays = rays_through(rng, vol.shape, 60)
    for perm in itertools.permutations(range(3)):
        pv = np.ascontiguousarray(np.transpose(vol, perm))
        for s, d in rays:
            r = d - s
            ar = np.sort(np.abs(r))
            if ar[2] - ar[1] < 1e-6:
                continue                      # tie-break is not permutation invariant (reading #8)
            base = oracle.ray_grid(vol, s, d)
            got = oracle.ray_grid(pv, s[list(perm)], d[list(perm)])
            assert abs(got["value"] - base["value"]) < 1e-13 * (1 + abs(base["value"]))
            assert perm[got["m"]] == base["m"]
            assert (got["i_first"], got["i_last"]) == (base["i_first"], base["i_last"])
    for ax in range(3):
        mv = np.ascontiguousarray(np.flip(vol, axis=ax))
        for s, d in rays:
            s2, d2 = s.copy(), d.copy()
            s2[ax] = vol.shape[ax] - 1 - s[ax]
            d2[ax] = vol.shape[ax] - 1 - d[ax]
            base = oracle.ray_grid(vol, s, d)
            got = oracle.ray_grid(mv, s2, d2)
            assert abs(got["value"] - base["value"]) < 1e-12 * (1 + abs(base["value"]))
            assert got["m"] == base["m"]


@pytest.mark.parametrize("m", [0, 1, 2])
def test_mass_conservation_parallel_rays(oracle, m):
    """north_star (e): partition of unity (Eq. 8) + zero padding (reading #2):
    parallel rays on a unit lattice in the plane perpendicular to m, with ANY fractional offset and
    covering (-1, N), sum to  ||r~|| * sum(vol)  (axis-aligned: ||r~|| = 1)."""
    rng = np.random.default_rng(30 + m)
    shape = (6, 7, 5)
    vol = rand_vol(rng, shape)
    t1, t2 = (m + 1) % 3, (m + 2) % 3
    total = float(vol.astype(np.float64).sum())
    for slope in ((0.0, 0.0), (0.31, -0.22), (-0.9, 0.77)):
        f1, f2 = rng.uniform(0, 1, 2)
        direction = np.zeros(3)
        direction[m], direction[t1], direction[t2] = 1.0, slope[0], slope[1]
        L = np.linalg.norm(direction)
        acc = 0.0
        reach = int(shape[m] * max(abs(slope[0]), abs(slope[1]))) + 3
        for j in range(-reach - 1, shape[t1] + reach + 1):
            for k in range(-reach - 1, shape[t2] + reach + 1):
                base = np.zeros(3)
                base[t1], base[t2] = j + f1, k + f2        # position on slice m = 0
                s = base - 25.0 * direction
                d = base + 40.0 * direction
                acc += oracle.ray_grid(vol, s, d)["value"]
        assert abs(acc - L * total) < 1e-10 * max(1.0, abs(total))


# ------------------------------------------------------------------- library routine pin

def test_against_scipy_trilinear(oracle):
    """PAPER.md:155 footnote: tri-linear interpolation at p(i) is identical to the 2x2 bilinear
    form because p_m is integer.  scipy.ndimage.map_coordinates(order=1) on the zero-padded volume
    is an independent implementation of the per-sample value."""
    from scipy.ndimage import map_coordinates
    rng = np.random.default_rng(12)
    vol = rand_vol(rng, (9, 7, 8))
    pad = 3
    vp = np.pad(vol.astype(np.float64), pad)
    for s, d in rays_through(rng, vol.shape, 150, spread=1.3):
        r = d - s
        m = int(np.argmax(np.abs(r)))
        rt = r / r[m]
        i = np.arange(vol.shape[m], dtype=np.float64)
        pts = s[:, None] + (i - s[m])[None, :] * rt[:, None]
        pts[m] = i
        ok = np.ones_like(i, dtype=bool)
        for t in range(3):
            if t != m:
                ok &= (pts[t] > -1) & (pts[t] < vol.shape[t])
        vals = map_coordinates(vp, pts[:, ok] + pad, order=1, mode="nearest")
        expect = np.linalg.norm(rt) * vals.sum()
        got = oracle.ray_grid(vol, s, d)
        assert abs(got["value"] - expect) < 1e-12 * (1 + abs(expect))
        if ok.any():
            assert (got["i_first"], got["i_last"]) == (int(i[ok][0]), int(i[ok][-1]))
        else:
            assert got["i_last"] < got["i_first"]


def test_dense_quadrature_of_the_voxel_model(oracle):
    """north_star (f): dense midpoint quadrature of the line integral of the model
    "nearest slice along m x zero-padded bilinear in the slice plane".  Joseph's sum is the
    one-point-per-slab midpoint rule of that integral, exact when the volume is affine in the
    transverse coordinates, otherwise close (loose tolerance)."""
    from scipy.ndimage import map_coordinates
    rng = np.random.default_rng(13)
    shape = (7, 6, 5)
    nq = 40000
    for affine in (True, False):
        if affine:
            idx = np.indices(shape)
            vol = (0.2 + 0.05 * idx[0] + 0.03 * idx[1] - 0.02 * idx[2]).astype(np.float32)
        else:
            vol = rand_vol(rng, shape)
        vp = np.pad(vol.astype(np.float64), 3)
        for s, d in rays_through(rng, shape, 12, spread=0.5):
            r = d - s
            m = int(np.argmax(np.abs(r)))
            rt = r / r[m]
            xm = -0.5 + (np.arange(nq * shape[m]) + 0.5) / nq        # dense positions along m
            pts = s[:, None] + (xm - s[m])[None, :] * rt[:, None]
            pts[m] = np.round(xm)                                     # nearest slice
            vals = map_coordinates(vp, pts + 3, order=1, mode="nearest")
            integral = np.linalg.norm(rt) * vals.sum() / nq
            got = oracle.ray_grid(vol, s, d)["value"]
            if affine and got != 0.0:
                # interior rays of an affine volume: the midpoint rule is exact; rays touching the
                # zero padding are not affine there, allow the loose bound
                tol = 1e-3
            else:
                tol = 2e-2
            assert abs(got - integral) <= tol * max(1.0, abs(integral))


# ------------------------------------------------------------------- set-up decisions

def test_driving_axis_ties_go_to_lowest_index(oracle):
    """Eq. 2 with reading #8."""
    vol = np.ones((4, 4, 4), dtype=np.float32)
    s = np.array([-5.0, -5.0, -2.0])
    assert oracle.ray_grid(vol, s, s + np.array([10.0, 10.0, 3.0]))["m"] == 0
    assert oracle.ray_grid(vol, s, s + np.array([10.0, -10.0, 10.0]))["m"] == 0
    assert oracle.ray_grid(vol, s, s + np.array([3.0, 10.0, 10.0]))["m"] == 1
    assert oracle.ray_grid(vol, s, s + np.array([3.0, 9.0, -10.0]))["m"] == 2
    z = oracle.ray_grid(vol, s, s)
    assert z["value"] == 0.0 and z["i_last"] < z["i_first"]


def test_entry_exit_indices_are_the_extreme_inside_slices(oracle):
    """Alg. 1 l.8 replaced by exact entry/exit: i_first / i_last are the least /
    greatest i with -1 < p_t(i) < N_t for both transverse axes; the set is an interval."""
    rng = np.random.default_rng(14)
    shape = (15, 9, 12)
    vol = np.ones(shape, dtype=np.float32)
    for s, d in rays_through(rng, shape, 300, spread=1.4):
        g = oracle.ray_grid(vol, s, d)
        m = g["m"]
        r = d - s
        rt = r / r[m]
        inside = []
        for i in range(shape[m]):
            ok = True
            for t in range(3):
                if t != m:
                    p = s[t] + (float(i) - s[m]) * rt[t]
                    ok &= (-1.0 < p < shape[t])
            inside.append(ok)
        where = np.flatnonzero(inside)
        if len(where) == 0:
            assert (g["i_first"], g["i_last"]) == (0, -1)
        else:
            assert (g["i_first"], g["i_last"]) == (where[0], where[-1])
            assert len(where) == where[-1] - where[0] + 1


def test_projection_level_equals_ray_level(oracle):
    """Geometry plumbing: pixel (iu, iv) centre = det_origin + iu*u + iv*v, world -> grid by
    (x - origin) / delta (PAPER.md:57 Fig. 1, :63); block, list and whole-projection entry
    points agree with the ray-level routine."""
    from paper_1609_00958_b200 import synth
    rng = np.random.default_rng(15)
    vol = rand_vol(rng, (10, 9, 8))
    delta = 0.7
    origin = np.array([-(n - 1) / 2 * delta for n in vol.shape]) + np.array([0.3, -0.2, 0.1])
    geom = synth.random_poses(3, 20.0, 33.0, 7, 5, 0.9, rng)
    vals, mfl, pl = oracle.project(vol, delta, origin, geom, 7, 5, threads=2)
    ids = np.array([(p, iv, iu) for p in range(3) for iv in range(5) for iu in range(7)], dtype=np.int32)
    v2, m2, p2, _ = oracle.project_rays(vol, delta, origin, geom, ids, threads=2)
    assert np.array_equal(vals.ravel(), v2) and np.array_equal(mfl.reshape(-1, 3), m2)
    assert np.array_equal(pl.ravel(), p2)
    for (p, iv, iu), v, mm in zip(ids, v2, m2):
        D = geom[p, 3:6] + iu * geom[p, 6:9] + iv * geom[p, 9:12]
        s = (geom[p, 0:3] - origin) / delta
        d = (D - origin) / delta
        g = oracle.ray_grid(vol, s, d)
        assert abs(v - delta * g["value"]) < 1e-12 * (1 + abs(v))
        assert tuple(mm) == (g["m"], g["i_first"], g["i_last"])
    assert np.count_nonzero(v2) > 20


def test_golden_regression(oracle):
    """tests/golden/oracle_regression.txt is written by tests/golden/make_golden.py, which calls
    only oracle/ -- guards the oracle against silent drift."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLDEN, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    lines = mg.compute_lines()
    with open(os.path.join(GOLDEN, "oracle_regression.txt")) as f:
        stored = [ln.rstrip("\n") for ln in f if not ln.startswith("#")]
    assert len(stored) == len(lines)
    for a, b in zip(stored, lines):
        fa, fb = a.split(), b.split()
        assert fa[:6] == fb[:6]
        assert abs(float(fa[6]) - float(fb[6])) <= 1e-12 * max(1.0, abs(float(fa[6])))


# ----------------------------------------------------------------------------- back-projection oracle

def _bp_poses(shape, delta, nu, nv):
    """Three poses whose rays are x-, y- and z-driven, detector slightly larger than the volume's shadow."""
    ctr = np.zeros(3)
    poses = []
    for src, u, v in [((-40.0, 3.0, 2.0), (0.0, 1.0, 0.1), (0.0, -0.1, 1.0)),
                      ((2.0, 38.0, -3.0), (1.0, 0.0, 0.2), (-0.2, 0.0, 1.0)),
                      ((3.0, -2.0, 41.0), (1.0, 0.15, 0.0), (-0.15, 1.0, 0.0))]:
        S = np.array(src)
        n = (ctr - S) / np.linalg.norm(ctr - S)
        C = S + 70.0 * n
        U = 0.9 * np.array(u) / np.linalg.norm(u)
        V = 0.9 * np.array(v) / np.linalg.norm(v)
        poses.append(np.concatenate([S, C - (nu - 1) / 2 * U - (nv - 1) / 2 * V, U, V]))
    return np.stack(poses)


@pytest.mark.parametrize("kernel", [0, 1])
def test_backprojection_is_the_transpose_voxel_by_voxel(oracle, kernel):
    """(A^T y)[v] = <A e_v, y> for EVERY voxel v of a tiny grid: the back-projection oracle against the
    pinned forward oracle applied to unit volumes (the definition of the transpose, nothing shared but
    the ray set-up)."""
    rng = np.random.default_rng(71)
    shape, delta, nu, nv = (4, 5, 3), 0.8, 9, 8
    origin = tuple(-(n - 1) / 2.0 * delta + 0.1 * k for k, n in enumerate(shape))
    geom = _bp_poses(shape, delta, nu, nv)
    y = rng.uniform(-1.0, 2.0, size=(len(geom), nv, nu))
    bp = oracle.backproject(y, shape, delta, origin, geom, kernel=kernel)
    assert bp.shape == shape
    seen_axes = set()
    for v in itertools.product(*[range(n) for n in shape]):
        e = np.zeros(shape, dtype=np.float32)
        e[v] = 1.0
        fwd, mfl, _ = oracle.project(e, delta, origin, geom, nu, nv, kernel=kernel)
        seen_axes |= set(np.unique(mfl[..., 0]))
        assert abs(bp[v] - float((fwd * y).sum())) <= 1e-12 * max(1.0, abs(bp[v])), v
    assert seen_axes == {0, 1, 2}
    assert np.abs(bp).max() > 0.1


def test_backprojection_adjoint_identity_and_linearity(oracle):
    rng = np.random.default_rng(72)
    shape, delta, nu, nv = (11, 9, 12), 0.7, 21, 17
    origin = tuple(-(n - 1) / 2.0 * delta for n in shape)
    geom = _bp_poses(shape, delta, nu, nv)
    x = rng.uniform(-1.0, 1.0, size=shape).astype(np.float32)
    y1 = rng.uniform(-1.0, 1.0, size=(len(geom), nv, nu))
    y2 = rng.uniform(-1.0, 1.0, size=(len(geom), nv, nu))
    ax, _, _ = oracle.project(x, delta, origin, geom, nu, nv)
    b1 = oracle.backproject(y1, shape, delta, origin, geom)
    b2 = oracle.backproject(y2, shape, delta, origin, geom, threads=3)
    lhs, rhs = float((ax * y1).sum()), float((x.astype(np.float64) * b1).sum())
    assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), 1.0)
    b12 = oracle.backproject(2.0 * y1 - 3.0 * y2, shape, delta, origin, geom)
    assert np.allclose(b12, 2.0 * b1 - 3.0 * b2, rtol=0, atol=1e-11)
    # weights are non-negative: a non-negative projection back-projects to a non-negative volume,
    # and <A 1, y> = sum(A^T y)
    ones = np.ones(shape, dtype=np.float32)
    a1, _, _ = oracle.project(ones, delta, origin, geom, nu, nv)
    bp = oracle.backproject(np.abs(y1), shape, delta, origin, geom)
    assert bp.min() >= 0.0
    assert abs(float((a1 * np.abs(y1)).sum()) - float(bp.sum())) <= 1e-10 * float(bp.sum())


# ---------------------------------------------------------------- given-axis rays (reading #8) and voxel-list transpose

def test_given_axis_equals_chosen_axis_and_axis_swap_on_ties(oracle):
    """jo_ray_grid_axis is pinned without calling itself twice: (1) with the axis Eq. 2 chooses it returns the
    bits of the pinned jo_ray_grid; (2) on an EXACT tie |r_x| = |r_y| the sum along y equals the chosen-axis sum
    of the problem with the x and y axes swapped (there Eq. 2's lowest-index rule picks the old y)."""
    rng = np.random.default_rng(81)
    vol = rand_vol(rng, (7, 6, 5))
    geom = np.array([[-30.0, 2.0, 1.0, 40.0, -8.0, -6.0, 0.0, 1.1, 0.0, 0.0, 0.0, 1.3]])
    ids = np.array([(0, iv, iu) for iv in range(10) for iu in range(14)], dtype=np.int32)
    origin, delta = (-3.1, -2.4, -2.2), 0.9
    val, mfl, pl, _ = oracle.project_rays(vol, delta, origin, geom, ids)
    val2, mfl2, pl2 = oracle.project_rays_axis(vol, delta, origin, geom, ids, mfl[:, 0])
    assert np.array_equal(val, val2) and np.array_equal(mfl, mfl2) and np.array_equal(pl, pl2)
    assert len(np.unique(mfl[:, 0])) >= 1 and np.abs(val).max() > 0.1
    # exact ties, grid coordinates: r = (a, +-a, c) with |c| < |a|
    n_checked = 0
    for _ in range(40):
        s = np.array([rng.uniform(-9, -4), rng.uniform(-3, 9), rng.uniform(-2, 7)])
        a = float(rng.integers(12, 24))
        sign = 1.0 if rng.random() < 0.5 else -1.0
        d = s + np.array([a, sign * a, rng.uniform(-0.4, 0.4) * a])
        if abs(d[0] - s[0]) != abs(d[1] - s[1]):
            continue                                                      # rounding broke the tie
        assert oracle.ray_grid(vol, s, d)["m"] == 0                        # Eq. 2, reading #8
        got = oracle.ray_grid_axis(vol, s, d, 1)
        pv = np.ascontiguousarray(np.transpose(vol, (1, 0, 2)))
        ref = oracle.ray_grid(pv, s[[1, 0, 2]], d[[1, 0, 2]])
        assert ref["m"] == 0
        assert abs(got["value"] - ref["value"]) <= 1e-13 * (1 + abs(ref["value"]))        # tap order differs
        assert (got["i_first"], got["i_last"]) == (ref["i_first"], ref["i_last"])
        n_checked += ref["i_last"] >= ref["i_first"]
    assert n_checked >= 10


@pytest.mark.parametrize("kernel", [0, 1])
def test_voxel_list_backprojection_equals_full_backprojection(oracle, kernel):
    """jo_backproject_voxels (the transpose by its definition, one hat product per ray and voxel, rays limited
    to a detector window) against the pinned jo_backproject on every voxel of small grids with all three
    driving axes -- which also shows that the window is wide enough for these magnifications."""
    rng = np.random.default_rng(82)
    shape, delta, nu, nv = (9, 7, 8), 0.8, 15, 13
    origin = tuple(-(n - 1) / 2.0 * delta + 0.05 * k for k, n in enumerate(shape))
    geom = _bp_poses(shape, delta, nu, nv)
    y = rng.uniform(-1.0, 2.0, size=(len(geom), nv, nu))
    full = oracle.backproject(y, shape, delta, origin, geom, kernel=kernel)
    vox = np.array(list(itertools.product(*[range(n) for n in shape])), dtype=np.int32)
    got = oracle.backproject_voxels(y, shape, delta, origin, geom, vox, halfwin=4, kernel=kernel, threads=2)
    assert np.abs(full).max() > 0.1
    assert np.allclose(got, full.reshape(-1), rtol=0, atol=1e-12 * np.abs(full).max())
    # a window that is too narrow must show up as a difference (the check above is not vacuous)
    narrow = oracle.backproject_voxels(y, shape, delta, origin, geom, vox, halfwin=0, kernel=kernel)
    assert np.abs(narrow - full.reshape(-1)).max() > 1e-3
