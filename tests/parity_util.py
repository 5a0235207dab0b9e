"""Shared helpers of the GPU parity tests: the tolerance of BASELINE.json's north_star and the
comparison of one batch of rays against the oracle."""
import numpy as np

REL_TOL = 2e-5      # max per-ray relative error
ABS_COEF = 1e-6     # x ray path length x max|voxel|
MARGIN = 1e-9       # rays whose fp64 decisions sit this close to a tie may take the other decision
MAX_TIE_FRACTION = 1e-4   # ... and there must be very few of them


def tolerance(oracle_values, pathlen, vol_absmax):
    return REL_TOL * np.abs(oracle_values) + ABS_COEF * pathlen * vol_absmax


def make_recompute(oracle, vol, voxel_size, origin, geom, ray_ids, kernel=0):
    """recompute(positions, axes) -> (values, mfl, pathlen) of the rays ray_ids[positions] with the driving axis
    GIVEN (oracle.project_rays_axis): what assert_parity needs for near-tie rays (reading #8)."""
    ids = np.asarray(ray_ids, dtype=np.int32).reshape(-1, 3)

    def recompute(positions, axes):
        return oracle.project_rays_axis(vol, voxel_size, origin, geom, ids[positions], axes, kernel=kernel)

    return recompute


def assert_parity(gpu_values, gpu_mfl, oracle_values, oracle_mfl, pathlen, margins, vol_absmax, what="",
                  recompute=None):
    """gpu_values f32[n], gpu_mfl i32[n][3]; oracle outputs as oracle.project_rays returns them.

    Indices (m, i_first, i_last) must match exactly except for rays whose decision margin is < MARGIN
    (DESIGN.md index-parity rule).  Such a ray is accepted with other indices only if
      - its driving axis differs (a tie of Eq. 2 within MARGIN): its value matches, inside the normal tolerance,
        the oracle RECOMPUTED ALONG THE GPU'S AXIS (`recompute`, see make_recompute), and its slice range is the
        oracle's for that axis (or sits on a boundary tie itself);
      - only its slice range differs (a transverse coordinate within MARGIN of -1 or N_t, where the boundary
        sample's weight is < MARGIN): its value matches the oracle's own value inside the normal tolerance;
    and such rays are fewer than MAX_TIE_FRACTION of the batch (at least 2 are allowed).
    Every ray is compared in value.  Misses are exactly +0.0.  Returns the worst error / tolerance ratio."""
    gv32 = np.asarray(gpu_values).ravel()
    gv = gv32.astype(np.float64)
    ov = np.asarray(oracle_values, dtype=np.float64).ravel().copy()
    gm = np.asarray(gpu_mfl).reshape(-1, 3)
    om = np.asarray(oracle_mfl).reshape(-1, 3).copy()
    pl = np.asarray(pathlen, dtype=np.float64).ravel().copy()
    mg = np.asarray(margins, dtype=np.float64).reshape(-1, 2)
    n = gv.shape[0]
    assert gv.shape == ov.shape and gm.shape == om.shape
    assert np.all(np.isfinite(gv)), what
    same = np.all(gm == om, axis=1)
    near_tie = (mg[:, 0] < MARGIN) | (mg[:, 1] < MARGIN)
    bad_idx = ~same & ~near_tie
    assert not bad_idx.any(), "%s: %d rays with different (m, i_first, i_last), first: gpu %s oracle %s" % (
        what, bad_idx.sum(), gm[bad_idx][0], om[bad_idx][0])
    other = np.nonzero(~same)[0]                          # near ties decided the other way
    assert len(other) <= max(2, int(MAX_TIE_FRACTION * n)), "%s: %d of %d rays on a decision tie" % (what, len(other), n)
    axis_diff = other[gm[other, 0] != om[other, 0]]
    if len(axis_diff):
        assert recompute is not None, "%s: %d rays took the other driving axis on a tie and no recompute was given" % (
            what, len(axis_diff))
        assert np.all(mg[axis_diff, 0] < MARGIN), what
        v2, m2, p2 = recompute(axis_diff, gm[axis_diff, 0])
        range_ok = np.all(m2 == gm[axis_diff], axis=1) | (mg[axis_diff, 1] < MARGIN)
        assert range_ok.all(), "%s: slice range along the GPU's axis differs: gpu %s oracle %s" % (
            what, gm[axis_diff][~range_ok][0], m2[~range_ok][0])
        ov[axis_diff], om[axis_diff], pl[axis_diff] = v2, m2, p2
    tol = tolerance(ov, pl, vol_absmax)
    err = np.abs(gv - ov)
    over = err > tol
    if over.any():
        q = int(np.argmax(err - tol))
        raise AssertionError("%s: %d rays outside tolerance; worst ray %d: gpu %.9g oracle %.9g err %.3g tol %.3g mfl %s"
                             % (what, over.sum(), q, gv[q], ov[q], err[q], tol[q], om[q]))
    # misses are exactly +0.0 (not -0.0)
    miss = (om[:, 2] < om[:, 1]) & (gm[:, 2] < gm[:, 1])
    assert np.all(gv32[miss] == 0.0) and not np.signbit(gv32[miss]).any(), what
    ratio = np.where(tol > 0, err / np.where(tol > 0, tol, 1), 0.0)
    return float(ratio.max()) if n else 0.0
