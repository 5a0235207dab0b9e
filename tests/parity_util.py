"""Shared helpers of the GPU parity tests: the tolerance of BASELINE.json's north_star and the
comparison of one batch of rays against the oracle."""
import numpy as np

REL_TOL = 2e-5      # max per-ray relative error
ABS_COEF = 1e-6     # x ray path length x max|voxel|
MARGIN = 1e-9       # rays whose fp64 decisions sit this close to a tie are compared under either decision


def tolerance(oracle_values, pathlen, vol_absmax):
    return REL_TOL * np.abs(oracle_values) + ABS_COEF * pathlen * vol_absmax


def assert_parity(gpu_values, gpu_mfl, oracle_values, oracle_mfl, pathlen, margins, vol_absmax, what=""):
    """gpu_values f32[n], gpu_mfl i32[n][3]; oracle outputs as oracle.project_rays returns them.
    Indices (m, i_first, i_last) must match exactly except for rays whose decision margin is < MARGIN
    (DESIGN.md index-parity rule); values must be inside the tolerance for every ray.
    Returns the worst error / tolerance ratio."""
    gv = np.asarray(gpu_values, dtype=np.float64).ravel()
    ov = np.asarray(oracle_values, dtype=np.float64).ravel()
    gm = np.asarray(gpu_mfl).reshape(-1, 3)
    om = np.asarray(oracle_mfl).reshape(-1, 3)
    pl = np.asarray(pathlen, dtype=np.float64).ravel()
    mg = np.asarray(margins, dtype=np.float64).reshape(-1, 2)
    assert gv.shape == ov.shape and gm.shape == om.shape
    assert np.all(np.isfinite(gv)), what
    same = np.all(gm == om, axis=1)
    near_tie = (mg[:, 0] < MARGIN) | (mg[:, 1] < MARGIN)
    bad_idx = ~same & ~near_tie
    assert not bad_idx.any(), "%s: %d rays with different (m, i_first, i_last), first: gpu %s oracle %s" % (
        what, bad_idx.sum(), gm[bad_idx][0], om[bad_idx][0])
    tol = tolerance(ov, pl, vol_absmax)
    err = np.abs(gv - ov)
    cmp = same                                   # near-tie rays with other indices: value checked loosely below
    over = cmp & (err > tol)
    if over.any():
        q = int(np.argmax(np.where(cmp, err - tol, -1)))
        raise AssertionError("%s: %d rays outside tolerance; worst ray %d: gpu %.9g oracle %.9g err %.3g tol %.3g mfl %s"
                             % (what, over.sum(), q, gv[q], ov[q], err[q], tol[q], om[q]))
    # misses are exactly +0.0
    miss = om[:, 2] < om[:, 1]
    assert np.all(gv[miss & same] == 0.0), what
    ratio = np.where(tol > 0, err / np.where(tol > 0, tol, 1), 0.0)
    return float(ratio[cmp].max()) if cmp.any() else 0.0
