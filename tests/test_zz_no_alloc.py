"""fp_project_static (include/fp.h): the projector for callers that may not allocate.  Its scratch is a static device
array, so nothing is cudaMalloc'ed inside the library.  Checked against the existing path (fp_project with
FP_KERNEL_DIRECT through a context) on two calls in a row that share the array.

Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from parity_util import REL_TOL, ABS_COEF

pytestmark = pytest.mark.gpu


def _existing_path(torch, fp, cfg, vol, geom, interp):
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_DIRECT)
        P.set_option(fp.OPT_INTERP, interp)
        P.set_option(fp.OPT_COUNT_SAMPLES, 1)
        ref = P.project(vol, geom, cfg.nu, cfg.nv).clone()
        torch.cuda.synchronize()
        return ref, P.last_sample_count()


def _assert_close(cfg, vol, got, ref, what):
    # the tolerance of the parity tests (tests/parity_util.py) with the path length bounded by the grid's diagonal
    pathlen = float(np.sqrt(3.0) * max(cfg.n) * cfg.voxel_size)
    tol = REL_TOL * ref.abs().double() + ABS_COEF * pathlen * float(vol.abs().max())
    err = (got.double() - ref.double()).abs()
    assert bool((err <= tol).all()), (what, float((err / tol.clamp_min(1e-300)).max()))
    assert float(ref.abs().max()) > 0.0, what


def test_static_entry_point_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    from paper_1609_00958_b200 import fp, synth

    cfg = synth.CONFIGS["C2"]
    vol = synth.make_volume(cfg, device="cuda")
    rng = np.random.default_rng(4242)
    # call 1: 24 poses -- circular ones and random ones (all three driving axes, z-driven rays read with a stride)
    geom1 = np.concatenate([synth.make_geometry(cfg)[::15],
                            synth.random_poses(12, cfg.sid, cfg.sdd, cfg.nu, cfg.nv, cfg.pitch, rng)])
    # call 2: fewer poses (the table keeps call 1's entries behind them), other poses, the other interpolation
    geom2 = synth.random_poses(7, cfg.sid, cfg.sdd, cfg.nu, cfg.nv, cfg.pitch, rng)
    ref1, cnt1 = _existing_path(torch, fp, cfg, vol, geom1, fp.INTERP_LINEAR)
    ref2, cnt2 = _existing_path(torch, fp, cfg, vol, geom2, fp.INTERP_SPLINE)

    out1 = torch.full((len(geom1), cfg.nv, cfg.nu), float("nan"), device="cuda")
    out2 = torch.full((len(geom2), cfg.nv, cfg.nu), float("nan"), device="cuda")
    n1 = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    n2 = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    # back to back on one stream, no synchronisation in between
    fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, geom1, cfg.nu, cfg.nv, fp.INTERP_LINEAR, out=out1, n_samples=n1)
    fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, geom2, cfg.nu, cfg.nv, fp.INTERP_SPLINE, out=out2, n_samples=n2)
    torch.cuda.synchronize()
    _assert_close(cfg, vol, out1, ref1, "first call")
    _assert_close(cfg, vol, out2, ref2, "second call")
    # the counter restarts with every call
    assert int(n1.item()) == cnt1 and int(n2.item()) == cnt2 and cnt1 > cnt2 > 0

    # a third call, identical to the second: same result again, and the device's free memory does not move
    free_before = torch.cuda.mem_get_info()[0]
    out3 = out1[: len(geom2)]                      # an existing buffer: the test itself allocates nothing here
    out3.fill_(float("nan"))
    fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, geom2, cfg.nu, cfg.nv, fp.INTERP_SPLINE, out=out3)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    assert torch.equal(out3, out2)


def test_static_entry_point_rejects_what_it_cannot_hold():
    import torch
    from paper_1609_00958_b200 import fp, synth

    cfg = synth.CONFIGS["C1"]
    vol = synth.make_volume(cfg, device="cuda")
    g = synth.make_geometry(cfg)
    too_many = np.repeat(g[:1], fp.STATIC_MAX_PROJ + 1, axis=0)
    out = torch.zeros((len(too_many), 4, 4), device="cuda")
    with pytest.raises(fp.FpError) as e:
        fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, too_many, 4, 4, out=out)
    assert e.value.status == 4 and "FP_STATIC_MAX_PROJ" in str(e.value)        # FP_ERR_UNSUPPORTED
    with pytest.raises(fp.FpError) as e:
        fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, g[:2], 4, 4, interp=7, out=out[:2])
    assert e.value.status == 1                                                   # FP_ERR_INVALID_ARG
    # exactly the maximum is accepted, and an empty call leaves the output alone and reports zero samples
    most = np.repeat(g[:1], fp.STATIC_MAX_PROJ, axis=0)
    fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, most, 4, 4, out=out[: fp.STATIC_MAX_PROJ])
    n = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    fp.project_static(cfg.n, cfg.voxel_size, cfg.origin, vol, np.zeros((0, 12)), 4, 4, out=out[:0], n_samples=n)
    torch.cuda.synchronize()
    assert int(n.item()) == 0
    assert torch.equal(out[0], out[fp.STATIC_MAX_PROJ - 1])
