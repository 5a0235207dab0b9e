"""Host logic of libfp.so that needs no device: which sampling kernel a pose gets and how wide the
aligned kernel's staging window must be (fp_plan, include/fp.h)."""
import math

import numpy as np
import pytest

from paper_1609_00958_b200 import fp, synth


def circular_pose(theta, sid, sdd, nu, nv, pitch):
    c, s = math.cos(theta), math.sin(theta)
    S = np.array([sid * c, sid * s, 0.0])
    C = S - sdd * np.array([c, s, 0.0])
    U = pitch * np.array([-s, c, 0.0])
    V = pitch * np.array([0.0, 0.0, 1.0])
    return np.concatenate([S, C - (nu - 1) / 2 * U - (nv - 1) / 2 * V, U, V])


@pytest.mark.parametrize("name,wmax", [("C1", 128), ("C2", 256), ("C3", 256), ("C5", 384), ("P1", 384)])
def test_circular_orbits_take_the_aligned_kernel(name, wmax):
    cfg = synth.CONFIGS[name]
    geom = synth.make_geometry(cfg)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        ws = []
        for p in range(0, cfg.n_proj, max(1, cfg.n_proj // 45)):
            k, w, z = P.plan(geom[p], cfg.nu, cfg.nv)
            assert k in (fp.KERNEL_ALIGNED, fp.KERNEL_TMA) and not z, (name, p)
            # the TMA-fed kernel only where its 256-voxel window holds the block's rows
            assert (k == fp.KERNEL_TMA) <= (w <= 256), (name, p, w)
            ws.append(w)
        # the window must hold the z extent of one block's rows (at most 256 of them)
        assert 16 <= max(ws) <= wmax, (name, max(ws))


def test_wide_cones_take_the_tma_kernel_with_narrower_row_blocks():
    """C5 / P1: the z window of 256 detector rows exceeds the largest TMA box (256 voxels); most poses fit with
    192-row blocks and are planned FP_KERNEL_TMA with that window, the rest (C5 near 45 degrees: more than 12 volume
    rows per slice) stay with the line-staging kernel and its wider window."""
    for name, lo_frac in (("C5", 0.6), ("P1", 0.7)):
        cfg = synth.CONFIGS[name]
        geom = synth.make_geometry(cfg)
        with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
            plans = [P.plan(geom[p], cfg.nu, cfg.nv) for p in range(0, cfg.n_proj, 4)]
        tma = [w for k, w, z in plans if k == fp.KERNEL_TMA]
        al = [w for k, w, z in plans if k == fp.KERNEL_ALIGNED]
        assert len(tma) + len(al) == len(plans)
        assert len(tma) >= lo_frac * len(plans) and len(al) > 0, (name, len(tma), len(al))
        assert max(tma) <= 256 < min(al), (name, max(tma), min(al))


def test_general_poses_take_the_tile_kernel_and_report_z_driven_rays():
    cfg = synth.CONFIGS["C4"]
    geom = synth.make_geometry(cfg)
    zs = 0
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        for p in range(cfg.n_proj):
            k, w, z = P.plan(geom[p], cfg.nu, cfg.nv)
            assert k == fp.KERNEL_TILE and w == 0
            zs += z
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_DIRECT)
        assert P.plan(geom[0], cfg.nu, cfg.nv)[0] == fp.KERNEL_DIRECT
    # a volume whose z rows are not a multiple of 4 voxels cannot be addressed by tensor maps: direct kernel
    with fp.Projector(30, 30, 30, 1.0, (-14.5, -14.5, -14.5)) as P:
        assert P.plan(geom[0], cfg.nu, cfg.nv)[0] == fp.KERNEL_DIRECT
    # ~70 degree cone: almost every pose has some z-driven rays, a few (source near the xy plane) have none
    assert 0.9 * cfg.n_proj < zs < cfg.n_proj


def test_aligned_kernel_is_refused_when_its_preconditions_fail():
    cfg = synth.CONFIGS["C2"]
    g = circular_pose(0.3, cfg.sid, cfg.sdd, cfg.nu, cfg.nv, cfg.pitch)
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        assert P.plan(g, cfg.nu, cfg.nv)[0] in (fp.KERNEL_ALIGNED, fp.KERNEL_TMA)
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_ALIGNED)
        assert P.plan(g, cfg.nu, cfg.nv)[0] == fp.KERNEL_ALIGNED
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_AUTO)
        # a rolled detector: u picks up a z component
        r = g.copy()
        r[6:9] = 0.999 * g[6:9] + 0.04 * g[9:12]
        assert P.plan(r, cfg.nu, cfg.nv)[0] == fp.KERNEL_TILE
        # a tilted rotation axis: v picks up an x component
        t = g.copy()
        t[9] = 1e-9
        assert P.plan(t, cfg.nu, cfg.nv)[0] == fp.KERNEL_TILE
        # a tall detector close to the source: the outer rows are z-driven
        tall = circular_pose(0.3, 100.0, 120.0, 64, 512, 1.5)
        k, w, z = P.plan(tall, 64, 512)
        assert k == fp.KERNEL_TILE and z
        # the forced direct kernel
        P.set_option(fp.OPT_KERNEL, fp.KERNEL_DIRECT)
        assert P.plan(g, cfg.nu, cfg.nv)[0] == fp.KERNEL_DIRECT
    # nz not a multiple of 4: no float4 loads along z
    with fp.Projector(128, 128, 126, 1.0, (-63.5, -63.5, -62.5)) as P:
        assert P.plan(g, cfg.nu, cfg.nv)[0] == fp.KERNEL_DIRECT


def test_window_grows_with_the_row_spacing():
    cfg = synth.CONFIGS["C3"]
    with fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin) as P:
        w1 = P.plan(circular_pose(0.1, cfg.sid, cfg.sdd, 768, 768, 1.0), 768, 768)[1]
        w2 = P.plan(circular_pose(0.1, cfg.sid, cfg.sdd, 768, 768, 1.6), 768, 768)[1]
        # a detector too coarse for the largest window falls back to the general-pose (tile) kernel
        k3, w3, _ = P.plan(circular_pose(0.1, cfg.sid, cfg.sdd, 768, 768, 4.0), 768, 768)
    assert 0 < w1 < w2 <= 512
    assert k3 == fp.KERNEL_TILE and w3 == 0
