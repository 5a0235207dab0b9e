#!/usr/bin/env python
"""Device-timed benchmark of the B200 Joseph cone-beam forward projector (libfp.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

One "step" is one pass of the whole hot path (geometry ingest, ray set-up, layout stage if the
pose needs it, sampling loop, weight + store) over one batch of synthetic
input: the full orbit of the configuration (C3: 360 projections of a 512^3 volume onto 768^2).
Prints ONE JSON line (rank 0).  DESIGN.md "Measurement" states how every number is formed.

The oracle (oracle/) is used only by the cpu_baseline leg and by --impl reference.
"""
from __future__ import annotations

import argparse
import datetime
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "512^3 cone-beam projections/s"
UNIT = "projections/s"
TAP_BYTES = 16           # 4 taps x 4 B per sample: the paper's "memory access rate"
FALLBACK_HBM_GBS = 6650.0
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")


def csrc_sha():
    """Hash of the library's sources: profiles/traffic.json records it with every ncu capture, and a capture is
    quoted only while the sources it was taken from are the ones being timed."""
    from paper_1609_00958_b200.ncu_traffic import csrc_sha as f
    return f()


def captured_traffic(config, kernel, interp):
    """(entry, stale) for this config / kernel from profiles/traffic.json (written by
    python -m paper_1609_00958_b200.ncu_traffic from an ncu --set full capture)."""
    try:
        db = json.load(open(TRAFFIC_JSON))
    except Exception:
        return None, False
    e = db.get("%s/%s/%s" % (config, kernel, interp))
    if e is None:
        return None, False
    return e, e.get("csrc_sha") != csrc_sha()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": FALLBACK_HBM_GBS}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""

    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        # started BEFORE the warm-up steps so that no idle gap (in which the clocks fall back) separates the
        # warm-up from the timed region; only the samples stamped inside [mark_start, mark_end] are reported
        self.t0 = self.t1 = None
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def mark_start(self):
        # nvidia-smi needs about 0.2 s to print its first sample: a run whose warm-up is shorter than that (C1, C2)
        # waits for it here, so that at least that sample stands in for a timed region of a few milliseconds
        t_end = time.time() + 1.0
        while self.p is not None and os.path.getsize(self.f.name) == 0 and time.time() < t_end:
            time.sleep(0.01)
        self.t0 = datetime.datetime.now()

    def mark_end(self):
        self.t1 = datetime.datetime.now()

    def _inside(self, stamp: str) -> bool:
        if self.t0 is None or self.t1 is None:
            return True
        try:
            t = datetime.datetime.strptime(stamp, "%Y/%m/%d %H:%M:%S.%f")
        except ValueError:
            return True
        slack = datetime.timedelta(milliseconds=50)
        return self.t0 - slack <= t <= self.t1 + slack

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        out = self.summarize(self.f.read())
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        return out

    def summarize(self, text: str) -> dict:
        """Median SM clock, maximum clock and throttle reasons of the nvidia-smi samples stamped inside
        [mark_start, mark_end] (host logic, covered by tests/test_bench_host.py)."""
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        lines = [[x.strip() for x in line.split(",")] for line in text.splitlines()]
        lines = [c for c in lines if len(c) >= 9]
        inside = [c for c in lines if self._inside(c[0])]
        # a timed region shorter than the sampling period (C1, C2) has no sample of its own: then the samples of
        # the warm-up steps right before it stand in, and the line says so
        out["window"] = "timed region" if inside else "whole run (timed region shorter than the sampling period)"
        sm, mx, reasons = [], [], set()
        for c in (inside or lines):
            try:
                sm.append(float(c[1]))
                mx.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def oracle_sample(cfg, geom, vol_np, max_seconds=20.0, kernel=0, threads=None):
    """Time the oracle, as it stands, on a bounded sample of the workload: whole detector rows of eight
    projections spread over the orbit (both driving axes and the switches between them for circular
    orbits), on `threads` host threads (default: every core).  Returns (projections/s, samples/s, cores,
    description, ids, values, mfl, pathlen, margins)."""
    import oracle
    cores = oracle.host_cores() if threads is None else threads
    # eight poses spread over the orbit: both driving axes, both signs, and the switches between them
    projs = sorted({(k * cfg.n_proj) // 8 + (cfg.n_proj // 16 if k % 2 else 0) for k in range(8)})
    # calibrate on a few rows, then size the sample for ~max_seconds of wall time
    rows_cal = max(1, min(cfg.nv, 4))
    def ids_for(rows):
        vs = np.linspace(0, cfg.nv - 1, rows).round().astype(np.int32)
        p, v, u = np.meshgrid(np.array(projs, dtype=np.int32), vs, np.arange(cfg.nu, dtype=np.int32), indexing="ij")
        return np.stack([p.ravel(), v.ravel(), u.ravel()], axis=1).astype(np.int32)
    ids = ids_for(rows_cal)
    t0 = time.perf_counter()
    oracle.project_rays(vol_np, cfg.voxel_size, cfg.origin, geom, ids, kernel=kernel, threads=cores)
    t_cal = time.perf_counter() - t0
    rows = int(max(rows_cal, min(cfg.nv, rows_cal * max_seconds / max(t_cal, 1e-3))))
    ids = ids_for(rows)
    t0 = time.perf_counter()
    val, mfl, pl, mg = oracle.project_rays(vol_np, cfg.voxel_size, cfg.origin, geom, ids, kernel=kernel, threads=cores)
    dt = time.perf_counter() - t0
    n_samples = int(np.maximum(mfl[:, 2] - mfl[:, 1] + 1, 0).sum())
    rays_per_proj = cfg.nu * cfg.nv
    proj_per_s = (len(ids) / rays_per_proj) / dt
    desc = "%d of %d detector rows (all %d columns) of %d projections %s: %d rays, %d samples in %.1f s" % (
        rows, cfg.nv, cfg.nu, len(projs), projs, len(ids), n_samples, dt)
    return proj_per_s, n_samples / dt, cores, desc, ids, val, mfl, pl, mg


def run_reference(args):
    """--impl reference: the fp64 CPU oracle as the reference arm (there is no reference code)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1609_00958_b200 import synth
    cfg = synth.CONFIGS[args.config]
    geom = synth.make_geometry(cfg)
    vol = synth.make_volume(cfg, device="cpu").numpy()
    budget = 60.0 / max(1, args.steps + args.warmup)
    vals = []
    desc, cores = "", 0
    for k in range(args.warmup + args.steps):
        pps, sps, cores, desc, *_ = oracle_sample(cfg, geom, vol, max_seconds=min(20.0, budget), kernel=1 if args.interp == "spline" else 0)
        if k >= args.warmup:
            vals.append((pps, sps))
    pps = statistics.median(v[0] for v in vals)
    sps = statistics.median(v[1] for v in vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": pps, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * cfg.n_proj / pps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "extrapolated": True},
        "gsamples_per_s": sps / 1e9,
        "cpu_baseline": {"value": pps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": pps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))
    return 0


def max_over_ranks(dist, value, device="cuda"):
    """MAX of a python float over all ranks (identity without a process group)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_throughput(world, units_per_rank, seconds_max):
    """Whole-job rate of `world` independent replicas: every rank processes the
    same number of units, the job takes as long as its slowest rank."""
    return world * units_per_rank / seconds_max


def workload_name(cfg):
    return "%s: %dx%dx%d fp32 volume, %d projections (%s orbit) onto %dx%d" % (
        cfg.name, *cfg.n, cfg.n_proj, cfg.orbit, cfg.nu, cfg.nv)


def run_backproject(args, torch, fp, cfg, geom, vol, proj, P, stream, world, rank, dist):
    """--op backproject: one step = fp_backproject of the whole orbit (A^T applied to the projections of the
    synthetic volume) into a volume-sized output; reported as back-projected projections per second."""
    P.project(vol, geom, cfg.nu, cfg.nv, out=proj, stream=stream)          # the input: A x
    bp = torch.empty_like(vol)

    def step():
        P.backproject(proj, geom, cfg.nu, cfg.nv, out=bp, stream=stream)
        return P.last_launch_count()

    clocks = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    launches = 0
    clocks.mark_start()
    ev[0].record(stream)
    for k in range(args.steps):
        launches += step()
        ev[k + 1].record(stream)
    torch.cuda.synchronize()
    clocks.mark_end()
    clk = clocks.stop()
    ms = max_over_ranks(dist, ev[0].elapsed_time(ev[args.steps])) / args.steps
    if rank != 0:
        return 0
    # adjoint identity on the timed data: <A x, A x> = <x, A^T A x>
    lhs = float((proj.double() ** 2).sum())
    rhs = float((vol.double() * bp.double()).sum())
    peaks, peak_kind = measured_peaks()
    vol_bytes, proj_bytes = vol.numel() * 4, cfg.nu * cfg.nv * 4
    algo = cfg.n_proj * (2 * vol_bytes + proj_bytes)        # read-modify-write of the volume once per projection
    achieved = algo / (ms * 1e-3) / 1e9
    # poses of the aligned class take the transpose of the TMA-fed kernel unless the direct kernel is forced
    aligned = P.plan(geom[0], cfg.nu, cfg.nv)[0] in (fp.KERNEL_ALIGNED, fp.KERNEL_TMA)
    bp_kernel = "fp_bp_aligned_kernel" if aligned else "fp_backproject_kernel"
    cap, stale = captured_traffic(cfg.name, bp_kernel, args.interp)
    line = {
        "metric": "512^3 cone-beam back-projections/s", "value": replicas_throughput(world, cfg.n_proj, ms * 1e-3),
        "unit": "projections/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "op": "backproject", "interpolation": args.interp},
        "clocks": clk, "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                     "frac": achieved / peaks["hbm_gbs"],
                     "traffic": cap["dram_bytes"] if (cap is not None and not stale) else None,
                     "traffic_source": (cap["source"] if (cap is not None and not stale) else None),
                     "peak_kind": peak_kind,
                     "kernel": bp_kernel, "algorithmic_bytes_per_launch": algo},
        "adjoint_check": {"lhs": lhs, "rhs": rhs, "rel_diff": abs(lhs - rhs) / abs(lhs)},
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3", choices=["C1", "C2", "C3", "C4", "C5", "P1"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-probes", action="store_true", help="skip the L2 / shared-memory read probes")
    ap.add_argument("--layout-prepared", action="store_true",
                    help="FP_OPT_VOLATILE = 0 and fp_prepare before the timed region: the layout stage is NOT timed")
    ap.add_argument("--kernel", type=int, default=0, help="FP_OPT_KERNEL value (0 = auto)")
    ap.add_argument("--group", type=int, default=-1, help="FP_OPT_GROUP (-1 = library default)")
    ap.add_argument("--op", default="project", choices=["project", "backproject"],
                    help="project: the headline forward projector; backproject: its exact transpose (SURVEY 8(f) #2)")
    ap.add_argument("--interp", default="linear", choices=["linear", "spline"],
                    help="interpolation kernel: GJP_lin (PAPER.md:150 Eq. 13, the headline) or GJP_spl (:152 Eq. 14)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)          # timing rule: at least three untimed warm-up steps
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # python bench.py --gpus N: start the N replicas ourselves, one process per GPU
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)

    import torch
    from paper_1609_00958_b200 import fp, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    fp.load()

    cfg = synth.CONFIGS[args.config]
    geom = synth.make_geometry(cfg)
    vol = synth.make_volume(cfg, device="cuda")
    batch = cfg.batch or cfg.n_proj
    out = torch.empty((cfg.n_proj, cfg.nv, cfg.nu), device="cuda", dtype=torch.float32)
    P = fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin)
    if args.kernel:
        P.set_option(fp.OPT_KERNEL, args.kernel)
    interp = fp.INTERP_SPLINE if args.interp == "spline" else fp.INTERP_LINEAR
    P.set_option(fp.OPT_INTERP, interp)
    if args.group >= 0:
        P.set_option(fp.OPT_GROUP, args.group)
    if cfg.cylinder:
        P.set_option(fp.OPT_FOV_CYLINDER, 1)       # the volume is zero outside the inscribed cylinder
    stream = torch.cuda.current_stream()
    if args.layout_prepared:
        P.set_option(fp.OPT_VOLATILE, 0)
        P.prepare(vol, stream=stream)

    if args.op == "backproject":
        return run_backproject(args, torch, fp, cfg, geom, vol, out, P, stream, world, rank, dist)

    def step():
        launches, samples = 0, None
        for p0 in range(0, cfg.n_proj, batch):
            p1 = min(cfg.n_proj, p0 + batch)
            P.project(vol, geom[p0:p1], cfg.nu, cfg.nv, out=out[p0:p1], stream=stream)
            launches += P.last_launch_count()
        return launches

    def barrier():
        if dist is not None:
            dist.barrier()

    # sample count of one step (outside the timed region: fp_last_sample_count synchronises, and the
    # count costs one exact fp64 ray set-up per ray that the sampling itself does not need)
    samples = 0
    clocks = ClockSampler(local_rank)
    P.set_option(fp.OPT_COUNT_SAMPLES, 1)
    for p0 in range(0, cfg.n_proj, batch):
        p1 = min(cfg.n_proj, p0 + batch)
        P.project(vol, geom[p0:p1], cfg.nu, cfg.nv, out=out[p0:p1], stream=stream)
        samples += P.last_sample_count()
    P.set_option(fp.OPT_COUNT_SAMPLES, 0)        # the library default: the timed path is the one a user gets
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()

    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    torch.cuda.synchronize()
    launches = 0
    clocks.mark_start()
    ev[0].record(stream)
    for k in range(args.steps):
        launches += step()
        ev[k + 1].record(stream)
    torch.cuda.synchronize()
    clocks.mark_end()
    barrier()
    clk = clocks.stop()
    P.check()                                    # no kernel found the host plan too small
    step_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[args.steps])
    total_ms = max_over_ranks(dist, total_ms)
    ms_per_step = total_ms / args.steps
    proj_per_s = replicas_throughput(world, cfg.n_proj, ms_per_step * 1e-3)
    samples_per_s = replicas_throughput(world, samples, ms_per_step * 1e-3)

    # ---- end to end through fp_project_host: pinned host volume in, pinned host projections out
    e2e = None
    if not args.no_e2e:
        vol_h = vol.cpu().pin_memory()
        out_h = torch.empty((cfg.n_proj, cfg.nv, cfg.nu), dtype=torch.float32).pin_memory()
        P2 = fp.Projector(*cfg.n, cfg.voxel_size, cfg.origin)
        P2.set_option(fp.OPT_INTERP, interp)
        if cfg.cylinder:
            P2.set_option(fp.OPT_FOV_CYLINDER, 1)
        if args.kernel:
            P2.set_option(fp.OPT_KERNEL, args.kernel)
        P2.project_host(vol_h, geom, cfg.nu, cfg.nv, out_host=out_h)          # warm-up (allocations)
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            P2.project_host(vol_h, geom, cfg.nu, cfg.nv, out_host=out_h)      # synchronises before returning
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dist, dt)
        e2e = {"value": replicas_throughput(world, cfg.n_proj * n_e2e, dt), "unit": UNIT,
               "h2d_bytes_per_step": int(vol_h.numel() * 4 + geom.size * 8),
               "d2h_bytes_per_step": int(out_h.numel() * 4), "steps": n_e2e,
               "same_result_as_device_path": bool(torch.equal(out_h, out.cpu()))}
        P2.close()
        del vol_h

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # which sampling kernel the library's plan picks for this workload (fp_plan, host only)
    plans = [P.plan(g, cfg.nu, cfg.nv)[0] for g in geom]
    names = {fp.KERNEL_DIRECT: "fp_direct_kernel", fp.KERNEL_ALIGNED: "fp_aligned_kernel", fp.KERNEL_TMA: "fp_tma_kernel",
             fp.KERNEL_TEX: "fp_tex_kernel", fp.KERNEL_TILE: "fp_tile_kernel", fp.KERNEL_HWLIN: "fp_tex_kernel (hardware filtering)"}
    # every pose is planned on its own; name the kernel that takes most of them and say how many
    kernel_name = names[max(set(plans), key=plans.count)]
    kernel_share = {names[k]: plans.count(k) for k in sorted(set(plans))}
    peaks, peak_kind = measured_peaks()
    vol_bytes = vol.numel() * 4
    out_bytes_per_proj = cfg.nu * cfg.nv * 4
    # algorithmic HBM bytes per projection: the voxels the cone can touch once + the projection written once
    # (DESIGN.md).  With FP_OPT_FOV_CYLINDER the method's own work is the inscribed cylinder, pi/4 of the box.
    vol_algo = vol_bytes * (math.pi / 4.0 if cfg.cylinder else 1.0)
    algo_bytes_per_step = cfg.n_proj * (vol_algo + out_bytes_per_proj)
    n_calls = max(1, (cfg.n_proj + batch - 1) // batch)
    kernel_ms = ms_per_step            # one sampling launch per fp_project; the step is that launch (or n_calls of them)
    achieved = algo_bytes_per_step / (kernel_ms * 1e-3) / 1e9
    cap, stale = captured_traffic(cfg.name, kernel_name, args.interp)
    use = cap is not None and not stale
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"],
                "traffic": cap["dram_bytes"] if use else None,
                "traffic_source": (cap["source"] if use else ("stale: sources changed since " + cap["source"] if cap else None)),
                "peak_kind": peak_kind, "kernel": kernel_name, "projections_per_kernel": kernel_share,
                "algorithmic_bytes_per_launch": algo_bytes_per_step / n_calls,
                "algorithmic_bytes_note": ("volume bytes x pi/4 (inscribed cylinder, FP_OPT_FOV_CYLINDER) + projection bytes"
                                           if cfg.cylinder else "volume bytes + projection bytes, per projection"),
                "median_ms": statistics.median(step_ms), "best_ms": min(step_ms),
                "frac_best": algo_bytes_per_step / (min(step_ms) * 1e-3) / 1e9 / peaks["hbm_gbs"]}
    # L2 and L1 / shared-memory rates against probed peaks (BASELINE.json metric: "achieved HBM/L2 GB/s vs peak")
    roofline_l2 = roofline_l1 = None
    if not args.no_probes:
        l2_peak = fp.probe_bandwidth(fp.PROBE_L2_READ)
        sh_peak = fp.probe_bandwidth(fp.PROBE_SHARED_READ)
        hbm_read = fp.probe_bandwidth(fp.PROBE_HBM_READ)
        l2_ach = (cap["l2_bytes"] / (kernel_ms / n_calls * 1e-3) / 1e9) if use and cap.get("l2_bytes") else None
        roofline_l2 = {"bound": "l2", "achieved": l2_ach, "peak": l2_peak, "unit": "GB/s",
                       "frac": (l2_ach / l2_peak) if l2_ach else None,
                       "achieved_kind": "32 B x lts__t_sectors_srcunit_tex of the kept ncu capture / live kernel time" if l2_ach else "no current capture",
                       "peak_kind": "fp_probe_bandwidth(L2_READ): 48 MiB re-read through ld.global.cg", "hbm_read_probe_gbs": hbm_read}
        tap_gbs = TAP_BYTES * samples_per_s / world / 1e9
        sh_ach = (cap["lsu_wavefronts"] * 128.0 / (kernel_ms / n_calls * 1e-3) / 1e9) if use and cap.get("lsu_wavefronts") else None
        roofline_l1 = {"bound": "shared", "achieved": tap_gbs, "peak": sh_peak, "unit": "GB/s", "frac": tap_gbs / sh_peak,
                       "achieved_kind": "16 B x samples / time: the four taps of every sample (PAPER.md:314)",
                       "wavefront_gbs": sh_ach, "wavefront_frac": (sh_ach / sh_peak) if sh_ach else None,
                       "peak_kind": "fp_probe_bandwidth(SHARED_READ): conflict-free 32-bit loads"}

    cpu_baseline = None
    parity = None
    if not args.no_cpu_baseline and world == 1:
        vol_np = vol.cpu().numpy()
        pps, sps, cores, desc, ids, val, mfl, pl, mg = oracle_sample(cfg, geom, vol_np, max_seconds=15.0, kernel=1 if args.interp == "spline" else 0)
        cpu_baseline = {"value": pps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                        "gsamples_per_s": sps / 1e9, "extrapolated_from_sample": True}
        # the same oracle on ONE thread, on a sample a tenth as long
        pps1, sps1, _, desc1, *_ = oracle_sample(cfg, geom, vol_np, max_seconds=4.0, kernel=1 if args.interp == "spline" else 0, threads=1)
        cpu_baseline["single_thread"] = {"value": pps1, "unit": UNIT, "cores": 1, "gsamples_per_s": sps1 / 1e9, "sample": desc1}
        g = out[torch.from_numpy(ids[:, 0].astype(np.int64)).cuda(), torch.from_numpy(ids[:, 1].astype(np.int64)).cuda(),
                torch.from_numpy(ids[:, 2].astype(np.int64)).cuda()].cpu().numpy().astype(np.float64)
        tol = 2e-5 * np.abs(val) + 1e-6 * pl * float(vol.abs().max().item())
        gm = P.ray_ranges(geom, cfg.nu, cfg.nv) if cfg.n_proj * cfg.nu * cfg.nv <= (1 << 28) else None
        idx_equal = None
        if gm is not None:
            gmr = gm[torch.from_numpy(ids[:, 0].astype(np.int64)).cuda(), torch.from_numpy(ids[:, 1].astype(np.int64)).cuda(),
                     torch.from_numpy(ids[:, 2].astype(np.int64)).cuda()].cpu().numpy()
            idx_equal = bool(np.array_equal(gmr, mfl))
            del gm
        miss = mfl[:, 2] < mfl[:, 1]
        parity = {"rays": int(len(ids)), "worst_err_over_tol": float(np.max(np.abs(g - val) / np.maximum(tol, 1e-300))),
                  "indices_equal": idx_equal, "misses_are_plus_zero": bool(np.all(g[miss] == 0.0) and not np.signbit(g[miss]).any())}

    line = {
        "metric": METRIC, "value": proj_per_s, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "projections_per_call": batch, "replicas": world,
                   "l2_policy": "inputs larger than L2 (volume %d MB, output %d MB per step; L2 126 MB)" % (
                       vol_bytes >> 20, (cfg.n_proj * out_bytes_per_proj) >> 20),
                   "layout_stage_in_timed_region": not args.layout_prepared, "interpolation": args.interp},
        "gsamples_per_s": samples_per_s / 1e9,
        "samples_per_step": samples,
        "tap_access_rate_gbs": TAP_BYTES * samples_per_s / 1e9,
        "step_ms": step_ms,
        "ms_median": statistics.median(step_ms), "ms_best": min(step_ms),
        "value_best": replicas_throughput(world, cfg.n_proj, min(step_ms) * 1e-3),
        "clocks": clk,
        "gpu_launches": launches,
        "e2e": e2e,
        "roofline": roofline,
        "roofline_l2": roofline_l2,
        "roofline_l1": roofline_l1,
        "cpu_baseline": cpu_baseline,
        "parity_check": parity,
        "paper_context": "GTX 970: 176 projections/s (GJP_lin, global memory), 292 GB/s tap access rate, "
                         "512^3 -> 512^2, 1.04e8 samples/projection (PAPER.md:331 Table 1)",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
