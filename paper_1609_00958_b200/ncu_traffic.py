"""Records what an `ncu --set full` capture of one sampling-kernel launch measured, for bench.py's roofline lines.

    python -m paper_1609_00958_b200.ncu_traffic <report.ncu-rep> --config C3 --kernel fp_tma_kernel \
        [--interp linear] --source profiles/r2_01_tma_kernel_c3.md

Reads the report with `ncu -i ... --page raw --csv` (no GPU needed) and writes, under the key
"<config>/<kernel>/<interp>" of profiles/traffic.json: DRAM bytes (read + write), L2 bytes (32 B x lts__t_sectors_srcunit_tex),
shared-memory / L1 data-pipe wavefronts, the kernel's duration under ncu, and the hash of the library sources
the capture belongs to.  bench.py quotes an entry only while that hash matches the sources it is timing.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import io
import json
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")


def csrc_sha() -> str:
    h = hashlib.sha256()
    d = os.path.join(HERE, "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def _to_bytes(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return float(value.replace(",", "")) * scale.get(unit, 1.0)


def read_report(path: str, launch: int = 0) -> dict:
    raw = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units, vals = rows[0], rows[1], rows[2 + launch]
    col = {h: i for i, h in enumerate(hdr)}

    def get(name):
        i = col[name]
        return vals[i], units[i]

    dur, dur_u = get("gpu__time_duration.sum")
    dur_ms = float(dur.replace(",", "")) * {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}[dur_u]
    out = {
        "kernel_name": vals[col["Kernel Name"]],
        "dram_bytes": _to_bytes(*get("dram__bytes_read.sum")) + _to_bytes(*get("dram__bytes_write.sum")),
        # sectors the SMs requested from L2 (32 B each): tile copies of the TMA engine, stores of the projections
        "l2_bytes": 32.0 * float(get("lts__t_sectors_srcunit_tex.sum")[0].replace(",", "")),
        "l2_hit_rate": float(get("lts__t_sectors_srcunit_tex_lookup_hit.sum")[0].replace(",", ""))
                       / max(1.0, float(get("lts__t_sectors_srcunit_tex.sum")[0].replace(",", ""))),
        "lsu_wavefronts": float(get("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")[0].replace(",", "")),
        "ncu_duration_ms": dur_ms,
    }
    return out


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--config", required=True)
    ap.add_argument("--kernel", required=True)
    ap.add_argument("--interp", default="linear")
    ap.add_argument("--source", required=True, help="the profiles/*.md summary that documents the capture")
    ap.add_argument("--launch", type=int, default=0, help="which captured launch of the report")
    args = ap.parse_args()
    e = read_report(args.report, args.launch)
    assert args.kernel in e["kernel_name"], "the report holds %s" % e["kernel_name"]
    e["csrc_sha"] = csrc_sha()
    e["source"] = args.source
    try:
        db = json.load(open(TRAFFIC_JSON))
    except Exception:
        db = {}
    db["%s/%s/%s" % (args.config, args.kernel, args.interp)] = e
    with open(TRAFFIC_JSON, "w") as f:
        json.dump(db, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps(e, indent=1))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
