"""Writes tests/golden/oracle_regression.txt.  Calls ONLY oracle/ (never the CUDA path).

Run from the repo root:  python tests/golden/make_golden.py
The inputs are exactly reproducible on any machine (integer-valued volume from numpy's
default_rng, dyadic geometry), so the file guards the oracle against silent drift.
Columns: proj iv iu m i_first i_last value(fp64, world units).
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def inputs():
    rng = np.random.default_rng(160900958)
    vol = rng.integers(0, 64, size=(12, 10, 9)).astype(np.float32) / 16.0
    delta = 0.5
    origin = np.array([-(n - 1) / 2.0 * delta for n in vol.shape])
    geom = np.array([
        # source             det origin (pixel 0,0)     u              v
        [-20.0, 1.0, 0.5, 12.0, -5.0, -4.0, 0.0, 1.25, 0.0, 0.0, 0.0, 1.0],
        [3.0, -18.0, -1.0, -6.0, 10.0, -3.5, 1.5, 0.25, 0.0, 0.0, 0.0, 0.875],
        [0.5, 2.0, 25.0, -4.0, -4.5, -9.0, 1.0, 0.125, 0.0, -0.125, 1.0, 0.0],
    ])
    nu, nv = 9, 8
    ids = np.array([(p, iv, iu) for p in range(3) for iv in range(nv) for iu in range(nu)], dtype=np.int32)
    return vol, delta, origin, geom, ids


def compute_lines():
    import oracle
    vol, delta, origin, geom, ids = inputs()
    val, mfl, _, _ = oracle.project_rays(vol, delta, origin, geom, ids)
    return ["%d %d %d %d %d %d %.17g" % (*ids[q], *mfl[q], val[q]) for q in range(len(ids))]


if __name__ == "__main__":
    with open(os.path.join(HERE, "oracle_regression.txt"), "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle only); proj iv iu m i_first i_last value\n")
        f.write("\n".join(compute_lines()) + "\n")
    print("wrote oracle_regression.txt")
