"""fp64 CPU oracle of the Generalized Joseph Projector -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product path
(``paper_1609_00958_b200``) never does, and this package never imports the product.

The arithmetic lives in ``joseph_oracle.c`` (plain C, fp64, no FMA contraction); this
file only compiles it with gcc, loads it with ctypes and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "joseph_oracle.c")
_LIB = os.path.join(_HERE, "libjoseph_oracle.so")

KERNEL_LIN = 0
KERNEL_SPL = 1

CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
          "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    """Compile joseph_oracle.c -> libjoseph_oracle.so (gcc).  Returns the .so path."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        fp = ctypes.POINTER(ctypes.c_float)
        cip = ctypes.POINTER(ctypes.c_int)
        L.jo_ray_grid.argtypes = [fp, cip, dp, dp, ctypes.c_int, dp, ip, dp, dp]
        L.jo_ray_grid.restype = None
        L.jo_ray_definition.argtypes = [fp, cip, dp, dp, ctypes.c_int, dp]
        L.jo_ray_definition.restype = None
        L.jo_project_rays.argtypes = [fp, cip, ctypes.c_double, dp, dp, ctypes.c_int,
                                      ctypes.c_long, ip, dp, ip, dp, dp]
        L.jo_project_rays.restype = None
        L.jo_project_block.argtypes = [fp, cip, ctypes.c_double, dp, dp, ctypes.c_int,
                                       ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       dp, ip, dp, dp]
        L.jo_project_block.restype = None
        L.jo_backproject.argtypes = [dp, cip, ctypes.c_double, dp, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, dp]
        L.jo_backproject.restype = None
        L.jo_ray_grid_axis.argtypes = [fp, cip, dp, dp, ctypes.c_int, ctypes.c_int, dp, ip, dp]
        L.jo_ray_grid_axis.restype = None
        L.jo_project_rays_axis.argtypes = [fp, cip, ctypes.c_double, dp, dp, ctypes.c_int, ctypes.c_long, ip, ip,
                                           dp, ip, dp]
        L.jo_project_rays_axis.restype = None
        L.jo_backproject_voxels.argtypes = [dp, cip, ctypes.c_double, dp, dp, ctypes.c_int, ctypes.c_int,
                                            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_long, ip, dp]
        L.jo_backproject_voxels.restype = None
        _lib = L
    return _lib


def _vol(vol):
    v = np.ascontiguousarray(vol, dtype=np.float32)
    assert v.ndim == 3
    n = (ctypes.c_int * 3)(*v.shape)
    return v, n


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _iptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _fptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def ray_grid(vol, s, d, kernel: int = KERNEL_LIN):
    """One ray in grid coordinates.  Returns dict(value, m, i_first, i_last, L, margins)."""
    v, n = _vol(vol)
    s = np.ascontiguousarray(s, dtype=np.float64)
    d = np.ascontiguousarray(d, dtype=np.float64)
    val = ctypes.c_double()
    L = ctypes.c_double()
    mfl = np.zeros(3, dtype=np.int32)
    mg = np.zeros(2, dtype=np.float64)
    lib().jo_ray_grid(_fptr(v), n, _dptr(s), _dptr(d), kernel, ctypes.byref(val), _iptr(mfl),
                      ctypes.byref(L), _dptr(mg))
    return dict(value=val.value, m=int(mfl[0]), i_first=int(mfl[1]), i_last=int(mfl[2]),
                L=L.value, margins=(float(mg[0]), float(mg[1])))


def ray_grid_axis(vol, s, d, m: int, kernel: int = KERNEL_LIN):
    """One ray in grid coordinates with the driving axis given (jo_ray_grid_axis)."""
    v, n = _vol(vol)
    s = np.ascontiguousarray(s, dtype=np.float64)
    d = np.ascontiguousarray(d, dtype=np.float64)
    val = ctypes.c_double()
    L = ctypes.c_double()
    mfl = np.zeros(3, dtype=np.int32)
    lib().jo_ray_grid_axis(_fptr(v), n, _dptr(s), _dptr(d), kernel, int(m), ctypes.byref(val), _iptr(mfl),
                           ctypes.byref(L))
    return dict(value=val.value, m=int(mfl[0]), i_first=int(mfl[1]), i_last=int(mfl[2]), L=L.value)


def ray_definition(vol, s, d, kernel: int = KERNEL_LIN) -> float:
    """The O(N^3) triple-sum definition of one ray sum (grid coordinates)."""
    v, n = _vol(vol)
    s = np.ascontiguousarray(s, dtype=np.float64)
    d = np.ascontiguousarray(d, dtype=np.float64)
    val = ctypes.c_double()
    lib().jo_ray_definition(_fptr(v), n, _dptr(s), _dptr(d), kernel, ctypes.byref(val))
    return val.value


def project_rays(vol, voxel_size, origin, geom, ray_ids, kernel: int = KERNEL_LIN, threads: int = 1):
    """World-unit ray sums for ray_ids[n][3] = (projection, iv, iu).

    Returns (values f64[n], mfl i32[n][3], pathlen f64[n], margins f64[n][2]).
    ``threads`` > 1 splits the list over a thread pool (ctypes releases the GIL).
    """
    v, n = _vol(vol)
    origin = np.ascontiguousarray(origin, dtype=np.float64)
    geom = np.ascontiguousarray(geom, dtype=np.float64).reshape(-1, 12)
    ids = np.ascontiguousarray(ray_ids, dtype=np.int32).reshape(-1, 3)
    nr = ids.shape[0]
    values = np.zeros(nr, dtype=np.float64)
    mfl = np.zeros((nr, 3), dtype=np.int32)
    pathlen = np.zeros(nr, dtype=np.float64)
    margins = np.zeros((nr, 2), dtype=np.float64)

    def run(lo, hi):
        if hi > lo:
            lib().jo_project_rays(_fptr(v), n, float(voxel_size), _dptr(origin), _dptr(geom), kernel,
                                  hi - lo, _iptr(ids[lo:hi]), _dptr(values[lo:hi]), _iptr(mfl[lo:hi]),
                                  _dptr(pathlen[lo:hi]), _dptr(margins[lo:hi]))

    lib()
    if threads <= 1 or nr < 4 * threads:
        run(0, nr)
    else:
        chunk = max(1, (nr + 16 * threads - 1) // (16 * threads))
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(lambda lo: run(lo, min(nr, lo + chunk)), range(0, nr, chunk)))
    return values, mfl, pathlen, margins


def project_rays_axis(vol, voxel_size, origin, geom, ray_ids, axis, kernel: int = KERNEL_LIN):
    """project_rays with the driving axis GIVEN per ray (jo_ray_grid_axis; reading #8: the parity
    harness evaluates near-tie rays along the axis the GPU took).  Returns (values, mfl, pathlen)."""
    v, n = _vol(vol)
    origin = np.ascontiguousarray(origin, dtype=np.float64)
    geom = np.ascontiguousarray(geom, dtype=np.float64).reshape(-1, 12)
    ids = np.ascontiguousarray(ray_ids, dtype=np.int32).reshape(-1, 3)
    ax = np.ascontiguousarray(axis, dtype=np.int32).reshape(-1)
    nr = ids.shape[0]
    assert ax.shape[0] == nr
    values = np.zeros(nr, dtype=np.float64)
    mfl = np.zeros((nr, 3), dtype=np.int32)
    pathlen = np.zeros(nr, dtype=np.float64)
    if nr:
        lib().jo_project_rays_axis(_fptr(v), n, float(voxel_size), _dptr(origin), _dptr(geom), kernel, nr,
                                   _iptr(ids), _iptr(ax), _dptr(values), _iptr(mfl), _dptr(pathlen))
    return values, mfl, pathlen


def project_block(vol, voxel_size, origin, geom_row, iu0, iu1, iv0, iv1, kernel: int = KERNEL_LIN):
    """Pixel rectangle [iv0,iv1) x [iu0,iu1) of one projection, outputs [iv][iu]."""
    v, n = _vol(vol)
    origin = np.ascontiguousarray(origin, dtype=np.float64)
    g = np.ascontiguousarray(geom_row, dtype=np.float64).reshape(12)
    h, w = iv1 - iv0, iu1 - iu0
    values = np.zeros((h, w), dtype=np.float64)
    mfl = np.zeros((h, w, 3), dtype=np.int32)
    pathlen = np.zeros((h, w), dtype=np.float64)
    margins = np.zeros((h, w, 2), dtype=np.float64)
    lib().jo_project_block(_fptr(v), n, float(voxel_size), _dptr(origin), _dptr(g), kernel,
                           iu0, iu1, iv0, iv1, _dptr(values), _iptr(mfl), _dptr(pathlen), _dptr(margins))
    return values, mfl, pathlen, margins


def project(vol, voxel_size, origin, geom, nu, nv, kernel: int = KERNEL_LIN, threads: int = 1):
    """Whole projections: returns (values f64[n_proj][nv][nu], mfl i32[n_proj][nv][nu][3],
    pathlen f64[n_proj][nv][nu]).  Work is split by (projection, row band) over threads."""
    v, _ = _vol(vol)
    geom = np.ascontiguousarray(geom, dtype=np.float64).reshape(-1, 12)
    n_proj = geom.shape[0]
    values = np.zeros((n_proj, nv, nu), dtype=np.float64)
    mfl = np.zeros((n_proj, nv, nu, 3), dtype=np.int32)
    pathlen = np.zeros((n_proj, nv, nu), dtype=np.float64)
    band = max(1, min(nv, 4096 // max(1, nu)))
    jobs = [(p, r0, min(nv, r0 + band)) for p in range(n_proj) for r0 in range(0, nv, band)]

    def run(job):
        p, r0, r1 = job
        a, b, c, _ = project_block(v, voxel_size, origin, geom[p], 0, nu, r0, r1, kernel)
        values[p, r0:r1], mfl[p, r0:r1], pathlen[p, r0:r1] = a, b, c

    lib()
    if threads <= 1:
        for j in jobs:
            run(j)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(run, jobs))
    return values, mfl, pathlen


def backproject(proj, shape, voxel_size, origin, geom, kernel: int = KERNEL_LIN, threads: int = 1):
    """Exact transpose of ``project`` (jo_backproject): proj f64[n_proj][nv][nu] -> volume f64[nx][ny][nz].
    ``threads`` > 1 splits the projections over a thread pool, each thread into its own accumulator."""
    y = np.ascontiguousarray(proj, dtype=np.float64)
    assert y.ndim == 3
    n_proj, nv, nu = y.shape
    geom = np.ascontiguousarray(geom, dtype=np.float64).reshape(-1, 12)
    assert geom.shape[0] == n_proj
    origin = np.ascontiguousarray(origin, dtype=np.float64)
    n = (ctypes.c_int * 3)(*[int(k) for k in shape])
    lib()

    def run(lo, hi):
        out = np.zeros(tuple(int(k) for k in shape), dtype=np.float64)
        if hi > lo:
            lib().jo_backproject(_dptr(y[lo:hi]), n, float(voxel_size), _dptr(origin), _dptr(geom[lo:hi]), kernel,
                                 hi - lo, nu, nv, _dptr(out))
        return out

    threads = max(1, min(threads, n_proj))
    if threads == 1:
        return run(0, n_proj)
    cuts = np.linspace(0, n_proj, threads + 1).astype(int)
    with ThreadPoolExecutor(max_workers=threads) as ex:
        parts = list(ex.map(lambda k: run(int(cuts[k]), int(cuts[k + 1])), range(threads)))
    return sum(parts[1:], parts[0])


def backproject_voxels(proj, shape, voxel_size, origin, geom, voxels, halfwin: int, kernel: int = KERNEL_LIN,
                       threads: int = 1):
    """(A^T proj)[v] for the listed voxels[n][3] = (ix, iy, iz) by the definition of the transpose
    (jo_backproject_voxels); halfwin = half width in pixels of the detector window visited around each voxel's
    projection.  Returns f64[n]."""
    y = np.ascontiguousarray(proj, dtype=np.float64)
    n_proj, nv, nu = y.shape
    geom = np.ascontiguousarray(geom, dtype=np.float64).reshape(-1, 12)
    assert geom.shape[0] == n_proj
    origin = np.ascontiguousarray(origin, dtype=np.float64)
    vox = np.ascontiguousarray(voxels, dtype=np.int32).reshape(-1, 3)
    out = np.zeros(vox.shape[0], dtype=np.float64)
    n = (ctypes.c_int * 3)(*[int(k) for k in shape])
    lib()

    def run(lo, hi):
        if hi > lo:
            lib().jo_backproject_voxels(_dptr(y), n, float(voxel_size), _dptr(origin), _dptr(geom), kernel, n_proj, nu,
                                        nv, int(halfwin), hi - lo, _iptr(vox[lo:hi]), _dptr(out[lo:hi]))

    nq = vox.shape[0]
    if threads <= 1 or nq < 4 * threads:
        run(0, nq)
    else:
        chunk = max(1, (nq + 8 * threads - 1) // (8 * threads))
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(lambda lo: run(lo, min(nq, lo + chunk)), range(0, nq, chunk)))
    return out


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1
