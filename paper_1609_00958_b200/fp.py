"""Thin ctypes binding of libfp.so (include/fp.h): argument marshalling only.

Every step of the projector runs in the library's CUDA kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: if the library cannot be loaded
or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfp.so")

FP_OK = 0
STATUS = {0: "FP_OK", 1: "FP_ERR_INVALID_ARG", 2: "FP_ERR_CUDA", 3: "FP_ERR_OOM", 4: "FP_ERR_UNSUPPORTED"}

OPT_KERNEL, OPT_VOLATILE, OPT_INTERP, OPT_PERMUTED_COPY, OPT_COUNT_SAMPLES, OPT_FOV_CYLINDER, OPT_GROUP = 1, 2, 3, 4, 5, 6, 7
OPT_TEST_FORCE_TMA = 100
KERNEL_AUTO, KERNEL_DIRECT, KERNEL_ALIGNED, KERNEL_TMA, KERNEL_TEX, KERNEL_HWLIN, KERNEL_TILE = 0, 1, 2, 3, 4, 5, 6
INTERP_LINEAR, INTERP_SPLINE = 0, 1

# every symbol include/fp.h declares (tests check the library exports all of them)
SYMBOLS = ["fp_create", "fp_destroy", "fp_set_option", "fp_get_option", "fp_prepare", "fp_project",
           "fp_project_host", "fp_backproject", "fp_ray_ranges", "fp_plan", "fp_check", "fp_last_sample_count",
           "fp_last_launch_count", "fp_probe_bandwidth", "fp_project_static", "fp_status_string", "fp_last_error", "fp_version"]
PROBE_HBM_READ, PROBE_L2_READ, PROBE_SHARED_READ = 0, 1, 2


class FpError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__("%s: %s" % (STATUS.get(status, status), msg))
        self.status = status


_lib = None


def load(build_if_missing: bool = True):
    """dlopen libfp.so (building it with nvcc first if it is missing and nvcc is present)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from . import build as _b
        try:
            _b.build()
        except Exception:
            if not os.path.exists(LIB_PATH):
                raise
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError("libfp.so is not built: run python -m paper_1609_00958_b200.build")
    L = ctypes.CDLL(LIB_PATH)
    vp, i, dp = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double)
    L.fp_create.argtypes = [i, i, i, ctypes.c_double, dp, ctypes.POINTER(vp)]
    L.fp_destroy.argtypes = [vp]
    L.fp_set_option.argtypes = [vp, i, i]
    L.fp_get_option.argtypes = [vp, i, ctypes.POINTER(i)]
    L.fp_prepare.argtypes = [vp, vp, vp]
    L.fp_project.argtypes = [vp, vp, i, dp, i, i, vp, vp]
    L.fp_project_host.argtypes = [vp, vp, i, dp, i, i, vp]
    L.fp_backproject.argtypes = [vp, vp, i, dp, i, i, vp, vp]
    L.fp_ray_ranges.argtypes = [vp, i, dp, i, i, vp, vp]
    L.fp_plan.argtypes = [vp, dp, i, i, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i)]
    L.fp_last_sample_count.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
    L.fp_last_launch_count.argtypes = [vp, ctypes.POINTER(i)]
    L.fp_check.argtypes = [vp]
    L.fp_probe_bandwidth.argtypes = [i, ctypes.POINTER(ctypes.c_double)]
    L.fp_probe_bandwidth.restype = i
    for name in ("fp_create", "fp_destroy", "fp_set_option", "fp_get_option", "fp_prepare", "fp_project", "fp_check",
                 "fp_project_host", "fp_backproject", "fp_ray_ranges", "fp_plan", "fp_last_sample_count", "fp_last_launch_count"):
        getattr(L, name).restype = i
    L.fp_project_static.argtypes = [i, i, i, ctypes.c_double, dp, vp, i, dp, i, i, i, vp, vp, vp, ctypes.c_char_p, ctypes.c_size_t]
    L.fp_project_static.restype = i
    L.fp_status_string.argtypes = [i]
    L.fp_status_string.restype = ctypes.c_char_p
    L.fp_last_error.argtypes = [vp]
    L.fp_last_error.restype = ctypes.c_char_p
    L.fp_version.argtypes = []
    L.fp_version.restype = ctypes.c_char_p
    _lib = L
    return L


def _geom(geom) -> np.ndarray:
    g = np.ascontiguousarray(geom, dtype=np.float64)
    if g.ndim == 1:
        g = g.reshape(-1, 12)
    if g.ndim != 2 or g.shape[1] != 12:
        raise ValueError("geometry must be [n_proj][12] float64")
    return g


def _stream_handle(stream) -> int:
    import torch
    if stream is None:
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


class Projector:
    """One fp_ctx: a voxel grid (nx, ny, nz, voxel_size, origin) and its device workspaces."""

    def __init__(self, nx: int, ny: int, nz: int, voxel_size: float, origin: Sequence[float]):
        self._L = load()
        self._h = ctypes.c_void_p()
        o = (ctypes.c_double * 3)(*[float(x) for x in origin])
        st = self._L.fp_create(int(nx), int(ny), int(nz), float(voxel_size), o, ctypes.byref(self._h))
        if st != FP_OK:
            self._h = ctypes.c_void_p()
            raise FpError(st, "fp_create")
        self.shape = (int(nx), int(ny), int(nz))

    # -- helpers
    def _check(self, st: int):
        if st != FP_OK:
            raise FpError(st, (self._L.fp_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.fp_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the ABI, same names
    def set_option(self, key: int, value: int):
        self._check(self._L.fp_set_option(self._h, key, value))

    def get_option(self, key: int) -> int:
        v = ctypes.c_int()
        self._check(self._L.fp_get_option(self._h, key, ctypes.byref(v)))
        return v.value

    def _check_vol(self, vol):
        import torch
        if not (isinstance(vol, torch.Tensor) and vol.is_cuda and vol.dtype == torch.float32
                and vol.is_contiguous() and tuple(vol.shape) == self.shape):
            raise ValueError("volume must be a contiguous CUDA float32 tensor of shape %s" % (self.shape,))

    def prepare(self, vol, stream=None):
        self._check_vol(vol)
        self._check(self._L.fp_prepare(self._h, vol.data_ptr(), _stream_handle(stream)))

    def project(self, vol, geom, nu: int, nv: int, out=None, stream=None):
        """fp_project: vol CUDA fp32 (nx,ny,nz); geom host float64 [n_proj][12]; returns CUDA fp32 [n_proj][nv][nu]."""
        import torch
        self._check_vol(vol)
        g = _geom(geom)
        n_proj = g.shape[0]
        if out is None:
            out = torch.empty((n_proj, nv, nu), device=vol.device, dtype=torch.float32)
        elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
                  and out.numel() == n_proj * nv * nu):
            raise ValueError("out must be a contiguous CUDA float32 tensor with n_proj*nv*nu elements")
        self._check(self._L.fp_project(self._h, vol.data_ptr(), n_proj,
                                       g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                       int(nu), int(nv), out.data_ptr(), _stream_handle(stream)))
        return out

    def project_host(self, vol_host, geom, nu: int, nv: int, out_host=None):
        """fp_project_host: vol a CPU fp32 tensor / ndarray (ideally pinned); returns a CPU tensor."""
        import torch
        if isinstance(vol_host, np.ndarray):
            vol_host = torch.from_numpy(np.ascontiguousarray(vol_host, dtype=np.float32))
        if not (vol_host.device.type == "cpu" and vol_host.dtype == torch.float32 and vol_host.is_contiguous()
                and tuple(vol_host.shape) == self.shape):
            raise ValueError("vol_host must be a contiguous CPU float32 tensor of shape %s" % (self.shape,))
        g = _geom(geom)
        n_proj = g.shape[0]
        if out_host is None:
            out_host = torch.empty((n_proj, nv, nu), dtype=torch.float32)
        self._check(self._L.fp_project_host(self._h, vol_host.data_ptr(), n_proj,
                                            g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                            int(nu), int(nv), out_host.data_ptr()))
        return out_host

    def backproject(self, proj, geom, nu: int, nv: int, out=None, stream=None):
        """fp_backproject: proj CUDA fp32 [n_proj][nv][nu] -> CUDA fp32 volume (nx,ny,nz) = A^T proj."""
        import torch
        g = _geom(geom)
        n_proj = g.shape[0]
        if not (isinstance(proj, torch.Tensor) and proj.is_cuda and proj.dtype == torch.float32 and proj.is_contiguous()
                and proj.numel() == n_proj * nv * nu):
            raise ValueError("proj must be a contiguous CUDA float32 tensor with n_proj*nv*nu elements")
        if out is None:
            out = torch.empty(self.shape, device=proj.device, dtype=torch.float32)
        else:
            self._check_vol(out)
        self._check(self._L.fp_backproject(self._h, proj.data_ptr(), n_proj,
                                           g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                           int(nu), int(nv), out.data_ptr(), _stream_handle(stream)))
        return out

    def ray_ranges(self, geom, nu: int, nv: int, device="cuda", stream=None):
        """fp_ray_ranges: CUDA int32 [n_proj][nv][nu][3] = (m, i_first, i_last)."""
        import torch
        g = _geom(geom)
        n_proj = g.shape[0]
        mfl = torch.empty((n_proj, nv, nu, 3), device=device, dtype=torch.int32)
        self._check(self._L.fp_ray_ranges(self._h, n_proj, g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                          int(nu), int(nv), mfl.data_ptr(), _stream_handle(stream)))
        return mfl

    def plan(self, geom_row, nu: int, nv: int):
        """fp_plan: (kernel, window, z_driven) the library would use for one pose; host only."""
        g = np.ascontiguousarray(geom_row, dtype=np.float64).reshape(12)
        k, w, z = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        self._check(self._L.fp_plan(self._h, g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(nu), int(nv),
                                    ctypes.byref(k), ctypes.byref(w), ctypes.byref(z)))
        return k.value, w.value, bool(z.value)

    def check(self) -> None:
        """fp_check: raises FpError if a kernel since the last check found the host plan too small."""
        self._check(self._L.fp_check(self._h))

    def last_sample_count(self) -> int:
        n = ctypes.c_ulonglong()
        self._check(self._L.fp_last_sample_count(self._h, ctypes.byref(n)))
        return int(n.value)

    def last_launch_count(self) -> int:
        n = ctypes.c_int()
        self._check(self._L.fp_last_launch_count(self._h, ctypes.byref(n)))
        return n.value


STATIC_MAX_PROJ = 512


def project_static(shape, voxel_size: float, origin, vol, geom, nu: int, nv: int, interp: int = INTERP_LINEAR,
                   out=None, n_samples=None, stream=None):
    """fp_project_static: the projector without a context and without any allocation inside the library (its
    scratch is a static device array).  `out` ([n_proj][nv][nu] fp32) and `n_samples` (one int64 word, optional)
    are the caller's device tensors; `out` is created here if not given."""
    import torch
    g = _geom(geom)
    n_proj = g.shape[0]
    if vol.dtype != torch.float32 or not vol.is_cuda or not vol.is_contiguous() or tuple(vol.shape) != tuple(shape):
        raise ValueError("vol must be a contiguous fp32 CUDA tensor of the grid's shape")
    if out is None:
        out = torch.empty((n_proj, nv, nu), dtype=torch.float32, device=vol.device)
    if out.dtype != torch.float32 or not out.is_contiguous() or tuple(out.shape) != (n_proj, nv, nu):
        raise ValueError("out must be a contiguous fp32 tensor [n_proj][nv][nu]")
    if n_samples is not None and (n_samples.dtype != torch.int64 or n_samples.numel() != 1 or not n_samples.is_cuda):
        raise ValueError("n_samples must be a one-element int64 CUDA tensor")
    o = (ctypes.c_double * 3)(*[float(x) for x in origin])
    err = ctypes.create_string_buffer(256)
    st = load().fp_project_static(int(shape[0]), int(shape[1]), int(shape[2]), float(voxel_size), o, vol.data_ptr(), n_proj,
                                  g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(nu), int(nv), int(interp),
                                  out.data_ptr(), n_samples.data_ptr() if n_samples is not None else None,
                                  _stream_handle(stream), err, len(err))
    if st != FP_OK:
        raise FpError(st, err.value.decode())
    return out


def probe_bandwidth(what: int) -> float:
    """fp_probe_bandwidth: GB/s of the harness's read probe `what` (PROBE_*) on the current device."""
    v = ctypes.c_double()
    st = load().fp_probe_bandwidth(int(what), ctypes.byref(v))
    if st != 0:
        raise FpError(st, "fp_probe_bandwidth(%d)" % what)
    return v.value


def version() -> str:
    return load().fp_version().decode()
