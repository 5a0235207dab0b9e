"""Simultaneous algebraic reconstruction with the matched projector pair (
PAPER.md:27 sec. 1.1, :308 sec. 3.1 "10 SART iterations", :367).

    x_{k+1} = x_k + lambda * A^T( (y - A x_k) / (A 1) ) / (A^T 1)

A is fp_project, A^T is fp_backproject (its exact transpose); A 1 and A^T 1 are the ray lengths through the
volume and the total weight every voxel receives.  All projections are used in every update (the "simultaneous"
form).  The projector and back-projector run in libfp.so; the residual, the two divisions and the update are
plain elementwise torch operations on the device (plumbing, not part of the measured hot path).
"""
from __future__ import annotations


def sart(P, y, geom, nu: int, nv: int, n_iter: int = 10, lam: float = 1.0, x0=None, eps: float = 1e-6):
    """P: fp.Projector; y: CUDA fp32 [n_proj][nv][nu].  Returns (x, residuals) where residuals[k] is
    sqrt(sum((y - A x_k)^2 / (A 1))) BEFORE update k (k = 0 .. n_iter-1) and residuals[n_iter] after the last."""
    import torch
    shape = P.shape
    ones_v = torch.ones(shape, device=y.device, dtype=torch.float32)
    row = P.project(ones_v, geom, nu, nv)                    # A 1
    col = P.backproject(torch.ones_like(y), geom, nu, nv)    # A^T 1
    inv_row = torch.where(row > eps, 1.0 / row.clamp_min(eps), torch.zeros_like(row))
    inv_col = torch.where(col > eps, 1.0 / col.clamp_min(eps), torch.zeros_like(col))
    x = torch.zeros(shape, device=y.device, dtype=torch.float32) if x0 is None else x0.clone()
    residuals = []
    ax = torch.empty_like(y)
    bp = torch.empty_like(x)
    for _ in range(n_iter):
        P.project(x, geom, nu, nv, out=ax)
        r = y - ax
        residuals.append(float(torch.sqrt((r.double() ** 2 * inv_row.double()).sum())))
        P.backproject(r * inv_row, geom, nu, nv, out=bp)
        x += lam * bp * inv_col
    P.project(x, geom, nu, nv, out=ax)
    r = y - ax
    residuals.append(float(torch.sqrt((r.double() ** 2 * inv_row.double()).sum())))
    return x, residuals
