"""`torch.autograd` glue for the projector pair: LIRE++ trains through P and P* (the
backward pass of a linear operator is its adjoint, SURVEY.md s.3 call stack B).  `cbct_bp_adjoint` is the EXACT
transpose of the matrix `cbct_fp` applies, so the gradients below are the gradients of the discrete operators, not
approximations.  Argument marshalling only: every value is computed by the library's kernels, on the current stream.

    y = project(geom, x)          # x[..., nz, ny, nx] -> y[..., n_views, nv, nu];  dL/dx = P^T dL/dy
    x = backproject(geom, y)      # y[..., n_views, nv, nu] -> x[..., nz, ny, nx];  dL/dy = P dL/dx

Leading axes (batch, channels) are flattened into the `channels` argument of one call.
"""
from __future__ import annotations

import torch

from . import cbct


def _run(fn, geom, src, tail_in, tail_out):
    if tuple(src.shape[-3:]) != tuple(tail_in):
        raise cbct.CbctError(f"expected trailing shape {tuple(tail_in)}, got {tuple(src.shape[-3:])}")
    if not src.is_cuda:
        raise cbct.CbctError("autograd wrappers take CUDA tensors (no CPU fallback)")
    lead = tuple(src.shape[:-3])
    c = 1
    for d in lead:
        c *= int(d)
    out = torch.empty(lead + tuple(tail_out), device=src.device, dtype=torch.float32)
    if c:
        fn(src.detach().to(torch.float32).contiguous(), out, c)
    return out


class _Project(torch.autograd.Function):
    @staticmethod
    def forward(ctx, vol, geom):
        ctx.geom = geom
        return _run(geom.fp, geom, vol, geom.vol_shape, geom.sino_shape)

    @staticmethod
    def backward(ctx, grad_sino):
        g = ctx.geom
        return _Backproject.apply(grad_sino, g), None


class _Backproject(torch.autograd.Function):
    @staticmethod
    def forward(ctx, sino, geom):
        ctx.geom = geom
        return _run(geom.bp_adjoint, geom, sino, geom.sino_shape, geom.vol_shape)

    @staticmethod
    def backward(ctx, grad_vol):
        g = ctx.geom
        return _Project.apply(grad_vol, g), None


def project(geom: cbct.Geometry, vol: torch.Tensor) -> torch.Tensor:
    """P vol (cbct_fp), differentiable; gradient = cbct_bp_adjoint."""
    return _Project.apply(vol, geom)


def backproject(geom: cbct.Geometry, sino: torch.Tensor) -> torch.Tensor:
    """P^T sino (cbct_bp_adjoint), differentiable; gradient = cbct_fp."""
    return _Backproject.apply(sino, geom)
