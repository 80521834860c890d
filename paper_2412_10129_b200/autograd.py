"""PyTorch operator wrappers (section 2.8: "TIGRE projectors ... treated as a linear differentiable operator
by the automatic differentiation engine").  A and A^T as torch.autograd Functions over the
library's kernels, with no trip through host memory (the paper's binding copies through NumPy; here the tensors stay on
the device).  The backward of A is the library's A^T and vice versa:
  * backprojector="exact" (default) uses the ray-driven exact transposes (TIGRE_ATB_EXACT_*): gradients are the true
    gradients of the forward computation (<Ax, y> = <x, A^T y> to fp32 rounding), A^T itself is differentiable through Ax;
  * backprojector="matched" / "fdk" uses the voxel-driven pair of the iterative methods: an approximate adjoint (the
    "mismatched backprojector" of PAPER.md:130), faster.
"""
from __future__ import annotations

import torch

import paper_2412_10129_b200 as tg


class _Ax(torch.autograd.Function):
    @staticmethod
    def forward(ctx, vol, op):
        ctx.op = op
        return tg.Ax(vol.contiguous(), op.geo, op.angles, op.ax_mode)

    @staticmethod
    def backward(ctx, grad_proj):
        op = ctx.op
        return _Atb.apply(grad_proj, op), None


class _Atb(torch.autograd.Function):
    @staticmethod
    def forward(ctx, proj, op):
        ctx.op = op
        return tg.Atb(proj.contiguous(), op.geo, op.angles, op.atb_mode)

    @staticmethod
    def backward(ctx, grad_vol):
        op = ctx.op
        return _Ax.apply(grad_vol, op), None


class Projector:
    """A(vol) -> projections and AT(proj) -> volume as differentiable operators on CUDA float32 tensors."""

    def __init__(self, geo, angles, ax_mode="siddon", backprojector="exact"):
        self.geo, self.angles, self.ax_mode = geo, angles, ax_mode
        self.atb_mode = ("exact_" + ax_mode) if backprojector == "exact" else backprojector

    def A(self, vol):
        return _Ax.apply(vol, self)

    def AT(self, proj):
        return _Atb.apply(proj, self)

    __call__ = A
