"""torch.autograd hookup of the four C-ABI operators (paper section IV-C).

The paper trains through the transforms with PyTorch autograd and obtains the backward pass from the adjoint
operators ("adjoint iSHT = Y^dagger, adjoint SHT = W Y", "reuse of forward and inverse transforms",
P:292).  Here the backward of `alm2map` IS `cuhpx_alm2map_adjoint` and the backward of `map2alm` IS
`cuhpx_map2alm_adjoint` (and vice versa, so double backward works): no arithmetic happens in Python, the
functions only pick which C-ABI call runs.

Gradient convention (include/cuhpx.h, R4): the stored complex tensor a[b, idx] is treated by PyTorch
as the pair (Re a, Im a), so the cotangent of a complex input is the complex number (dL/dRe a) + i (dL/dIm a) --
exactly what S^T and A^T return.  Im a_l0 carries no gradient (it is ignored on input; the adjoint returns 0).
"""
from __future__ import annotations

import torch

from .binding import Transform


class _Alm2Map(torch.autograd.Function):
    @staticmethod
    def forward(ctx, alm, T: Transform):
        ctx.T = T
        return T.alm2map(alm.contiguous())

    @staticmethod
    def backward(ctx, gmap):
        return _Alm2MapAdjoint.apply(gmap, ctx.T), None


class _Alm2MapAdjoint(torch.autograd.Function):
    @staticmethod
    def forward(ctx, gmap, T: Transform):
        ctx.T = T
        return T.alm2map_adjoint(gmap.contiguous())

    @staticmethod
    def backward(ctx, galm):
        return _Alm2Map.apply(galm, ctx.T), None


class _Map2Alm(torch.autograd.Function):
    @staticmethod
    def forward(ctx, hmap, T: Transform):
        ctx.T = T
        return T.map2alm(hmap.contiguous())

    @staticmethod
    def backward(ctx, galm):
        return _Map2AlmAdjoint.apply(galm, ctx.T), None


class _Map2AlmAdjoint(torch.autograd.Function):
    @staticmethod
    def forward(ctx, galm, T: Transform):
        ctx.T = T
        return T.map2alm_adjoint(galm.contiguous())

    @staticmethod
    def backward(ctx, gmap):
        return _Map2Alm.apply(gmap, ctx.T), None


def alm2map(alm: torch.Tensor, T: Transform) -> torch.Tensor:
    """Differentiable synthesis S (Eq. 24): complex [batch, nalm] -> real [batch, npix]."""
    return _Alm2Map.apply(alm, T)


def map2alm(hmap: torch.Tensor, T: Transform) -> torch.Tensor:
    """Differentiable analysis A (Eq. 26): real [batch, npix] -> complex [batch, nalm]."""
    return _Map2Alm.apply(hmap, T)


class SHT(torch.nn.Module):
    """Analysis as a module (the paper's "SHT" layer)."""

    def __init__(self, T: Transform):
        super().__init__()
        self.T = T

    def forward(self, hmap):
        return map2alm(hmap, self.T)


class ISHT(torch.nn.Module):
    """Synthesis as a module (the paper's "iSHT" layer, used in its one-layer training demo)."""

    def __init__(self, T: Transform):
        super().__init__()
        self.T = T

    def forward(self, alm):
        return alm2map(alm, self.T)
