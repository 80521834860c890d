"""oracle/prox.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

fp64 numpy oracle of the TV proximal operator and of FISTA ("Proximal
algorithms ... For the 2-norm and TV proximal operators, TIGRE provides the Fast Iterative Shrinkage-Thresholding
Algorithm (FISTA) [42]", used in PAPER.md:308-314 and 377-393: FISTA(proj, geo, angles, 20, 'hyper', 2e2, 'init',
'FDK', 'tviter', 50)).  Only tests/ may import this module; it shares nothing with paper_2412_10129_b200/.

The paper names both and cites [42]; it prints neither, so both are READINGS:

P24  TV proximal operator  prox(f) = argmin_u 1/2 ||u - f||^2 + lam * TV(u),  TV isotropic with forward differences
     (zero at the upper border of every axis; an axis of length 1 drops out), computed by n_iter steps of the
     dual projection iteration
         p <- (p + tau * grad(div p - f/lam)) / (1 + tau * |grad(div p - f/lam)|),   p = 0 at the start,
         u  = f - lam * div p,
     grad = forward differences, div = -grad^T (backward differences of p with p = 0 outside), |.| the Euclidean norm
     of the three components at a voxel, tau = 1/12 (three dimensions) unless given.  lam = 0 returns f.
P25  FISTA for ||A x - b||^2 + 2 lam TV(x) with step 1/L ('hyper' = L):
         y_0 = x_0, t_0 = 1
         x_{k+1} = prox_{lam}( y_k + (2/L) A^T (b - A y_k) )
         t_{k+1} = (1 + sqrt(1 + 4 t_k^2)) / 2
         y_{k+1} = x_{k+1} + ((t_k - 1) / t_{k+1}) (x_{k+1} - x_k)
     resid[k] = ||b - A y_k||_2 (the residual the step is built from).
"""
from __future__ import annotations

import numpy as np

from . import oracle as orc


def grad(d):
    """Forward differences along z, y, x of d[nz][ny][nx]; zero at the upper border; returns (gz, gy, gx)."""
    out = []
    for ax in range(3):
        g = np.zeros_like(d)
        if d.shape[ax] > 1:
            sl_lo = [slice(None)] * 3
            sl_hi = [slice(None)] * 3
            sl_lo[ax], sl_hi[ax] = slice(0, -1), slice(1, None)
            g[tuple(sl_lo)] = d[tuple(sl_hi)] - d[tuple(sl_lo)]
        out.append(g)
    return out


def div(p):
    """div = -grad^T: backward differences of the components (pz, py, px), p = 0 outside."""
    acc = np.zeros_like(p[0])
    for ax in range(3):
        q = p[ax]
        if q.shape[ax] == 1:
            continue
        sl_lo = [slice(None)] * 3
        sl_hi = [slice(None)] * 3
        sl_lo[ax], sl_hi[ax] = slice(0, -1), slice(1, None)
        qq = q.copy()
        last = [slice(None)] * 3
        last[ax] = slice(-1, None)
        qq[tuple(last)] = 0.0                 # the forward difference at the upper border is zero: that p never acts
        acc += qq
        acc[tuple(sl_hi)] -= qq[tuple(sl_lo)]
    return acc


def tv_forward(u):
    gz, gy, gx = grad(np.asarray(u, dtype=np.float64))
    return float(np.sum(np.sqrt(gx * gx + gy * gy + gz * gz)))


def tv_prox(f, lam, n_iter, tau=1.0 / 12.0):
    """P24."""
    f = np.asarray(f, dtype=np.float64)
    if lam == 0.0:
        return f.copy()
    p = [np.zeros_like(f) for _ in range(3)]
    for _ in range(n_iter):
        g = grad(div(p) - f / lam)
        nrm = np.sqrt(g[0] ** 2 + g[1] ** 2 + g[2] ** 2)
        p = [(p[a] + tau * g[a]) / (1.0 + tau * nrm) for a in range(3)]
    return f - lam * div(p)


def fista(b, geo, angles, n_iter, L, lam, tv_iter, ax_mode=orc.SIDDON, atb_mode=orc.MATCHED, x0=None, exact_adjoint=False,
          tau=1.0 / 12.0):
    """P25.  Returns (x, resid[n_iter])."""
    AT = (lambda y: orc.atb_exact(y, geo, angles, ax_mode)) if exact_adjoint else (lambda y: orc.atb(y, geo, angles, atb_mode))
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(geo.vol_shape) if x0 is None else np.array(x0, dtype=np.float64)
    y = x.copy()
    t = 1.0
    resid = np.zeros(n_iter)
    for k in range(n_iter):
        r = b - orc.ax(y, geo, angles, ax_mode)
        resid[k] = np.sqrt(float(np.sum(r * r)))
        x_new = tv_prox(y + (2.0 / L) * AT(r), lam, tv_iter, tau)
        t_new = 0.5 * (1.0 + np.sqrt(1.0 + 4.0 * t * t))
        y = x_new + ((t - 1.0) / t_new) * (x_new - x)
        x, t = x_new, t_new
    return x, resid
