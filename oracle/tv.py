"""oracle/tv.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

fp64 numpy oracle of the (adaptive-weighted) total-variation term and its gradient-descent minimiser
(SURVEY.md section 8(f).2).  Source: section 2.2.3, eq. (7) (AwTV, printed for two
dimensions) and eq. (8) (weights), "a gradient descend minimizer of the function is available"; the TV norm
is the limit delta -> infinity.  Only tests/ may import this module; it shares nothing with
paper_2412_10129_b200/.

Readings (listed in DESIGN.md section 2, P20-P22):
  P20  three dimensions: backward differences along x, y and z under one root, summed over the voxels that have
       all their backward neighbours (index >= 1 along every axis longer than 1; an axis of length 1 drops out,
       which makes nz = 1 exactly the printed 2-D formula);  eps >= 0 is added under the root so that the
       gradient exists where all differences vanish (the paper prints none: eps = 0 reproduces eq. 7).
  P21  "gradient" is the true gradient of eq. (7), the weights of eq. (8) differentiated along with the
       differences:  d/dd [ w(d) d^2 ] = 2 d w(d) (1 - d^2/delta^2).
  P22  minimiser: n_steps of  x <- x - alpha * g / ||g||_2  (g = gradient at the current x; stop if ||g|| = 0).
"""
from __future__ import annotations

import numpy as np


def _diffs(x):
    """Backward differences d[a][p] = x[p] - x[p - e_a] on the summation domain (all axes of length > 1 have
    index >= 1).  x is [nz][ny][nx]; returns (dz, dy, dx, domain_slices) with absent axes giving zeros."""
    x = np.asarray(x, dtype=np.float64)
    sl = tuple(slice(1, None) if n > 1 else slice(None) for n in x.shape)
    core = x[sl]
    d = []
    for ax, n in enumerate(x.shape):
        if n > 1:
            back = list(sl)
            back[ax] = slice(0, -1)
            d.append(core - x[tuple(back)])
        else:
            d.append(np.zeros_like(core))
    return d[0], d[1], d[2], sl


def _w(d, delta):
    if not np.isfinite(delta):
        return np.ones_like(d)
    return np.exp(-(d / delta) ** 2)          # eq. (8)


def awtv(x, delta=np.inf, eps=0.0):
    """AwTV(x) of eq. (7) in three dimensions (P20); delta = inf is the TV norm."""
    dz, dy, dx, _ = _diffs(x)
    q = _w(dx, delta) * dx ** 2 + _w(dy, delta) * dy ** 2 + _w(dz, delta) * dz ** 2 + eps
    return float(np.sum(np.sqrt(q)))


def awtv_gradient(x, delta=np.inf, eps=1e-8):
    """Gradient of awtv(x, delta, eps) with respect to every voxel (P21), same shape as x."""
    x = np.asarray(x, dtype=np.float64)
    dz, dy, dx, sl = _diffs(x)
    wz, wy, wx = _w(dz, delta), _w(dy, delta), _w(dx, delta)
    T = np.sqrt(wx * dx ** 2 + wy * dy ** 2 + wz * dz ** 2 + eps)

    def a(d, w):                              # d T / d d  =  d w (1 - d^2/delta^2) / T
        f = 1.0 if not np.isfinite(delta) else (1.0 - (d / delta) ** 2)
        with np.errstate(invalid="ignore", divide="ignore"):
            out = np.where(T > 0, d * w * f / T, 0.0)
        return out

    g = np.zeros_like(x)
    for ax, (d, w) in enumerate(((dz, wz), (dy, wy), (dx, wx))):
        if x.shape[ax] == 1:
            continue
        aa = a(d, w)
        g[sl] += aa                           # x[p] enters its own term with +1 ...
        back = list(sl)
        back[ax] = slice(0, -1)
        g[tuple(back)] -= aa                  # ... and the term of p + e_a with -1
    return g


def minimize_awtv(x, n_steps, alpha, delta=np.inf, eps=1e-8):
    """P22: n_steps of normalised steepest descent on awtv."""
    x = np.array(x, dtype=np.float64)
    for _ in range(n_steps):
        g = awtv_gradient(x, delta, eps)
        nrm = float(np.sqrt(np.sum(g * g)))
        if nrm == 0.0:
            break
        x = x - alpha * g / nrm
    return x
