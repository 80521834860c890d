"""oracle/pocs.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

fp64 numpy oracle of the ASD-POCS family: ASD-POCS, its ordered-subsets version
OS-ASD-POCS and their adaptive-weighted variants (AwASD-POCS), PAPER.md:116 ("Projection Onto Convex Sets ...
Adaptive Steepest Descend version (ASD-POCS) [30] ... Versions of these two algorithms exists for the Adaptive
weighed TV norm [32, 33], and OS versions exist for the first with both TV norms"), PAPER.md:141-149 (OS
counterparts, Snippet 1) and PAPER.md:169 ("The AwTV norm can be now used with any POCS-type algorithm").
Only tests/ may import this module; it shares nothing with paper_2412_10129_b200/.

The paper names the algorithm and cites [30] for it but prints no pseudo-code, so the loop below is a READING
(P23 in DESIGN.md section 2): the adaptive-steepest-descent / projection-onto-convex-sets alternation of [30]
restated with the pieces this oracle already has,

  for it = 0 .. n_iter-1:
      x0 = x
      (data step, "POCS")   one OS-SART sweep over the subsets with relaxation beta, nonnegativity on
                            (oracle.ossart, eq. 6 with the row / column weights; single-view subsets = SART)
      beta  <- beta * beta_red
      dd    = || A x - b ||_2                      (a fresh forward projection of the new iterate, all views)
      dp    = || x - x0 ||_2
      if it == 0:  dtvg = alpha * dp               (the TV step length is tied to the first data step)
      xp = x
      (regulariser step)    ng steps of  x <- x - dtvg * g / ||g||_2,  g = gradient of (Aw)TV   (oracle.tv, P20-P22)
      dg    = || x - xp ||_2
      if dg > r_max * dp and dd > epsilon:  dtvg <- dtvg * alpha_red
      c     = <x - xp, xp - x0> / (dg * dp)        (cosine between the two steps; 0 if either vanishes)
      stop after this iteration if (c < -0.99 and dd <= epsilon) or beta < 0.005

hist[it] = (dd, dp, dg, dtvg used in this iteration's TV step, c).
"""
from __future__ import annotations

import numpy as np

from . import oracle as orc
from . import tv as otv


def asd_pocs(b, geo, angles, subsets, n_iter, beta=1.0, beta_red=0.99, ng=20, alpha=0.002, alpha_red=0.95,
             r_max=0.95, epsilon=0.0, delta=np.inf, tv_eps=1e-8, ax_mode=orc.SIDDON, atb_mode=orc.MATCHED, x0=None):
    """Returns (x, hist[n_done][5]).  subsets: list of view-index lists (ASD-POCS: one view each; OS-ASD-POCS:
    blocks).  delta finite = AwASD-POCS."""
    angles = np.asarray(angles, dtype=np.float64).reshape(-1, 3)
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(geo.vol_shape) if x0 is None else np.array(x0, dtype=np.float64)
    subsets = [np.asarray(s, dtype=np.int64) for s in subsets]
    Ws = [orc.row_weights(orc._sub_geo(geo, s), angles[s], ax_mode) for s in subsets]
    Vs = [orc.col_weights(orc._sub_geo(geo, s), angles[s], atb_mode) for s in subsets]
    hist = []
    dtvg = 0.0
    for it in range(n_iter):
        xstart = x.copy()
        # ---- data step: one OS-SART sweep with relaxation beta
        for s, W, V in zip(subsets, Ws, Vs):
            gs = orc._sub_geo(geo, s)
            r = W * (b[s] - orc.ax(x, gs, angles[s], ax_mode))
            x = np.maximum(x + beta * V * orc.atb(r, gs, angles[s], atb_mode), 0.0)
        beta *= beta_red
        d = orc.ax(x, geo, angles, ax_mode) - b
        dd = float(np.sqrt(np.sum(d * d)))
        dpv = x - xstart
        dp = float(np.sqrt(np.sum(dpv * dpv)))
        if it == 0:
            dtvg = alpha * dp
        xp = x.copy()
        # ---- regulariser step: ng normalised steepest-descent steps on (Aw)TV with step length dtvg
        used = dtvg
        x = otv.minimize_awtv(x, ng, dtvg, delta, tv_eps)
        dgv = x - xp
        dg = float(np.sqrt(np.sum(dgv * dgv)))
        if dg > r_max * dp and dd > epsilon:
            dtvg *= alpha_red
        c = float(np.sum(dgv * dpv) / (dg * dp)) if dg > 0.0 and dp > 0.0 else 0.0
        hist.append((dd, dp, dg, used, c))
        if (c < -0.99 and dd <= epsilon) or beta < 0.005:
            break
    return x, np.array(hist, dtype=np.float64).reshape(-1, 5)


def sart_tv(b, geo, angles, subsets, n_iter, lam=1.0, lam_red=1.0, tv_lambda=0.0, tv_iter=10, ax_mode=orc.SIDDON,
            atb_mode=orc.MATCHED, x0=None):
    """SART-TV ("TIGRE also includes the SART-TV algorithm [44] ... can also be interpreted as a proximal
    method", used at PAPER.md:365): reading P31: per iteration one OS-SART sweep with relaxation lam (single-view subsets:
    SART), then the TV proximal operator of oracle/prox.py (P24) with weight tv_lambda and tv_iter dual iterations;
    lam <- lam * lam_red.  Returns (x, resid) with resid[it] the running residual of the sweep (as oracle.ossart)."""
    from . import prox as oprox
    angles = np.asarray(angles, dtype=np.float64).reshape(-1, 3)
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(geo.vol_shape) if x0 is None else np.array(x0, dtype=np.float64)
    subsets = [np.asarray(s, dtype=np.int64) for s in subsets]
    Ws = [orc.row_weights(orc._sub_geo(geo, s), angles[s], ax_mode) for s in subsets]
    Vs = [orc.col_weights(orc._sub_geo(geo, s), angles[s], atb_mode) for s in subsets]
    resid = np.zeros(n_iter)
    for it in range(n_iter):
        acc = 0.0
        for s, W, V in zip(subsets, Ws, Vs):
            gs = orc._sub_geo(geo, s)
            d = b[s] - orc.ax(x, gs, angles[s], ax_mode)
            acc += float(np.sum(d * d))
            x = np.maximum(x + lam * V * orc.atb(W * d, gs, angles[s], atb_mode), 0.0)
        resid[it] = np.sqrt(acc)
        x = oprox.tv_prox(x, tv_lambda, tv_iter)
        lam *= lam_red
    return x, resid
