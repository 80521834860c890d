"""oracle/curved.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

fp64 numpy oracle of the curved-detector "flattening" ("Curved detectors ...
(with equidistant source-detector distance in each pixel) ... TIGRE now allows to consider curved detectors by applying
a 'flattening' transformation").  The paper gives no formula; reading P30: the curved detector
is the cylinder of radius DSD about the axis through the source parallel to the detector's v axis; its pixel (i, j)
sits at arc length s_i = (i + 1/2) du - nu du/2 from the central ray (fan angle s_i/DSD) and height
v_j = (j + 1/2) dv - nv dv/2.  The ray to the FLAT pixel at (u, v) (plane at distance DSD) has fan angle
gamma = atan(u/DSD) and meets the cylinder at arc length DSD gamma and height v cos(gamma); the flattened image is the
curved one interpolated bilinearly there (zero outside).  offDetector, rotDetector shift / rotate both detectors alike
and drop out.  Only tests/ may import this module.
"""
from __future__ import annotations

import numpy as np


def flatten(curved, geo, n_angles=None):
    """curved [nA][nv][nu] -> flat [nA][nv][nu] (same pixel counts and pitches on both detectors)."""
    p = np.asarray(curved, dtype=np.float64)
    nA = p.shape[0]
    nu, nv = geo.nDetector
    du, dv = geo.dDetector
    dsd_a = getattr(geo, "DSD_a", None)
    DSD = np.full(nA, float(geo.DSD)) if dsd_a is None else np.asarray(dsd_a, dtype=np.float64).reshape(nA)
    u = (np.arange(nu) + 0.5) * du - 0.5 * nu * du
    v = (np.arange(nv) + 0.5) * dv - 0.5 * nv * dv
    out = np.zeros_like(p)
    for a in range(nA):
        gamma = np.arctan(u / DSD[a])
        fi = (DSD[a] * gamma + 0.5 * nu * du) / du - 0.5                     # continuous column index on the arc
        fj = (np.multiply.outer(v, np.cos(gamma)) + 0.5 * nv * dv) / dv - 0.5   # [nv][nu] continuous row index
        i0 = np.floor(fi).astype(int)
        ai = fi - i0
        j0 = np.floor(fj).astype(int)
        aj = fj - j0
        acc = np.zeros((nv, nu))
        for cj in (0, 1):
            for ci in (0, 1):
                ii = np.broadcast_to(i0 + ci, (nv, nu))
                jj = j0 + cj
                w = np.broadcast_to(ai if ci else 1.0 - ai, (nv, nu)) * (aj if cj else 1.0 - aj)
                ok = (ii >= 0) & (ii < nu) & (jj >= 0) & (jj < nv)
                acc += np.where(ok, w * p[a][np.clip(jj, 0, nv - 1), np.clip(ii, 0, nu - 1)], 0.0)
        out[a] = acc
    return out
