"""oracle/fdk_ext.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

fp64 numpy oracle of the FDK variants of SURVEY.md section 8(f).4: the filter family and the two redundancy weightings
the paper names ("FBP and FDK [24], with various filter types and geometric correction methods, such as
Wang [25] and Parker [26] weights for detector displacement and angular range corrections, respectively"; a
Shepp-Logan filtered FDK is used at PAPER.md:359, a 200-degree arc at 281).  Only tests/ may import this module.

The paper prints none of the formulas; the readings:

P26  filters: the Ram-Lak taps of P12 (h0 = 1/(4 tau^2), h_odd = -1/(pi n tau)^2) on a grid of L = 2^ceil(log2(2 nu))
     samples, transformed to frequency, multiplied by a window W(omega), omega_k = 2 pi k / L in [0, pi] (mirrored), and
     applied by circular convolution to the zero-padded, cosine-weighted row (L >= 2 nu: no wrap):
         ram_lak 1;  shepp_logan sin(omega/2)/(omega/2);  cosine cos(omega/2);
         hamming 0.54 + 0.46 cos(omega);  hann 0.5 + 0.5 cos(omega).
P27  Parker weights (angular range Theta = |theta_last - theta_first| = pi + 2 eps < 2 pi, monotone angles): with
     beta = |theta - theta_first| and gamma = -dir * atan(u / DSD) (u = detector coordinate of the column incl.
     offDetector_u, dir = sign of the rotation; the sign makes (beta + pi + 2 gamma, -gamma) the conjugate ray),
         w = sin^2(pi/4 * beta / (eps - gamma))                 0 <= beta < 2 eps - 2 gamma
             1                                                  2 eps - 2 gamma <= beta <= pi - 2 gamma
             sin^2(pi/4 * (pi + 2 eps - beta) / (eps + gamma))  pi - 2 gamma < beta <= pi + 2 eps
     and the FDK sum is scaled by dtheta = Theta/(nA - 1) (no factor 1/2: every line is counted once).
P28  Wang weights (detector displaced along u, full circle): the columns |u| <= u_ov = nu du/2 - |offDetector_u| are
     measured twice, the rest once or never:
         w(u) = 1/2 (sin(pi/2 * atan(u s / DSD) / atan(u_ov / DSD)) + 1)  for |u| <= u_ov,  1 for u s > u_ov,  0 else
     (s = sign of the displacement), and the projections are multiplied by 2 w before the full-circle FDK of P12.
"""
from __future__ import annotations

import numpy as np

from . import oracle as orc

FILTERS = ("ram_lak", "shepp_logan", "cosine", "hamming", "hann")


def window(name, L):
    """W(omega_k), k = 0..L-1 (mirrored about L/2)."""
    k = np.arange(L)
    k = np.minimum(k, L - k)
    om = 2.0 * np.pi * k / L
    if name == "ram_lak":
        return np.ones(L)
    if name == "shepp_logan":
        w = np.ones(L)
        nz = om > 0
        w[nz] = np.sin(om[nz] / 2) / (om[nz] / 2)
        return w
    if name == "cosine":
        return np.cos(om / 2)
    if name == "hamming":
        return 0.54 + 0.46 * np.cos(om)
    if name == "hann":
        return 0.5 + 0.5 * np.cos(om)
    raise ValueError(name)


def pad_length(nu):
    return 1 << int(np.ceil(np.log2(2 * nu)))


def filter_response(nu, tau, name):
    """Frequency response H(omega_k) * W(omega_k) on L samples (real: the taps are even)."""
    L = pad_length(nu)
    n = np.arange(L)
    n = np.where(n <= L // 2, n, n - L)                      # 0, 1, ..., L/2, -(L/2 - 1), ..., -1
    h = np.zeros(L)
    h[n == 0] = 1.0 / (4.0 * tau * tau)
    odd = (n % 2) != 0
    h[odd] = -1.0 / (np.pi * n[odd] * tau) ** 2
    return np.real(np.fft.fft(h)) * window(name, L)


def _per_view(geo, name, scalar, nA):
    a = getattr(geo, name + "_a", None)
    return np.full(nA, float(scalar)) if a is None else np.asarray(a, dtype=np.float64).reshape(nA)


def _u_coords(geo, nA):
    """Detector coordinate of every column, per view, including offDetector_u: [nA][nu]."""
    nu, du = geo.nDetector[0], geo.dDetector[0]
    u = (np.arange(nu) + 0.5) * du - 0.5 * nu * du
    off = getattr(geo, "offDetector_a", None)
    offu = np.full(nA, float(geo.offDetector[0])) if off is None else np.asarray(off, dtype=np.float64).reshape(nA, 2)[:, 0]
    return u[None, :] + offu[:, None]


def parker_weights(geo, angles):
    """P27: [nA][nu]."""
    th = np.asarray(angles, dtype=np.float64).reshape(-1, 3)[:, 0]
    nA = th.size
    DSD = _per_view(geo, "DSD", geo.DSD, nA)
    d = np.diff(th)
    if not (np.all(d > 0) or np.all(d < 0)):
        raise ValueError("Parker weights need monotone angles")
    direction = 1.0 if th[-1] > th[0] else -1.0
    Theta = abs(th[-1] - th[0])
    eps = 0.5 * (Theta - np.pi)
    beta = np.abs(th - th[0])[:, None]
    gamma = -direction * np.arctan(_u_coords(geo, nA) / DSD[:, None])
    w = np.ones_like(gamma)
    lo = beta < 2 * eps - 2 * gamma
    hi = beta > np.pi - 2 * gamma
    with np.errstate(divide="ignore", invalid="ignore"):
        wl = np.sin(np.pi / 4 * beta / (eps - gamma)) ** 2
        wh = np.sin(np.pi / 4 * (np.pi + 2 * eps - beta) / (eps + gamma)) ** 2
    w = np.where(lo, wl, w)
    w = np.where(hi, wh, w)
    return w


def wang_weights(geo, nA):
    """P28: [nA][nu] (the factor 2 not included)."""
    nu, du = geo.nDetector[0], geo.dDetector[0]
    DSD = _per_view(geo, "DSD", geo.DSD, nA)[:, None]
    uu = _u_coords(geo, nA)
    offu = uu[:, :1] - ((0 + 0.5) * du - 0.5 * nu * du)
    s = np.where(offu >= 0, 1.0, -1.0)
    u_ov = 0.5 * nu * du - np.abs(offu)
    t = uu * s
    w = 0.5 * (np.sin(0.5 * np.pi * np.arctan(t / DSD) / np.arctan(u_ov / DSD)) + 1.0)
    w = np.where(t > u_ov, 1.0, w)
    w = np.where(t < -u_ov, 0.0, w)
    return w


def fdk_filter(proj, geo, angles, filt="ram_lak", colw=None):
    """q = tau * ((proj * cos * colw) conv h_filt) per detector row, by zero padding to L and the FFT (P26)."""
    ang = np.asarray(angles, dtype=np.float64).reshape(-1, 3)
    nA = ang.shape[0]
    nu, nv = geo.nDetector
    du, dv = geo.dDetector
    DSD = _per_view(geo, "DSD", geo.DSD, nA)
    DSO = _per_view(geo, "DSO", geo.DSO, nA)
    u = (np.arange(nu) + 0.5) * du - 0.5 * nu * du
    v = (np.arange(nv) + 0.5) * dv - 0.5 * nv * dv
    offa = getattr(geo, "offDetector_a", None)
    offD = np.broadcast_to(np.asarray(geo.offDetector, dtype=np.float64), (nA, 2)) if offa is None else np.asarray(offa, dtype=np.float64).reshape(nA, 2)
    p = np.asarray(proj, dtype=np.float64).reshape(nA, nv, nu)
    out = np.zeros_like(p)
    L = pad_length(nu)
    par = getattr(geo, "mode", "cone") == "parallel"       # P29: no magnification, no cosine weight
    for a in range(nA):
        tau = du if par else du * DSO[a] / DSD[a]
        # P34: (u, v) of the cosine weight are measured from the principal ray, i.e. include offDetector
        cosw = 1.0 if par else DSD[a] / np.sqrt(DSD[a] ** 2 + (u[None, :] + offD[a, 0]) ** 2 + (v[:, None] + offD[a, 1]) ** 2)
        row = p[a] * cosw
        if colw is not None:
            row = row * colw[a][None, :]
        H = filter_response(nu, tau, filt)
        F = np.fft.fft(row, n=L, axis=1)
        out[a] = tau * np.real(np.fft.ifft(F * H[None, :], axis=1))[:, :nu]
    return out


def fdk(proj, geo, angles, filt="ram_lak", weighting=None):
    """FDK with a filter of P26 and weighting None (full circle, P12), 'parker' (P27) or 'wang' (P28)."""
    ang = np.asarray(angles, dtype=np.float64).reshape(-1, 3)
    nA = ang.shape[0]
    if weighting == "parker":
        colw = parker_weights(geo, ang)
        scale = abs(ang[-1, 0] - ang[0, 0]) / (nA - 1)
    elif weighting == "wang":
        colw = 2.0 * wang_weights(geo, nA)
        scale = (2.0 * np.pi / nA) / 2.0
    else:
        colw = None
        scale = (2.0 * np.pi / nA) / 2.0
    q = fdk_filter(proj, geo, ang, filt, colw)
    return scale * orc.atb(q, geo, ang, orc.FDK)
