"""Independent geometry and closed forms used to PIN the oracle (tests only).

Nothing here calls oracle/ or the CUDA path.  Rotations come from scipy's Rotation
(a library routine), positions are written from the definitions of PAPER.md App. B
Table B1 (lines 543-566) under the readings P2-P6 of DESIGN.md; the voxel -> detector
map is solved as a WORLD-frame ray/plane intersection (the oracle works in the detector
frame), the Siddon pin is a per-voxel ray/box intersection (the oracle merges sorted
plane crossings).
"""
import numpy as np
from scipy.spatial.transform import Rotation as Rot


def view_params(geo, angles, ia):
    def pick(s, a):
        return np.asarray(s if a is None else np.asarray(a)[ia], dtype=np.float64)
    return dict(DSD=float(pick(geo.DSD, geo.DSD_a)), DSO=float(pick(geo.DSO, geo.DSO_a)),
                COR=float(pick(geo.COR, geo.COR_a)), offO=pick(geo.offOrigin, geo.offOrigin_a),
                offD=pick(geo.offDetector, geo.offDetector_a),
                rotD=pick(geo.rotDetector, geo.rotDetector_a),
                ang=np.asarray(angles, dtype=np.float64).reshape(-1, 3)[ia])


def world_frame(geo, angles, ia):
    """Source S, detector centre Dc, unit pixel axes eu, ev and normal n, all in world coords."""
    p = view_params(geo, angles, ia)
    Rg = Rot.from_euler("ZYZ", p["ang"]).as_matrix()                  # intrinsic z-y'-z''
    Rd = Rot.from_euler("ZYX", [p["rotD"][2], p["rotD"][1], p["rotD"][0]]).as_matrix()
    shift = np.array([0.0, -p["COR"], 0.0])
    S = Rg @ (np.array([p["DSO"], 0.0, 0.0]) + shift)
    Dc = Rg @ (np.array([p["DSO"] - p["DSD"], p["offD"][0], p["offD"][1]]) + shift)
    eu = Rg @ Rd @ np.array([0.0, 1.0, 0.0])
    ev = Rg @ Rd @ np.array([0.0, 0.0, 1.0])
    n = Rg @ Rd @ np.array([1.0, 0.0, 0.0])
    return S, Dc, eu, ev, n, p


def pixel_world(geo, angles, ia, iu, iv):
    S, Dc, eu, ev, n, p = world_frame(geo, angles, ia)
    u = (np.asarray(iu) + 0.5) * geo.dDetector[0] - 0.5 * geo.nDetector[0] * geo.dDetector[0]
    v = (np.asarray(iv) + 0.5) * geo.dDetector[1] - 0.5 * geo.nDetector[1] * geo.dDetector[1]
    return S, Dc + np.multiply.outer(u, eu) + np.multiply.outer(v, ev)


def parallel_rays(geo, angles, ia, iu, iv):
    """Parallel-beam mode (reading P29), independently of the oracle: start and end points of the rays of pixels
    (iu, iv): every ray runs along the gantry-rotated x axis and ends at its pixel, starting DSD in front of it."""
    S, Dc, eu, ev, n, p = world_frame(geo, angles, ia)
    u = (np.asarray(iu) + 0.5) * geo.dDetector[0] - 0.5 * geo.nDetector[0] * geo.dDetector[0]
    v = (np.asarray(iv) + 0.5) * geo.dDetector[1] - 0.5 * geo.nDetector[1] * geo.dDetector[1]
    P = Dc + np.multiply.outer(u, eu) + np.multiply.outer(v, ev)
    ex = Rot.from_euler("ZYZ", p["ang"]).as_matrix() @ np.array([1.0, 0.0, 0.0])
    return P + p["DSD"] * ex, P


def parallel_voxel_to_detector(geo, angles, ia, X):
    """Parallel-beam mode: continuous pixel index of the point where the ray through X (direction: gantry x axis) meets
    the detector plane, and the cosine between ray and detector normal."""
    S, Dc, eu, ev, n, p = world_frame(geo, angles, ia)
    ex = Rot.from_euler("ZYZ", p["ang"]).as_matrix() @ np.array([1.0, 0.0, 0.0])
    t = ((Dc - X) @ n) / (ex @ n)
    hit = X + t[..., None] * ex
    fu = ((hit - Dc) @ eu + 0.5 * geo.nDetector[0] * geo.dDetector[0]) / geo.dDetector[0] - 0.5
    fv = ((hit - Dc) @ ev + 0.5 * geo.nDetector[1] * geo.dDetector[1]) / geo.dDetector[1] - 0.5
    return fu, fv, abs(float(ex @ n))


def vol_box(geo, offO):
    s = np.array(geo.nVoxel) * np.array(geo.dVoxel)
    b0 = np.asarray(offO) - 0.5 * s
    return b0, b0 + s


def voxel_centres(geo, offO):
    """[nz][ny][nx][3] world coordinates of the voxel centres."""
    b0, _ = vol_box(geo, offO)
    ax = [b0[k] + (np.arange(geo.nVoxel[k]) + 0.5) * geo.dVoxel[k] for k in range(3)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return np.stack([X, Y, Z], -1)


def segment_box_length(S, P, lo, hi):
    """Length of segment S->P inside each axis-aligned box [lo_j, hi_j] (vectorised over boxes)."""
    d = P - S
    L = np.linalg.norm(d)
    tmin = np.zeros(lo.shape[:-1])
    tmax = np.ones(lo.shape[:-1])
    for k in range(3):
        if d[k] == 0.0:
            inside = (S[k] >= lo[..., k]) & (S[k] <= hi[..., k])
            tmin = np.where(inside, tmin, 1.0)
            tmax = np.where(inside, tmax, 0.0)
        else:
            t1 = (lo[..., k] - S[k]) / d[k]
            t2 = (hi[..., k] - S[k]) / d[k]
            tmin = np.maximum(tmin, np.minimum(t1, t2))
            tmax = np.minimum(tmax, np.maximum(t1, t2))
    return np.maximum(tmax - tmin, 0.0) * L


def segment_box_params(S, P, lo, hi):
    """Entry and exit parameters (t in [0,1] along S->P) of the segment in each box; exit <= entry where it misses."""
    d = P - S
    tmin = np.zeros(lo.shape[:-1])
    tmax = np.ones(lo.shape[:-1])
    for k in range(3):
        if d[k] == 0.0:
            inside = (S[k] >= lo[..., k]) & (S[k] <= hi[..., k])
            tmin = np.where(inside, tmin, 1.0)
            tmax = np.where(inside, tmax, 0.0)
        else:
            t1 = (lo[..., k] - S[k]) / d[k]
            t2 = (hi[..., k] - S[k]) / d[k]
            tmin = np.maximum(tmin, np.minimum(t1, t2))
            tmax = np.minimum(tmax, np.maximum(t1, t2))
    return tmin, tmax


def brute_force_ax(vol, geo, angles):
    """Sum over ALL voxels of (segment length inside that voxel's box) * value."""
    nA = np.asarray(angles).reshape(-1, 3).shape[0]
    nu, nv = geo.nDetector
    out = np.zeros((nA, nv, nu))
    h = np.array(geo.dVoxel)
    for ia in range(nA):
        p = view_params(geo, angles, ia)
        c = voxel_centres(geo, p["offO"])
        lo, hi = c - 0.5 * h, c + 0.5 * h
        for iv in range(nv):
            for iu in range(nu):
                S, P = pixel_world(geo, angles, ia, iu, iv)
                out[ia, iv, iu] = np.sum(segment_box_length(S, P, lo, hi) * vol)
    return out


def ellipsoid_line_integrals(ell, S, P):
    """Closed-form line integral of additive homogeneous ellipsoids along the infinite line
    through S and P (P: [...,3]); textbook quadratic: chord = 2 sqrt(B^2 - AC)/A."""
    w = P - S
    w = w / np.linalg.norm(w, axis=-1, keepdims=True)
    tot = np.zeros(w.shape[:-1])
    for c, a, Q, rho in zip(ell["centre"], ell["axes"], ell["Q"], ell["rho"]):
        m = (Q.T @ (S - c)) / a
        d = (w @ Q) / a
        A = np.sum(d * d, -1)
        B = d @ m
        Cc = m @ m - 1.0
        disc = B * B - A * Cc
        tot += rho * np.where(disc > 0, 2.0 * np.sqrt(np.maximum(disc, 0.0)) / A, 0.0)
    return tot


def voxel_to_detector(geo, angles, ia, X):
    """World-frame ray/plane intersection: continuous pixel index (fu,fv) of voxel centres X[...,3],
    plus R=|hit-S|, r=|X-S|, cos(gamma) and the FDK depth DSO - X'_x."""
    S, Dc, eu, ev, n, p = world_frame(geo, angles, ia)
    d = X - S
    t = ((Dc - S) @ n) / (d @ n)
    hit = S + t[..., None] * d
    u = (hit - Dc) @ eu
    v = (hit - Dc) @ ev
    fu = (u + 0.5 * geo.nDetector[0] * geo.dDetector[0]) / geo.dDetector[0] - 0.5
    fv = (v + 0.5 * geo.nDetector[1] * geo.dDetector[1]) / geo.dDetector[1] - 0.5
    R = np.linalg.norm(hit - S, axis=-1)
    r = np.linalg.norm(d, axis=-1)
    cosg = np.abs((hit - S) @ n) / R
    Rg = Rot.from_euler("ZYZ", p["ang"]).as_matrix()
    depth = p["DSO"] - (X @ Rg)[..., 0]          # (Rg^T X)_x ; COR only shifts y
    return fu, fv, R, r, cosg, depth


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
