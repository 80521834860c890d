"""oracle/oracle.py — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Python face of the fp64 CPU oracle (oracle/tigre_oracle.c) plus the iteration drivers
written out in numpy, step by step in the order of SURVEY.md §8(c) O-D..O-F (DESIGN.md
"Readings of the paper").  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this module.  It imports nothing from
paper_2412_10129_b200/ and shares no code with it; inputs come from workloads/.

Citations: eq. 1 (b = Ax, line integrals); 102 eq. 4 (gradient step);
115 (SART/OS-SART/SIRT: row/column reweighting, nonnegativity); 135 eq. 6 (subset update);
90, 114 (FDK); 117, 130 (CGLS); 179-197, 543-566 (geometry).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

SIDDON, INTERP = 0, 1
MATCHED, FDK = 0, 1


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("nu", C.c_int32), ("nv", C.c_int32), ("parallel", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("du", C.c_double), ("dv", C.c_double), ("accuracy", C.c_double)]


_VIEW_DOUBLES = 3 + 3 + 2 + 3 + 3   # DSD DSO COR offO[3] offD[2] rotD[3] ang[3]
_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_ax.restype = C.c_int
        _lib.orc_atb.restype = C.c_int
        _lib.orc_atb_exact.restype = C.c_int
        _lib.orc_fdk_filter.restype = C.c_int
        _lib.orc_siddon_segments.restype = C.c_int
        _lib.orc_siddon_index.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def set_num_threads(n: int) -> None:
    """OpenMP threads the C routines use from now on (bench.py's single-thread leg)."""
    lib().orc_set_num_threads(int(n))


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _grid(geo) -> _Grid:
    return _Grid(geo.nVoxel[0], geo.nVoxel[1], geo.nVoxel[2], geo.nDetector[0], geo.nDetector[1],
                 1 if getattr(geo, "mode", "cone") == "parallel" else 0,
                 geo.dVoxel[0], geo.dVoxel[1], geo.dVoxel[2], geo.dDetector[0], geo.dDetector[1],
                 geo.accuracy)


def _views(geo, angles) -> np.ndarray:
    """[nA][14] table of per-view parameters (marshalling of the per-angle overrides only)."""
    angles = np.ascontiguousarray(angles, dtype=np.float64).reshape(-1, 3)
    nA = angles.shape[0]
    t = np.zeros((nA, _VIEW_DOUBLES), dtype=np.float64)

    def pick(scalar, arr, width):
        if arr is None:
            return np.broadcast_to(np.asarray(scalar, dtype=np.float64).reshape(1, width), (nA, width))
        return np.asarray(arr, dtype=np.float64).reshape(nA, width)

    t[:, 0:1] = pick(geo.DSD, geo.DSD_a, 1)
    t[:, 1:2] = pick(geo.DSO, geo.DSO_a, 1)
    t[:, 2:3] = pick(geo.COR, geo.COR_a, 1)
    t[:, 3:6] = pick(geo.offOrigin, geo.offOrigin_a, 3)
    t[:, 6:8] = pick(geo.offDetector, geo.offDetector_a, 2)
    t[:, 8:11] = pick(geo.rotDetector, geo.rotDetector_a, 3)
    t[:, 11:14] = angles
    return np.ascontiguousarray(t)


def _as_in(a):
    a = np.ascontiguousarray(a)
    if a.dtype == np.float32:
        return a, 1
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, 0


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


# ------------------------------------------------------------------ projectors
def ax(vol, geo, angles, mode=SIDDON, ray_ids=None, info=False):
    """Forward projection (O-A Siddon / O-B interpolated).  Returns float64 [nA][nv][nu],
    or [n] for the sampled rays `ray_ids` (linear ids (ia*nv+iv)*nu+iu).
    info=True also returns dict(nseg, first_vox, last_vox)."""
    g = _grid(geo)
    v = _views(geo, angles)
    nA = v.shape[0]
    vol, f32 = _as_in(vol)
    assert vol.size == np.prod(geo.vol_shape)
    if ray_ids is None:
        n = nA * g.nu * g.nv
        ids = None
        shape = (nA, g.nv, g.nu)
    else:
        ids = np.ascontiguousarray(ray_ids, dtype=np.int64)
        n = ids.size
        shape = (n,)
    out = np.zeros(n, dtype=np.float64)
    nseg = np.zeros(n, dtype=np.int64) if info else None
    fv = np.zeros(n, dtype=np.int64) if info else None
    lv = np.zeros(n, dtype=np.int64) if info else None
    rc = lib().orc_ax(_ptr(vol), f32, C.byref(g), _ptr(v), nA, int(mode), _ptr(ids), C.c_int64(n),
                      _ptr(out), _ptr(nseg), _ptr(fv), _ptr(lv))
    assert rc == 0
    out = out.reshape(shape)
    if info:
        return out, dict(nseg=nseg.reshape(shape), first_vox=fv.reshape(shape), last_vox=lv.reshape(shape))
    return out


def atb(proj, geo, angles, mode=MATCHED, vox_ids=None, return_fuv=False):
    """Voxel-driven backprojection (O-C).  proj=None means all-ones projections (A^T 1).
    Returns float64 [nz][ny][nx] or [n] for sampled voxels (linear ids (iz*ny+iy)*nx+ix)."""
    g = _grid(geo)
    v = _views(geo, angles)
    nA = v.shape[0]
    unit = proj is None
    if unit:
        p, f32 = None, 0
    else:
        p, f32 = _as_in(proj)
        assert p.size == nA * g.nu * g.nv
    if vox_ids is None:
        n, ids, shape = g.nx * g.ny * g.nz, None, geo.vol_shape
    else:
        ids = np.ascontiguousarray(vox_ids, dtype=np.int64)
        n, shape = ids.size, (ids.size,)
    out = np.zeros(n, dtype=np.float64)
    fuv = np.zeros((n, nA, 2), dtype=np.float64) if return_fuv else None
    rc = lib().orc_atb(_ptr(p), f32, int(unit), C.byref(g), _ptr(v), nA, int(mode), _ptr(ids),
                       C.c_int64(n), _ptr(out), _ptr(fuv))
    if rc != 0:
        raise ValueError("geometry error: a voxel lies at or behind the source plane")
    out = out.reshape(shape)
    return (out, fuv) if return_fuv else out


def atb_exact(proj, geo, angles, ax_mode=SIDDON):
    """Exact transpose of ax(.., ax_mode): ray-driven scatter of the same weights (P11)."""
    g = _grid(geo)
    v = _views(geo, angles)
    p, f32 = _as_in(proj)
    out = np.zeros(g.nx * g.ny * g.nz, dtype=np.float64)
    rc = lib().orc_atb_exact(_ptr(p), f32, C.byref(g), _ptr(v), v.shape[0], int(ax_mode), _ptr(out))
    assert rc == 0
    return out.reshape(geo.vol_shape)


def siddon_index(geo, angles, ray_ids):
    """Reading P19(a): per ray the segment count, the voxel index of the first / second / second-to-last / last segment, the
    parameter lengths of the first and last segment and the smallest gap between consecutive crossings (knife-edge flags)."""
    g = _grid(geo)
    v = _views(geo, angles)
    ids = np.ascontiguousarray(ray_ids, dtype=np.int64)
    n = ids.size
    nseg = np.zeros(n, dtype=np.int64)
    vox4 = np.zeros((n, 4), dtype=np.int64)
    ft, lt, mg = np.zeros(n), np.zeros(n), np.zeros(n)
    rc = lib().orc_siddon_index(C.byref(g), _ptr(v), v.shape[0], _ptr(ids), C.c_int64(n), _ptr(nseg), _ptr(vox4), _ptr(ft), _ptr(lt), _ptr(mg))
    assert rc == 0
    return dict(nseg=nseg, first=vox4[:, 0], second=vox4[:, 1], second_last=vox4[:, 2], last=vox4[:, 3], first_t=ft, last_t=lt,
                min_gap=mg)


def siddon_segments(geo, angles, ia, iu, iv):
    g = _grid(geo)
    v = _views(geo, angles)
    cap = g.nx + g.ny + g.nz + 8
    idx = np.zeros(cap, dtype=np.int64)
    ln = np.zeros(cap, dtype=np.float64)
    n = lib().orc_siddon_segments(C.byref(g), _ptr(v), int(ia), int(iu), int(iv), _ptr(idx), _ptr(ln), cap)
    assert n >= 0
    return idx[:n].copy(), ln[:n].copy()


def source_pixel(geo, angles, ia, iu, iv):
    g = _grid(geo)
    v = _views(geo, angles)
    S = np.zeros(3)
    P = np.zeros(3)
    lib().orc_source_pixel(C.byref(g), _ptr(v), int(ia), C.c_double(iu), C.c_double(iv), _ptr(S), _ptr(P))
    return S, P


def voxel_map(geo, angles, ia, ix, iy, iz):
    g = _grid(geo)
    v = _views(geo, angles)
    X = np.zeros(3)
    fuv = np.zeros(2)
    lib().orc_voxel_map(C.byref(g), _ptr(v), int(ia), int(ix), int(iy), int(iz), _ptr(X), _ptr(fuv))
    return X, fuv


# ------------------------------------------------------------------ O-D FDK (P12)
def fdk_filter(proj, geo, angles):
    g = _grid(geo)
    v = _views(geo, angles)
    p, f32 = _as_in(proj)
    out = np.zeros(p.size, dtype=np.float64)
    rc = lib().orc_fdk_filter(_ptr(p), f32, C.byref(g), _ptr(v), v.shape[0], _ptr(out))
    assert rc == 0
    return out.reshape(v.shape[0], g.nv, g.nu)


def fdk(proj, geo, angles):
    """x = (dtheta/2) * sum_a w_F * bilinear(q_a), dtheta = 2 pi / nAngles (full circle)."""
    nA = np.asarray(angles).reshape(-1, 3).shape[0]
    q = fdk_filter(proj, geo, angles)
    return (2.0 * np.pi / nA) / 2.0 * atb(q, geo, angles, FDK)


# ------------------------------------------------------------------ O-E SIRT / OS-SART
def row_weights(geo, angles, ax_mode):
    """W = 1/(A 1) where (A 1) > eps_W = 1e-2*min(dVoxel), else 0 (P13)."""
    a1 = ax(np.ones(geo.vol_shape), geo, angles, ax_mode)
    eps = 1e-2 * min(geo.dVoxel)
    W = np.zeros_like(a1)
    np.divide(1.0, a1, out=W, where=a1 > eps)
    return W


def col_weights(geo, angles, atb_mode):
    """V = 1/(A^T 1) where (A^T 1) > eps_V = 1e-6 * max_j (A^T 1)_j, else 0 (P13, P16)."""
    at1 = atb(None, geo, angles, atb_mode)
    eps = 1e-6 * at1.max()
    V = np.zeros_like(at1)
    np.divide(1.0, at1, out=V, where=at1 > eps)
    return V


def _sub_geo(geo, idx):
    """Geometry restricted to the views idx (slices the per-angle arrays: marshalling only)."""
    kw = {}
    for name in ("DSD_a", "DSO_a", "COR_a", "offOrigin_a", "offDetector_a", "rotDetector_a"):
        a = getattr(geo, name)
        if a is not None:
            kw[name] = np.asarray(a)[idx]
    return geo.copy(**kw) if kw else geo


def ossart(b, geo, angles, subsets, n_iter, lam=1.0, nonneg=True, ax_mode=SIDDON, atb_mode=MATCHED,
           x0=None, trace=None, row_scale=None):
    """for it, for s:  r = W_s*(b_s - A_s x);  x += lam * V_s * A_s^T r;  x = max(x,0).
    SIRT is one subset holding all views.  resid[it] = sqrt(sum_s ||b_s - A_s x||^2) from the
    A_s x computed during the sweep (running residual).  Returns (x, resid)."""
    angles = np.asarray(angles, dtype=np.float64).reshape(-1, 3)
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(geo.vol_shape) if x0 is None else np.array(x0, dtype=np.float64)
    subsets = [np.asarray(s, dtype=np.int64) for s in subsets]
    Ws = [row_weights(_sub_geo(geo, s), angles[s], ax_mode) for s in subsets]
    if row_scale is not None:
        # data-redundancy weighting (reading P17): the row weights of view a, column u are multiplied
        # by row_scale[a][u] (the displaced-detector weights of oracle/fdk_ext.py, P28)
        rs = np.asarray(row_scale, dtype=np.float64)
        Ws = [W * rs[s][:, None, :] for W, s in zip(Ws, subsets)]
    Vs = [col_weights(_sub_geo(geo, s), angles[s], atb_mode) for s in subsets]
    resid = np.zeros(n_iter)
    for it in range(n_iter):
        acc = 0.0
        for s, W, V in zip(subsets, Ws, Vs):
            gs = _sub_geo(geo, s)
            d = b[s] - ax(x, gs, angles[s], ax_mode)
            acc += float(np.sum(d * d))
            r = W * d
            x = x + lam * V * atb(r, gs, angles[s], atb_mode)
            if nonneg:
                x = np.maximum(x, 0.0)
            if trace is not None:
                trace.append(x.copy())
        resid[it] = np.sqrt(acc)
    return x, resid


def sirt(b, geo, angles, n_iter, **kw):
    nA = np.asarray(angles).reshape(-1, 3).shape[0]
    return ossart(b, geo, angles, [np.arange(nA)], n_iter, **kw)


# ------------------------------------------------------------------ O-F CGLS (textbook, PAPER.md:463 ref [35])
def cgls(b, geo, angles, n_iter, ax_mode=SIDDON, atb_mode=MATCHED, exact_adjoint=False):
    """r = b - A x0 (x0 = 0); s = A^T r; p = s; gamma = ||s||^2; repeat: q = A p;
    alpha = gamma/||q||^2; x += alpha p; r -= alpha q; s = A^T r; gamma' = ||s||^2;
    beta = gamma'/gamma; p = s + beta p.  resid[it] = ||r|| after the update."""
    AT = (lambda y: atb_exact(y, geo, angles, ax_mode)) if exact_adjoint else \
         (lambda y: atb(y, geo, angles, atb_mode))
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(geo.vol_shape)
    r = b.copy()
    s = AT(r)
    p = s.copy()
    gamma = float(np.sum(s * s))
    resid = np.zeros(n_iter)
    for it in range(n_iter):
        q = ax(p, geo, angles, ax_mode)
        alpha = gamma / float(np.sum(q * q))
        x = x + alpha * p
        r = r - alpha * q
        s = AT(r)
        gamma_new = float(np.sum(s * s))
        beta = gamma_new / gamma
        p = s + beta * p
        gamma = gamma_new
        resid[it] = np.sqrt(float(np.sum(r * r)))
    return x, resid


# ------------------------------------------------------------------ gradient descent, eq. (4)
def gradient_descent(b, geo, angles, n_iter, lam, ax_mode=SIDDON, atb_mode=MATCHED, exact_adjoint=False, x0=None):
    """x^k = x^{k-1} + lam A^T (b - A x^{k-1}) (eq. 4; the paper prints the residual as (Ax - b): with that sign the
    iteration ascends, so the descent sign is taken: reading P32).  resid[k] = ||b - A x^{k-1}||_2."""
    AT = (lambda y: atb_exact(y, geo, angles, ax_mode)) if exact_adjoint else (lambda y: atb(y, geo, angles, atb_mode))
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(geo.vol_shape) if x0 is None else np.array(x0, dtype=np.float64)
    resid = np.zeros(n_iter)
    for k in range(n_iter):
        r = b - ax(x, geo, angles, ax_mode)
        resid[k] = np.sqrt(float(np.sum(r * r)))
        x = x + lam * AT(r)
    return x, resid


# ------------------------------------------------------------------ MLEM / OSEM, eq. (5); 118-120, 139
def osem(b, geo, angles, subsets, n_iter, ax_mode=SIDDON, atb_mode=MATCHED, exact_adjoint=False, x0=None):
    """x <- x / (A_s^T 1) * A_s^T (b_s / (A_s x)) for every subset s in turn (one subset holding all views: MLEM, eq. 5).
    Reading P33: the quotient is 0 where A_s x <= 0 (rays that miss the support), the column normalisation 1/(A_s^T 1) is
    0 where A_s^T 1 <= 1e-6 max (as V in P13); x0 = ones unless given."""
    angles = np.asarray(angles, dtype=np.float64).reshape(-1, 3)
    b = np.asarray(b, dtype=np.float64)
    x = np.ones(geo.vol_shape) if x0 is None else np.array(x0, dtype=np.float64)
    subsets = [np.asarray(s, dtype=np.int64) for s in subsets]

    def AT(y, gs, a):
        return atb_exact(y, gs, a, ax_mode) if exact_adjoint else atb(y, gs, a, atb_mode)

    Vs = []
    for s in subsets:
        gs = _sub_geo(geo, s)
        at1 = AT(np.ones((len(s),) + geo.proj_shape), gs, angles[s])
        V = np.zeros_like(at1)
        np.divide(1.0, at1, out=V, where=at1 > 1e-6 * at1.max())
        Vs.append(V)
    for _ in range(n_iter):
        for s, V in zip(subsets, Vs):
            gs = _sub_geo(geo, s)
            p = ax(x, gs, angles[s], ax_mode)
            ratio = np.zeros_like(p)
            np.divide(b[s], p, out=ratio, where=p > 0.0)
            x = x * V * AT(ratio, gs, angles[s])
    return x


def mlem(b, geo, angles, n_iter, **kw):
    nA = np.asarray(angles).reshape(-1, 3).shape[0]
    return osem(b, geo, angles, [np.arange(nA)], n_iter, **kw)
