"""Thin Python binding of libtigre_b200 (include/tigre_b200.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library; PyTorch is used for device memory
and streams.  There is no CPU fallback and no import of oracle/: if the shared library is
missing or no CUDA device is present, calls raise.

Functions mirror the C ABI names: Ax, Atb, row_weights, col_weights, residual, update,
ossart, sirt, cgls, fdk, fdk_filter, Ax_count.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtigre_b200.so")

AX_SIDDON, AX_INTERP = 0, 1
ATB_MATCHED, ATB_FDK = 0, 1
_AX_MODES = {"siddon": 0, "interp": 1, "interpolated": 1, 0: 0, 1: 1}
_ATB_MODES = {"matched": 0, "fdk": 1, "FDK": 1, "exact_siddon": 2, "exact_interp": 3, 0: 0, 1: 1, 2: 2, 3: 3}

_dp = C.POINTER(C.c_double)


class tigre_geo(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32),
        ("nVoxel", C.c_int32 * 3), ("dVoxel", C.c_double * 3),
        ("nDetector", C.c_int32 * 2), ("dDetector", C.c_double * 2),
        ("DSD", C.c_double), ("DSO", C.c_double), ("COR", C.c_double),
        ("offOrigin", C.c_double * 3), ("offDetector", C.c_double * 2), ("rotDetector", C.c_double * 3),
        ("DSD_a", _dp), ("DSO_a", _dp), ("COR_a", _dp),
        ("offOrigin_a", _dp), ("offDetector_a", _dp), ("rotDetector_a", _dp),
        ("accuracy", C.c_double), ("mode", C.c_int32),
    ]


class TigreError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = _lib().tigre_strerror(code).decode()
        if code == -5:
            msg += ": " + _lib().tigre_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} [{code}]")


_LIB = None
EXPORTS = ["tigre_Ax", "tigre_Atb", "tigre_Ax_slab", "tigre_Atb_slab", "tigre_slab_row_band", "tigre_row_weights", "tigre_col_weights", "tigre_residual",
           "tigre_update", "tigre_ossart", "tigre_cgls", "tigre_gradient_descent", "tigre_fdk", "tigre_fdk_filter", "tigre_fdk_ex", "tigre_fdk_filter_ex", "tigre_fdk_weights", "tigre_flatten_detector",
           "tigre_awtv", "tigre_awtv_gradient", "tigre_minimize_awtv", "tigre_tv_prox", "tigre_fista", "tigre_Ax_count", "tigre_plan_create", "tigre_plan_create_ex", "tigre_plan_ossart", "tigre_plan_asd_pocs", "tigre_plan_osem", "tigre_plan_sart_tv", "tigre_plan_destroy",
           "tigre_plan_bytes", "tigre_profile", "tigre_profile_read", "tigre_workspace_bytes", "tigre_set_chunk_budget", "tigre_chunk_stats", "tigre_set_atb_path", "tigre_set_tv_path", "tigre_strerror",
           "tigre_last_cuda_error", "tigre_version", "tigre_Ax_index", "tigre_set_index_path", "tigre_set_workspace", "tigre_plan_workspace_bytes",
           "tigre_workspace_stats", "tigre_sirt_chunked", "tigre_microbench", "tigre_set_ax_path", "tigre_set_plan_v_path", "tigre_plan_ossart_subsets", "tigre_Atb_boxes", "tigre_set_fdk_path", "tigre_residual_noalloc", "tigre_set_siddon_path", "tigre_band_z_range", "tigre_set_plan_fuse"]


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2412_10129_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.tigre_strerror.restype = C.c_char_p
        lib.tigre_last_cuda_error.restype = C.c_char_p
        lib.tigre_workspace_bytes.restype = C.c_size_t
        lib.tigre_plan_bytes.restype = C.c_size_t
        lib.tigre_plan_workspace_bytes.restype = C.c_size_t
        lib.tigre_set_workspace.argtypes = [C.c_void_p, C.c_size_t]
        lib.tigre_plan_bytes.argtypes = [C.c_void_p]
        lib.tigre_plan_destroy.argtypes = [C.c_void_p]
        for name in EXPORTS:
            getattr(lib, name)
        _LIB = lib
    return _LIB


def _check(code, where):
    if code != 0:
        raise TigreError(code, where)


class _Geo:
    """Marshals a workloads.Geometry (or anything with the same attributes) to the C struct and
    keeps the numpy arrays behind the optional per-angle pointers alive."""

    def __init__(self, geo, nA):
        g = tigre_geo()
        g.struct_size = C.sizeof(tigre_geo)
        g.nVoxel[:] = [int(v) for v in geo.nVoxel]
        g.dVoxel[:] = [float(v) for v in geo.dVoxel]
        g.nDetector[:] = [int(v) for v in geo.nDetector]
        g.dDetector[:] = [float(v) for v in geo.dDetector]
        g.DSD, g.DSO, g.COR = float(geo.DSD), float(geo.DSO), float(geo.COR)
        g.offOrigin[:] = [float(v) for v in geo.offOrigin]
        g.offDetector[:] = [float(v) for v in geo.offDetector]
        g.rotDetector[:] = [float(v) for v in geo.rotDetector]
        g.accuracy = float(geo.accuracy)
        g.mode = 1 if getattr(geo, "mode", "cone") == "parallel" else 0
        self.keep = []
        for name, width in (("DSD_a", 1), ("DSO_a", 1), ("COR_a", 1), ("offOrigin_a", 3),
                            ("offDetector_a", 2), ("rotDetector_a", 3)):
            a = getattr(geo, name, None)
            if a is not None:
                a = np.ascontiguousarray(a, dtype=np.float64).reshape(nA, width)
                self.keep.append(a)
                setattr(g, name, a.ctypes.data_as(_dp))
        self.c = g

    @property
    def ref(self):
        return C.byref(self.c)


def _angles(angles):
    a = np.ascontiguousarray(angles, dtype=np.float64)
    if a.ndim == 1:
        a = np.stack([a, np.zeros_like(a), np.zeros_like(a)], 1)
    a = np.ascontiguousarray(a.reshape(-1, 3))
    return a, a.shape[0]


def _stream(t=None):
    import torch
    if t is not None and t.is_cuda:
        return C.c_void_p(torch.cuda.current_stream(t.device).cuda_stream)
    if torch.cuda.is_available():
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(0)


def _f32(t, shape=None, name="tensor"):
    import torch
    if not isinstance(t, torch.Tensor):
        raise TypeError(f"{name}: expected a torch.Tensor (device memory), got {type(t)}")
    if t.dtype != torch.float32 or not t.is_contiguous():
        raise ValueError(f"{name}: need contiguous float32")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return C.c_void_p(t.data_ptr())


def _new(shape, like=None, device=None):
    import torch
    if like is not None:
        if like.is_cuda:
            return torch.empty(shape, dtype=torch.float32, device=like.device)
        return torch.empty(shape, dtype=torch.float32, pin_memory=True)   # chunked path: pinned in, pinned out
    return torch.empty(shape, dtype=torch.float32, device=device or "cuda")


class _Registered:
    """Keeps a cudaHostRegister'ed range registered for as long as the tensor that owns it lives."""

    def __init__(self, ptr):
        self.ptr = ptr

    def __del__(self):
        try:
            import torch
            torch.cuda.cudart().cudaHostUnregister(self.ptr)
        except Exception:
            pass


def pinned_empty(shape):
    """A float32 host tensor of exactly prod(shape) * 4 bytes, page-locked with cudaHostRegister: what the chunked path wants
    for arrays of tens of GB (torch's own pinned allocator rounds every request up to a power of two: 116 GB would take 128 GiB)."""
    import torch
    t = torch.empty(shape, dtype=torch.float32)
    if t.numel():
        rc = torch.cuda.cudart().cudaHostRegister(t.data_ptr(), t.numel() * 4, 0)
        if int(rc) != 0:
            raise RuntimeError(f"cudaHostRegister failed ({rc}) for {t.numel() * 4} bytes")
        t._tigre_registration = _Registered(t.data_ptr())
    return t


def vol_shape(geo):
    return (geo.nVoxel[2], geo.nVoxel[1], geo.nVoxel[0])


def proj_shape(geo, nA):
    return (nA, geo.nDetector[1], geo.nDetector[0])


# ------------------------------------------------------------------ the projector pair
def Ax(vol, geo, angles, mode="siddon", out=None):
    """b = A x.  vol: float32 [nz][ny][nx] CUDA tensor (or pinned host tensor -> chunked path)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    pv = _f32(vol, vol_shape(geo), "vol")
    if out is None:
        out = _new(proj_shape(geo, nA), like=vol)
    po = _f32(out, proj_shape(geo, nA), "out")
    _check(_lib().tigre_Ax(pv, G.ref, a.ctypes.data_as(_dp), nA, _AX_MODES[mode], po, _stream(vol)), "tigre_Ax")
    return out


def slab_row_band(geo, angles, z0, nzs):
    """(row0, nrows): detector rows the z-slab [z0, z0 + nzs) can reach in any view (host arithmetic)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    r0, nr = C.c_int(0), C.c_int(0)
    _check(_lib().tigre_slab_row_band(G.ref, a.ctypes.data_as(_dp), nA, int(z0), int(nzs), C.byref(r0), C.byref(nr)),
           "tigre_slab_row_band")
    return r0.value, nr.value


def Ax_slab(vol_slab, geo, angles, z0, mode="siddon", out=None):
    """Partial line integrals of the z-slices [z0, z0 + vol_slab.shape[0]) of a volume described by geo (full size)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    nzs = int(vol_slab.shape[0])
    pv = _f32(vol_slab, (nzs,) + tuple(vol_shape(geo)[1:]), "vol_slab")
    if out is None:
        out = _new(proj_shape(geo, nA), like=vol_slab)
    po = _f32(out, proj_shape(geo, nA), "out")
    _check(_lib().tigre_Ax_slab(pv, G.ref, a.ctypes.data_as(_dp), nA, _AX_MODES[mode], int(z0), nzs, po, _stream(vol_slab)),
           "tigre_Ax_slab")
    return out


def Atb_slab(proj, geo, angles, z0, nzs, mode="matched", out=None):
    """Slices [z0, z0 + nzs) of A^T b (voxel-driven modes)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    pp = _f32(proj, proj_shape(geo, nA), "proj")
    shape = (int(nzs),) + tuple(vol_shape(geo)[1:])
    if out is None:
        out = _new(shape, like=proj)
    po = _f32(out, shape, "out")
    _check(_lib().tigre_Atb_slab(pp, G.ref, a.ctypes.data_as(_dp), nA, _ATB_MODES[mode], int(z0), int(nzs), po, _stream(proj)),
           "tigre_Atb_slab")
    return out


def Atb(proj, geo, angles, mode="matched", out=None):
    """x = A^T b.  mode: "matched" / "fdk" (voxel-driven) or "exact_siddon" / "exact_interp" (the exact transpose of
    Ax in that mode, ray-driven scatter).  proj: float32 [nA][nv][nu]."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    pp = _f32(proj, proj_shape(geo, nA), "proj")
    if out is None:
        out = _new(vol_shape(geo), like=proj)
    po = _f32(out, vol_shape(geo), "out")
    _check(_lib().tigre_Atb(pp, G.ref, a.ctypes.data_as(_dp), nA, _ATB_MODES[mode], po, _stream(proj)), "tigre_Atb")
    return out


def row_weights(geo, angles, ax_mode="siddon", device="cuda"):
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    W = _new(proj_shape(geo, nA), device=device)
    _check(_lib().tigre_row_weights(G.ref, a.ctypes.data_as(_dp), nA, _AX_MODES[ax_mode], _f32(W), _stream(W)),
           "tigre_row_weights")
    return W


def col_weights(geo, angles, atb_mode="matched", device="cuda"):
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    V = _new(vol_shape(geo), device=device)
    _check(_lib().tigre_col_weights(G.ref, a.ctypes.data_as(_dp), nA, _ATB_MODES[atb_mode], _f32(V), _stream(V)),
           "tigre_col_weights")
    return V


def residual(b, ax, W=None, return_norm=False):
    r = _new(tuple(b.shape), like=b)
    nrm = C.c_double(0.0)
    _check(_lib().tigre_residual(_f32(b), _f32(ax, b.shape, "Ax"), _f32(W, b.shape, "W") if W is not None else None,
                                 _f32(r), C.c_size_t(b.numel()), C.byref(nrm) if return_norm else None, _stream(b)),
           "tigre_residual")
    return (r, nrm.value) if return_norm else r


RESIDUAL_NOALLOC_MAX_N = 1 << 28   # TIGRE_RESIDUAL_NOALLOC_MAX_N


def residual_noalloc(b, ax, r, W=None, nrm2=None):
    """tigre_residual_noalloc: r <- W .* (b - ax), nrm2[0] <- ||b - ax||^2, with no allocation and no synchronisation inside the
    library (scratch: a file-scope device array, so numel <= RESIDUAL_NOALLOC_MAX_N; calls that overlap on the GPU race on it).
    The caller passes the outputs: r (float32, b's shape) and, optionally, nrm2 (a float64 device tensor of one element)."""
    import torch
    if nrm2 is not None and (not isinstance(nrm2, torch.Tensor) or nrm2.dtype != torch.float64 or not nrm2.is_cuda or nrm2.numel() != 1):
        raise ValueError("nrm2: need a float64 device tensor of one element")
    _check(_lib().tigre_residual_noalloc(_f32(b), _f32(ax, b.shape, "Ax"), _f32(W, b.shape, "W") if W is not None else None,
                                         _f32(r, b.shape, "r"), C.c_size_t(b.numel()),
                                         C.c_void_p(nrm2.data_ptr()) if nrm2 is not None else None, _stream(b)),
           "tigre_residual_noalloc")
    return r


def update(x, g, V=None, lam=1.0, nonneg=True):
    """In place: x <- max(0, x + lam * V .* g)."""
    _check(_lib().tigre_update(_f32(x), _f32(g, x.shape, "g"), _f32(V, x.shape, "V") if V is not None else None,
                               C.c_float(lam), int(bool(nonneg)), C.c_size_t(x.numel()), _stream(x)), "tigre_update")
    return x


# ------------------------------------------------------------------ drivers
def ossart(b, geo, angles, subsets, n_iter, lam=1.0, nonneg=True, ax_mode="siddon", atb_mode="matched", x0=None):
    """OS-SART; `subsets` is a list of view-index lists.  Returns (x, resid_hist)."""
    import torch
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    idx = np.ascontiguousarray(np.concatenate([np.asarray(s, dtype=np.int32) for s in subsets]))
    off = np.zeros(len(subsets) + 1, dtype=np.int32)
    off[1:] = np.cumsum([len(s) for s in subsets])
    x = torch.zeros(vol_shape(geo), dtype=torch.float32, device=b.device) if x0 is None else x0.clone()
    hist = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(_lib().tigre_ossart(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA,
                               idx.ctypes.data_as(C.POINTER(C.c_int32)), off.ctypes.data_as(C.POINTER(C.c_int32)),
                               len(subsets), int(n_iter), C.c_float(lam), int(bool(nonneg)), _AX_MODES[ax_mode],
                               _ATB_MODES[atb_mode], _f32(x), hist.ctypes.data_as(_dp), _stream(b)), "tigre_ossart")
    return x, hist[:n_iter]


class OssartPlan:
    """tigre_plan_*: view tables and the SART weights computed once; iterate() runs sweeps."""

    def __init__(self, geo, angles, subsets, ax_mode="siddon", atb_mode="matched", redundancy=False):
        a, nA = _angles(angles)
        G = _Geo(geo, nA)
        idx = np.ascontiguousarray(np.concatenate([np.asarray(s, dtype=np.int32) for s in subsets]))
        off = np.zeros(len(subsets) + 1, dtype=np.int32)
        off[1:] = np.cumsum([len(s) for s in subsets])
        self.geo, self.nA = geo, nA
        self._h = C.c_void_p(None)
        _check(_lib().tigre_plan_create_ex(G.ref, a.ctypes.data_as(_dp), nA, idx.ctypes.data_as(C.POINTER(C.c_int32)),
                                           off.ctypes.data_as(C.POINTER(C.c_int32)), len(subsets), _AX_MODES[ax_mode],
                                           _ATB_MODES[atb_mode], int(bool(redundancy)), _stream(), C.byref(self._h)),
               "tigre_plan_create_ex")

    @property
    def nbytes(self):
        return int(_lib().tigre_plan_bytes(self._h))

    def iterate(self, b, x, n_iter=1, lam=1.0, nonneg=True, want_resid=True):
        """In place on x.  b, x: CUDA tensors, or both pinned host tensors (end-to-end path)."""
        hist = np.zeros(max(n_iter, 1), dtype=np.float64)
        _check(_lib().tigre_plan_ossart(self._h, _f32(b, proj_shape(self.geo, self.nA), "b"),
                                        _f32(x, vol_shape(self.geo), "x"), int(n_iter), C.c_float(lam),
                                        int(bool(nonneg)), hist.ctypes.data_as(_dp) if want_resid else None,
                                        _stream(b)), "tigre_plan_ossart")
        return hist[:n_iter]

    def iterate_subsets(self, b, x, s_begin, s_end, lam=1.0, nonneg=True):
        """The subset steps [s_begin, s_end) of one sweep, in place on x."""
        _check(_lib().tigre_plan_ossart_subsets(self._h, _f32(b, proj_shape(self.geo, self.nA), "b"), _f32(x, vol_shape(self.geo), "x"),
                                                int(s_begin), int(s_end), C.c_float(lam), int(bool(nonneg)), _stream(b)),
               "tigre_plan_ossart_subsets")
        return x

    def asd_pocs(self, b, x, n_iter, beta=1.0, beta_red=0.99, ng=20, alpha=0.002, alpha_red=0.95, r_max=0.95,
                 epsilon=0.0, delta=None, tv_eps=1e-8):
        """ASD-POCS family in place on x (single-view subsets: ASD-POCS; blocks: OS-ASD-POCS; delta: AwTV).
        Returns hist[n_done][5] = dd, dp, dg, dtvg, c."""
        hist = np.zeros((max(n_iter, 1), 5), dtype=np.float64)
        done = C.c_int(0)
        _check(_lib().tigre_plan_asd_pocs(self._h, _f32(b, proj_shape(self.geo, self.nA), "b"),
                                          _f32(x, vol_shape(self.geo), "x"), int(n_iter), C.c_float(beta),
                                          C.c_float(beta_red), int(ng), C.c_float(alpha), C.c_float(alpha_red),
                                          C.c_float(r_max), C.c_float(epsilon), _delta(delta), C.c_float(tv_eps),
                                          hist.ctypes.data_as(_dp), C.byref(done), _stream(b)), "tigre_plan_asd_pocs")
        return hist[:done.value]

    def osem(self, b, x, n_iter):
        """MLEM (one subset of all views) / OSEM in place on x (positive start)."""
        _check(_lib().tigre_plan_osem(self._h, _f32(b, proj_shape(self.geo, self.nA), "b"), _f32(x, vol_shape(self.geo), "x"),
                                      int(n_iter), _stream(b)), "tigre_plan_osem")
        return x

    def sart_tv(self, b, x, n_iter, lam=1.0, lam_red=1.0, tv_lambda=0.0, tv_iter=10, tau=1.0 / 12.0):
        """SART-TV in place on x: OS-SART sweep + TV prox per iteration; returns the residual history."""
        hist = np.zeros(max(n_iter, 1), dtype=np.float64)
        _check(_lib().tigre_plan_sart_tv(self._h, _f32(b, proj_shape(self.geo, self.nA), "b"),
                                         _f32(x, vol_shape(self.geo), "x"), int(n_iter), C.c_float(lam), C.c_float(lam_red),
                                         C.c_float(tv_lambda), int(tv_iter), C.c_float(tau), hist.ctypes.data_as(_dp),
                                         _stream(b)), "tigre_plan_sart_tv")
        return hist[:n_iter]

    def close(self):
        if self._h:
            _lib().tigre_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sirt(b, geo, angles, n_iter, **kw):
    _, nA = _angles(angles)
    return ossart(b, geo, angles, [np.arange(nA)], n_iter, **kw)


def cgls(b, geo, angles, n_iter, ax_mode="siddon", atb_mode="matched"):
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    x = _new(vol_shape(geo), like=b)
    hist = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(_lib().tigre_cgls(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, int(n_iter),
                             _AX_MODES[ax_mode], _ATB_MODES[atb_mode], _f32(x), hist.ctypes.data_as(_dp), _stream(b)),
           "tigre_cgls")
    return x, hist[:n_iter]


_FILTERS = {"ram_lak": 0, "shepp_logan": 1, "cosine": 2, "hamming": 3, "hann": 4}
_WEIGHTINGS = {None: 0, "full": 0, "parker": 1, "wang": 2}


def gradient_descent(b, geo, angles, n_iter, lam, ax_mode="siddon", atb_mode="matched", x0=None):
    """Eq. (4): x += lam A^T (b - A x); returns (x, resid)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    x = _new(vol_shape(geo), like=b)
    if x0 is None:
        x.zero_()
    else:
        x.copy_(x0)
    hist = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(_lib().tigre_gradient_descent(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, int(n_iter),
                                         C.c_float(lam), _AX_MODES[ax_mode], _ATB_MODES[atb_mode], _f32(x),
                                         hist.ctypes.data_as(_dp), _stream(b)), "tigre_gradient_descent")
    return x, hist[:n_iter]


def fdk_ex(b, geo, angles, filt="ram_lak", weighting=None):
    """FDK with a windowed ramp filter and Parker (short scan) or Wang (displaced detector) weights."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    x = _new(vol_shape(geo), like=b)
    _check(_lib().tigre_fdk_ex(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, _FILTERS[filt],
                               _WEIGHTINGS[weighting], _f32(x), _stream(b)), "tigre_fdk_ex")
    return x


def fdk_filter_ex(b, geo, angles, filt="ram_lak", weighting=None):
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    q = _new(proj_shape(geo, nA), like=b)
    _check(_lib().tigre_fdk_filter_ex(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, _FILTERS[filt],
                                      _WEIGHTINGS[weighting], _f32(q), _stream(b)), "tigre_fdk_filter_ex")
    return q


def flatten_detector(curved, geo, angles):
    """Projections measured on a curved (cylindrical, radius DSD) detector resampled onto the flat detector of geo."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    flat = _new(proj_shape(geo, nA), like=curved)
    _check(_lib().tigre_flatten_detector(_f32(curved, proj_shape(geo, nA), "curved"), G.ref, a.ctypes.data_as(_dp), nA,
                                         _f32(flat), _stream(curved)), "tigre_flatten_detector")
    return flat


def fdk_weights(geo, angles, weighting):
    """Parker / Wang weight table [nA][nu] (host, fp64; Wang without the factor 2)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    w = np.zeros((nA, geo.nDetector[0]), dtype=np.float64)
    _check(_lib().tigre_fdk_weights(G.ref, a.ctypes.data_as(_dp), nA, _WEIGHTINGS[weighting], w.ctypes.data_as(_dp)),
           "tigre_fdk_weights")
    return w


def fdk(b, geo, angles):
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    x = _new(vol_shape(geo), like=b)
    _check(_lib().tigre_fdk(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, _f32(x), _stream(b)),
           "tigre_fdk")
    return x


def fdk_filter(b, geo, angles):
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    q = _new(tuple(b.shape), like=b)
    _check(_lib().tigre_fdk_filter(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, _f32(q),
                                   _stream(b)), "tigre_fdk_filter")
    return q


def Ax_count(geo, angles, mode="siddon", return_counts=False, device="cuda"):
    """Exact number of ray-samples of one Ax call (the BASELINE metric's unit)."""
    import torch
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    total = C.c_uint64(0)
    counts = torch.empty(proj_shape(geo, nA), dtype=torch.int32, device=device) if return_counts else None
    _check(_lib().tigre_Ax_count(G.ref, a.ctypes.data_as(_dp), nA, _AX_MODES[mode],
                                 C.c_void_p(counts.data_ptr()) if return_counts else None, C.byref(total),
                                 _stream(counts)), "tigre_Ax_count")
    return (total.value, counts) if return_counts else total.value


def Atb_boxes(proj, geo, angles, mode="matched"):
    """Reading P19(b): (vol, meta, boxes) of the TMA-staged backprojector: meta = dict(tile=(x, y, z), box=(u, v), tiles=(x, y, z)) or
    None when the problem takes the gather kernel; boxes int32 [tz][ty][tx][nA][4] = (u0, v0, fits, 0)."""
    import torch
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    pp = _f32(proj, proj_shape(geo, nA), "proj")
    vol = _new(vol_shape(geo), like=proj)
    meta = (C.c_int32 * 8)()
    _check(_lib().tigre_Atb_boxes(pp, G.ref, a.ctypes.data_as(_dp), nA, _ATB_MODES[mode], _f32(vol), meta, None, _stream(proj)),
           "tigre_Atb_boxes")
    m = [int(v) for v in meta]
    if m[0] == 0:
        return Atb(proj, geo, angles, mode), None, None
    boxes = torch.empty((m[7], m[6], m[5], nA, 4), dtype=torch.int32, device=proj.device)
    _check(_lib().tigre_Atb_boxes(pp, G.ref, a.ctypes.data_as(_dp), nA, _ATB_MODES[mode], _f32(vol), meta,
                                  C.c_void_p(boxes.data_ptr()), _stream(proj)), "tigre_Atb_boxes")
    return vol, dict(tile=tuple(m[0:3]), box=tuple(m[3:5]), tiles=tuple(m[5:8])), boxes


def Ax_index(geo, angles, device="cuda"):
    """Reading P19(a): (first_last int64 [nA][nv][nu][2], nseg int32 [nA][nv][nu]) of the Siddon march itself: linear index of
    the first / last voxel each ray gives a non-zero length to (-1: the ray misses) and the number of such voxels."""
    import torch
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    fl = torch.empty(proj_shape(geo, nA) + (2,), dtype=torch.int64, device=device)
    ns = torch.empty(proj_shape(geo, nA), dtype=torch.int32, device=device)
    _check(_lib().tigre_Ax_index(G.ref, a.ctypes.data_as(_dp), nA, C.c_void_p(fl.data_ptr()), C.c_void_p(ns.data_ptr()), _stream(fl)),
           "tigre_Ax_index")
    return fl, ns


def set_index_path(path):
    """0 = 32-bit element offsets below 2^31 voxels (default), 1 = always the 64-bit instantiations of the ray-driven kernels."""
    _check(_lib().tigre_set_index_path(int(path)), "tigre_set_index_path")


_WORKSPACE = None


def set_workspace(buf):
    """Give the library a caller-owned workspace (a CUDA uint8 / any-dtype tensor, kept alive here) or None to return to the
    stream-ordered pool."""
    global _WORKSPACE
    if buf is None:
        _check(_lib().tigre_set_workspace(None, 0), "tigre_set_workspace")
        _WORKSPACE = None
        return
    _check(_lib().tigre_set_workspace(C.c_void_p(buf.data_ptr()), C.c_size_t(buf.numel() * buf.element_size())), "tigre_set_workspace")
    _WORKSPACE = buf


def plan_workspace_bytes(geo, nA, n_subsets, max_subset_views, host_data=False):
    G = _Geo(geo, nA)
    return int(_lib().tigre_plan_workspace_bytes(G.ref, int(nA), int(n_subsets), int(max_subset_views), int(bool(host_data))))


def workspace_stats():
    """(bytes in use, high-water mark, pool allocations since set_workspace)."""
    a, b, c = C.c_size_t(0), C.c_size_t(0), C.c_uint64(0)
    _check(_lib().tigre_workspace_stats(C.byref(a), C.byref(b), C.byref(c)), "tigre_workspace_stats")
    return a.value, b.value, c.value


def sirt_chunked(b, geo, angles, x, n_iter=1, lam=1.0, nonneg=True, ax_mode="siddon", atb_mode="matched", r_scratch=None):
    """SIRT on PINNED host tensors larger than the device (in place on x).  r_scratch: pinned, shaped like b (None: b itself is
    overwritten by the weighted residual, n_iter == 1 only).  Returns the residual history."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    r = b if r_scratch is None else r_scratch
    hist = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(_lib().tigre_sirt_chunked(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, int(n_iter), C.c_float(lam),
                                     int(bool(nonneg)), _AX_MODES[ax_mode], _ATB_MODES[atb_mode], _f32(x, vol_shape(geo), "x"),
                                     _f32(r, proj_shape(geo, nA), "r_scratch"), hist.ctypes.data_as(_dp), _stream()), "tigre_sirt_chunked")
    return hist[:n_iter]


PEAK_KINDS = {"ffma": 0, "smem": 1, "l1_lines": 2, "l2": 3, "h2d": 4, "d2h": 5, "hbm_copy": 6, "sm_hz": 7}


def microbench(kind):
    """One of the step-0 machine rates (see tigre_microbench in the header); kind: a key of PEAK_KINDS."""
    v = C.c_double(0.0)
    _check(_lib().tigre_microbench(PEAK_KINDS[kind], C.byref(v), _stream()), "tigre_microbench")
    return v.value


def workspace_bytes(geo, nA, op):
    G = _Geo(geo, nA)
    return int(_lib().tigre_workspace_bytes(G.ref, int(nA), int(op)))


def set_chunk_budget(nbytes):
    _check(_lib().tigre_set_chunk_budget(C.c_size_t(int(nbytes))), "tigre_set_chunk_budget")


def profile(enable=True):
    _check(_lib().tigre_profile(int(bool(enable))), "tigre_profile")


def profile_read():
    """{'ms': {'ax','atb','ew'}, 'launches': {...}} accumulated since profile(True)."""
    ms = (C.c_double * 3)()
    n = (C.c_uint64 * 3)()
    _check(_lib().tigre_profile_read(ms, n), "tigre_profile_read")
    k = ("ax", "atb", "ew")
    return dict(ms=dict(zip(k, [float(v) for v in ms])), launches=dict(zip(k, [int(v) for v in n])))


def version():
    return int(_lib().tigre_version())


def set_tv_path(path):
    """0 = float4 TV gradient kernel when the shape qualifies (default), 1 = scalar kernel only."""
    _check(_lib().tigre_set_tv_path(int(path)), "tigre_set_tv_path")


def set_fdk_path(path):
    """0 = tensor-core FDK pre-filter when the problem qualifies (default), 1 = CUDA-core convolution only."""
    _check(_lib().tigre_set_fdk_path(int(path)), "tigre_set_fdk_path")


def set_plan_v_path(path):
    """0 = plans store V_s per subset when that fits (default), 1 = always store, 2 = always recompute per subset step."""
    _check(_lib().tigre_set_plan_v_path(int(path)), "tigre_set_plan_v_path")


def set_ax_path(path):
    """0 = TMA-staged interpolated Ax kernel for narrow beams that qualify (default), 1 = L1 gather kernel only, 2 = TMA kernel
    for wide beams too."""
    _check(_lib().tigre_set_ax_path(int(path)), "tigre_set_ax_path")


def band_z_range(geo, angles, row0, row1):
    """(zlo, zhi): z-slices that rays of detector rows [row0, row1) of these views can meet (zlo > zhi: none); None if no bound is
    formed.  Host only."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    lo, hi = C.c_int32(0), C.c_int32(-1)
    rc = _lib().tigre_band_z_range(C.byref(G.c), a.ctypes.data_as(_dp), nA, int(row0), int(row1), C.byref(lo), C.byref(hi))
    if rc == 1:
        return None
    _check(rc, "tigre_band_z_range")
    return lo.value, hi.value


def set_plan_fuse(on):
    """1 = OS-SART update in the backprojector's epilogue where the TMA kernel runs (default), 0 = as its own kernel."""
    _check(_lib().tigre_set_plan_fuse(int(bool(on))), "tigre_set_plan_fuse")


def set_siddon_path(path):
    """0 = L1 gather Siddon Ax kernel (default), 1 = TMA-staged Siddon kernel where the problem qualifies (slower; A/B hook)."""
    _check(_lib().tigre_set_siddon_path(int(path)), "tigre_set_siddon_path")


def set_atb_path(path):
    """0 = TMA-staged A^T b kernel when the problem qualifies (default), 1 = gather kernel only, 2 = TMA kernel with an undersized box
    (test hook), 3 = TMA kernel without the linearised z-runs of tilted views."""
    _check(_lib().tigre_set_atb_path(int(path)), "tigre_set_atb_path")


def chunk_stats():
    """(h2d_bytes, d2h_bytes, n_slabs, n_batches) of the most recent chunked Ax / Atb call."""
    a, b, c, d = C.c_uint64(0), C.c_uint64(0), C.c_int(0), C.c_int(0)
    _check(_lib().tigre_chunk_stats(C.byref(a), C.byref(b), C.byref(c), C.byref(d)), "tigre_chunk_stats")
    return a.value, b.value, c.value, d.value


# ------------------------------------------------------------------ TV / AwTV
def _dims(x):
    if x.dim() != 3:
        raise ValueError("expected a [nz][ny][nx] volume")
    return int(x.shape[2]), int(x.shape[1]), int(x.shape[0])


def _delta(delta):
    return C.c_float(0.0 if delta is None or not np.isfinite(delta) else float(delta))


def awtv(x, delta=None, eps=0.0):
    """AwTV(x) of PAPER.md eq. 7 in 3-D (delta None / inf: the TV norm)."""
    nx, ny, nz = _dims(x)
    v = C.c_double(0.0)
    _check(_lib().tigre_awtv(_f32(x), nx, ny, nz, _delta(delta), C.c_float(eps), C.byref(v), _stream(x)), "tigre_awtv")
    return v.value


def awtv_gradient(x, delta=None, eps=1e-8, return_scalars=False):
    """dAwTV/dx; with return_scalars also (AwTV(x), ||g||^2) from the same pass."""
    nx, ny, nz = _dims(x)
    g = _new(tuple(x.shape), like=x)
    v, n2 = C.c_double(0.0), C.c_double(0.0)
    _check(_lib().tigre_awtv_gradient(_f32(x), nx, ny, nz, _delta(delta), C.c_float(eps), _f32(g),
                                      C.byref(v) if return_scalars else None, C.byref(n2) if return_scalars else None,
                                      _stream(x)), "tigre_awtv_gradient")
    return (g, v.value, n2.value) if return_scalars else g


def tv_prox(f, lam, n_iter, tau=1.0 / 12.0, out=None):
    """TV proximal operator (ROF denoising by the dual projection iteration); out may be f itself."""
    nx, ny, nz = _dims(f)
    u = _new(tuple(f.shape), like=f) if out is None else out
    _check(_lib().tigre_tv_prox(_f32(f), nx, ny, nz, C.c_float(lam), int(n_iter), C.c_float(tau), _f32(u), _stream(f)),
           "tigre_tv_prox")
    return u


def fista(b, geo, angles, n_iter, L, tv_lambda, tv_iter, ax_mode="siddon", atb_mode="matched", x0=None, tau=1.0 / 12.0):
    """FISTA with the TV prox; returns (x, resid)."""
    a, nA = _angles(angles)
    G = _Geo(geo, nA)
    x = _new(vol_shape(geo), like=b)
    if x0 is None:
        x.zero_()
    else:
        x.copy_(x0)
    hist = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(_lib().tigre_fista(_f32(b, proj_shape(geo, nA), "b"), G.ref, a.ctypes.data_as(_dp), nA, int(n_iter), C.c_float(L),
                              C.c_float(tv_lambda), int(tv_iter), C.c_float(tau), _AX_MODES[ax_mode], _ATB_MODES[atb_mode],
                              _f32(x), hist.ctypes.data_as(_dp), _stream(b)), "tigre_fista")
    return x, hist[:n_iter]


def minimize_awtv(x, n_steps, alpha, delta=None, eps=1e-8):
    """In place: n_steps of x <- x - alpha g/||g||_2."""
    nx, ny, nz = _dims(x)
    _check(_lib().tigre_minimize_awtv(_f32(x), nx, ny, nz, _delta(delta), C.c_float(eps), C.c_float(alpha), int(n_steps),
                                      _stream(x)), "tigre_minimize_awtv")
    return x
