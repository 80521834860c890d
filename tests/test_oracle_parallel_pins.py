"""Pins of the oracle's parallel-beam mode (reading P29; the synchrotron parallel-beam workload) against
independent geometry (tests/helpers.py) and mathematics: brute-force per-voxel intersection lengths, closed-form chords
of ellipsoids (exact for parallel rays: no divergence), the cone-beam limit DSO -> infinity, the adjoint identity, the
voxel -> detector map, the closed-form sum of weights, the normalisation of the matched weight against the exact
transpose, and FBP of an analytic ball."""
import numpy as np
import pytest

from oracle import fdk_ext as fx
from oracle import oracle as orc
from tests import helpers as H
from workloads.geometry import Geometry, circular_angles


def chords(ell, S, P):
    """Closed-form chord x density of one ellipsoid along the lines through S[...,3] and P[...,3] (per-ray origins)."""
    c, a, rho = ell["centre"][0], ell["axes"][0], ell["rho"][0]
    w = P - S
    w = w / np.linalg.norm(w, axis=-1, keepdims=True)
    m, d = (S - c) / a, w / a
    A, B, Cc = np.sum(d * d, -1), np.sum(d * m, -1), np.sum(m * m, -1) - 1.0
    disc = B * B - A * Cc
    return rho * np.where(disc > 0, 2.0 * np.sqrt(np.maximum(disc, 0.0)) / A, 0.0)


def par_geo(**kw):
    base = dict(nVoxel=(6, 5, 7), dVoxel=(1.0, 1.2, 0.9), nDetector=(10, 9), dDetector=(1.1, 1.3), DSD=60.0, DSO=35.0,
                mode="parallel")
    base.update(kw)
    return Geometry(**base)


def brute_ax(vol, geo, ang):
    out = np.zeros((len(ang), geo.nDetector[1], geo.nDetector[0]))
    iu, iv = np.meshgrid(np.arange(geo.nDetector[0]), np.arange(geo.nDetector[1]))
    c = H.voxel_centres(geo, geo.offOrigin).reshape(-1, 3)
    h = np.array(geo.dVoxel)
    for ia in range(len(ang)):
        S, P = H.parallel_rays(geo, ang, ia, iu, iv)
        for jv in range(geo.nDetector[1]):
            for ju in range(geo.nDetector[0]):
                L = H.segment_box_length(S[jv, ju], P[jv, ju], c - 0.5 * h, c + 0.5 * h)
                out[ia, jv, ju] = L @ vol.ravel()
    return out


def test_siddon_parallel_equals_brute_force_with_every_parameter_nonzero():
    geo = par_geo(offOrigin=(0.4, -0.3, 0.2), offDetector=(0.7, -0.5), rotDetector=(0.05, -0.04, 0.03), COR=0.6)
    ang = np.array([[0.3, 0.1, -0.2], [1.9, -0.15, 0.1], [4.0, 0.0, 0.0]])
    vol = np.random.default_rng(0).random(geo.vol_shape)
    assert np.allclose(orc.ax(vol, geo, ang, orc.SIDDON), brute_ax(vol, geo, ang), rtol=0, atol=1e-12)


def test_ellipsoid_chords_are_exact_in_the_limit_and_interp_converges():
    n = 48
    geo = Geometry(nVoxel=(n, n, n), dVoxel=(0.5,) * 3, nDetector=(40, 36), dDetector=(0.7, 0.7), DSD=90.0, DSO=50.0,
                   mode="parallel")
    ang = circular_angles(3)
    ell = dict(centre=np.array([[1.0, -2.0, 0.5]]), axes=np.array([[7.0, 5.0, 6.0]]), Q=np.eye(3)[None], rho=np.array([0.02]))
    c = H.voxel_centres(geo, (0, 0, 0))
    vol = 0.02 * (np.sum(((c - ell["centre"][0]) / ell["axes"][0]) ** 2, -1) < 1.0)
    iu, iv = np.meshgrid(np.arange(40), np.arange(36))
    ref = np.stack([chords(ell, *H.parallel_rays(geo, ang, ia, iu, iv)) for ia in range(3)])
    for mode in (orc.SIDDON, orc.INTERP):
        p = orc.ax(vol, geo, ang, mode)
        assert abs(p.sum() / ref.sum() - 1.0) < 0.01                # first order in the voxel size (voxelised ellipsoid)
    # mirrored detector coordinate gives a different image: the sign of u matters
    assert abs(orc.ax(vol, geo, ang, orc.SIDDON)[0] - ref[0]).max() < 0.3 * ref.max()
    assert abs(orc.ax(vol, geo, ang, orc.SIDDON)[0][:, ::-1] - ref[0]).max() > 0.3 * ref.max()


def test_cone_beam_tends_to_parallel_beam():
    geo = par_geo()
    ang = circular_angles(4)
    vol = np.random.default_rng(1).random(geo.vol_shape)
    y = np.random.default_rng(2).random((4, 9, 10))
    far = 1e7
    cone = geo.copy(mode="cone", DSO=far, DSD=far + (geo.DSD - geo.DSO))      # same detector position, source far away
    for mode in (orc.SIDDON, orc.INTERP):
        assert H.rel_l2(orc.ax(vol, cone, ang, mode), orc.ax(vol, geo, ang, mode)) < 1e-5
    for mode in (orc.MATCHED, orc.FDK):
        assert H.rel_l2(orc.atb(y, cone, ang, mode), orc.atb(y, geo, ang, mode)) < 1e-5


def test_adjoint_identity_parallel():
    geo = par_geo(rotDetector=(0.02, 0.03, -0.01), offDetector=(0.3, 0.2))
    ang = circular_angles(5)
    rng = np.random.default_rng(3)
    x, y = rng.random(geo.vol_shape), rng.random((5, 9, 10))
    for mode in (orc.SIDDON, orc.INTERP):
        lhs = np.sum(orc.ax(x, geo, ang, mode) * y)
        rhs = np.sum(x * orc.atb_exact(y, geo, ang, mode))
        assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_voxel_map_unit_projection_and_weight_normalisation():
    geo = par_geo(offOrigin=(0.4, -0.3, 0.2), offDetector=(0.7, -0.5), rotDetector=(0.05, -0.04, 0.03), COR=0.6)
    ang = np.array([[0.3, 0.1, -0.2], [1.9, -0.15, 0.1]])
    X = H.voxel_centres(geo, geo.offOrigin)
    ones = np.ones((2, 9, 10))
    ref_m = np.zeros(geo.vol_shape)
    cvol = np.prod(geo.dVoxel) / np.prod(geo.dDetector)
    for ia in range(2):
        fu, fv, cosn = H.parallel_voxel_to_detector(geo, ang, ia, X)
        _, got = orc.voxel_map(geo, ang, ia, 2, 3, 4)
        assert got[0] == pytest.approx(fu[4, 3, 2], abs=1e-12) and got[1] == pytest.approx(fv[4, 3, 2], abs=1e-12)
        # bilinear of an all-ones image with zero border: product of the in-range tap weights
        def cov(f, n):
            fl = np.floor(f)
            a = f - fl
            lo_in = (fl >= 0) & (fl < n)
            hi_in = (fl + 1 >= 0) & (fl + 1 < n)
            return (1 - a) * lo_in + a * hi_in
        ref_m += cvol / cosn * cov(fu, 10) * cov(fv, 9)
    assert np.allclose(orc.atb(ones, geo, ang, orc.MATCHED), ref_m, rtol=1e-12, atol=1e-14)
    # normalisation: on a fine detector the matched weights sum like the exact transpose does
    fine = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(64, 64), dDetector=(0.25, 0.25), DSD=40.0, DSO=20.0,
                    mode="parallel")
    a1 = circular_angles(3)
    m = orc.atb(None, fine, a1, orc.MATCHED)[2:-2, 2:-2, 2:-2]
    e = orc.atb_exact(np.ones((3, 64, 64)), fine, a1, orc.SIDDON)[2:-2, 2:-2, 2:-2]
    assert abs(m.sum() / e.sum() - 1.0) < 0.01


def test_fbp_reconstructs_analytic_ball_over_half_and_full_circle():
    n, nd = 40, 64
    geo = Geometry(nVoxel=(n, n, n), dVoxel=(1.0,) * 3, nDetector=(nd, nd), dDetector=(1.0, 1.0), DSD=200.0, DSO=100.0,
                   mode="parallel")
    rho, rad, cen = 0.02, 12.0, np.array([3.0, -2.0, 1.0])
    ell = dict(centre=cen[None], axes=np.full((1, 3), rad), Q=np.eye(3)[None], rho=np.array([rho]))
    iu, iv = np.meshgrid(np.arange(nd), np.arange(nd))
    c = H.voxel_centres(geo, (0, 0, 0))
    d = np.linalg.norm(c - cen, axis=-1)
    for span, nA in ((np.pi, 90), (2 * np.pi, 120)):
        ang = circular_angles(nA, span=span)
        proj = np.stack([chords(ell, *H.parallel_rays(geo, ang, ia, iu, iv)) for ia in range(nA)])
        x = orc.fdk(proj, geo, ang)                               # (pi / nA) sum: right for [0, pi) and for [0, 2 pi)
        inside, outside = x[d < rad - 2.5].mean(), x[(d > rad + 2.5) & (d < 18)].mean()
        assert abs(inside / rho - 1.0) < 0.01, (span, inside / rho)
        assert abs(outside) < 0.01 * rho
        assert np.allclose(fx.fdk_filter(proj[:2], geo, ang[:2], "ram_lak"), orc.fdk_filter(proj[:2], geo, ang[:2]), atol=1e-12)
