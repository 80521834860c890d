"""Pins of the curved-detector flattening oracle (oracle/curved.py; reading P30): line integrals of an
analytic ball evaluated at the CURVED detector's pixel positions (built here from first principles) and flattened must
equal the line integrals at the flat pixels up to the interpolation error, which falls as h^2; the central column and
row are fixed points; a curved image that depends on the fan angle only maps by u -> DSD atan(u/DSD)."""
import numpy as np
import pytest

from oracle import curved
from tests import helpers as H
from workloads.geometry import Geometry


def curved_pixel_world(geo, nu, nv, du, dv):
    """World positions of the curved detector's pixels for the view at angle 0, no offsets: source S = (DSO, 0, 0), the
    cylinder of radius DSD about the vertical axis through S; fan angle = arc length / DSD, measured from the central ray
    towards +y."""
    S = np.array([geo.DSO, 0.0, 0.0])
    s = (np.arange(nu) + 0.5) * du - 0.5 * nu * du
    v = (np.arange(nv) + 0.5) * dv - 0.5 * nv * dv
    g = s / geo.DSD
    P = np.zeros((nv, nu, 3))
    P[..., 0] = S[0] - geo.DSD * np.cos(g)[None, :]
    P[..., 1] = geo.DSD * np.sin(g)[None, :]
    P[..., 2] = v[:, None]
    return S, P


def ball(S, P, cen, rad, rho):
    ell = dict(centre=cen[None], axes=np.full((1, 3), rad), Q=np.eye(3)[None], rho=np.array([rho]))
    return H.ellipsoid_line_integrals(ell, S, P)


def test_flattened_ball_projection_converges_to_the_flat_one():
    cen, rad, rho = np.array([10.0, 25.0, -12.0]), 40.0, 0.02
    errs = []
    for n, d in ((96, 4.0), (192, 2.0), (384, 1.0)):
        geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(n, n), dDetector=(d, d), DSD=600.0, DSO=400.0)
        S, Pc = curved_pixel_world(geo, n, n, d, d)
        iu, iv = np.meshgrid(np.arange(n), np.arange(n))
        Sf, Pf = H.pixel_world(geo, np.zeros((1, 3)), 0, iu, iv)
        flat_ref = ball(Sf, Pf, cen, rad, rho)
        got = curved.flatten(ball(S, Pc, cen, rad, rho)[None], geo)[0]
        m = flat_ref > 0.6 * flat_ref.max()                          # away from the ball's silhouette (a square-root edge)
        # the flat detector is wider than the arc: its outermost columns fall off the curved one (zero there)
        inside = np.abs(600.0 * np.arctan(((np.arange(n) + 0.5) * d - 0.5 * n * d) / 600.0)) < 0.5 * n * d - d
        m &= inside[None, :]
        errs.append(np.abs(got - flat_ref)[m].max() / flat_ref.max())
    assert errs[2] < 5e-4 and errs[1] < errs[0] / 2 and errs[2] < errs[0] / 5   # falls with the pixel size (interpolation error)
    # without flattening the curved image is visibly not the flat one
    assert np.abs(ball(S, Pc, cen, rad, rho) - flat_ref)[m].max() / flat_ref.max() > 20 * errs[2]


def test_fixed_points_and_pure_fan_angle_images():
    n, d, DSD = 65, 1.5, 300.0                                        # odd sizes: a pixel sits exactly on the central ray
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(n, n), dDetector=(d, d), DSD=DSD, DSO=200.0)
    rng = np.random.default_rng(0)
    img = rng.random((1, n, n))
    out = curved.flatten(img, geo)
    assert out[0, n // 2, n // 2] == pytest.approx(img[0, n // 2, n // 2], abs=1e-14)    # u = v = 0 maps to itself
    s = (np.arange(n) + 0.5) * d - 0.5 * n * d
    lin = np.broadcast_to((3.0 + 0.01 * s)[None, None, :], (1, n, n))                     # linear in arc length, constant in v
    u = s
    expect = 3.0 + 0.01 * DSD * np.arctan(u / DSD)
    got = curved.flatten(lin, geo)[0]
    rows = slice(3, n - 3)
    assert np.allclose(got[rows], np.broadcast_to(expect, (n, n))[rows], atol=1e-12)     # bilinear is exact on linear data
    # per-view DSD is honoured
    geo2 = geo.copy(DSD_a=np.array([300.0, 500.0]))
    two = curved.flatten(np.concatenate([lin, lin]), geo2)
    assert np.allclose(two[0], got) and not np.allclose(two[1], got)
