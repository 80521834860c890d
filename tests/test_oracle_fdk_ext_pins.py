"""Pins of the FDK-variants oracle (oracle/fdk_ext.py; readings P26-P28) against what is fixed
independently of it: the FFT formulation with the Ram-Lak window IS the direct convolution of the pinned C oracle; Hann
and Hamming windows are three-tap averages of the Ram-Lak taps (shift theorem); cosine^2 = Hann; the Shepp-Logan taps
tend to the textbook closed form -2/(pi^2 tau^2 (4n^2-1)); Parker / Wang weights of geometrically conjugate rays (found
with the independent geometry of tests/helpers.py) sum to one; short-scan and displaced-detector FDK reconstruct an
analytic ball to rho, and fail to without the weights."""
import numpy as np
import pytest

from oracle import fdk_ext as fx
from oracle import oracle as orc
from tests import helpers as H
from workloads.geometry import Geometry, circular_angles


def taps_from_response(nu, tau, name):
    L = fx.pad_length(nu)
    return np.real(np.fft.ifft(fx.filter_response(nu, tau, name))), L


def test_ram_lak_fft_formulation_is_the_direct_convolution():
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(37, 5), dDetector=(1.3, 1.1), DSD=700.0, DSO=450.0)
    ang = circular_angles(3)
    p = np.random.default_rng(0).random((3, 5, 37))
    assert np.allclose(fx.fdk_filter(p, geo, ang, "ram_lak"), orc.fdk_filter(p, geo, ang), rtol=0, atol=1e-12)


def test_hann_and_hamming_are_three_tap_averages_cosine_squared_is_hann():
    nu, tau = 50, 0.7
    h, L = taps_from_response(nu, tau, "ram_lak")
    for name, a0, a1 in (("hann", 0.5, 0.25), ("hamming", 0.54, 0.23)):
        g, _ = taps_from_response(nu, tau, name)
        ref = a0 * h + a1 * (np.roll(h, 1) + np.roll(h, -1))     # cos(omega) in frequency = mean of the two unit shifts
        assert np.allclose(g, ref, rtol=0, atol=1e-13)
    assert np.allclose(fx.window("cosine", L) ** 2, fx.window("hann", L), atol=1e-15)
    assert fx.window("shepp_logan", L)[0] == 1.0 and fx.window("shepp_logan", L)[L // 2] == pytest.approx(2 / np.pi)
    assert h[0] == pytest.approx(1 / (4 * tau * tau)) and h[1] == pytest.approx(-1 / (np.pi * tau) ** 2) and abs(h[2]) < 1e-15


def test_shepp_logan_taps_tend_to_the_textbook_kernel():
    tau = 1.0
    g, L = taps_from_response(2048, tau, "shepp_logan")          # L = 4096
    n = np.arange(0, 20)
    ref = -2.0 / (np.pi ** 2 * tau ** 2 * (4.0 * n ** 2 - 1.0))
    assert np.allclose(g[:20], ref, rtol=0, atol=2e-6)


def _ray_line(geo, ang, ia, iu):
    S, P = H.pixel_world(geo, ang, ia, np.array([iu]), np.array([geo.nDetector[1] // 2]))
    # central row is at v = +dv/2 for an even detector: use the exact mid-plane by dropping z
    d = (P[0] - S)[:2]
    d = d / np.linalg.norm(d)
    off = S[0] * d[1] - S[1] * d[0]                              # signed distance of the line from the origin
    return d, off


def test_parker_weights_of_conjugate_rays_sum_to_one():
    nu, du, DSD, DSO = 64, 2.0, 1500.0, 1000.0
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(nu, 2), dDetector=(du, 1.0), DSD=DSD, DSO=DSO)
    Gamma = np.arctan(0.5 * nu * du / DSD)
    for direction in (1.0, -1.0):
        eps = Gamma + 0.1
        nA = 721
        th = direction * np.linspace(0.0, np.pi + 2 * eps, nA) + 0.3
        ang = np.stack([th, np.zeros(nA), np.zeros(nA)], 1)
        w = fx.parker_weights(geo, ang)
        assert np.all((w >= 0) & (w <= 1))
        u = (np.arange(nu) + 0.5) * du - 0.5 * nu * du
        checked = 0
        for ia in (0, 40, 200, 333):
            for iu in (3, 20, 45, 60):
                # the conjugate of (theta, u) is the ray at column -u of the view where the reversed line is seen
                d0, off0 = _ray_line(geo, ang, ia, iu)
                ju = nu - 1 - iu
                cands = [ja for ja in range(nA) if np.dot(_ray_line(geo, ang, ja, ju)[0], d0) < -0.99999]
                if not cands:
                    continue
                ja = min(cands, key=lambda j: abs(_ray_line(geo, ang, j, ju)[1] + off0))
                d1, off1 = _ray_line(geo, ang, ja, ju)
                assert abs(off1 + off0) < 0.05 * du               # the same line, traversed the other way
                # weights vary smoothly: allow for the angular grid (one step of 0.5 % of the ramp)
                assert w[ia, iu] + w[ja, ju] == pytest.approx(1.0, abs=0.02)
                checked += 1
        assert checked >= 8
        assert w[nA // 2, nu // 2] == 1.0 and w[0, nu // 2] == 0.0 and w[-1, nu // 2] == pytest.approx(0.0, abs=1e-12)


def test_wang_weights_complement_and_limits():
    nu, du, DSD = 100, 1.5, 1200.0
    for off in (12.0, -21.0):
        geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(nu, 2), dDetector=(du, 1.0), DSD=DSD, DSO=800.0,
                       offDetector=(off, 0.0))
        w = fx.wang_weights(geo, 4)[0]
        u = (np.arange(nu) + 0.5) * du - 0.5 * nu * du + off
        u_ov = 0.5 * nu * du - abs(off)
        s = np.sign(off)
        assert np.all(w[u * s > u_ov] == 1.0)
        assert np.all(np.diff(w) * s >= -1e-15)                  # monotone towards the long side
        # a full circle sees every line of the overlap twice, at +u and -u: the two weights sum to one
        inside = np.abs(u) < u_ov
        wi = np.interp(-u[inside], u if s > 0 else u, w)         # weight at the mirrored coordinate
        assert np.allclose(w[inside] + wi, 1.0, atol=2e-3)
        assert w[np.argmin(np.abs(u))] == pytest.approx(0.5, abs=0.02)


def _ball_projections(geo, ang, rho, rad, cen):
    nu, nv = geo.nDetector
    ell = dict(centre=cen[None], axes=np.full((1, 3), rad), Q=np.eye(3)[None], rho=np.array([rho]))
    iu, iv = np.meshgrid(np.arange(nu), np.arange(nv))
    proj = np.zeros((len(ang), nv, nu))
    for ia in range(len(ang)):
        S, P = H.pixel_world(geo, ang, ia, iu, iv)
        proj[ia] = H.ellipsoid_line_integrals(ell, S, P)
    return proj


def _ball_levels(x, geo, rad, cen):
    c = H.voxel_centres(geo, (0, 0, 0))
    d = np.linalg.norm(c - cen, axis=-1)
    mid = np.abs(c[..., 2]) < 4.0
    return x[(d < rad - 2.5) & mid].mean(), x[(d > rad + 2.5) & (d < 18) & mid].mean()


def test_short_scan_fdk_with_parker_weights_reconstructs_the_ball():
    n, nd = 40, 64
    geo = Geometry(nVoxel=(n, n, n), dVoxel=(1.0,) * 3, nDetector=(nd, nd), dDetector=(1.5, 1.5), DSD=1536.0, DSO=1000.0)
    Gamma = np.arctan(0.5 * nd * 1.5 / 1536.0)
    nA = 90
    th = np.linspace(0.0, np.pi + 2 * (Gamma + 0.05), nA) + 0.4
    ang = np.stack([th, np.zeros(nA), np.zeros(nA)], 1)
    rho, rad, cen = 0.02, 12.0, np.array([3.0, -2.0, 0.0])
    proj = _ball_projections(geo, ang, rho, rad, cen)
    for filt, tol in (("ram_lak", 0.015), ("shepp_logan", 0.02), ("hann", 0.03)):
        inside, outside = _ball_levels(fx.fdk(proj, geo, ang, filt, "parker"), geo, rad, cen)
        assert abs(inside / rho - 1.0) < tol, (filt, inside / rho)
        assert abs(outside) < 0.02 * rho
    # without the weights the doubly measured lines count twice: the level is off by far more than the tolerance
    q = fx.fdk_filter(proj, geo, ang, "ram_lak")
    naive = (th[-1] - th[0]) / (nA - 1) * orc.atb(q, geo, ang, orc.FDK)
    assert abs(_ball_levels(naive, geo, rad, cen)[0] / rho - 1.0) > 0.05


def test_displaced_detector_fdk_with_wang_weights_reconstructs_the_ball():
    n, nd = 40, 48
    geo = Geometry(nVoxel=(n, n, n), dVoxel=(1.0,) * 3, nDetector=(nd, 64), dDetector=(1.5, 1.5), DSD=1536.0, DSO=1000.0,
                   offDetector=(20.0, 0.0))                       # detector spans u in [-16, 56], the ball shadow +-24: half-fan
    ang = circular_angles(120)
    rho, rad, cen = 0.02, 12.0, np.array([3.0, -2.0, 0.0])
    proj = _ball_projections(geo, ang, rho, rad, cen)
    inside, outside = _ball_levels(fx.fdk(proj, geo, ang, "ram_lak", "wang"), geo, rad, cen)
    assert abs(inside / rho - 1.0) < 0.015, inside / rho          # (the narrower the overlap, the rougher: 7 % at 10 mm)
    assert abs(outside) < 0.1 * rho
    plain_in, _ = _ball_levels(fx.fdk(proj, geo, ang, "ram_lak", None), geo, rad, cen)
    assert abs(plain_in / rho - 1.0) > 0.1                       # truncated rows through the ramp filter: wrong level


# ------------------------------------------------------------------ the cosine pre-weight of P12 / P34
def _cosine_weight_from_geometry(geo, ang, ia, iu, iv):
    """cos of the angle between the ray source -> pixel and the detector normal, from the independent WORLD-frame geometry of
    tests/helpers.py: for an unrotated detector this is the textbook FDK pre-weight DSD / sqrt(DSD^2 + u^2 + v^2) with (u, v)
    measured from the foot of the source's perpendicular on the detector."""
    S, Dc, eu, ev, n, p = H.world_frame(geo, ang, ia)
    _, P = H.pixel_world(geo, ang, ia, np.array([iu]), np.array([iv]))
    d = P[0] - S
    return abs(d @ n) / np.linalg.norm(d)


@pytest.mark.parametrize("offD", [(0.0, 0.0), (25.0, -10.0)])
def test_fdk_filter_impulse_response_pins_the_cosine_weight(offD):
    """A single bright pixel far off the axis of a SHORT geometry (weight ~ 0.85): the filtered row is
    tau * cos * h[n] (h the Ram-Lak taps of P12), every other row stays zero.  With a displaced detector the weight is
    centred on the principal ray, not on the detector (reading P34)."""
    nu, nv, du, dv = 40, 30, 4.0, 4.0
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(nu, nv), dDetector=(du, dv), DSD=150.0, DSO=100.0,
                   offDetector=offD)
    ang = circular_angles(3, start=0.4)
    tau = du * geo.DSO / geo.DSD
    for ia, iu0, iv0 in ((1, 29, 26), (2, 2, 3), (0, 20, 15)):
        p = np.zeros((3, nv, nu))
        p[ia, iv0, iu0] = 1.0
        cosw = _cosine_weight_from_geometry(geo, ang, ia, iu0, iv0)
        u0 = (iu0 + 0.5) * du - 0.5 * nu * du + offD[0]
        v0 = (iv0 + 0.5) * dv - 0.5 * nv * dv + offD[1]
        assert cosw == pytest.approx(geo.DSD / np.sqrt(geo.DSD ** 2 + u0 ** 2 + v0 ** 2), rel=1e-13)
        if (iu0, iv0) != (20, 15):
            assert cosw < 0.95                                      # far from 1: a dropped weight is a >5 % error here
        n = np.arange(nu) - iu0
        h = np.where(n == 0, 1.0 / (4 * tau * tau), np.where(n % 2 != 0, -1.0 / (np.pi * np.where(n == 0, 1, n) * tau) ** 2, 0.0))
        want = np.zeros((3, nv, nu))
        want[ia, iv0] = tau * cosw * h
        for got in (orc.fdk_filter(p, geo, ang), fx.fdk_filter(p, geo, ang, "ram_lak")):
            assert np.allclose(got, want, rtol=0, atol=1e-12 * abs(want).max())


def _wide_fan_problem(offu=0.0, nu=168):
    # source 200 mm from the axis: short geometry, wide fan
    geo = Geometry(nVoxel=(96, 96, 2), dVoxel=(1.5, 1.5, 1.0), nDetector=(nu, 4), dDetector=(2.5, 2.5), DSD=300.0, DSO=200.0,
                   offDetector=(offu, 0.0))
    ang = circular_angles(240)
    rho, rad, cen = 0.02, 12.0, np.array([52.0, -25.0, 0.0])       # a small ball far off the axis: seen at fan angles up to 20 deg
    return geo, ang, rho, rad, cen


def _wide_levels(x, geo, rad, cen):
    c = H.voxel_centres(geo, (0, 0, 0))
    d = np.linalg.norm(c - cen, axis=-1)
    return x[d < rad - 4.0].mean(), x[(d > rad + 4.0) & (d < rad + 9.0)].mean()


def test_wide_fan_fdk_needs_the_cosine_weight():
    """Mid-plane FDK is exact fan-beam FBP: an analytic ball seen under fan angles up to 20 degrees comes back at rho; without
    the cosine pre-weight the level is 2 % off (the pin that a 1536 mm geometry cannot give: there the weight
    is 0.999)."""
    geo, ang, rho, rad, cen = _wide_fan_problem()
    proj = _ball_projections(geo, ang, rho, rad, cen)
    inside, outside = _wide_levels(orc.fdk(proj, geo, ang), geo, rad, cen)
    assert abs(inside / rho - 1.0) < 0.005, inside / rho
    assert abs(outside) < 0.01 * rho
    # the same reconstruction with the weight divided out again
    nu, nv = geo.nDetector
    u = (np.arange(nu) + 0.5) * 2.5 - 0.5 * nu * 2.5
    v = (np.arange(nv) + 0.5) * 2.5 - 0.5 * nv * 2.5
    cosw = geo.DSD / np.sqrt(geo.DSD ** 2 + u[None, :] ** 2 + v[:, None] ** 2)
    naive, _ = _wide_levels(orc.fdk(proj / cosw[None], geo, ang), geo, rad, cen)
    assert abs(naive / rho - 1.0) > 0.015, naive / rho            # 2.1 %: four times the tolerance above


def test_displaced_wide_fan_fdk_centres_the_cosine_weight_on_the_principal_ray():
    """Detector displaced by a quarter of its width (the case Wang weights exist for): the level inside the ball
    is right to 0.5 % only if the cosine weight is centred on the principal ray (u + offDetector_u), reading P34."""
    nu = 120
    geo, ang, rho, rad, cen = _wide_fan_problem(offu=0.25 * nu * 2.5, nu=nu)
    proj = _ball_projections(geo, ang, rho, rad, cen)
    inside, outside = _wide_levels(fx.fdk(proj, geo, ang, "ram_lak", "wang"), geo, rad, cen)
    assert abs(inside / rho - 1.0) < 0.005, inside / rho
    assert abs(outside) < 0.02 * rho
