"""Pins of the TV / AwTV oracle (oracle/tv.py; eqs. 7-8) against what the paper and the mathematics
fix: the printed 2-D formula evaluated pixel by pixel, closed forms, the TV limit, finite differences."""
import numpy as np
import pytest

from oracle import tv


def awtv_2d_printed(x, delta):
    """eq. (7)/(8) exactly as printed: two dimensions, i, j = 1..n-1, pixel by pixel."""
    total = 0.0
    for i in range(1, x.shape[0]):
        for j in range(1, x.shape[1]):
            di, dj = x[i, j] - x[i - 1, j], x[i, j] - x[i, j - 1]
            wi, wj = np.exp(-(di / delta) ** 2), np.exp(-(dj / delta) ** 2)
            total += np.sqrt(wj * dj ** 2 + wi * di ** 2)
    return total


def test_nz1_is_the_printed_two_dimensional_formula():
    img = np.random.default_rng(0).random((9, 7))
    for delta in (0.05, 0.3, 5.0):
        assert tv.awtv(img[None], delta) == pytest.approx(awtv_2d_printed(img, delta), rel=1e-13)


def test_single_bright_pixel_closed_form():
    # 3x3 image, x[1,1] = h: terms at (1,1): sqrt(2 w) h, at (2,1) and (1,2): sqrt(w) h, at (2,2): 0
    h, delta = 0.7, 0.9
    img = np.zeros((1, 3, 3))
    img[0, 1, 1] = h
    w = np.exp(-(h / delta) ** 2)
    assert tv.awtv(img, delta) == pytest.approx(h * np.sqrt(w) * (2 + np.sqrt(2)), rel=1e-14)
    assert tv.awtv(img, np.inf) == pytest.approx(h * (2 + np.sqrt(2)), rel=1e-14)      # TV


def test_tv_limit_and_linear_ramp():
    # delta -> infinity gives TV; for x = a i + b j + c k every term is sqrt(a^2+b^2+c^2)
    nz, ny, nx = 5, 6, 7
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    a, b, c = 0.3, -0.2, 0.5
    x = a * i + b * j + c * k
    assert tv.awtv(x) == pytest.approx((nx - 1) * (ny - 1) * (nz - 1) * np.sqrt(a * a + b * b + c * c), rel=1e-13)
    y = np.random.default_rng(1).random((4, 5, 6))
    assert tv.awtv(y, 1e12) == pytest.approx(tv.awtv(y, np.inf), rel=1e-12)
    assert tv.awtv(y, 0.2) < tv.awtv(y, np.inf)             # weights <= 1 only ever lower the norm
    assert np.allclose(tv.awtv_gradient(y, 1e12), tv.awtv_gradient(y, np.inf), rtol=1e-10, atol=1e-12)


def test_constant_image():
    x = np.full((3, 4, 5), 2.5)
    assert tv.awtv(x, 0.1, eps=1e-8) == pytest.approx(2 * 3 * 4 * 1e-4)
    assert np.all(tv.awtv_gradient(x, 0.1, 1e-8) == 0)


@pytest.mark.parametrize("delta", [np.inf, 0.5, 0.08])
def test_gradient_against_central_finite_differences(delta):
    # catches a dropped neighbour term, a wrong sign, frozen weights (P21), a shifted domain
    rng = np.random.default_rng(2)
    x = rng.random((4, 5, 6)) * 0.3
    g = tv.awtv_gradient(x, delta, eps=1e-6)
    h = 1e-6
    for idx in [(0, 0, 0), (0, 2, 3), (1, 0, 4), (2, 3, 0), (3, 4, 5), (1, 1, 1), (2, 2, 2), (3, 0, 0), (0, 4, 5)]:
        xp, xm = x.copy(), x.copy()
        xp[idx] += h
        xm[idx] -= h
        fd = (tv.awtv(xp, delta, 1e-6) - tv.awtv(xm, delta, 1e-6)) / (2 * h)
        assert g[idx] == pytest.approx(fd, rel=1e-5, abs=1e-7), idx
    g2 = tv.awtv_gradient(x[:1], delta, eps=1e-6)           # nz = 1: the 2-D case
    xp, xm = x[:1].copy(), x[:1].copy()
    xp[0, 2, 2] += h
    xm[0, 2, 2] -= h
    assert g2[0, 2, 2] == pytest.approx((tv.awtv(xp, delta, 1e-6) - tv.awtv(xm, delta, 1e-6)) / (2 * h), rel=1e-5)


def test_gradient_sums_to_zero_and_minimiser_descends():
    # every difference enters with +1 and -1: the gradient of a translation-invariant functional sums to zero
    x = np.random.default_rng(3).random((6, 7, 8))
    for delta in (np.inf, 0.3):
        assert abs(tv.awtv_gradient(x, delta).sum()) < 1e-10
    vals = [tv.awtv(tv.minimize_awtv(x, n, 0.05, 0.3), 0.3) for n in (0, 1, 5, 20)]
    assert vals[0] > vals[1] > vals[2] > vals[3]
    x1 = tv.minimize_awtv(x, 1, 0.05, np.inf)
    assert np.sqrt(np.sum((x1 - x) ** 2)) == pytest.approx(0.05, rel=1e-12)         # P22: step length alpha
