"""Pins of the TV-prox / FISTA oracle (oracle/prox.py; readings P24, P25) against
what the mathematics fixes: div = -grad^T; the closed-form TV denoising of a 1-D two-level step; optimality of the
prox against perturbations and against scipy's minimiser of the smoothed objective on a tiny volume; mean
preservation; the O(1/k^2) bound of [42] on an explicit least-squares problem and convergence to its lstsq solution;
the first iterate written out by hand."""
import numpy as np
import pytest
from scipy.optimize import minimize

from oracle import oracle as orc
from oracle import prox
from workloads import make_config


def test_div_is_minus_grad_transpose():
    rng = np.random.default_rng(0)
    for shape in ((4, 5, 6), (1, 7, 3), (5, 1, 1), (2, 2, 2)):
        d = rng.standard_normal(shape)
        p = [rng.standard_normal(shape) for _ in range(3)]
        g = prox.grad(d)
        lhs = sum(float(np.sum(g[a] * p[a])) for a in range(3))
        assert lhs == pytest.approx(-float(np.sum(d * prox.div(p))), rel=1e-12, abs=1e-12)


def test_one_dimensional_step_closed_form():
    # f = a on n1 samples then b on n2 samples (a < b): the minimiser of 1/2||u-f||^2 + lam*sum|du| keeps two plateaus,
    # raised by lam/n1 and lowered by lam/n2 (as long as they do not meet)
    n1, n2, a, b, lam = 5, 8, 0.2, 1.0, 0.3
    f = np.concatenate([np.full(n1, a), np.full(n2, b)])[None, None, :]
    u = prox.tv_prox(f, lam, 4000, tau=0.25)                 # one dimension: tau <= 1/4
    ref = np.concatenate([np.full(n1, a + lam / n1), np.full(n2, b - lam / n2)])
    assert np.allclose(u[0, 0], ref, atol=1e-6)
    # the same signal laid along y and along z (catches a transposed axis)
    assert np.allclose(prox.tv_prox(f.reshape(1, -1, 1), lam, 4000, tau=0.25)[0, :, 0], ref, atol=1e-6)
    assert np.allclose(prox.tv_prox(f.reshape(-1, 1, 1), lam, 4000, tau=0.25)[:, 0, 0], ref, atol=1e-6)
    # lam large enough for the plateaus to meet: the mean
    big = prox.tv_prox(f, 50.0, 20000, tau=0.25)
    assert np.allclose(big, f.mean(), atol=1e-5)


def test_trivial_cases_and_mean_preservation():
    rng = np.random.default_rng(1)
    f = rng.random((4, 5, 6))
    assert np.array_equal(prox.tv_prox(f, 0.0, 10), f)
    c = np.full((3, 4, 5), 1.7)
    assert np.allclose(prox.tv_prox(c, 0.4, 25), c, atol=1e-14)
    u = prox.tv_prox(f, 0.1, 30)
    assert u.sum() == pytest.approx(f.sum(), rel=1e-13)         # div p sums to zero
    assert prox.tv_forward(u) < prox.tv_forward(f)


def test_prox_is_the_minimiser_on_a_tiny_volume():
    rng = np.random.default_rng(2)
    f = rng.random((3, 3, 4))
    lam = 0.15
    u = prox.tv_prox(f, lam, 6000)

    def energy(v):
        v = v.reshape(f.shape)
        return 0.5 * float(np.sum((v - f) ** 2)) + lam * prox.tv_forward(v)

    e = energy(u)
    assert e < energy(f)
    for _ in range(50):                                          # no nearby point is better
        assert e <= energy(u + 1e-3 * rng.standard_normal(f.shape)) + 1e-12

    def smooth(v):                                               # scipy on the smoothed objective lands at the same energy
        v = v.reshape(f.shape)
        g = prox.grad(v)
        return 0.5 * float(np.sum((v - f) ** 2)) + lam * float(np.sum(np.sqrt(g[0] ** 2 + g[1] ** 2 + g[2] ** 2 + 1e-12)))

    res = minimize(smooth, f.ravel(), method="L-BFGS-B", options={"maxiter": 5000, "ftol": 1e-15, "gtol": 1e-10})
    assert e == pytest.approx(energy(res.x), rel=2e-4)
    assert e <= energy(res.x) + 1e-9


@pytest.fixture(scope="module")
def tiny_system():
    geo, ang, rec = make_config("C1", scale=16, n_angles=6)      # 4^3 volume, 6x6 detector, 6 views
    n = int(np.prod(geo.vol_shape))
    A = np.zeros((6 * 6 * 6, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        A[:, j] = orc.ax(e.reshape(geo.vol_shape), geo, ang, orc.SIDDON).ravel()
    rng = np.random.default_rng(4)
    xt = rng.random(n)
    b = (A @ xt + 0.01 * rng.standard_normal(A.shape[0])).reshape(6, 6, 6)
    return geo, ang, A, b


def test_fista_rate_bound_and_limit(tiny_system):
    # lam = 0 (prox = identity), exact adjoint: F(x_k) - F* <= 2 L ||x0 - x*||^2 / (k+1)^2 with F = ||Ax-b||^2 and
    # L >= its gradient's Lipschitz constant 2 sigma_max^2 (Beck & Teboulle, Theorem 4.4), and x_k -> lstsq solution
    geo, ang, A, b = tiny_system
    xs, *_ = np.linalg.lstsq(A, b.ravel(), rcond=None)
    Fs = float(np.sum((A @ xs - b.ravel()) ** 2))
    L = 2.0 * np.linalg.svd(A, compute_uv=False)[0] ** 2
    for k in (1, 2, 5, 10, 40):
        x, _ = prox.fista(b, geo, ang, k, L, 0.0, 0, exact_adjoint=True)
        F = float(np.sum((A @ x.ravel() - b.ravel()) ** 2))
        assert F - Fs <= 2.0 * L * float(np.sum(xs ** 2)) / (k + 1) ** 2 + 1e-12
    x, resid = prox.fista(b, geo, ang, 3000, L, 0.0, 0, exact_adjoint=True)
    assert np.linalg.norm(A @ x.ravel() - b.ravel()) == pytest.approx(np.sqrt(Fs), rel=1e-3)
    assert resid[0] == pytest.approx(np.linalg.norm(b), rel=1e-14)                 # y_0 = 0
    # momentum matters: plain gradient steps (one FISTA iteration restarted k times) are slower at k = 40
    xi = np.zeros(geo.vol_shape)
    for _ in range(40):
        xi, _ = prox.fista(b, geo, ang, 1, L, 0.0, 0, exact_adjoint=True, x0=xi)
    x40, _ = prox.fista(b, geo, ang, 40, L, 0.0, 0, exact_adjoint=True)
    assert np.sum((A @ x40.ravel() - b.ravel()) ** 2) < np.sum((A @ xi.ravel() - b.ravel()) ** 2)


def test_fista_first_iterates_by_hand(tiny_system):
    geo, ang, A, b = tiny_system
    L, lam, nit = 50.0, 0.02, 7
    x1, _ = prox.fista(b, geo, ang, 1, L, lam, nit)
    At = lambda r: orc.atb(r, geo, ang, orc.MATCHED)
    x1_ref = prox.tv_prox((2.0 / L) * At(b), lam, nit)
    assert np.allclose(x1, x1_ref, atol=1e-15)
    x2, resid = prox.fista(b, geo, ang, 2, L, lam, nit)
    t1 = (1 + np.sqrt(5.0)) / 2
    y1 = x1_ref + 0.0 * x1_ref                                  # (t_0 - 1)/t_1 = 0: no momentum yet
    r1 = b - orc.ax(y1, geo, ang, orc.SIDDON)
    x2_ref = prox.tv_prox(y1 + (2.0 / L) * At(r1), lam, nit)
    assert np.allclose(x2, x2_ref, atol=1e-14)
    assert resid[1] == pytest.approx(np.linalg.norm(r1), rel=1e-13)
    x3, _ = prox.fista(b, geo, ang, 3, L, lam, nit)
    t2 = (1 + np.sqrt(1 + 4 * t1 * t1)) / 2
    y2 = x2_ref + (t1 - 1) / t2 * (x2_ref - x1_ref)
    x3_ref = prox.tv_prox(y2 + (2.0 / L) * At(b - orc.ax(y2, geo, ang, orc.SIDDON)), lam, nit)
    assert np.allclose(x3, x3_ref, atol=1e-14)


def test_gradient_descent_is_fista_without_momentum_and_converges(tiny_system):
    # eq. (4) (reading P32): one FISTA iteration with lam_tv = 0 IS a gradient step of length 2/L; iterating it from its own
    # result reproduces gradient descent with lam = 2/L; with lam < 2/sigma_max^2 the residual decreases monotonically to
    # the least-squares residual
    geo, ang, A, b = tiny_system
    smax = np.linalg.svd(A, compute_uv=False)[0]
    lam = 1.0 / smax ** 2
    x, resid = orc.gradient_descent(b, geo, ang, 4, lam, exact_adjoint=True)
    xi = np.zeros(geo.vol_shape)
    for _ in range(4):
        xi, _ = prox.fista(b, geo, ang, 1, 2.0 / lam, 0.0, 0, exact_adjoint=True, x0=xi)
    assert np.allclose(x, xi, rtol=1e-13, atol=1e-15)
    _, resid = orc.gradient_descent(b, geo, ang, 300, lam, exact_adjoint=True)
    assert np.all(np.diff(resid) <= 1e-12)
    xs, *_ = np.linalg.lstsq(A, b.ravel(), rcond=None)
    assert resid[-1] >= np.linalg.norm(A @ xs - b.ravel()) - 1e-12
    # and by hand: the first step from zero is lam A^T b
    x1, r1 = orc.gradient_descent(b, geo, ang, 1, lam, exact_adjoint=True)
    assert np.allclose(x1.ravel(), lam * (A.T @ b.ravel()), rtol=1e-12, atol=1e-15)
    assert r1[0] == pytest.approx(np.linalg.norm(b), rel=1e-14)


def test_mlem_eq5_by_hand_fixed_point_and_kl_descent(tiny_system):
    # eq. (5): the first iterate from x = 1 written with the explicit matrix; a consistent solution is a fixed point; with
    # the exact adjoint the Kullback-Leibler distance KL(b, Ax) never increases (the classical EM property); one subset of
    # all views = MLEM, and OSEM with the subsets visited in turn equals chained single-subset calls
    geo, ang, A, b = tiny_system
    b = np.abs(b) + 0.05
    bv = b.ravel()
    x1 = orc.mlem(b, geo, ang, 1, exact_adjoint=True)
    hit = (A @ np.ones(A.shape[1])) > 0                      # rays that meet the volume (the others have a zero row)
    q = np.zeros_like(bv)
    q[hit] = bv[hit] / (A @ np.ones(A.shape[1]))[hit]
    ref = (1.0 / (A.T @ np.ones(A.shape[0]))) * (A.T @ q)
    assert np.allclose(x1.ravel(), ref, rtol=1e-12)
    xs = np.random.default_rng(5).random(A.shape[1]) + 0.1
    bc = (A @ xs).reshape(b.shape)
    keep = orc.mlem(bc, geo, ang, 3, exact_adjoint=True, x0=xs.reshape(geo.vol_shape))
    assert np.allclose(keep.ravel(), xs, rtol=1e-12)

    def kl(x):
        p = (A @ x.ravel())[hit]
        return float(np.sum(bv[hit] * np.log(bv[hit] / p) - bv[hit] + p))

    vals = [kl(orc.mlem(b, geo, ang, k, exact_adjoint=True)) for k in range(1, 9)]
    assert all(vals[i + 1] <= vals[i] + 1e-12 for i in range(7)) and vals[-1] < 0.5 * vals[0]
    subs = [[0, 2, 4], [1, 3, 5]]
    full = orc.osem(b, geo, ang, subs, 1, exact_adjoint=True)
    step = orc.osem(b, geo, ang, [subs[0]], 1, exact_adjoint=True)
    step = orc.osem(b, geo, ang, [subs[1]], 1, exact_adjoint=True, x0=step)
    assert np.allclose(full, step, rtol=1e-13)
