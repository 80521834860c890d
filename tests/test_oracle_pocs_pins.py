"""Pins of the ASD-POCS oracle (oracle/pocs.py; reading P23) against what is fixed
independently of it: with the TV step switched off it IS OS-SART (oracle.ossart, itself pinned in
test_oracle_pins.py); one iteration is the hand-written composition "OS-SART sweep, then ng TV descent steps of
length alpha*||first data step||"; the logged norms are recomputed from the iterates; the step-length rule is
re-derived from the log; on noisy data it lowers the TV of the iterate relative to OS-SART."""
import numpy as np
import pytest

from oracle import oracle as orc
from oracle import pocs
from oracle import tv as otv
from workloads import make_config, phantom_for


@pytest.fixture(scope="module")
def case():
    geo, ang, rec = make_config("C1", scale=4, n_angles=12)      # 16^3, 24x24 detector, 12 views
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON)
    rng = np.random.default_rng(3)
    b = b + 0.02 * b.max() * rng.standard_normal(b.shape)           # noisy data: what the TV step is for
    subsets = [list(range(s, 12, 4)) for s in range(4)]
    return geo, ang, b, subsets


def test_without_tv_step_it_is_ossart(case):
    geo, ang, b, subsets = case
    x, hist = pocs.asd_pocs(b, geo, ang, subsets, 3, beta=0.8, beta_red=1.0, ng=0)
    ref, _ = orc.ossart(b, geo, ang, subsets, 3, lam=0.8)
    assert np.array_equal(x, ref)
    assert np.all(hist[:, 2] == 0)                                  # no TV movement


def test_one_iteration_is_the_handwritten_composition(case):
    geo, ang, b, subsets = case
    alpha, ng, delta = 0.01, 7, 0.05
    x, hist = pocs.asd_pocs(b, geo, ang, subsets, 1, beta=1.0, ng=ng, alpha=alpha, delta=delta)
    x1, _ = orc.ossart(b, geo, ang, subsets, 1, lam=1.0)
    dp = np.linalg.norm(x1)                                        # x0 = 0
    ref = otv.minimize_awtv(x1, ng, alpha * dp, delta, 1e-8)
    assert np.allclose(x, ref, rtol=0, atol=1e-14)
    d = orc.ax(x1, geo, ang, orc.SIDDON) - b
    assert hist[0, 0] == pytest.approx(np.linalg.norm(d), rel=1e-13)           # dd: fresh residual of the data step
    assert hist[0, 1] == pytest.approx(dp, rel=1e-13)
    assert hist[0, 2] == pytest.approx(np.linalg.norm(ref - x1), rel=1e-12)
    assert hist[0, 3] == pytest.approx(alpha * dp, rel=1e-13)


def test_relaxation_shrinks_and_step_rule_follows_the_log(case):
    geo, ang, b, subsets = case
    beta_red, alpha_red, r_max, eps = 0.9, 0.5, 0.1, 0.0
    x, hist = pocs.asd_pocs(b, geo, ang, subsets, 5, beta=1.0, beta_red=beta_red, ng=5, alpha=0.05,
                            alpha_red=alpha_red, r_max=r_max, epsilon=eps)
    assert hist.shape == (5, 5)
    for it in range(1, 5):                                          # dtvg used at it = dtvg used at it-1, reduced iff the rule fired
        dd, dp, dg, used = hist[it - 1, :4]
        fired = dg > r_max * dp and dd > eps
        assert hist[it, 3] == pytest.approx(used * (alpha_red if fired else 1.0), rel=1e-14)
    assert any(hist[it, 3] < hist[it - 1, 3] for it in range(1, 5))            # the rule does fire in this case
    # with a huge r_max it never fires
    _, h2 = pocs.asd_pocs(b, geo, ang, subsets, 4, ng=5, alpha=0.05, alpha_red=0.5, r_max=1e9)
    assert np.all(h2[:, 3] == h2[0, 3])
    # with epsilon above every residual it never fires either
    _, h3 = pocs.asd_pocs(b, geo, ang, subsets, 4, ng=5, alpha=0.05, alpha_red=0.5, r_max=0.1, epsilon=1e9)
    assert np.all(h3[:, 3] == h3[0, 3])
    assert np.all(np.abs(hist[:, 4]) <= 1 + 1e-12)                               # a cosine


def test_stops_when_relaxation_is_exhausted(case):
    geo, ang, b, subsets = case
    _, hist = pocs.asd_pocs(b, geo, ang, subsets, 10, beta=1.0, beta_red=0.05, ng=1)
    assert hist.shape[0] == 2                                       # beta: 1 -> 0.05 -> 0.0025 < 0.005 after the 2nd iteration


def test_lowers_tv_relative_to_ossart_and_keeps_the_fit(case):
    geo, ang, b, subsets = case
    x, hist = pocs.asd_pocs(b, geo, ang, subsets, 6, ng=10, alpha=0.02)
    ref, _ = orc.ossart(b, geo, ang, subsets, 6)
    assert otv.awtv(x) < 0.9 * otv.awtv(ref)
    assert hist[-1, 0] < 1.5 * np.linalg.norm(orc.ax(ref, geo, ang, orc.SIDDON) - b)


def test_sart_tv_reductions(case):
    # SART-TV (reading P31): with tv_lambda = 0 it IS OS-SART (bitwise); one iteration is the hand-written composition
    # "sweep, then TV prox"; the prox lowers the TV of the iterate
    from oracle import prox as oprox
    geo, ang, b, subsets = case
    x, r = pocs.sart_tv(b, geo, ang, subsets, 3, lam=0.9, tv_lambda=0.0)
    ref, rr = orc.ossart(b, geo, ang, subsets, 3, lam=0.9)
    assert np.array_equal(x, ref) and np.array_equal(r, rr)
    x1, _ = pocs.sart_tv(b, geo, ang, subsets, 1, tv_lambda=2e-3, tv_iter=15)
    s1, _ = orc.ossart(b, geo, ang, subsets, 1)
    assert np.allclose(x1, oprox.tv_prox(s1, 2e-3, 15), atol=1e-15)
    x4, _ = pocs.sart_tv(b, geo, ang, subsets, 4, tv_lambda=2e-3, tv_iter=15)
    s4, _ = orc.ossart(b, geo, ang, subsets, 4)
    assert oprox.tv_forward(x4) < 0.9 * oprox.tv_forward(s4)
    # relaxation reduction: the second sweep runs with lam * lam_red
    xa, _ = pocs.sart_tv(b, geo, ang, subsets, 2, lam=1.0, lam_red=0.5, tv_lambda=0.0)
    first, _ = orc.ossart(b, geo, ang, subsets, 1, lam=1.0)
    second, _ = orc.ossart(b, geo, ang, subsets, 1, lam=0.5, x0=first)
    assert np.array_equal(xa, second)
