"""GPU parity of the ASD-POCS family (tigre_plan_asd_pocs, PAPER.md:116, 141-149, 169;
reading P23) against oracle/pocs.py on the same seeded inputs.  Tolerance: the data step is the OS-SART sweep
(1e-5 per projector call), the regulariser step the TV minimiser (1e-5); a few iterations of both compound to
<= 1e-4 rel-L2 on the iterate and on the logged norms.  The step-length rule compares floating-point norms: the
cases are chosen away from its knife edge and the test checks that both sides took the same decisions."""
import numpy as np
import pytest

from oracle import oracle as orc
from oracle import pocs as opocs
from tests import helpers as H
from workloads import make_config, phantom_for

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2412_10129_b200 as m
    m.version()
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


def noisy_case(scale, n_angles, seed):
    geo, ang, rec = make_config("C1", scale=scale, n_angles=n_angles)
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON)
    b = b + 0.02 * b.max() * np.random.default_rng(seed).standard_normal(b.shape)
    return geo, ang, b.astype(np.float32)


def decisions(hist, r_max, eps):
    return [(h[2] > r_max * h[1]) and (h[0] > eps) for h in hist]


@pytest.mark.parametrize("delta", [None, 0.004])
def test_os_asd_pocs_matches_oracle(tg, delta):
    geo, ang, b = noisy_case(2, 24, 5)                       # 32^3, 48x48 detector, 24 views, 4 blocks of 6
    subsets = [list(range(s, 24, 4)) for s in range(4)]
    kw = dict(beta=1.0, beta_red=0.9, ng=8, alpha=0.02, alpha_red=0.6, r_max=0.2, epsilon=0.0)
    ref, href = opocs.asd_pocs(b, geo, ang, subsets, 4, delta=np.inf if delta is None else delta, **kw)
    plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched")
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    hist = plan.asd_pocs(dev(b), x, 4, delta=delta, **kw)
    plan.close()
    assert hist.shape == href.shape
    assert decisions(hist, 0.2, 0.0) == decisions(href, 0.2, 0.0)
    assert np.allclose(hist[:, :4], href[:, :4], rtol=1e-4)
    assert np.allclose(hist[:, 4], href[:, 4], atol=1e-3)
    assert H.rel_l2(host(x), ref) <= 1e-4


def test_asd_pocs_single_view_subsets_interp_fdk_weights(tg):
    # ASD-POCS proper: every view its own subset (SART data step); the other projector pair
    geo, ang, b = noisy_case(4, 10, 6)                       # 16^3, 24x24 detector, 10 views
    subsets = [[a] for a in range(10)]
    kw = dict(beta=0.7, beta_red=0.95, ng=5, alpha=0.01, alpha_red=0.5, r_max=0.5, epsilon=0.0)
    ref, href = opocs.asd_pocs(b, geo, ang, subsets, 3, ax_mode=orc.INTERP, atb_mode=orc.FDK, **kw)
    plan = tg.OssartPlan(geo, ang, subsets, "interp", "fdk")
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    hist = plan.asd_pocs(dev(b), x, 3, **kw)
    plan.close()
    assert decisions(hist, 0.5, 0.0) == decisions(href, 0.5, 0.0)
    assert np.allclose(hist[:, :4], href[:, :4], rtol=2e-4)
    assert H.rel_l2(host(x), ref) <= 2e-4                    # interpolated / FDK-weighted pair: 1e-4 per call


def test_no_tv_steps_is_the_ossart_sweep_and_early_stop(tg):
    geo, ang, b = noisy_case(2, 24, 7)
    subsets = [list(range(s, 24, 4)) for s in range(4)]
    plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched")
    bd = dev(b)
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    hist = plan.asd_pocs(bd, x, 2, beta=0.8, beta_red=1.0, ng=0)
    y = torch.zeros_like(x)
    plan.iterate(bd, y, 2, lam=0.8)
    assert torch.equal(x, y)
    assert np.all(hist[:, 2] == 0)
    # relaxation exhausted: 1 -> 0.05 -> 0.0025 < 0.005 stops after the second iteration
    z = torch.zeros_like(x)
    h2 = plan.asd_pocs(bd, z, 10, beta=1.0, beta_red=0.05, ng=1)
    assert h2.shape[0] == 2
    plan.close()


def test_larger_problem_composition_and_tv_drop(tg):
    # C3 at half size (256^3, 360 views of 512x384, 20 subsets): one iteration equals the composition of the
    # library's own OS-SART sweep and TV minimiser; the TV of the iterate drops
    geo, ang, rec = make_config("C3", scale=2)
    vol = dev(phantom_for(rec, geo))
    b = tg.Ax(vol, geo, ang, "siddon")
    gen = torch.Generator(device="cuda").manual_seed(3)
    b = b + 0.02 * float(b.max()) * torch.randn(b.shape, generator=gen, device="cuda")
    nA = len(ang)
    subsets = [list(range(s, nA, 20)) for s in range(20)]
    plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched")
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    hist = plan.asd_pocs(b, x, 1, ng=10, alpha=0.01)
    y = torch.zeros_like(x)
    plan.iterate(b, y, 1)
    dp = float(y.double().norm())
    assert hist[0, 1] == pytest.approx(dp, rel=1e-6)
    assert hist[0, 3] == pytest.approx(0.01 * dp, rel=1e-6)
    assert hist[0, 0] == pytest.approx(float((tg.Ax(y, geo, ang, "siddon") - b).double().norm()), rel=1e-5)
    tv0 = tg.awtv(y, None, 1e-8)
    tg.minimize_awtv(y, 10, float(np.float32(hist[0, 3])), None, 1e-8)
    assert float((x - y).double().norm()) <= 1e-6 * float(y.double().norm())
    assert tg.awtv(x, None, 1e-8) < tv0
    plan.close()


def test_sart_tv_matches_oracle(tg):
    geo, ang, b = noisy_case(2, 24, 9)
    subsets = [list(range(s, 24, 4)) for s in range(4)]
    ref, rref = opocs.sart_tv(b, geo, ang, subsets, 3, lam=1.0, lam_red=0.9, tv_lambda=1e-3, tv_iter=12)
    plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched")
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    res = plan.sart_tv(dev(b), x, 3, lam=1.0, lam_red=0.9, tv_lambda=1e-3, tv_iter=12)
    assert H.rel_l2(host(x), ref) <= 1e-4
    assert np.allclose(res, rref, rtol=1e-4)
    y = torch.zeros_like(x)
    plan.sart_tv(dev(b), y, 2, lam=0.8, tv_lambda=0.0)                 # no regularisation: the plain sweeps
    z = torch.zeros_like(x)
    plan.iterate(dev(b), z, 2, lam=0.8)
    assert torch.equal(y, z)
    plan.close()


def test_mlem_and_osem_match_oracle(tg):
    geo, ang, b = noisy_case(2, 24, 10)
    b = np.abs(b) + 0.01
    for subsets in ([list(range(24))], [list(range(s, 24, 4)) for s in range(4)]):       # MLEM, OSEM
        ref = orc.osem(b, geo, ang, subsets, 3)
        plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched")
        x = torch.ones(geo.vol_shape, dtype=torch.float32, device="cuda")
        plan.osem(dev(b), x, 3)
        plan.close()
        assert H.rel_l2(host(x), ref) <= 1e-4
        assert float(x.min()) >= 0.0


def test_argument_errors(tg):
    geo, ang, b = noisy_case(4, 4, 8)
    plan = tg.OssartPlan(geo, ang, [[0, 1], [2, 3]], "siddon", "matched")
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    with pytest.raises(tg.TigreError) as e:
        plan.asd_pocs(dev(b), x, 1, ng=-1)
    assert e.value.code == -1
    with pytest.raises(tg.TigreError) as e:
        plan.asd_pocs(torch.from_numpy(b), x, 1)              # host projections
    assert e.value.code == -3
    plan.close()
