"""GPU parity of the TV proximal operator and FISTA (tigre_tv_prox, tigre_fista; SURVEY.md section 8(f).2;
PAPER.md:122, 308-314, 377-393; readings P24, P25) against oracle/prox.py.  Tolerances (none stated by north_star for
this row; from the arithmetic): one dual iteration is a handful of fp32 operations per voxel and the iteration is
non-expansive, so n iterations stay within ~n ulp: 1e-5 rel-L2 on u; FISTA compounds the projector pair (1e-5 per
call for Siddon / matched) with the prox: 1e-4 on the iterate and the residual history."""
import numpy as np
import pytest

from oracle import oracle as orc
from oracle import prox as oprox
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


# (nz, ny, nx): ragged scalar path, 2-D, 1-D, and nx % 4 == 0 (four voxels per thread) incl. a multi-row / multi-plane case
SHAPES = [(13, 17, 21), (1, 19, 23), (1, 1, 40), (7, 1, 5), (6, 10, 32), (20, 33, 64), (3, 5, 4)]


@pytest.mark.parametrize("shape", SHAPES)
def test_prox_matches_oracle(tg, shape):
    rng = np.random.default_rng(sum(shape))
    f = rng.random(shape).astype(np.float32)
    f[: shape[0] // 2 + 1, : shape[1] // 2 + 1] += 1.0                 # an edge plus noise
    for lam, n in ((0.1, 25), (0.5, 60)):
        ref = oprox.tv_prox(f, lam, n)
        u = tg.tv_prox(dev(f), lam, n)
        assert H.rel_l2(host(u), ref) <= 1e-5
    assert torch.equal(tg.tv_prox(dev(f), 0.0, 10), dev(f))           # lam = 0 copies
    t = dev(f)
    tg.tv_prox(t, 0.1, 25, out=t)                                     # in place
    assert H.rel_l2(host(t), oprox.tv_prox(f, 0.1, 25)) <= 1e-5


def test_prox_one_dimensional_step_closed_form_on_gpu(tg):
    n1, n2, a, b, lam = 5, 8, 0.2, 1.0, 0.3
    f = np.concatenate([np.full(n1, a), np.full(n2, b)]).astype(np.float32)
    ref = np.concatenate([np.full(n1, a + lam / n1), np.full(n2, b - lam / n2)])
    for shape in ((1, 1, -1), (1, -1, 1), (-1, 1, 1)):
        u = tg.tv_prox(dev(f.reshape(shape)), lam, 4000, tau=0.25)
        assert np.allclose(host(u).ravel(), ref, atol=2e-5)


def test_prox_full_size_properties(tg):
    # C3's volume size: properties that hold at any size + a sub-block against the oracle (n dual iterations reach n voxels)
    g = torch.Generator(device="cuda").manual_seed(9)
    f = torch.rand((512, 512, 512), generator=g, device="cuda")
    n = 6
    u = tg.tv_prox(f, 0.2, n)
    assert float(u.double().sum()) == pytest.approx(float(f.double().sum()), rel=1e-7)      # div p sums to zero (each u is rounded to fp32: 6e-8)
    blk = f[100:140, 200:240, 300:364].cpu().numpy()
    ref = oprox.tv_prox(blk, 0.2, n)[n + 1:-n - 1, n + 1:-n - 1, n + 1:-n - 1]
    got = host(u[100:140, 200:240, 300:364])[n + 1:-n - 1, n + 1:-n - 1, n + 1:-n - 1]
    assert H.rel_l2(got, ref) <= 1e-5


@pytest.mark.parametrize("modes", [("siddon", "matched", False), ("interp", "fdk", False), ("siddon", "exact_siddon", True)])
def test_fista_matches_oracle(tg, modes):
    axm, atm, exact = modes
    geo, ang, rec = make_config("C1", scale=2, n_angles=16)             # 32^3, 48x48 detector, 16 views
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON)
    b = (b + 0.02 * b.max() * np.random.default_rng(11).standard_normal(b.shape)).astype(np.float32)
    oax = orc.SIDDON if axm == "siddon" else orc.INTERP
    oat = orc.FDK if atm == "fdk" else orc.MATCHED
    # L: a safe upper bound of 2 ||A||^2 from ||A^T A 1||_inf (row sums of a nonnegative matrix)
    At = (lambda y: orc.atb_exact(y, geo, ang, oax)) if exact else (lambda y: orc.atb(y, geo, ang, oat))
    L = 2.0 * float(At(orc.ax(np.ones(geo.vol_shape), geo, ang, oax)).max())
    lam = 2e-4
    ref, rref = oprox.fista(b, geo, ang, 5, L, lam, 10, ax_mode=oax, atb_mode=oat, exact_adjoint=exact)
    x, resid = tg.fista(dev(b), geo, ang, 5, L, lam, 10, ax_mode=axm, atb_mode=atm)
    tol = 1e-4 if axm == "siddon" else 2e-4
    assert np.allclose(resid, rref, rtol=tol)
    assert H.rel_l2(host(x), ref) <= tol
    assert rref[-1] < rref[0]


def test_gradient_descent_eq4_matches_oracle(tg):
    geo, ang, rec = make_config("C1", scale=2, n_angles=16)
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON).astype(np.float32)
    lam = 1.0 / float(orc.atb(orc.ax(np.ones(geo.vol_shape), geo, ang, orc.SIDDON), geo, ang, orc.MATCHED).max())
    for atm, exact in (("matched", False), ("exact_siddon", True)):
        ref, rref = orc.gradient_descent(b, geo, ang, 5, lam, exact_adjoint=exact)
        x, resid = tg.gradient_descent(dev(b), geo, ang, 5, lam, atb_mode=atm)
        assert H.rel_l2(host(x), ref) <= 1e-4 and np.allclose(resid, rref, rtol=1e-4)
        assert resid[-1] < resid[0]


def test_fista_init_and_argument_errors(tg):
    geo, ang, rec = make_config("C1", scale=4, n_angles=6)
    vol = phantom_for(rec, geo).astype(np.float32)
    b = tg.Ax(dev(vol), geo, ang, "siddon")
    x0 = dev(vol * 0.5)
    ref, _ = oprox.fista(host(b), geo, ang, 2, 500.0, 1e-3, 5, x0=vol * 0.5)
    x, _ = tg.fista(b, geo, ang, 2, 500.0, 1e-3, 5, x0=x0)
    assert H.rel_l2(host(x), ref) <= 1e-4
    with pytest.raises(tg.TigreError) as e:
        tg.fista(b, geo, ang, 1, 0.0, 1e-3, 5)                        # L must be positive
    assert e.value.code == -1
    with pytest.raises(tg.TigreError) as e:
        tg.tv_prox(torch.zeros((4, 4, 4)), 0.1, 3, out=torch.zeros((4, 4, 4)))   # host tensors
    assert e.value.code == -3
