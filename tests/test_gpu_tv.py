"""GPU parity of the TV / AwTV kernels (eqs. 7-8) against oracle/tv.py.
Tolerances (none is stated by north_star for this row; derived from the arithmetic): fp32 terms with 2-ulp SFU
exp / rsqrt summed in fp64 -> value to 1e-6 relative; gradient (six O(1) terms per voxel) and the minimiser's
iterate to 1e-5 rel-L2."""
import numpy as np
import pytest

from oracle import tv as otv
from tests import helpers as H

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


SHAPES = [(53, 61, 70), (8, 8, 32), (1, 45, 37), (9, 1, 33), (17, 20, 1), (1, 1, 5), (3, 9, 100),   # (nz, ny, nx): ragged, 2-D, 1-D
          # nx % 4 == 0: the four-voxels-per-thread kernel; several x tiles (edge warp), ragged y tiles, three z chunks
          (70, 37, 264), (5, 23, 128), (130, 12, 132), (2, 2, 4)]


@pytest.mark.parametrize("delta", [None, 0.25, 0.02])
@pytest.mark.parametrize("shape", SHAPES)
def test_value_and_gradient_match_oracle(tg, shape, delta):
    x = (np.random.default_rng(hash(shape) % 1000).random(shape) * 0.3).astype(np.float32)
    d = np.inf if delta is None else delta
    v_ref = otv.awtv(x, d, eps=1e-8)
    g_ref = otv.awtv_gradient(x, d, eps=1e-8)
    assert tg.awtv(dev(x), delta, eps=1e-8) == pytest.approx(v_ref, rel=1e-6)
    g, v, n2 = tg.awtv_gradient(dev(x), delta, eps=1e-8, return_scalars=True)
    assert v == pytest.approx(v_ref, rel=1e-6)
    if np.linalg.norm(g_ref) > 0:
        assert H.rel_l2(host(g), g_ref) <= 1e-5
        assert n2 == pytest.approx(float(np.sum(g_ref ** 2)), rel=1e-5)
    else:
        assert np.all(host(g) == 0)


def test_piecewise_constant_phantom_and_eps_zero(tg):
    # flat regions (all differences zero) with eps = 0: T = 0 there, gradient terms must be 0, not NaN
    x = np.zeros((20, 24, 40), np.float32)
    x[5:15, 6:18, 10:30] = 1.0
    x[8:12, 10:14, 15:25] = 0.4
    for delta in (None, 0.5):
        d = np.inf if delta is None else delta
        g = host(tg.awtv_gradient(dev(x), delta, eps=0.0))
        assert np.all(np.isfinite(g))
        assert H.rel_l2(g, otv.awtv_gradient(x, d, eps=0.0)) <= 1e-5
        assert tg.awtv(dev(x), delta, eps=0.0) == pytest.approx(otv.awtv(x, d, 0.0), rel=1e-6)


@pytest.mark.parametrize("delta", [None, 0.1])
def test_minimiser_matches_oracle_and_descends(tg, delta):
    rng = np.random.default_rng(5)
    x = np.zeros((24, 30, 36), np.float32)
    x[6:18, 8:22, 9:27] = 0.5
    x += (0.02 * rng.standard_normal(x.shape)).astype(np.float32)          # a noisy block
    d = np.inf if delta is None else delta
    ref = otv.minimize_awtv(x, 15, 0.05, d, eps=1e-8)
    t = dev(x)
    tg.minimize_awtv(t, 15, 0.05, delta, eps=1e-8)
    assert H.rel_l2(host(t), ref) <= 1e-5
    assert tg.awtv(t, delta, 1e-8) < 0.9 * tg.awtv(dev(x), delta, 1e-8)


def test_full_size_properties_512(tg):
    # at C3's volume size: properties that hold at any size, and sampled voxels against the oracle on a sub-block
    g = torch.Generator(device="cuda").manual_seed(7)
    x = torch.rand((512, 512, 512), generator=g, device="cuda") * 0.3
    grad, v, n2 = tg.awtv_gradient(x, 0.2, eps=1e-8, return_scalars=True)
    assert abs(float(grad.double().sum())) <= 1e-6 * float(grad.double().abs().sum())     # translation invariance
    assert n2 == pytest.approx(float((grad.double() ** 2).sum()), rel=1e-9)
    # interior voxels of a sub-block depend only on the block plus one voxel around it
    blk = x[100:140, 200:240, 300:364].cpu().numpy()
    ref = otv.awtv_gradient(blk, 0.2, eps=1e-8)[1:-1, 1:-1, 1:-1]
    got = host(grad[101:139, 201:239, 301:363])
    assert H.rel_l2(got, ref) <= 1e-5


def test_vector_and_scalar_kernels_agree_at_full_size(tg):
    # the two gradient kernels (tigre_set_tv_path) form the same sums; compared on the whole 512^3 volume
    g = torch.Generator(device="cuda").manual_seed(11)
    x = torch.rand((512, 512, 512), generator=g, device="cuda") * 0.3
    try:
        for delta in (None, 0.2):
            tg.set_tv_path(0)
            g4, v4, n4 = tg.awtv_gradient(x, delta, eps=1e-8, return_scalars=True)
            tg.set_tv_path(1)
            g1, v1, n1 = tg.awtv_gradient(x, delta, eps=1e-8, return_scalars=True)
            assert float((g4 - g1).double().norm()) <= 1e-6 * float(g1.double().norm())
            assert v4 == pytest.approx(v1, rel=1e-6) and n4 == pytest.approx(n1, rel=1e-6)
    finally:
        tg.set_tv_path(0)


def test_argument_errors(tg):
    with pytest.raises(tg.TigreError) as e:
        tg.awtv(torch.zeros((4, 4, 4)), None)                 # host tensor
    assert e.value.code == -3
    with pytest.raises(tg.TigreError) as e:
        tg.awtv(torch.zeros((4, 4, 4), device="cuda"), None, eps=-1.0)
    assert e.value.code == -1
