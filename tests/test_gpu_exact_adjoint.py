"""GPU parity of the exact-adjoint backprojectors: tigre_Atb modes EXACT_SIDDON /
EXACT_INTERP are the transposes of tigre_Ax in those modes (ray-driven scatter of the same weights).
Checked against the oracle's scatter transposes (themselves pinned to 1e-12 by <Ax,y> = <x,A^T y> in fp64,
tests/test_oracle_pins.py), by the adjoint identity of the GPU pair itself, and through CGLS."""
import numpy as np
import pytest

from oracle import oracle as orc
from tests import helpers as H
from workloads import Geometry, circular_angles, make_config, phantom_for

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


def general_geometry(nA=5, seed=41):
    rng = np.random.default_rng(seed)
    geo = Geometry(nVoxel=(37, 29, 23), dVoxel=(1.0, 1.3, 0.8), nDetector=(45, 31), dDetector=(2.1, 2.6),
                   DSD=400.0, DSO=250.0, COR=0.7, offOrigin=(0.4, -0.6, 0.3), offDetector=(1.1, -0.9),
                   rotDetector=(0.05, -0.04, 0.08))
    angles = np.stack([rng.uniform(0, 2 * np.pi, nA), rng.uniform(-0.4, 0.4, nA), rng.uniform(-0.5, 0.5, nA)], 1)
    geo.rotDetector_a = np.asarray(geo.rotDetector) + 0.03 * rng.standard_normal((nA, 3))
    return geo, angles


CASES = [("exact_siddon", "siddon", orc.SIDDON, 1e-5), ("exact_interp", "interp", orc.INTERP, 1e-4)]


@pytest.mark.parametrize("mode,ax_mode,omode,tol", CASES)
def test_exact_adjoint_matches_oracle_scatter(tg, mode, ax_mode, omode, tol):
    for geo, ang in (general_geometry(),
                     (Geometry(nVoxel=(70, 61, 53), dVoxel=(1.0, 1.0, 1.0), nDetector=(101, 67), dDetector=(1.5, 1.5),
                               DSD=600.0, DSO=380.0), circular_angles(16, start=0.05))):   # all octants, x- and y-dominant
        y = np.random.default_rng(42).random((len(ang),) + geo.proj_shape, dtype=np.float32)
        ref = orc.atb_exact(y, geo, ang, omode)
        got = host(tg.Atb(dev(y), geo, ang, mode))
        assert H.rel_l2(got, ref) <= tol
        assert np.array_equal(got == 0, ref == 0)           # the same voxels are never met


@pytest.mark.parametrize("mode,ax_mode,omode,tol", CASES)
def test_adjoint_identity_of_the_gpu_pair(tg, mode, ax_mode, omode, tol):
    # <A x, y> = <x, A^T y> for the GPU's own pair, up to fp32 rounding (the voxel-driven pair misses it by ~1e-2)
    geo, ang, rec = make_config("C1")
    rng = np.random.default_rng(43)
    x = rng.random(geo.vol_shape, dtype=np.float32)
    y = rng.random((len(ang),) + geo.proj_shape, dtype=np.float32)
    lhs = float(np.sum(host(tg.Ax(dev(x), geo, ang, ax_mode)) * y))
    rhs = float(np.sum(x.astype(np.float64) * host(tg.Atb(dev(y), geo, ang, mode))))
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs)
    gap_voxel_driven = abs(lhs - float(np.sum(x.astype(np.float64) * host(tg.Atb(dev(y), geo, ang, "matched"))))) / abs(lhs)
    assert gap_voxel_driven > 10 * max(abs(lhs - rhs) / abs(lhs), 1e-7)   # what the exact modes are for


def test_adjoint_identity_full_size_c3_subset(tg):
    # a property that holds at any size: one ordered subset of C3 (36 views of 1024x768 through 512^3)
    geo, ang, _ = make_config("C3")
    ang = ang[3::20]
    g = torch.Generator(device="cuda").manual_seed(44)
    x = torch.rand(geo.vol_shape, generator=g, device="cuda")
    y = torch.rand((len(ang),) + geo.proj_shape, generator=g, device="cuda")
    lhs = float((tg.Ax(x, geo, ang, "siddon").double() * y.double()).sum())
    rhs = float((x.double() * tg.Atb(y, geo, ang, "exact_siddon").double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs)


def test_cgls_with_exact_adjoint(tg):
    geo, ang, rec = make_config("C1", scale=2, n_angles=24)      # 32^3, 48x48
    vol = phantom_for(rec, geo)
    b = orc.ax(vol, geo, ang, orc.SIDDON).astype(np.float32)
    xr, rr = orc.cgls(b, geo, ang, 6, orc.SIDDON, exact_adjoint=True)
    xg, rg = tg.cgls(dev(b), geo, ang, 6, "siddon", "exact_siddon")
    assert H.rel_l2(host(xg), xr) <= 1e-3
    assert np.allclose(rg, rr, rtol=1e-3)
    assert np.all(np.diff(rg) < 0)                            # with a true adjoint CGLS residuals decrease
    with pytest.raises(tg.TigreError) as e:                   # the transpose must be that of the Ax in use
        tg.cgls(dev(b), geo, ang, 1, "siddon", "exact_interp")
    assert e.value.code == -1


def test_exact_siddon_scatter_across_the_dominance_boundary(tg):
    """Lanes of one warp on both sides of |dx| = |dy| scatter into different arrays (the volume and its (x,y)-transposed
    copy), where EQUAL offsets are different voxels (on the diagonal x = y they coincide numerically): the pairwise merge
    of the scatter must not join such lanes.  Views at and around 45 degrees, the boundary moved pixel by pixel over the
    detector row so that it falls inside an (even, odd) lane pair as well as between pairs."""
    for offu in (0.0, 1.0, 2.0, 0.5):
        geo = Geometry(nVoxel=(64, 64, 40), dVoxel=(1.0, 1.0, 1.0), nDetector=(96, 48), dDetector=(1.0, 1.0),
                       DSD=500.0, DSO=300.0, offDetector=(offu, 0.0))
        ang = np.zeros((5, 3))
        ang[:, 0] = [np.pi / 4, np.pi / 4 + 1e-3, 3 * np.pi / 4 - 2e-3, 5 * np.pi / 4, 7 * np.pi / 4 + 5e-4]
        y = np.random.default_rng(7).random((len(ang),) + geo.proj_shape, dtype=np.float32)
        ref = orc.atb_exact(y, geo, ang, orc.SIDDON)
        got = host(tg.Atb(dev(y), geo, ang, "exact_siddon"))
        assert H.rel_l2(got, ref) <= 1e-5
        assert np.abs(got - ref).max() <= 1e-4 * np.abs(ref).max()
