"""GPU parity on the degenerate cases of the projector pair (rays that miss return 0; zero border
of both interpolants; §8(b): error behaviour), element by element against the fp64 oracle through the C ABI.

  * no views at all                           -> TIGRE_ERR_ARG, nothing launched
  * a volume of ONE voxel, ONE view           -> the chord of that box (Siddon) / the tent samples (interpolated)
  * a detector of ONE pixel                   -> one ray; A^T b is the tent footprint of that pixel
  * every ray misses the volume               -> Ax identically 0 (bit-exact), A^T b identically 0
  * an all-zero input                         -> an all-zero output (bit-exact; no NaN from 0 * weight)
  * sizes of 1 along single axes, odd sizes   -> ragged tiles in every direction, rows not 16-byte aligned
"""
import numpy as np
import pytest

from oracle import oracle as orc
from tests import helpers as H
from workloads import Geometry, circular_angles

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

AX = [("siddon", orc.SIDDON, 1e-5), ("interp", orc.INTERP, 1e-4)]
ATB = [("matched", orc.MATCHED, 1e-5), ("fdk", orc.FDK, 1e-4)]


@pytest.fixture(scope="module")
def tg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2412_10129_b200 as m
    m.version()          # fails loudly if the .so is missing
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


def _check_pair(tg, geo, ang, seed):
    rng = np.random.default_rng(seed)
    vol = rng.uniform(0.0, 1.0, geo.vol_shape).astype(np.float32)
    proj = rng.uniform(0.0, 1.0, (len(ang),) + tuple(geo.proj_shape[-2:])).astype(np.float32)
    for name, mode, tol in AX:
        ref = orc.ax(vol, geo, ang, mode)
        got = host(tg.Ax(dev(vol), geo, ang, name))
        assert got.shape == ref.shape
        assert np.isfinite(got).all()
        assert H.rel_l2(got, ref) <= tol, (name, H.rel_l2(got, ref))
        if name == "siddon":
            assert np.array_equal(got == 0, ref == 0)
    for name, mode, tol in ATB:
        ref = orc.atb(proj, geo, ang, mode)
        got = host(tg.Atb(dev(proj), geo, ang, name))
        assert got.shape == ref.shape
        assert np.isfinite(got).all()
        assert H.rel_l2(got, ref) <= tol, (name, H.rel_l2(got, ref))


def test_no_views_is_an_argument_error(tg):
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0, 1.0, 1.0), nDetector=(12, 12), dDetector=(1.6, 1.6), DSD=600.0, DSO=400.0)
    ang = np.zeros((0, 3))
    with pytest.raises(tg.TigreError) as e:
        tg.Ax(torch.zeros(geo.vol_shape, device="cuda"), geo, ang)
    assert e.value.code == -1
    with pytest.raises(tg.TigreError) as e:
        tg.Atb(torch.zeros((0, 12, 12), device="cuda"), geo, ang)
    assert e.value.code == -1


def test_single_voxel_single_view(tg):
    geo = Geometry(nVoxel=(1, 1, 1), dVoxel=(2.0, 3.0, 1.5), nDetector=(9, 7), dDetector=(0.9, 1.1), DSD=300.0, DSO=200.0)
    _check_pair(tg, geo, circular_angles(1, start=0.3), seed=1)


def test_single_pixel_detector(tg):
    geo = Geometry(nVoxel=(11, 9, 7), dVoxel=(1.0, 1.0, 1.0), nDetector=(1, 1), dDetector=(2.0, 2.0), DSD=300.0, DSO=200.0,
                   offDetector=(1.3, -0.7))
    _check_pair(tg, geo, circular_angles(3, start=0.1), seed=2)


@pytest.mark.parametrize("n,det", [((1, 13, 5), (17, 6)), ((13, 1, 5), (18, 7)), ((13, 5, 1), (19, 3)), ((33, 17, 19), (1, 23)),
                                    ((33, 17, 19), (23, 1))])
def test_unit_extent_along_one_axis(tg, n, det):
    geo = Geometry(nVoxel=n, dVoxel=(1.0, 1.2, 0.9), nDetector=det, dDetector=(1.7, 1.9), DSD=420.0, DSO=260.0,
                   rotDetector=(0.03, -0.02, 0.04), COR=0.4)
    ang = np.stack([np.array([0.2, 1.9, 4.4]), np.array([0.1, -0.2, 0.3]), np.array([0.0, 0.3, -0.1])], 1)
    _check_pair(tg, geo, ang, seed=3)


def test_every_ray_misses_the_volume(tg):
    # the detector is shifted by 40 of its own widths: no ray meets the volume, no voxel projects onto it
    geo = Geometry(nVoxel=(16, 16, 16), dVoxel=(1.0, 1.0, 1.0), nDetector=(20, 12), dDetector=(1.5, 1.5), DSD=600.0, DSO=400.0,
                   offDetector=(1200.0, 0.0))
    ang = circular_angles(4)
    rng = np.random.default_rng(4)
    vol = rng.uniform(0.5, 1.0, geo.vol_shape).astype(np.float32)
    proj = rng.uniform(0.5, 1.0, (4, 12, 20)).astype(np.float32)
    for name, mode, _ in AX:
        assert not orc.ax(vol, geo, ang, mode).any()
        assert not host(tg.Ax(dev(vol), geo, ang, name)).any()
    for name, mode, _ in ATB:
        assert not orc.atb(proj, geo, ang, mode).any()
        assert not host(tg.Atb(dev(proj), geo, ang, name)).any()


def test_zero_in_zero_out(tg):
    geo = Geometry(nVoxel=(21, 18, 10), dVoxel=(1.0, 1.0, 1.0), nDetector=(28, 16), dDetector=(1.5, 1.5), DSD=600.0, DSO=400.0)
    ang = circular_angles(5, start=0.2)
    for name, _, _ in AX:
        assert not host(tg.Ax(torch.zeros(geo.vol_shape, device="cuda"), geo, ang, name)).any()
    for name, _, _ in ATB:
        assert not host(tg.Atb(torch.zeros((5, 16, 28), device="cuda"), geo, ang, name)).any()
