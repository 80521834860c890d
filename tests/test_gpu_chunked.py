"""GPU parity of the host-chunking path: volume and projections in PINNED host
memory, z-slabs and view batches streamed through a deliberately tiny device budget so that several
slabs, several batches, ragged last chunks and partial detector-row bands all occur.  Compared with the
fp64 oracle at the same tolerances as the in-HBM path, and with the in-HBM result of the same library.
"""
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
    yield m
    m.set_chunk_budget(0)


def pinned(a):
    t = torch.empty(a.shape, dtype=torch.float32, pin_memory=True)
    t.copy_(torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)))
    return t


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


def cone_geometry():
    # wide cone (volume close to the source) so that z-slabs map to clearly different detector-row bands;
    # ragged sizes; detector offset so some rows see nothing
    return Geometry(nVoxel=(45, 38, 53), dVoxel=(1.0, 1.1, 0.9), nDetector=(72, 90), dDetector=(1.4, 1.2),
                    DSD=330.0, DSO=200.0, offDetector=(3.0, -6.0), offOrigin=(1.0, -2.0, 3.0))


@pytest.mark.parametrize("mode,tol", [("siddon", 1e-5), ("interp", 1e-4)])
@pytest.mark.parametrize("budget_kb", [200, 1500])
def test_chunked_ax_matches_oracle(tg, mode, tol, budget_kb):
    geo = cone_geometry()
    ang = circular_angles(11, start=0.1)
    vol = np.random.default_rng(21).random(geo.vol_shape, dtype=np.float32)
    ref = orc.ax(vol, geo, ang, orc.SIDDON if mode == "siddon" else orc.INTERP)
    # 200 kB: a slab is ~6 slices (45*38*4 B = 6.8 kB per slice) and a view batch 1-2 views (25 kB per view);
    # 1500 kB: all views resident, volume in a few slabs
    tg.set_chunk_budget(budget_kb * 1024)
    got = tg.Ax(pinned(vol), geo, ang, mode)
    assert not got.is_cuda and got.is_pinned()
    assert H.rel_l2(host(got), ref) <= tol
    tg.set_chunk_budget(0)
    inhbm = host(tg.Ax(torch.from_numpy(vol).cuda(), geo, ang, mode))
    assert H.rel_l2(host(got), inhbm) <= 2e-6


@pytest.mark.parametrize("mode,tol", [("matched", 1e-5), ("fdk", 1e-4)])
@pytest.mark.parametrize("budget_kb", [200, 1500])
def test_chunked_atb_matches_oracle(tg, mode, tol, budget_kb):
    geo = cone_geometry()
    ang = circular_angles(11, start=0.1)
    proj = np.random.default_rng(22).random((11, 90, 72), dtype=np.float32)
    ref = orc.atb(proj, geo, ang, orc.MATCHED if mode == "matched" else orc.FDK)
    tg.set_chunk_budget(budget_kb * 1024)
    got = tg.Atb(pinned(proj), geo, ang, mode)
    assert not got.is_cuda
    assert H.rel_l2(host(got), ref) <= tol
    tg.set_chunk_budget(0)
    inhbm = host(tg.Atb(torch.from_numpy(proj).cuda(), geo, ang, mode))
    assert H.rel_l2(host(got), inhbm) <= 2e-6


def test_chunked_general_geometry(tg):
    # tilted gantry and detector, per-view offsets: the row-band bound must still contain every contribution
    rng = np.random.default_rng(23)
    nA = 6
    geo = Geometry(nVoxel=(37, 29, 41), dVoxel=(1.0, 1.3, 0.8), nDetector=(45, 61), dDetector=(2.1, 1.6),
                   DSD=400.0, DSO=250.0, COR=0.7, offOrigin=(0.4, -0.6, 0.3), offDetector=(1.1, -0.9),
                   rotDetector=(0.05, -0.04, 0.08))
    ang = np.stack([rng.uniform(0, 2 * np.pi, nA), rng.uniform(-0.4, 0.4, nA), rng.uniform(-0.5, 0.5, nA)], 1)
    geo.rotDetector_a = np.asarray(geo.rotDetector) + 0.03 * rng.standard_normal((nA, 3))
    vol = rng.random(geo.vol_shape, dtype=np.float32)
    proj = rng.random((nA, 61, 45), dtype=np.float32)
    tg.set_chunk_budget(120 * 1024)
    try:
        assert H.rel_l2(host(tg.Ax(pinned(vol), geo, ang, "siddon")), orc.ax(vol, geo, ang, orc.SIDDON)) <= 1e-5
        assert H.rel_l2(host(tg.Ax(pinned(vol), geo, ang, "interp")), orc.ax(vol, geo, ang, orc.INTERP)) <= 1e-4
        assert H.rel_l2(host(tg.Atb(pinned(proj), geo, ang, "matched")), orc.atb(proj, geo, ang, orc.MATCHED)) <= 1e-5
    finally:
        tg.set_chunk_budget(0)


@pytest.mark.parametrize("ax_mode,atb_mode,tol", [("siddon", "matched", 1e-5), ("interp", "fdk", 1e-4)])
def test_chunked_sirt_driver_matches_oracle(tg, ax_mode, atb_mode, tol):
    # configs[4] in miniature: one and three SIRT iterations through tigre_sirt_chunked with every array in pinned host
    # memory and a budget that forces several slabs and batches in both passes, against the oracle's SIRT
    geo, ang, rec = make_config("C5", scale=96, n_angles=20)      # 32^3, 32x32 detector
    vol = phantom_for(rec, geo)
    om = dict(ax_mode=orc.SIDDON if ax_mode == "siddon" else orc.INTERP, atb_mode=orc.MATCHED if atb_mode == "matched" else orc.FDK)
    b = orc.ax(vol, geo, ang, om["ax_mode"]).astype(np.float32)
    x0 = (0.5 * vol).astype(np.float32)
    tg.set_chunk_budget(200 * 1024)
    try:
        for n_iter in (1, 3):
            xr, rr = orc.ossart(b, geo, ang, [np.arange(20)], n_iter, lam=1.0, x0=x0.astype(np.float64), **om)
            x, bb, r = pinned(x0), pinned(b), pinned(np.zeros_like(b))
            hist = tg.sirt_chunked(bb, geo, ang, x, n_iter, lam=1.0, ax_mode=ax_mode, atb_mode=atb_mode, r_scratch=r)
            assert H.rel_l2(host(x), xr) <= tol * (1 if n_iter == 1 else 3)
            assert np.allclose(hist, rr, rtol=1e-4)
            assert np.array_equal(bb.numpy(), b)                    # the data are untouched when a scratch array is given
        # in-place variant: b doubles as the residual scratch (one iteration only)
        x, bb = pinned(x0), pinned(b)
        tg.sirt_chunked(bb, geo, ang, x, 1, ax_mode=ax_mode, atb_mode=atb_mode)
        xr, _ = orc.ossart(b, geo, ang, [np.arange(20)], 1, lam=1.0, x0=x0.astype(np.float64), **om)
        assert H.rel_l2(host(x), xr) <= tol
        with pytest.raises(tg.TigreError):
            tg.sirt_chunked(bb, geo, ang, x, 2)                     # in place needs n_iter == 1
        # and the same step with everything resident on the device
        tg.set_chunk_budget(0)
        plan = tg.OssartPlan(geo, ang, [np.arange(20)], ax_mode, atb_mode)
        xd = torch.from_numpy(x0).cuda()
        plan.iterate(torch.from_numpy(b).cuda(), xd, 1)
        plan.close()
        assert H.rel_l2(host(x), host(xd)) <= 3e-6
    finally:
        tg.set_chunk_budget(0)


def test_chunked_budget_too_small_and_mixed_memory(tg):
    geo = cone_geometry()
    ang = circular_angles(3)
    vol = pinned(np.zeros(geo.vol_shape, np.float32))
    tg.set_chunk_budget(1024)
    try:
        with pytest.raises(tg.TigreError) as e:
            tg.Ax(vol, geo, ang, "siddon")
        assert e.value.code == -4
    finally:
        tg.set_chunk_budget(0)
    with pytest.raises(tg.TigreError) as e:               # pinned in, device out: not a supported mix
        tg.Ax(vol, geo, ang, "siddon", out=torch.empty((3, 90, 72), device="cuda"))
    assert e.value.code == -3
