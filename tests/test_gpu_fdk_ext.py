"""GPU parity of the FDK variants (tigre_fdk_filter_ex, tigre_fdk_ex; PAPER.md:114, 281, 359;
readings P26-P28) against oracle/fdk_ext.py.  Tolerance: north_star's 1e-4 rel-L2 for the FDK-weighted path (the filter
is an fp32 convolution of nu terms with fp64-built taps)."""
import numpy as np
import pytest

from oracle import fdk_ext as fx
from oracle import oracle as orc
from tests import helpers as H
from workloads import make_config, phantom_for
from workloads.geometry import Geometry

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


@pytest.mark.parametrize("filt", fx.FILTERS)
def test_filters_match_oracle(tg, filt):
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(83, 7), dDetector=(1.3, 1.1), DSD=700.0, DSO=450.0)
    geo.DSD_a = np.array([700.0, 650.0, 720.0])                       # per-view distances: tau differs per view
    ang = np.stack([np.array([0.1, 1.0, 2.5]), np.zeros(3), np.zeros(3)], 1)
    p = np.random.default_rng(1).random((3, 7, 83)).astype(np.float32)
    q = tg.fdk_filter_ex(dev(p), geo, ang, filt)
    assert H.rel_l2(host(q), fx.fdk_filter(p, geo, ang, filt)) <= 1e-5


def short_scan_case():
    geo, _, rec = make_config("C2", scale=8, n_angles=4)               # 32^3, 64x64 detector
    Gamma = np.arctan(0.5 * geo.nDetector[0] * geo.dDetector[0] / geo.DSD)
    nA = 50
    th = np.linspace(0.0, np.pi + 2 * (Gamma + 0.06), nA) + 0.25
    ang = np.stack([th, np.zeros(nA), np.zeros(nA)], 1)
    vol = phantom_for(rec, geo).astype(np.float64)
    return geo, ang, vol


@pytest.mark.parametrize("filt", ["ram_lak", "shepp_logan", "hamming"])
def test_short_scan_parker_fdk_matches_oracle(tg, filt):
    geo, ang, vol = short_scan_case()
    b = orc.ax(vol, geo, ang, orc.INTERP).astype(np.float32)
    ref = fx.fdk(b, geo, ang, filt, "parker")
    x = tg.fdk_ex(dev(b), geo, ang, filt, "parker")
    assert H.rel_l2(host(x), ref) <= 1e-4
    q = tg.fdk_filter_ex(dev(b), geo, ang, filt, "parker")
    assert H.rel_l2(host(q), fx.fdk_filter(b, geo, ang, filt, fx.parker_weights(geo, ang))) <= 1e-5
    # the reconstruction is a reconstruction: close to the phantom in the mid-plane region
    mid = slice(geo.nVoxel[2] // 2 - 2, geo.nVoxel[2] // 2 + 2)
    assert H.rel_l2(host(x)[mid], vol[mid]) < 0.5


def test_displaced_detector_wang_fdk_matches_oracle(tg):
    geo, ang, rec = make_config("C3", scale=16)                         # 32^3, 64x48 detector displaced by +20 mm, 45 views
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON).astype(np.float32)
    for filt in ("ram_lak", "hann"):
        ref = fx.fdk(b, geo, ang, filt, "wang")
        x = tg.fdk_ex(dev(b), geo, ang, filt, "wang")
        assert H.rel_l2(host(x), ref) <= 1e-4
    plain = tg.fdk_ex(dev(b), geo, ang, "ram_lak", None)
    assert torch.equal(plain, tg.fdk(dev(b), geo, ang))                # FULL + RAM_LAK is tigre_fdk


def test_full_size_c2_filter_sampled_rows(tg):
    # C2's detector (512 columns), 6 of its views, every filter: sampled rows against the oracle
    geo, ang, rec = make_config("C2")
    ang = ang[::60]
    gen = torch.Generator(device="cuda").manual_seed(4)
    b = torch.rand((len(ang), geo.nDetector[1], geo.nDetector[0]), generator=gen, device="cuda")
    bh = b.cpu().numpy()
    rows = [0, 17, 255, 256, 511]
    for filt in ("shepp_logan", "cosine", "hann"):
        q = host(tg.fdk_filter_ex(b, geo, ang, filt))
        # the cosine weight depends on v: filter the sampled rows one by one with a one-row detector placed at that v
        for r in rows:
            one = Geometry(nVoxel=geo.nVoxel, dVoxel=geo.dVoxel, nDetector=(geo.nDetector[0], 1), dDetector=geo.dDetector,
                           DSD=geo.DSD, DSO=geo.DSO)
            v = (r + 0.5) * geo.dDetector[1] - 0.5 * geo.nDetector[1] * geo.dDetector[1]
            u = (np.arange(geo.nDetector[0]) + 0.5) * geo.dDetector[0] - 0.5 * geo.nDetector[0] * geo.dDetector[0]
            # a one-row detector sits at v = 0: fold the row's cosine weight in by hand (ratio of the two weights)
            ratio = np.sqrt(geo.DSD ** 2 + u ** 2) / np.sqrt(geo.DSD ** 2 + u ** 2 + v ** 2)
            ref = fx.fdk_filter(bh[:, r:r + 1, :] * ratio[None, None, :], one, ang, filt)[:, 0, :]
            assert H.rel_l2(q[:, r, :], ref) <= 1e-5


def test_argument_errors(tg):
    geo, ang, vol = short_scan_case()
    b = torch.zeros((len(ang), geo.nDetector[1], geo.nDetector[0]), device="cuda")
    with pytest.raises(tg.TigreError) as e:
        tg.fdk_ex(b, geo, ang[::-1][[0, 2, 1] + list(range(3, len(ang)))], "ram_lak", "parker")   # not monotone
    assert e.value.code == -1
    with pytest.raises(KeyError):
        tg.fdk_ex(b, geo, ang, "butterworth", None)                   # unknown filter name: refused by the binding
    with pytest.raises(tg.TigreError) as e:
        tg.fdk_ex(b.cpu(), geo, ang, "hann", None)
    assert e.value.code == -3


def test_redundancy_weighting_inside_ossart_matches_oracle(tg):
    # the displaced-detector weights inside the iteration (plan created with redundancy on; reading P17)
    geo, ang, rec = make_config("C3", scale=16, n_angles=40)           # 32^3, 64x48 detector displaced by +20 mm (the case of test_ossart_scaled_c3)
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON).astype(np.float32)
    nA = len(ang)
    subsets = [list(range(s, nA, 5)) for s in range(5)]
    w = fx.wang_weights(geo, nA)
    ref, rres = orc.ossart(b, geo, ang, subsets, 3, row_scale=w)
    plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched", redundancy=True)
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    res = plan.iterate(dev(b), x, 3)
    plan.close()
    assert H.rel_l2(host(x), ref) <= 1e-4
    assert np.allclose(res, rres, rtol=1e-4)
    plain, _ = orc.ossart(b, geo, ang, subsets, 3)
    assert H.rel_l2(host(x), plain) > 1e-3                             # and it is not the unweighted iteration


def test_curved_detector_flattening_matches_oracle(tg):
    from oracle import curved as ocurved
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(157, 93), dDetector=(1.3, 1.7), DSD=420.0, DSO=300.0)
    geo.DSD_a = np.array([420.0, 380.0, 505.0])
    ang = np.stack([np.array([0.0, 1.0, 2.0]), np.zeros(3), np.zeros(3)], 1)
    img = np.random.default_rng(5).random((3, 93, 157)).astype(np.float32)
    ref = ocurved.flatten(img, geo)
    got = host(tg.flatten_detector(dev(img), geo, ang))
    # fp32 coordinates: a tap index can differ where the continuous index sits on an integer; compare in rel-L2
    assert H.rel_l2(got, ref) <= 1e-4
    # C4's detector size, one view: sampled pixels
    big = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(1536, 1536), dDetector=(0.2, 0.2), DSD=1536.0, DSO=1000.0)
    gen = torch.Generator(device="cuda").manual_seed(6)
    b = torch.rand((2, 1536, 1536), generator=gen, device="cuda")
    refb = ocurved.flatten(b.cpu().numpy(), big)
    assert H.rel_l2(host(tg.flatten_detector(b, big, ang[:2])), refb) <= 1e-4


# ------------------------------------------------------------------ the tensor-core pre-filter (fdk_tc.cu) against the CUDA-core one
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("nu,nv,nA", [(96, 9, 5), (332, 37, 7), (1024, 6, 3)])
def test_fdk_filter_kernel_paths_match_oracle(tg, path, nu, nv, nA):
    """tigre_set_fdk_path: 0 = Toeplitz GEMM on tcgen05 (3 x tf32 split products, fp32 accumulator in tensor memory), 1 = CUDA-core
    convolution.  Widths below one N tile (96), ragged in every tile dimension (332 = 256 + 76 columns, 7 x 37 = 259 rows = 2 row
    tiles + 3), C3's width (1024: 4 passes x 32 K blocks), displaced detector + per-view distances, every filter, Wang and
    Parker column weights: both kernels within 1e-5 of the oracle's fp64 filter."""
    rng = np.random.default_rng(nu)
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(nu, nv), dDetector=(0.4 * 1024 / nu, 1.1), DSD=700.0, DSO=450.0,
                   offDetector=(0.11 * nu * 0.4 * 1024 / nu, -1.7))
    geo.DSD_a = 700.0 + rng.uniform(-40, 40, nA)
    ang = np.stack([np.linspace(0.1, 2 * np.pi, nA, endpoint=False), np.zeros(nA), np.zeros(nA)], 1)
    p = rng.random((nA, nv, nu)).astype(np.float32)
    tg.set_fdk_path(path)
    try:
        for filt in ("ram_lak", "hann", "shepp_logan"):
            assert H.rel_l2(host(tg.fdk_filter_ex(dev(p), geo, ang, filt)), fx.fdk_filter(p, geo, ang, filt)) <= 1e-5, filt
        assert H.rel_l2(host(tg.fdk_filter(dev(p), geo, ang)), orc.fdk_filter(p, geo, ang)) <= 1e-5
        w = 2.0 * fx.wang_weights(geo, nA)
        assert H.rel_l2(host(tg.fdk_filter_ex(dev(p), geo, ang, "hamming", "wang")), fx.fdk_filter(p, geo, ang, "hamming", w)) <= 1e-5
        # smooth data: the ramp filter cancels two to three digits of the sum, so the fp32 rounding of the taps and of the
        # accumulation (6e-8 of the terms) shows as up to 1e-4 of the RESULT in either kernel: north_star's FDK tolerance
        u = np.linspace(-1, 1, nu)[None, None, :]
        smooth = (np.sqrt(np.maximum(1.0 - u * u, 0.0)) * (1.0 + 0.1 * rng.random((nA, nv, 1)))).astype(np.float32)
        ref = orc.fdk_filter(smooth, geo, ang)
        got = host(tg.fdk_filter(dev(smooth), geo, ang))
        assert np.linalg.norm(ref) < 0.2 * np.linalg.norm(smooth) / (4 * (geo.dDetector[0] * 450 / 700) ** 1)    # cancellation is real
        assert H.rel_l2(got, ref) <= 2e-4
    finally:
        tg.set_fdk_path(0)
