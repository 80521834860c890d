"""tigre_band_z_range (host only): the z-slices that rays of a band of detector rows can meet.  tigre_plan_ossart's
end-to-end path sends the iterate up in that order and starts each band of the first projection when its slices have arrived, so a
slice the bound leaves out would be read before it is there.  Checked against the oracle's first / last voxel per ray (reading
P19(a); the voxels of a ray between those two lie between them in z): every ray of every band, on C3's half-fan geometry, tilted and
offset detectors, an anisotropic volume, and views from every side; and the bound must be worth having where rows map to z."""
import numpy as np
import pytest

from oracle import oracle as orc
from workloads import Geometry, circular_angles, make_config

tg = pytest.importorskip("paper_2412_10129_b200")


def _lib_or_skip():
    try:
        tg.version()
    except Exception as e:   # no built library on this machine
        pytest.skip(str(e))


def _check(geo, ang, nbands=4, align=4):
    nu, nv = geo.nDetector
    nx, ny, _ = geo.nVoxel
    rows = -(-(-(-nv // nbands)) // align) * align
    ids = np.arange(len(ang) * nu * nv, dtype=np.int64)
    r = orc.siddon_index(geo, ang, ids)
    hit = r["nseg"] > 0
    zf, zl = r["first"] // (nx * ny), r["last"] // (nx * ny)
    row = (ids // nu) % nv
    spans = []
    for b in range(nbands):
        r0, r1 = min(b * rows, nv), min((b + 1) * rows, nv)
        if r1 <= r0:
            continue
        got = tg.band_z_range(geo, ang, r0, r1)
        assert got is not None
        zlo, zhi = got
        m = hit & (row >= r0) & (row < r1)
        if m.any():
            lo, hi = min(zf[m].min(), zl[m].min()), max(zf[m].max(), zl[m].max())
            assert zlo <= lo and hi <= zhi, (b, zlo, zhi, lo, hi)
        spans.append(max(0, zhi - zlo + 1))
    return spans


def test_band_z_range_contains_every_voxel_the_oracle_meets():
    _lib_or_skip()
    geo, ang, _ = make_config("C3", scale=8, n_angles=12)                  # 64^3, 128 x 96, offDetector 20 mm
    spans = _check(geo, ang)
    assert max(spans) <= 0.45 * geo.nVoxel[2]                               # a quarter of the rows needs well under half of the slices
    rng = np.random.default_rng(5)
    g2 = Geometry(nVoxel=(40, 56, 48), dVoxel=(1.0, 0.8, 1.3), nDetector=(72, 64), dDetector=(1.6, 1.9), DSD=700.0, DSO=450.0,
                  COR=0.6, offOrigin=(2.0, -1.5, 3.0), offDetector=(4.0, -6.0), rotDetector=(0.2, -0.05, 0.1))
    a2 = np.stack([rng.uniform(0, 2 * np.pi, 9), rng.uniform(-0.3, 0.3, 9), rng.uniform(-0.3, 0.3, 9)], 1)
    g2.rotDetector_a = np.asarray(g2.rotDetector) + 0.05 * rng.standard_normal((9, 3))
    _check(g2, a2)
    g3 = Geometry(nVoxel=(32, 32, 80), dVoxel=(1.0, 1.0, 0.5), nDetector=(48, 120), dDetector=(1.5, 0.7), DSD=500.0, DSO=300.0,
                  rotDetector=(1.2, 0.0, 0.0))                                # detector rolled by 69 degrees: rows no longer map to z
    _check(g3, circular_angles(7, start=0.3))


def test_band_z_range_declines_where_it_has_no_bound():
    _lib_or_skip()
    geo, ang, _ = make_config("C3", scale=8, n_angles=6)
    par = geo.copy(mode="parallel")
    assert tg.band_z_range(par, ang, 0, 24) is None
    near = Geometry(nVoxel=(64, 64, 32), dVoxel=(1.0, 1.0, 1.0), nDetector=(64, 32), dDetector=(1.0, 1.0), DSD=60.0, DSO=20.0)
    assert tg.band_z_range(near, circular_angles(4), 0, 8) is None          # source over the volume's footprint
    with pytest.raises(tg.TigreError):
        tg.band_z_range(geo, ang, 10, 10)
