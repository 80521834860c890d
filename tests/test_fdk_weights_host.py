"""Host logic of the FDK variants (no GPU): tigre_fdk_weights (Parker / Wang tables, built in fp64 on the host by the
library) against oracle/fdk_ext.py (readings P27, P28), and its argument errors."""
import numpy as np
import pytest

import paper_2412_10129_b200 as tg
from oracle import fdk_ext as fx
from workloads.geometry import Geometry


def short_scan(direction, nA=50, nu=40, off=0.0):
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(nu, 4), dDetector=(1.7, 1.0), DSD=900.0, DSO=600.0,
                   offDetector=(off, 0.0))
    Gamma = np.arctan((0.5 * nu * 1.7 + abs(off)) / 900.0)
    th = direction * np.linspace(0.0, np.pi + 2 * (Gamma + 0.07), nA) - 0.8
    return geo, np.stack([th, np.zeros(nA), np.zeros(nA)], 1)


@pytest.mark.parametrize("direction", [1.0, -1.0])
@pytest.mark.parametrize("off", [0.0, 3.5])
def test_parker_table_matches_oracle(direction, off):
    geo, ang = short_scan(direction, off=off)
    w = tg.fdk_weights(geo, ang, "parker")
    ref = fx.parker_weights(geo, ang)
    assert w.shape == ref.shape
    assert np.allclose(w, ref, rtol=0, atol=1e-13)


@pytest.mark.parametrize("off", [11.0, -7.25])
def test_wang_table_matches_oracle(off):
    geo = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(64, 4), dDetector=(1.5, 1.0), DSD=1200.0, DSO=800.0,
                   offDetector=(off, 0.0))
    ang = np.stack([np.linspace(0, 2 * np.pi, 12, endpoint=False), np.zeros(12), np.zeros(12)], 1)
    assert np.allclose(tg.fdk_weights(geo, ang, "wang"), fx.wang_weights(geo, 12), rtol=0, atol=1e-13)
    assert np.all(tg.fdk_weights(geo, ang, None) == 1.0)


def test_weighting_errors():
    geo, ang = short_scan(1.0)
    bad = ang.copy()
    bad[[3, 4]] = bad[[4, 3]]                                        # not monotone
    with pytest.raises(tg.TigreError) as e:
        tg.fdk_weights(geo, bad, "parker")
    assert e.value.code == -1
    full = np.stack([np.linspace(0, 2 * np.pi, 20), np.zeros(20), np.zeros(20)], 1)   # Theta = 2 pi: not a short scan
    with pytest.raises(tg.TigreError):
        tg.fdk_weights(geo, full, "parker")
    wide = Geometry(nVoxel=(8, 8, 8), dVoxel=(1.0,) * 3, nDetector=(16, 4), dDetector=(1.0, 1.0), DSD=900.0, DSO=600.0,
                    offDetector=(9.0, 0.0))                          # displaced by more than half the detector: no overlap
    with pytest.raises(tg.TigreError):
        tg.fdk_weights(wide, full, "wang")


def test_oracle_ossart_row_scale_pins():
    # the redundancy weighting of the iterative methods (reading P17) enters oracle.ossart as a scale of the row weights:
    # ones change nothing (bitwise); a constant c scales the first SIRT step by c (the update is linear in W); a scale
    # that zeroes some columns equals running on data whose residual is zeroed there
    from oracle import oracle as orc
    from workloads import make_config, phantom_for
    geo, ang, rec = make_config("C3", scale=32, n_angles=8)           # 16^3, 32x24 detector displaced by +20 mm
    vol = phantom_for(rec, geo).astype(np.float64)
    b = orc.ax(vol, geo, ang, orc.SIDDON)
    subsets = [list(range(0, 8, 2)), list(range(1, 8, 2))]
    nu = geo.nDetector[0]
    x_plain, _ = orc.ossart(b, geo, ang, subsets, 2)
    x_ones, _ = orc.ossart(b, geo, ang, subsets, 2, row_scale=np.ones((8, nu)))
    assert np.array_equal(x_plain, x_ones)
    x1, _ = orc.ossart(b, geo, ang, [list(range(8))], 1, nonneg=False)
    xc, _ = orc.ossart(b, geo, ang, [list(range(8))], 1, nonneg=False, row_scale=np.full((8, nu), 0.25))
    assert np.allclose(xc, 0.25 * x1, rtol=1e-13, atol=0)
    mask = np.ones((8, nu))
    mask[:, : nu // 3] = 0.0
    xm, _ = orc.ossart(b, geo, ang, [list(range(8))], 1, nonneg=False, row_scale=mask)
    W = orc.row_weights(geo, ang, orc.SIDDON) * mask[:, None, :]
    ref = orc.col_weights(geo, ang, orc.MATCHED) * orc.atb(W * b, geo, ang, orc.MATCHED)
    assert np.allclose(xm, ref, rtol=1e-13, atol=1e-18)
