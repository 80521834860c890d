"""GPU side of the multi-GPU sharding: the slab entry points tigre_Ax_slab / tigre_Atb_slab
that every rank would call, exercised on ONE device (this box has one): the partial projections of a z-partition add up
to tigre_Ax of the whole volume and to the oracle, slabs of A^T b concatenate to tigre_Atb, rows outside a slab's band are
zero, and ZSlabShards with world = 1 is the plain pair.  (The exchange step itself runs under gloo in
tests/test_sharded_host.py; ranks whose kernels wait on one another are not emulated on one GPU.)"""
import numpy as np
import pytest

from oracle import oracle as orc
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


@pytest.mark.parametrize("cfg,axm,atm,world", [("C1", "siddon", "matched", 3), ("C2", "interp", "fdk", 2), ("C3", "siddon", "matched", 4)])
def test_slab_partition_reproduces_the_whole(tg, cfg, axm, atm, world):
    from paper_2412_10129_b200.sharded import ZSlabShards
    scale = {"C1": 2, "C2": 8, "C3": 16}[cfg]
    geo, ang, rec = make_config(cfg, scale=scale, n_angles=12)
    vol = phantom_for(rec, geo).astype(np.float32) + 0.001
    oax = orc.SIDDON if axm == "siddon" else orc.INTERP
    oat = orc.MATCHED if atm == "matched" else orc.FDK
    ref_p = orc.ax(vol, geo, ang, oax)
    whole = tg.Ax(dev(vol), geo, ang, axm)
    total = torch.zeros_like(whole)
    back = []
    b = dev(ref_p)
    for r in range(world):
        sh = ZSlabShards(geo, ang, r, world)
        part = tg.Ax_slab(dev(vol[sh.z0:sh.z1]), geo, ang, sh.z0, axm)
        lo, hi = sh.band
        assert float(part[:, :lo].abs().sum()) == 0.0 and float(part[:, hi:].abs().sum()) == 0.0
        total += part
        back.append(sh.Atb(b, atm))
    tol = 1e-5 if axm == "siddon" else 1e-4
    assert H.rel_l2(host(total), ref_p) <= tol
    assert H.rel_l2(host(total), host(whole)) <= 1e-6
    cat = torch.cat(back, 0)
    assert H.rel_l2(host(cat), orc.atb(ref_p, geo, ang, oat)) <= tol
    assert H.rel_l2(host(cat), host(tg.Atb(b, geo, ang, atm))) <= 1e-6


def test_world_one_is_the_plain_pair_and_full_size_bands(tg):
    from paper_2412_10129_b200.sharded import ZSlabShards
    geo, ang, rec = make_config("C1", scale=2)
    vol = dev(phantom_for(rec, geo))
    sh = ZSlabShards(geo, ang, 0, 1)
    p = sh.Ax(vol, "siddon")
    assert torch.equal(p, tg.Ax(vol, geo, ang, "siddon"))
    assert torch.equal(sh.Atb(p, "matched"), tg.Atb(p, geo, ang, "matched"))
    assert sh.proj_dot(p, p) == pytest.approx(float((p.double() ** 2).sum()), rel=1e-12)
    # C3 at full size over 8 ranks: bands are ordered, overlap their neighbours and cover the detector
    geo3, ang3, _ = make_config("C3")
    shards = [ZSlabShards(geo3, ang3, r, 8) for r in range(8)]
    bands = shards[0].bands
    assert all(bands[i][0] <= bands[i + 1][0] and bands[i][1] <= bands[i + 1][1] for i in range(7))
    assert all(bands[i][1] > bands[i + 1][0] for i in range(7))
    assert bands[0][0] == 0 and bands[-1][1] == geo3.nDetector[1]
    own = shards[0].owned
    assert own[0][0] == 0 and own[-1][1] == geo3.nDetector[1] and all(own[i][1] == own[i + 1][0] for i in range(7))
    assert all(bands[i][0] <= own[i][0] and own[i][1] <= bands[i][1] for i in range(8))


def test_slab_argument_errors(tg):
    geo, ang, rec = make_config("C1", scale=4)
    vol = dev(phantom_for(rec, geo))
    with pytest.raises(tg.TigreError) as e:
        tg.Ax_slab(vol[:4], geo, ang, geo.nVoxel[2] - 2, "siddon")     # slab sticks out of the volume
    assert e.value.code == -1
    with pytest.raises(tg.TigreError) as e:
        tg.slab_row_band(geo, ang, 0, 0)
    assert e.value.code == -1
