"""Multi-GPU sharding logic (paper_2412_10129_b200/sharded.py) on CPU: a world_size-2 gloo
group with the oracle's projectors injected as the local slab operators.  Checks the z-partition, the row bands (the
library's host arithmetic, tigre_slab_row_band) against the rows the partial projections really touch, the banded
point-to-point exchange and the all-reduce variant against the unsharded oracle, the collective-free A^T b, and the
once-per-row reductions."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")


def _sub_geo(geo, z0, nzs):
    nz, dz = geo.nVoxel[2], geo.dVoxel[2]
    shift = ((z0 + 0.5 * nzs) - 0.5 * nz) * dz
    off = tuple(geo.offOrigin)
    return geo.copy(nVoxel=(geo.nVoxel[0], geo.nVoxel[1], nzs), offOrigin=(off[0], off[1], off[2] + shift))


def _ops():
    from oracle import oracle as orc

    def ax_slab(vol_slab, geo, angles, z0, mode="siddon"):
        g = _sub_geo(geo, z0, vol_slab.shape[0])
        return torch.from_numpy(orc.ax(vol_slab.numpy(), g, angles, orc.SIDDON if mode == "siddon" else orc.INTERP))

    def atb_slab(proj, geo, angles, z0, nzs, mode="matched"):
        g = _sub_geo(geo, z0, nzs)
        return torch.from_numpy(orc.atb(proj.numpy(), g, angles, orc.MATCHED if mode == "matched" else orc.FDK))

    return ax_slab, atb_slab


def _case():
    from workloads import make_config, phantom_for
    geo, ang, rec = make_config("C1", scale=4, n_angles=8)          # 16^3, 24x24 detector
    vol = phantom_for(rec, geo).astype(np.float64) + 0.01           # no empty slab
    return geo, ang, vol


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import paper_2412_10129_b200 as tg
    from paper_2412_10129_b200.sharded import ZSlabShards
    from oracle import oracle as orc
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    geo, ang, vol = _case()
    ax_slab, atb_slab = _ops()
    sh = ZSlabShards(geo, ang, rank, world, ax_slab=ax_slab, atb_slab=atb_slab, row_band=tg.slab_row_band)
    full = orc.ax(vol, geo, ang, orc.SIDDON)
    slab = torch.from_numpy(vol[sh.z0:sh.z1].copy())
    part = ax_slab(slab, geo, ang, sh.z0).numpy()
    lo, hi = sh.band
    res = {"band": sh.band, "owned": sh.owned, "overlaps": sh.overlaps()}
    res["outside_band_zero"] = bool(np.all(part[:, :lo] == 0) and np.all(part[:, hi:] == 0))
    pb = sh.Ax(slab, "siddon", banded=True).numpy()
    res["banded_err"] = float(np.abs(pb[:, lo:hi] - full[:, lo:hi]).max())
    pr = sh.Ax(slab, "siddon", banded=False).numpy()
    res["replicated_err"] = float(np.abs(pr - full).max())
    back = sh.Atb(torch.from_numpy(pb), "matched").numpy()          # only this rank's band of pb is valid: enough
    ref = orc.atb(full, geo, ang, orc.MATCHED)[sh.z0:sh.z1]
    res["atb_err"] = float(np.abs(back - ref).max() / np.abs(ref).max())
    res["dot"] = sh.proj_dot(torch.from_numpy(pb), torch.from_numpy(pb))
    res["dot_ref"] = float(np.sum(full * full))
    res["vdot"] = sh.vol_dot(slab, slab)
    res["vdot_ref"] = float(np.sum(vol * vol))
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_pair_world2_gloo():
    import torch.multiprocessing as mp
    port = 31500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    for r in (0, 1):
        assert res[r]["outside_band_zero"]                          # the band bounds every row the slab touches
        assert res[r]["banded_err"] < 1e-12
        assert res[r]["replicated_err"] < 1e-12
        assert res[r]["atb_err"] < 1e-12
        assert res[r]["dot"] == pytest.approx(res[r]["dot_ref"], rel=1e-12)
        assert res[r]["vdot"] == pytest.approx(res[r]["vdot_ref"], rel=1e-12)
    (lo0, hi0), (lo1, hi1) = res[0]["band"], res[1]["band"]
    assert lo0 == 0 or lo0 < lo1                                     # slabs ordered in z -> bands ordered in v
    assert hi0 > lo1                                                 # the cone makes neighbouring slabs share rows
    assert res[0]["overlaps"] == [(1, lo1, hi0)] and res[1]["overlaps"] == [(0, lo1, hi0)]
    assert res[0]["owned"] == res[1]["owned"]
    (a0, b0), (a1, b1) = res[0]["owned"]
    assert a0 == 0 and b0 == a1 and lo1 <= b0 <= hi0                 # a partition, cut inside the overlap


def test_partition_and_ownership_units():
    sys.path.insert(0, ROOT)
    from paper_2412_10129_b200.sharded import owned_rows, z_partition
    assert z_partition(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert z_partition(2, 4) == [(0, 1), (1, 2), (2, 2), (2, 2)]
    own = owned_rows([(0, 40), (30, 70), (60, 96)], 96)
    assert own == [(0, 35), (35, 65), (65, 96)]
    assert owned_rows([(5, 90)], 96) == [(0, 96)]


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    import paper_2412_10129_b200 as tg
    from paper_2412_10129_b200.sharded import ZSlabShards
    from oracle import oracle as orc
    geo, ang, vol = _case()
    ax_slab, atb_slab = _ops()
    # two shards evaluated one after the other in one process: their partial projections add up to the whole
    parts = []
    for r in range(2):
        sh = ZSlabShards(geo, ang, r, 2, ax_slab=ax_slab, atb_slab=atb_slab, row_band=tg.slab_row_band)
        parts.append(ax_slab(torch.from_numpy(vol[sh.z0:sh.z1].copy()), geo, ang, sh.z0).numpy())
    assert np.abs(parts[0] + parts[1] - orc.ax(vol, geo, ang, orc.SIDDON)).max() < 1e-12
    one = ZSlabShards(geo, ang, 0, 1, ax_slab=ax_slab, atb_slab=atb_slab, row_band=tg.slab_row_band)
    assert np.abs(one.Ax(torch.from_numpy(vol.copy())).numpy() - orc.ax(vol, geo, ang, orc.SIDDON)).max() < 1e-12
