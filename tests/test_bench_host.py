"""Host logic of bench.py that needs no GPU: the N > 1 aggregation (replicas only) under a
world_size-2 gloo process group, the roofline model, the subset recipe, and the reference arm's rank gating."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, "cpu")          # rank 1 is the slow one
    out[rank] = (ms, bench.whole_job_value(1.0e9, ms, world))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    import torch.multiprocessing as mp
    port = 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0] == res[1]                                         # every rank sees the same numbers
    ms, value = res[0]
    assert ms == 15.0                                               # the slowest rank's device time
    assert value == pytest.approx(2 * 1.0e9 / 15.0e-3 / 1e9)        # N x units / max time, in G units/s


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(2.0e9, 1000.0, 1) == pytest.approx(2.0)


def test_roofline_model_and_subsets():
    sys.path.insert(0, ROOT)
    import bench
    # DESIGN.md section 6 with the nominal machine rates (the run itself uses the measured ones): issue slots / algorithmic
    # instructions per unit, or the on-chip gather bound where lower
    r = bench.NOMINAL_PEAKS
    assert bench.model_peak("atb", r) == pytest.approx(148 * 128 * 1965e6 / 22 / 1e9)                  # 1.69 T updates/s (smem: 2.3)
    assert bench.model_peak("ax_siddon", r) == pytest.approx(148 * 128 * 1965e6 / 18 / 1e9)            # 2.07 T samples/s: issue binds
    assert bench.model_bounds("ax_siddon", r)["l1"] == pytest.approx(148 * 1965e6 * 32 / 2.84 / 1e9)   # (L1 at the measured 2.84 wavefronts)
    assert bench.model_peak("ax_interp", r) == pytest.approx(148 * 1965e6 / 16 * 32 / 1e9)             # 0.58 T samples/s: L1 binds
    assert "binding = issue" in bench.peak_source("ax_siddon", r, False)
    subs = bench.subsets_for({"name": "C3"}, 720)                   # reading P15: 20 interleaved subsets
    assert len(subs) == 20 and all(len(s) == 36 for s in subs)
    assert np.array_equal(subs[3][:3], [3, 23, 43])
    assert np.array_equal(np.sort(np.concatenate(subs)), np.arange(720))
    assert len(bench.subsets_for({"name": "C1"}, 64)) == 1          # SIRT


def test_reference_arm_rank_gating_and_line():
    # under torchrun only rank 0 runs the oracle; the other ranks exit 0 without output
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
