"""tigre_set_workspace ("the library allocates nothing persistent ... workspace memory is the
caller's"): with a caller-owned block set, drivers and plans run bitwise as with the stream-ordered pool and make no
allocation of their own; too small a block fails cleanly."""
import numpy as np
import pytest

from workloads import make_config, phantom_for

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2412_10129_b200 as m
    m.version()
    yield m
    m.set_workspace(None)


def test_ossart_cgls_fdk_bitwise_with_and_without_workspace(tg):
    geo, ang, rec = make_config("C3", scale=8)
    vol = torch.from_numpy(phantom_for(rec, geo)).cuda()
    nA = len(ang)
    subsets = [np.arange(s, nA, 5) for s in range(5)]
    b = tg.Ax(vol, geo, ang, "siddon")

    def run():
        plan = tg.OssartPlan(geo, ang, subsets)
        x = torch.zeros_like(vol)
        hist = plan.iterate(b, x, 3)
        plan.close()
        xc, _ = tg.cgls(b, geo, ang, 3, "siddon", "matched")
        xf = tg.fdk(b, geo, ang)
        xe = tg.Atb(b, geo, ang, "exact_siddon")
        return x, hist, xc, xf, tg.Ax(vol, geo, ang, "interp"), xe

    tg.set_workspace(None)
    ref = run()
    need = tg.plan_workspace_bytes(geo, nA, len(subsets), max(len(s) for s in subsets)) + tg.workspace_bytes(geo, nA, 3)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    tg.set_workspace(ws)
    try:
        got = run()
        in_use, high, pool_allocs = tg.workspace_stats()
        assert pool_allocs == 0                      # not one cudaMallocAsync while the workspace was set
        assert in_use == 0 and 0 < high <= need      # everything handed back; the stated bound held
    finally:
        tg.set_workspace(None)
    torch.cuda.synchronize()
    for a, r in zip(got[:1] + got[2:5], ref[:1] + ref[2:5]):
        assert torch.equal(a, r)                     # same kernels, same order: bitwise
    assert np.allclose(got[1], ref[1], rtol=1e-12, atol=0)     # the norm is summed with fp64 atomics: block order only
    assert float((got[5] - ref[5]).norm() / ref[5].norm()) < 2e-6   # atomics: order of summation only


def test_workspace_too_small_fails_cleanly_and_plans_pin_it(tg):
    geo, ang, rec = make_config("C1", scale=2)
    vol = torch.from_numpy(phantom_for(rec, geo)).cuda()
    b = tg.Ax(vol, geo, ang, "siddon")
    small = torch.empty(8192, dtype=torch.uint8, device="cuda")
    tg.set_workspace(small)
    try:
        with pytest.raises(tg.TigreError) as e:
            tg.cgls(b, geo, ang, 1)                  # needs two projection-sized and two volume-sized buffers
        assert e.value.code == -4
        assert tg.workspace_stats()[0] == 0          # the failed call left nothing behind
    finally:
        tg.set_workspace(None)
    ws = torch.empty(tg.plan_workspace_bytes(geo, len(ang), 1, len(ang)), dtype=torch.uint8, device="cuda")
    tg.set_workspace(ws)
    plan = tg.OssartPlan(geo, ang, [np.arange(len(ang))])
    with pytest.raises(tg.TigreError):
        tg.set_workspace(None)                       # a live plan holds blocks of it
    plan.close()
    tg.set_workspace(None)
    with pytest.raises(tg.TigreError):
        tg.set_workspace(torch.empty(16, dtype=torch.uint8, device="cuda"))      # below the minimum
    host = torch.empty(1 << 20, dtype=torch.uint8).pin_memory()
    with pytest.raises(tg.TigreError) as e:
        tg.set_workspace(host)
    assert e.value.code == -3


def test_chunked_path_sizes_itself_to_the_workspace(tg):
    from oracle import oracle as orc
    geo, ang, rec = make_config("C5", scale=96)
    vol = phantom_for(rec, geo)
    hv = torch.from_numpy(vol).pin_memory()
    ws = torch.empty(400 << 10, dtype=torch.uint8, device="cuda")      # budget = half of it: several slabs and batches
    tg.set_workspace(ws)
    try:
        p = tg.Ax(hv, geo, ang, "siddon")
        _, _, n_slabs, n_batches = tg.chunk_stats()
        assert tg.workspace_stats()[2] == 0 and n_slabs * n_batches > 1
    finally:
        tg.set_workspace(None)
    ref = orc.ax(vol, geo, ang, orc.SIDDON)
    assert np.linalg.norm(p.numpy().astype(np.float64) - ref) <= 1e-5 * np.linalg.norm(ref)


def test_plan_recomputes_column_weights_when_they_do_not_fit(tg):
    """Single-view subsets (SART, the data step of ASD-POCS / SART-TV): the plan keeps one volume of column weights and refills it
    per subset step instead of nSubsets volumes; same kernels, same numbers as the stored variant, and the oracle's SART."""
    from oracle import oracle as orc
    geo, ang, rec = make_config("C3", scale=16, n_angles=24)
    vol = phantom_for(rec, geo)
    b = tg.Ax(torch.from_numpy(vol).cuda(), geo, ang, "siddon")
    subsets = [np.array([a]) for a in range(len(ang))]
    out = {}
    for path in (1, 2):
        tg.set_plan_v_path(path)
        try:
            plan = tg.OssartPlan(geo, ang, subsets)
            out[path] = (plan.nbytes, torch.zeros_like(b[0, :1, :1]))
            x = torch.zeros(tg.vol_shape(geo), dtype=torch.float32, device="cuda")
            plan.iterate(b, x, 2, lam=0.5)
            xo = torch.ones_like(x)
            plan.osem(b, xo, 1)
            out[path] = (plan.nbytes, x, xo)
            plan.close()
        finally:
            tg.set_plan_v_path(0)
    nvox = int(np.prod(geo.nVoxel))
    assert out[1][0] - out[2][0] == 4 * nvox * (len(subsets) - 1)
    assert torch.equal(out[1][1], out[2][1]) and torch.equal(out[1][2], out[2][2])
    xr, _ = orc.ossart(b.cpu().numpy(), geo, ang, subsets, 2, lam=0.5)
    got = out[2][1].cpu().numpy().astype(np.float64)
    assert np.linalg.norm(got - xr) <= 3e-5 * np.linalg.norm(xr)
