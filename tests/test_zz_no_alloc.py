"""tigre_residual_noalloc (include/tigre_b200.h; csrc/noalloc.cu): the residual for callers that cannot call cudaMalloc.
Checked against the existing path (tigre_residual) on calls in a row that share the file-scope scratch array: a large call,
then a smaller one (the large call's partial sums stay in the array beyond the slots the small one uses), then the large one
again; r must be bitwise the existing path's, nrm2 within the 1e-6 of tests/test_gpu_parity.py::test_residual_and_update
(and in fact to fp64 rounding), and bitwise the same when a call is repeated.  Named test_zz_* so that pytest collects it
last: the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def tg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2412_10129_b200 as m
    m.version()
    return m


def _inputs(n, seed, offset=0):
    """seeded uniform inputs; offset = 1 gives views that are only 4-byte aligned (the scalar instantiation of the kernel)"""
    g = torch.Generator(device="cuda").manual_seed(seed)
    return [torch.rand(n + offset, generator=g, device="cuda", dtype=torch.float32)[offset:] for _ in range(3)]


def _one_call(tg, n, seed, with_w, offset=0):
    b, a, w = _inputs(n, seed, offset)
    w = w if with_w else None
    r_ref, nrm_ref = tg.residual(b.contiguous(), a.contiguous(), w.contiguous() if with_w else None, return_norm=True)   # the existing path
    r = torch.full((n + offset,), float("nan"), device="cuda")[offset:]
    nrm = torch.full((1,), float("nan"), device="cuda", dtype=torch.float64)
    tg.residual_noalloc(b, a, r, W=w, nrm2=nrm)
    torch.cuda.synchronize()
    assert torch.equal(r, r_ref)
    got = float(nrm.item())
    assert abs(got - nrm_ref) <= 1e-6 * max(nrm_ref, 1e-30)
    assert abs(got - nrm_ref) <= 1e-11 * max(nrm_ref, 1e-30)        # two fp64 summation orders of the same terms
    ref64 = float(((b.double() - a.double()) ** 2).sum().item())      # (fp32 difference squared in fp64 on the device, vs all-fp64)
    assert abs(got - ref64) <= 1e-6 * max(ref64, 1e-30)
    # the same call again: same slots of the shared array, fixed summation order -> bitwise the same number
    nrm_again = torch.zeros(1, device="cuda", dtype=torch.float64)
    tg.residual_noalloc(b, a, r, W=w, nrm2=nrm_again)
    torch.cuda.synchronize()
    assert nrm_again.item() == nrm.item()
    return got


def test_noalloc_residual_matches_the_existing_path_on_calls_in_a_row(tg):
    big, small = 3_000_003, 100_003            # 184 and 7 CTAs' worth of partials, ragged tails
    first = _one_call(tg, big, seed=11, with_w=True)
    _one_call(tg, small, seed=12, with_w=True)          # the big call's partials are still in slots 7..183
    _one_call(tg, small, seed=13, with_w=False, offset=1)   # unaligned views: scalar kernel
    _one_call(tg, 1, seed=14, with_w=False)
    assert _one_call(tg, big, seed=11, with_w=True) == first   # and the big call is unaffected by what ran in between


def test_noalloc_residual_without_norm_and_empty(tg):
    b, a, w = _inputs(70_001, 21)
    r = torch.empty_like(b)
    tg.residual_noalloc(b, a, r, W=w)                     # nrm2 = NULL: only r
    assert torch.equal(r, tg.residual(b, a, w))
    nrm = torch.full((1,), 5.0, device="cuda", dtype=torch.float64)
    e = torch.empty(0, device="cuda")
    tg.residual_noalloc(e, e, torch.empty(0, device="cuda"), nrm2=nrm)   # empty input: an empty sum
    assert nrm.item() == 0.0


def test_noalloc_residual_rejects_sizes_beyond_its_scratch(tg):
    b, a, _ = _inputs(1024, 31)
    r = torch.full((1024,), 7.0, device="cuda")
    lib = tg._lib()
    args = lambda n: (C.c_void_p(b.data_ptr()), C.c_void_p(a.data_ptr()), None, C.c_void_p(r.data_ptr()), C.c_size_t(n), None,
                      C.c_void_p(torch.cuda.current_stream().cuda_stream))
    code = lib.tigre_residual_noalloc(*args(tg.RESIDUAL_NOALLOC_MAX_N + 1))
    assert code == -7 and b"TIGRE_RESIDUAL_NOALLOC_MAX_N" in lib.tigre_strerror(code)
    torch.cuda.synchronize()
    assert bool((r == 7.0).all())                          # nothing was launched
    with pytest.raises(tg.TigreError, match="no-allocation"):
        tg._check(code, "tigre_residual_noalloc")
    assert lib.tigre_residual_noalloc(*args(1024)) == 0    # and the entry point still works afterwards


def test_noalloc_residual_leaves_device_memory_as_it_found_it(tg):
    b, a, w = _inputs(1_000_000, 41)
    r = torch.empty_like(b)
    nrm = torch.zeros(1, device="cuda", dtype=torch.float64)
    tg.residual_noalloc(b, a, r, W=w, nrm2=nrm)            # (first use on this device looks the scratch address up)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ws0 = tg.workspace_stats() if hasattr(tg, "workspace_stats") else None
    for _ in range(20):
        tg.residual_noalloc(b, a, r, W=w, nrm2=nrm)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    if ws0 is not None:
        assert tg.workspace_stats() == ws0
    ref = tg.residual(b, a, w, return_norm=True)[1]
    assert abs(nrm.item() - ref) <= 1e-6 * ref
