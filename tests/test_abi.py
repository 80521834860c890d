"""CPU-side checks of the boundary: the shared library loads, exports every symbol that
include/tigre_b200.h declares, and fails loudly (no CPU fallback) when there is no device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2412_10129_b200 import build
    return build.build()


def declared_symbols():
    names = set()
    for fn in os.listdir(os.path.join(ROOT, "include")):
        if fn.endswith(".h"):
            txt = open(os.path.join(ROOT, "include", fn)).read()
            names |= set(re.findall(r"TIGRE_API[^;(]*?\b(tigre_\w+)\s*\(", txt))
    return names


def test_header_declares_the_boundary():
    names = declared_symbols()
    for need in ("tigre_Ax", "tigre_Atb", "tigre_row_weights", "tigre_col_weights", "tigre_residual",
                 "tigre_update", "tigre_ossart", "tigre_cgls", "tigre_fdk", "tigre_strerror"):
        assert need in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_binding_lists_every_declared_symbol(lib_path):
    import paper_2412_10129_b200 as tg
    assert set(tg.EXPORTS) == declared_symbols()
    assert ctypes.sizeof(tg.tigre_geo) == 200 or ctypes.sizeof(tg.tigre_geo) > 0
    assert tg.version() >= 100


def test_struct_layout_matches_header(lib_path, tmp_path):
    # compile a tiny C program against the header and compare sizeof / offsets with the ctypes mirror
    import subprocess
    import paper_2412_10129_b200 as tg
    src = tmp_path / "o.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "tigre_b200.h"\n'
                   'int main(){printf("%zu %zu %zu %zu %zu\\n", sizeof(tigre_geo), offsetof(tigre_geo,dVoxel),'
                   'offsetof(tigre_geo,DSD), offsetof(tigre_geo,DSD_a), offsetof(tigre_geo,accuracy));return 0;}\n')
    exe = tmp_path / "o"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(v) for v in subprocess.check_output([str(exe)]).split()]
    G = tg.tigre_geo
    assert got == [ctypes.sizeof(G), G.dVoxel.offset, G.DSD.offset, G.DSD_a.offset, G.accuracy.offset]


def test_no_cpu_fallback(lib_path):
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("device present")
    import paper_2412_10129_b200 as tg
    from workloads import make_config
    geo, ang, _ = make_config("C1", scale=4)
    vol = torch.zeros(geo.vol_shape)
    out = torch.zeros((len(ang), geo.nDetector[1], geo.nDetector[0]))
    with pytest.raises(tg.TigreError) as e:
        tg.Ax(vol, geo, ang, out=out)
    assert e.value.code == -6           # TIGRE_ERR_NO_DEVICE


def test_argument_errors_need_no_device(lib_path):
    import paper_2412_10129_b200 as tg
    lib = ctypes.CDLL(lib_path)
    assert lib.tigre_Ax(None, None, None, 0, 0, None, None) == -1
    lib.tigre_strerror.restype = ctypes.c_char_p
    assert b"argument" in lib.tigre_strerror(-1)
    assert b"no CPU fallback" in lib.tigre_strerror(-6)


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2412_10129_b200")):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2412_10129_b200", txt, flags=re.M), fn
            assert "libtigre_b200" not in txt and "#include \"../" not in txt, fn


def test_no_alloc_entry_point_rejects_oversize_without_a_device(lib_path):
    """tigre_residual_noalloc: the size limit of its fixed scratch array is checked before anything else (no device needed), the
    header's constant is the binding's, and the error has its own code and text."""
    import paper_2412_10129_b200 as tg
    hdr = open(os.path.join(ROOT, "include", "tigre_b200.h")).read()
    m = re.search(r"#define\s+TIGRE_RESIDUAL_NOALLOC_MAX_N\s+(\d+)ull", hdr)
    assert m and int(m.group(1)) == tg.RESIDUAL_NOALLOC_MAX_N == 1 << 28
    lib = ctypes.CDLL(lib_path)
    lib.tigre_strerror.restype = ctypes.c_char_p
    code = lib.tigre_residual_noalloc(None, None, None, None, ctypes.c_size_t(tg.RESIDUAL_NOALLOC_MAX_N + 1), None, None)
    assert code == -7 and b"no-allocation" in lib.tigre_strerror(code)
    src = open(os.path.join(ROOT, "paper_2412_10129_b200", "csrc", "noalloc.cu")).read()
    body = src[src.index('extern "C"'):]
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "TempBuf", "cudaStreamCreate", "cudaEventCreate", "Synchronize"):
        assert banned not in body, banned                     # the entry point allocates nothing and never synchronises
    assert "static __device__ __align__(256)" in src and "cudaGetSymbolAddress" in src
