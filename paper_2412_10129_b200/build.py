"""Build libtigre_b200.so in-tree with nvcc for sm_100a (run: python -m paper_2412_10129_b200.build).

TIGRE_NVCC_EXTRA="-DAXTU=64 -DAXTV=2" python -m paper_2412_10129_b200.build --force   builds a tuning variant (the macros are
listed at the top of csrc/ax_common.cuh, csrc/ax_tma.cu, csrc/fdk_tc.cu); profiles/ names such builds by this command line."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtigre_b200.so")
SOURCES = ["geometry.cu", "ax.cu", "ax_tma.cu", "ax_siddon_tma.cu", "atb.cu", "atb_tma.cu", "elementwise.cu", "tv.cu", "prox.cu", "fdk.cu", "fdk_tc.cu", "chunked.cu", "peaks.cu", "noalloc.cu", "api.cu"]
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--fmad=true", "-cudart", "static"]


def _sources():
    return [os.path.join(CSRC, s) for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    import glob
    deps = _sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")) + [os.path.join(HERE, "..", "include", "tigre_b200.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    objs = []
    procs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for src in _sources():
        obj = os.path.join(HERE, "build", os.path.basename(src) + ".o")
        cmd = ["nvcc", "-c", src, "-o", obj] + FLAGS + os.environ.get("TIGRE_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else [])
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(obj)
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    subprocess.check_call(["nvcc", "-shared", "-o", LIB] + objs + ["-cudart", "static"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
