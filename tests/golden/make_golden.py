"""Writes tests/golden/c1_oracle_samples.txt: values of the fp64 ORACLE (oracle/ only; the CUDA path is never
involved) on BASELINE.json configs[0] "C1" (64^3 head phantom, 64 views of 96x96) at seeded sample points:
Siddon and interpolated line integrals of 48 rays, matched and FDK backprojections of 48 voxels (of the oracle's own
Siddon projections).  The paper prints no worked numerical example (PAPER.md gives definitions only, eq. 1 at
lines 80-84), so this file is a regression anchor for the oracle, not a pin: the pins are the closed forms and
brute-force checks in tests/test_oracle_pins.py.

    python tests/golden/make_golden.py        (from the repo root)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from workloads import make_config, phantom_for  # noqa: E402


def main():
    geo, ang, rec = make_config("C1")
    vol = phantom_for(rec, geo)
    rng = np.random.default_rng(20241210)
    n_rays = len(ang) * geo.nDetector[0] * geo.nDetector[1]
    # rays through the central half of the detector (so most of them hit the phantom)
    ia = rng.integers(0, len(ang), 48)
    iv = rng.integers(24, 72, 48)
    iu = rng.integers(24, 72, 48)
    rid = (ia * geo.nDetector[1] + iv) * geo.nDetector[0] + iu
    assert rid.max() < n_rays
    sid = orc.ax(vol, geo, ang, orc.SIDDON, ray_ids=rid)
    itp = orc.ax(vol, geo, ang, orc.INTERP, ray_ids=rid)
    proj = orc.ax(vol, geo, ang, orc.SIDDON).astype(np.float32)
    vid = rng.integers(0, vol.size, 48)
    mat = orc.atb(proj, geo, ang, orc.MATCHED, vox_ids=vid)
    fdk = orc.atb(proj, geo, ang, orc.FDK, vox_ids=vid)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle_samples.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ (fp64 CPU oracle) only; config C1, seed 20241210\n")
        f.write("# kind id value_a value_b   (ray: id = (ia*nv+iv)*nu+iu, a = Siddon, b = interpolated [mm * 1/mm];\n")
        f.write("#                            vox: id = (iz*ny+iy)*nx+ix, a = matched A^T b, b = FDK-weighted A^T b)\n")
        for i in range(48):
            f.write(f"ray {int(rid[i])} {sid[i]:.17g} {itp[i]:.17g}\n")
        for i in range(48):
            f.write(f"vox {int(vid[i])} {mat[i]:.17g} {fdk[i]:.17g}\n")
    print(path)


if __name__ == "__main__":
    main()
