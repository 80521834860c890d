"""The five BASELINE.json configs (C1..C5 = configs[0..4]) as Geometry + angle arrays.

Fields BASELINE.json leaves open are completed as SURVEY.md §8(d) proposes (all with
DSO = 1000 mm, DSD = 1536 mm) and restated in DESIGN.md "Input recipe".
No method arithmetic here: only parameter values and seeded random draws.
"""
from __future__ import annotations

import numpy as np

from .geometry import Geometry, circular_angles

# name -> recipe.  seed = config index.
CONFIGS = {
    "C1": dict(n=64, d=1.0, nA=64, det=(96, 96), ddet=1.6, seed=0,
               ax="siddon", atb="matched", phantom="head"),
    "C2": dict(n=256, d=0.5, nA=360, det=(512, 512), ddet=0.8, seed=1,
               ax="interp", atb="fdk", phantom="rand32"),
    "C3": dict(n=512, d=0.5, nA=720, det=(1024, 768), ddet=0.4, seed=2,
               ax="siddon", atb="matched", phantom="head+rand64", offDetector=(20.0, 0.0)),
    "C4": dict(n=1024, d=0.125, nA=1600, det=(1536, 1536), ddet=0.2, seed=3,
               ax="interp", atb="matched", phantom="pores", COR=0.3, rot_sigma_deg=0.5),
    "C5": dict(n=3072, d=0.04, nA=2400, det=(3072, 3072), ddet=0.1, seed=4,
               ax="siddon", atb="matched", phantom="rand64"),
}


def make_config(name: str, scale: int = 1, n_angles: int | None = None):
    """Return (geo, angles, recipe) for config `name`.

    scale > 1 gives a geometrically similar copy: voxel and pixel counts divided by
    `scale`, voxel and pixel pitches multiplied by it (same FOV, same fan/cone angles),
    angle count divided by it unless n_angles is given.  Used for parity cases the
    oracle finishes in seconds (e.g. the 1/4-scale C3 of SURVEY.md §8(d)).
    """
    r = dict(CONFIGS[name])
    n = r["n"] // scale
    nu, nv = r["det"][0] // scale, r["det"][1] // scale
    nA = n_angles if n_angles is not None else max(1, r["nA"] // scale)
    geo = Geometry(
        nVoxel=(n, n, n), dVoxel=(r["d"] * scale,) * 3,
        nDetector=(nu, nv), dDetector=(r["ddet"] * scale,) * 2,
        DSD=1536.0, DSO=1000.0, COR=r.get("COR", 0.0),
        offDetector=tuple(r.get("offDetector", (0.0, 0.0))), accuracy=0.5)
    angles = circular_angles(nA)
    if "rot_sigma_deg" in r:
        rng = np.random.default_rng(1000 + r["seed"])
        geo.rotDetector_a = np.deg2rad(r["rot_sigma_deg"]) * rng.standard_normal((nA, 3))
    r.update(name=name, scale=scale, nA=nA)
    return geo, angles, r


def scaled_config(name: str, scale: int, n_angles: int | None = None):
    return make_config(name, scale=scale, n_angles=n_angles)


def c5_like(n: int, n_angles: int):
    """configs[4]'s geometry at n^3 voxels and an n x n detector over the SAME field of view (pitches scaled by 3072 / n),
    with n_angles views over 2 pi: what the host-chunking runs use when the box cannot hold the full 207 GB."""
    r = CONFIGS["C5"]
    f = r["n"] / float(n)
    geo = Geometry(nVoxel=(n, n, n), dVoxel=(r["d"] * f,) * 3, nDetector=(n, n), dDetector=(r["ddet"] * f,) * 2,
                   DSD=1536.0, DSO=1000.0, accuracy=0.5)
    rec = dict(r, name="C5", scale=f, nA=n_angles)
    return geo, circular_angles(n_angles), rec
