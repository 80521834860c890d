"""Plain parameter container for the cone-beam geometry of PAPER.md App. B Table B1
(lines 543-566) and §2.4 (lines 179-197).  No transforms live here: the oracle and
the CUDA library each turn these numbers into source / detector positions themselves.

Units: mm and radians.  Axis order everywhere: volume (x, y, z), detector (u, v).
Arrays: vol[iz][iy][ix] (x fastest), proj[ia][iv][iu] (u fastest).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np


@dataclass
class Geometry:
    nVoxel: tuple            # (nx, ny, nz)
    dVoxel: tuple            # (dx, dy, dz) mm
    nDetector: tuple         # (nu, nv)
    dDetector: tuple         # (du, dv) mm
    DSD: float = 1536.0
    DSO: float = 1000.0
    COR: float = 0.0
    offOrigin: tuple = (0.0, 0.0, 0.0)
    offDetector: tuple = (0.0, 0.0)
    rotDetector: tuple = (0.0, 0.0, 0.0)     # (phi, theta, psi)
    accuracy: float = 0.5                    # interpolated-mode step, in voxels
    mode: str = "cone"                       # "cone" or "parallel" (synchrotron parallel-beam data)
    # optional per-angle overrides ("defined individually for each projection")
    DSD_a: Optional[np.ndarray] = None       # [nA]
    DSO_a: Optional[np.ndarray] = None       # [nA]
    COR_a: Optional[np.ndarray] = None       # [nA]
    offOrigin_a: Optional[np.ndarray] = None     # [nA][3]
    offDetector_a: Optional[np.ndarray] = None   # [nA][2]
    rotDetector_a: Optional[np.ndarray] = None   # [nA][3]

    @property
    def vol_shape(self):
        """numpy shape of the volume array (z, y, x)."""
        return (self.nVoxel[2], self.nVoxel[1], self.nVoxel[0])

    @property
    def proj_shape(self):
        """numpy shape of ONE projection (v, u)."""
        return (self.nDetector[1], self.nDetector[0])

    def copy(self, **kw) -> "Geometry":
        return replace(self, **kw)


def circular_angles(n: int, span: float = 2 * np.pi, start: float = 0.0) -> np.ndarray:
    """[n][3] Euler ZYZ array for a circular orbit: (theta, 0, 0), theta uniform in
    [start, start+span) (BASELINE.json configs "uniform in [0,2pi)")."""
    a = np.zeros((n, 3), dtype=np.float64)
    a[:, 0] = start + span * np.arange(n, dtype=np.float64) / n
    return a
