"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package holds NONE of the method's arithmetic (no projector, no weights,
no geometry transforms): only the plain `Geometry` parameter container
(App. B Table B1), the BASELINE.json config recipes, and the
phantom voxeliser (point-sampled ellipsoid membership).  Both `oracle/` and
`paper_2412_10129_b200/` take their inputs from here; neither imports the other.
"""
from .geometry import Geometry, circular_angles
from .configs import CONFIGS, c5_like, make_config, scaled_config
from .phantoms import (head_ellipsoids, random_ellipsoids, voxelise,
                       voxelise_slab, porous_cylinder, poisson_noise, phantom_for,
                       concat_ellipsoids, voxelise_slab_torch)

__all__ = ["Geometry", "circular_angles", "CONFIGS", "make_config", "scaled_config",
           "head_ellipsoids", "random_ellipsoids", "voxelise", "voxelise_slab",
           "porous_cylinder", "poisson_noise", "phantom_for", "concat_ellipsoids", "voxelise_slab_torch", "c5_like"]
