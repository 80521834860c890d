"""Seeded synthetic phantoms (input synthesis only — SURVEY.md §8(c) "Input synthesis").

An ellipsoid list is a dict of arrays:
    centre [n][3] mm, axes [n][3] mm (semi-axes), Q [n][3][3] (columns = ellipsoid axes
    in world coordinates), rho [n] mm^-1 (additive intensities).
Voxelisation point-samples membership at voxel centres.  The same lists feed the
closed-form chord pins in tests/ (which own that arithmetic).
"""
from __future__ import annotations

import os

import numpy as np

_DATA = os.path.join(os.path.dirname(__file__), "data", "head_phantom.txt")


def _rotz(deg):
    c, s = np.cos(np.deg2rad(deg)), np.sin(np.deg2rad(deg))
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])


def head_ellipsoids(half_fov_mm: float):
    """The repo-owned 10-ellipsoid head-like phantom scaled to a cube of half-size half_fov_mm."""
    t = np.loadtxt(_DATA)
    return dict(
        rho=t[:, 0].copy(),
        axes=t[:, 1:4] * half_fov_mm,
        centre=t[:, 4:7] * half_fov_mm,
        Q=np.stack([_rotz(p) for p in t[:, 7]]),
    )


def _random_rotations(rng, n):
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    return np.stack([
        np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], -1),
        np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], -1),
        np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], -1),
    ], 1)


def random_ellipsoids(n: int, fov_mm: float, seed: int):
    """BASELINE.json configs[1]: centres U(-0.8,0.8)*half-FOV, semi-axes U(0.05,0.3)*FOV,
    attenuation U(0,0.02) mm^-1, random rotations; numpy PCG64 seeded with `seed`."""
    rng = np.random.default_rng(seed)
    half = 0.5 * fov_mm
    return dict(
        centre=rng.uniform(-0.8, 0.8, (n, 3)) * half,
        axes=rng.uniform(0.05, 0.3, (n, 3)) * fov_mm,
        rho=rng.uniform(0.0, 0.02, n),
        Q=_random_rotations(rng, n),
    )


def concat_ellipsoids(*lists):
    return {k: np.concatenate([l[k] for l in lists]) for k in ("centre", "axes", "rho", "Q")}


def voxelise_slab(ell, geo, z0: int, z1: int, dtype=np.float32):
    """Voxelise z-slices [z0, z1) of the volume described by geo (offOrigin scalar form).
    Membership ((Q^T (X-c)) / axes)^2 summed <= 1 is evaluated in float64 at voxel centres, inside
    each ellipsoid's axis-aligned bounding box only."""
    nx, ny, nz = geo.nVoxel
    dx, dy, dz = geo.dVoxel
    ox, oy, oz = geo.offOrigin
    x = ox + (np.arange(nx) + 0.5) * dx - 0.5 * nx * dx
    y = oy + (np.arange(ny) + 0.5) * dy - 0.5 * ny * dy
    z = oz + (np.arange(z0, z1) + 0.5) * dz - 0.5 * nz * dz
    out = np.zeros((z1 - z0, ny, nx), dtype=dtype)
    for c, ax, Q, rho in zip(ell["centre"], ell["axes"], ell["Q"], ell["rho"]):
        ext = np.sqrt(((Q * ax[None, :]) ** 2).sum(axis=1))      # half-extent of the bounding box per world axis
        sel = []
        for coord, ck, ek in ((x, c[0], ext[0]), (y, c[1], ext[1]), (z, c[2], ext[2])):
            k = np.nonzero(np.abs(coord - ck) <= ek)[0]
            sel.append(k)
        if any(k.size == 0 for k in sel):
            continue
        sx, sy, sz = (slice(k[0], k[-1] + 1) for k in sel)
        X = x[sx][None, None, :] - c[0]
        Y = y[sy][None, :, None] - c[1]
        Z = z[sz][:, None, None] - c[2]
        s = 0.0
        for k in range(3):
            lk = (Q[0, k] * X + Q[1, k] * Y + Q[2, k] * Z) / ax[k]
            s = s + lk * lk
        out[sz, sy, sx] += (rho * (s <= 1.0)).astype(dtype)
    return out


def voxelise_slab_torch(ell, geo, z0: int, z1: int, device="cuda"):
    """voxelise_slab evaluated with torch on `device` (the same membership test in float64, the same bounding boxes): for
    volumes of tens of GB, where the numpy loop would take an hour.  Returns a float32 tensor [z1 - z0][ny][nx] on `device`.
    Input synthesis only; the consumer copies it wherever both sides read it from."""
    import torch
    nx, ny, nz = geo.nVoxel
    dx, dy, dz = geo.dVoxel
    ox, oy, oz = geo.offOrigin
    x = ox + (np.arange(nx) + 0.5) * dx - 0.5 * nx * dx
    y = oy + (np.arange(ny) + 0.5) * dy - 0.5 * ny * dy
    z = oz + (np.arange(z0, z1) + 0.5) * dz - 0.5 * nz * dz
    tx, ty, tz = (torch.from_numpy(a).to(device) for a in (x, y, z))
    out = torch.zeros((z1 - z0, ny, nx), dtype=torch.float32, device=device)
    for c, ax, Q, rho in zip(ell["centre"], ell["axes"], ell["Q"], ell["rho"]):
        ext = np.sqrt(((Q * ax[None, :]) ** 2).sum(axis=1))
        sel = [np.nonzero(np.abs(coord - ck) <= ek)[0] for coord, ck, ek in ((x, c[0], ext[0]), (y, c[1], ext[1]), (z, c[2], ext[2]))]
        if any(k.size == 0 for k in sel):
            continue
        sx, sy, sz = (slice(int(k[0]), int(k[-1]) + 1) for k in sel)
        X = tx[sx][None, None, :] - float(c[0])
        Y = ty[sy][None, :, None] - float(c[1])
        Z = tz[sz][:, None, None] - float(c[2])
        s = None
        for k in range(3):
            lk = (float(Q[0, k]) * X + float(Q[1, k]) * Y + float(Q[2, k]) * Z) / float(ax[k])
            s = lk * lk if s is None else s + lk * lk
        out[sz, sy, sx] += (s <= 1.0).to(torch.float32) * float(np.float32(rho))
    return out


def voxelise(ell, geo, dtype=np.float32, slab: int = 64):
    nz = geo.nVoxel[2]
    return np.concatenate([voxelise_slab(ell, geo, z0, min(nz, z0 + slab), dtype)
                           for z0 in range(0, nz, slab)], axis=0)


def porous_cylinder(geo, n_pores: int, seed: int, rho: float = 0.02, dtype=np.float32):
    """BASELINE.json configs[3]: cylinder (axis z, radius 0.45*FOV) of `rho` with
    spherical pores of radius U(2,20) voxels set to 0."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = geo.nVoxel
    dx, dy, dz = geo.dVoxel
    fov = nx * dx
    R = 0.45 * fov
    x = (np.arange(nx) + 0.5) * dx - 0.5 * nx * dx
    y = (np.arange(ny) + 0.5) * dy - 0.5 * ny * dy
    z = (np.arange(nz) + 0.5) * dz - 0.5 * nz * dz
    inside = (x[None, :] ** 2 + y[:, None] ** 2) <= R * R
    vol = np.broadcast_to(inside[None] * rho, (nz, ny, nx)).astype(dtype).copy()
    r = rng.uniform(2.0, 20.0, n_pores) * dx
    ang = rng.uniform(0, 2 * np.pi, n_pores)
    rad = R * np.sqrt(rng.uniform(0, 1, n_pores))
    cz = rng.uniform(-0.5 * nz * dz, 0.5 * nz * dz, n_pores)
    cx, cy = rad * np.cos(ang), rad * np.sin(ang)
    for k in range(n_pores):
        ix = np.nonzero(np.abs(x - cx[k]) <= r[k])[0]
        iy = np.nonzero(np.abs(y - cy[k]) <= r[k])[0]
        iz = np.nonzero(np.abs(z - cz[k]) <= r[k])[0]
        if ix.size == 0 or iy.size == 0 or iz.size == 0:
            continue
        sx, sy, sz = slice(ix[0], ix[-1] + 1), slice(iy[0], iy[-1] + 1), slice(iz[0], iz[-1] + 1)
        m = ((x[sx][None, None, :] - cx[k]) ** 2 + (y[sy][None, :, None] - cy[k]) ** 2
             + (z[sz][:, None, None] - cz[k]) ** 2) <= r[k] ** 2
        vol[sz, sy, sx][m] = 0
    return vol


def phantom_for(recipe, geo, dtype=np.float32):
    """Volume for a config recipe from workloads.configs (C1..C5)."""
    fov = geo.nVoxel[0] * geo.dVoxel[0]
    kind, seed = recipe["phantom"], recipe["seed"]
    if kind == "head":
        return voxelise(head_ellipsoids(0.5 * fov), geo, dtype)
    if kind == "rand32":
        return voxelise(random_ellipsoids(32, fov, seed), geo, dtype)
    if kind == "rand64":
        return voxelise(random_ellipsoids(64, fov, seed), geo, dtype)
    if kind == "head+rand64":
        return voxelise(concat_ellipsoids(head_ellipsoids(0.5 * fov),
                                          random_ellipsoids(64, fov, seed)), geo, dtype)
    if kind == "pores":
        return porous_cylinder(geo, 2000, seed, dtype=dtype)
    raise ValueError(kind)


def poisson_noise(b, I0: float, seed: int):
    """BASELINE.json configs[2] / SURVEY.md P18: b_noisy = -log(max(Poisson(I0 e^-b),1)/I0),
    generated once on the host and handed to both sides."""
    rng = np.random.default_rng(seed)
    counts = rng.poisson(I0 * np.exp(-np.asarray(b, dtype=np.float64)))
    return (-np.log(np.maximum(counts, 1) / I0)).astype(np.float32)
