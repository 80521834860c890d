"""Multi-GPU sharding of the projector pair over NCCL / NVLink ("split
... by image slabs", "scales linearly with the number of GPUs").  One process per GPU (torch.distributed).

Layout: the volume is sharded by z-slab (rank r owns slices [z0_r, z1_r)); every rank holds the detector rows of the
projections that ITS slab can reach (its row band), for all views.
  A^T b  needs no exchange: a slab's voxels read only the slab's row band (tigre_Atb_slab).
  Ax     has ONE exchange step: each rank forms the partial line integrals of its slab (tigre_Ax_slab; zero outside its
         band); where the bands of two ranks overlap (the cone makes neighbouring slabs share rows) the partial sums are
         exchanged and added.  banded=True sends exactly those overlaps point to point (batch_isend_irecv: NCCL P2P over
         NVLink on a GPU box) and leaves each rank with correct rows inside its own band; banded=False all-reduces the
         whole projection array (replicated result, more bytes).
Reductions over projection space (residual norms) count every row once through `owned_rows`: a partition of the
detector rows among the ranks (overlaps cut at their middle).

The local operators default to the library's slab entry points; tests inject CPU callables with the same signature
so that the partition / exchange logic runs under gloo without a GPU.
"""
from __future__ import annotations

import numpy as np


def z_partition(nz, world):
    """Contiguous, near-even z-slabs: [(z0, z1)] * world (ranks beyond nz get empty slabs)."""
    base, rem = divmod(nz, world)
    out, z = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((z, z + n))
        z += n
    return out


def owned_rows(bands, nv):
    """Partition [0, nv) among the ranks given their row bands [(lo, hi)] (ordered like the slabs): every row goes to
    exactly one rank whose band contains it (overlaps are cut at their middle); rows in no band go to the nearest."""
    world = len(bands)
    cuts = [0]
    for r in range(world - 1):
        lo_next, hi_this = bands[r + 1][0], bands[r][1]
        cuts.append(int(np.clip((lo_next + hi_this) // 2, cuts[-1], nv)))
    cuts.append(nv)
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


class ZSlabShards:
    def __init__(self, geo, angles, rank, world, group=None, ax_slab=None, atb_slab=None, row_band=None):
        self.geo, self.angles, self.rank, self.world, self.group = geo, angles, rank, world, group
        if ax_slab is None or atb_slab is None or row_band is None:
            import paper_2412_10129_b200 as tg            # the CUDA path; fails loudly without the extension
            ax_slab = ax_slab or tg.Ax_slab
            atb_slab = atb_slab or tg.Atb_slab
            row_band = row_band or tg.slab_row_band
        self._ax, self._atb = ax_slab, atb_slab
        nz, nv = geo.nVoxel[2], geo.nDetector[1]
        self.slabs = z_partition(nz, world)
        self.z0, self.z1 = self.slabs[rank]
        self.bands = []
        for (a, b) in self.slabs:                          # every rank computes every band: same host arithmetic
            if b > a:
                r0, nr = row_band(geo, angles, a, b - a)
                self.bands.append((r0, r0 + nr))
            else:
                self.bands.append((0, 0))
        self.band = self.bands[rank]
        self.owned = owned_rows(self.bands, nv)

    # ------------------------------------------------------------------ A^T b: no collective
    def Atb(self, proj, mode="matched"):
        """This rank's slab of A^T b.  proj: full-size array, valid at least on this rank's row band."""
        return self._atb(proj, self.geo, self.angles, self.z0, self.z1 - self.z0, mode)

    # ------------------------------------------------------------------ Ax: one exchange step
    def overlaps(self):
        """[(peer, lo, hi)]: rows this rank must exchange with each peer (intersection of the two bands)."""
        out = []
        for s in range(self.world):
            if s == self.rank:
                continue
            lo, hi = max(self.band[0], self.bands[s][0]), min(self.band[1], self.bands[s][1])
            if hi > lo:
                out.append((s, lo, hi))
        return out

    def Ax(self, vol_slab, mode="siddon", banded=True):
        """Projections of the WHOLE volume from this rank's slab: correct on this rank's row band (banded=True) or
        everywhere (banded=False)."""
        import torch
        import torch.distributed as dist
        part = self._ax(vol_slab, self.geo, self.angles, self.z0, mode)
        if self.world == 1:
            return part
        if not banded:
            dist.all_reduce(part, op=dist.ReduceOp.SUM, group=self.group)
            return part
        ops, recv = [], []
        for peer, lo, hi in self.overlaps():
            send = part[:, lo:hi, :].contiguous()          # my partial sums on the rows we share (snapshot before adding)
            buf = torch.empty_like(send)
            ops.append(dist.P2POp(dist.isend, send, peer, group=self.group))
            ops.append(dist.P2POp(dist.irecv, buf, peer, group=self.group))
            recv.append((lo, hi, buf))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        for lo, hi, buf in recv:
            part[:, lo:hi, :] += buf
        return part

    # ------------------------------------------------------------------ reductions over projection space
    def proj_dot(self, a, b):
        """<a, b> over all projection elements, every detector row counted once (on the rank that owns it)."""
        import torch
        import torch.distributed as dist
        lo, hi = self.owned[self.rank]
        s = (a[:, lo:hi, :].double() * b[:, lo:hi, :].double()).sum().reshape(1)
        if self.world > 1:
            dist.all_reduce(s, op=dist.ReduceOp.SUM, group=self.group)
        return float(s)

    def vol_dot(self, a_slab, b_slab):
        import torch
        import torch.distributed as dist
        s = (a_slab.double() * b_slab.double()).sum().reshape(1)
        if self.world > 1:
            dist.all_reduce(s, op=dist.ReduceOp.SUM, group=self.group)
        return float(s)
