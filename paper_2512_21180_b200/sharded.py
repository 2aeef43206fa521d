"""One batch of the cone-beam operators split over several GPUs (one process per GPU).

Call sequencing only -- every value is computed by the library's kernels through `cbct.Geometry`; the collectives
are `torch.distributed` (NCCL over NVLink on GPUs, gloo in the CPU tests of the partition logic).  Two splits:

* `channel_split` (s.8(e) item 1): channels are independent, so rank r runs the plain whole-volume calls on its
  contiguous share of the channels (`dist.channel_shard`).  No data-path collective; results stay sharded by
  channel.  The split to use whenever the batch has at least as many channels as there are ranks.
* `ShardedGeometry` (s.8(e) item 2), for batches with fewer channels than ranks (LIRE++ calls P on 4 + 1 and P* on
  4 and 1 channels): the FORWARD projector is sharded by VIEWS -- rank r owns views r, r + W,
  r + 2W, ... through its own handle with that strided angle list (reading R14: such a handle reproduces exactly
  those rows; the stride keeps the quarter-turn symmetry between a rank's views whenever n_views / W is a multiple
  of 4) and needs the whole volume -- and the BACKPROJECTORS by PLANES -- rank r owns a range of z-planes (on
  geometries symmetric under z -> -z: a range of the lower half together with its mirror image, which shares every
  weight) through `cbct_bp_adjoint_slab` / `cbct_bp_fdk_slab` and needs the whole sinogram.  A forward projection
  followed by a backprojection therefore costs exactly ONE exchange step: an all-gather of the sinogram rows
  (100 MiB per channel at 400 x 256 x 256; ~0.1-0.2 ms over NVSwitch against >= 5 ms of kernels).

Unmeasured on hardware: this pool hands out one GPU at a time.  The partition arithmetic and the reassembly are
covered by world-size-2 gloo tests on CPU (tests/test_dist_cpu.py); on one GPU, tests/test_gpu_sharded.py runs the
ranks' calls one after the other and checks the reassembled results against the unsharded calls and the oracle.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import dist as cdist


# ---------------------------------------------------------------------------------------------------------------
# partition arithmetic (pure integers; shared by the ranks' code, the CPU tests and the 1-GPU emulation)
# ---------------------------------------------------------------------------------------------------------------
def view_shard(n_views: int, rank: int, world: int) -> List[int]:
    """Views owned by `rank`: rank, rank + world, rank + 2 world, ...  Every view belongs to exactly one rank."""
    if n_views < 1 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad shard request")
    return list(range(rank, n_views, world))


def views_per_rank_padded(n_views: int, world: int) -> int:
    """Rows of a rank's block in the all-gather (blocks are padded to equal size when world does not divide n)."""
    return -(-n_views // world)


def plane_shard(nz: int, rank: int, world: int, mirror: bool) -> Tuple[int, int]:
    """Planes [z0, z1) owned by `rank` (possibly empty: z0 == z1).  mirror = False: a balanced contiguous split of
    [0, nz).  mirror = True: a balanced contiguous split of the LOWER half [0, ceil(nz / 2)); the rank also owns the
    mirror images [nz - z1, nz - z0) (the middle plane of an odd nz, its own image, once).  Boundaries are even
    numbers where possible so that the kernels' pairing of consecutive planes is the same as in the unsharded call."""
    if nz < 1 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad shard request")
    total = (nz + 1) // 2 if mirror else nz
    def cut(i):
        c = (total * i) // world
        c -= c % 2 if 0 < i < world else 0
        return min(max(c, 0), total)
    return cut(rank), cut(rank + 1)


def owned_planes(nz: int, rank: int, world: int, mirror: bool) -> List[int]:
    """All plane indices `rank` owns, in the order its slab buffer stores them (cbct_bp_*_slab layout)."""
    z0, z1 = plane_shard(nz, rank, world, mirror)
    planes = list(range(z0, z1))
    if mirror and z1 > z0:
        skip = 1 if nz - z1 < z1 else 0
        planes += list(range(nz - z1 + skip, nz - z0))
    return planes


def assemble_views(blocks, n_views: int):
    """blocks[r][C, m_pad, nv, nu] (rank r's rows, views r, r + W, ..., zero-padded to m_pad) -> the sinogram
    [C, n_views, nv, nu] in view order.  Pure data movement (a permuted copy)."""
    import torch
    world = len(blocks)
    C, m_pad = blocks[0].shape[0], blocks[0].shape[1]
    stacked = torch.stack(list(blocks), dim=2)                       # [C, m_pad, W, nv, nu]: view = k W + r
    full = stacked.reshape(C, m_pad * world, *blocks[0].shape[2:])
    return full[:, :n_views].contiguous()


# ---------------------------------------------------------------------------------------------------------------
# channel split (no collective)
# ---------------------------------------------------------------------------------------------------------------
def channel_split(geom, op: str, src, dst, channels: int, rank: int, world: int, stream=None) -> Tuple[int, int]:
    """Run `op` ('fp', 'bp_adjoint', 'bp_fdk') of `geom` on this rank's share of the `channels` channels of the
    batch: src / dst are the WHOLE batch tensors [channels, ...] (replicated or not -- only the rank's channels are
    read and written).  Returns (first_channel, count)."""
    first, count = cdist.channel_shard(channels, rank, world)
    if count:
        getattr(geom, op)(src[first:first + count], dst[first:first + count], count, stream=stream)
    return first, count


# ---------------------------------------------------------------------------------------------------------------
# view-sharded forward / plane-sharded backprojection
# ---------------------------------------------------------------------------------------------------------------
class ShardedGeometry:
    """The handles of one rank: a strided-view handle for the forward projector and a full-view handle for the
    plane ranges of the backprojectors.  `geom_kwargs` are the keyword arguments of `cbct.Geometry` for the WHOLE
    geometry (angles_rad optional)."""

    def __init__(self, geom_kwargs: dict, rank: int, world: int, group=None, max_workset_bytes: int = 0):
        from . import cbct
        kw = dict(geom_kwargs)
        n = int(kw["n_views"])
        ang = kw.pop("angles_rad", None)
        if ang is None:
            ang = [2.0 * np.pi * i / n for i in range(n)]     # the library's own default, same expression
        self.rank, self.world, self.group = rank, world, group
        self.n_views = n
        self.my_views = view_shard(n, rank, world)
        self.m_pad = views_per_rank_padded(n, world)
        self.full = cbct.Geometry(**kw, angles_rad=list(ang), max_workset_bytes=max_workset_bytes)
        self.part = None
        if self.my_views:
            self.part = cbct.Geometry(**dict(kw, n_views=len(self.my_views)), angles_rad=[ang[i] for i in self.my_views],
                                      max_workset_bytes=max_workset_bytes)
        nz = int(kw["vol_nz"])
        _, mirror = self.full.symmetry()
        self.mirror = bool(mirror) and nz > 1
        self.z0, self.z1 = plane_shard(nz, rank, world, self.mirror)
        self.planes = owned_planes(nz, rank, world, self.mirror)
        self.vol_shape, self.sino_shape = self.full.vol_shape, self.full.sino_shape

    # --- forward: this rank's rows, then the exchange step ---------------------------------------------------
    def fp_local(self, vol, channels: int, out=None, stream=None):
        """This rank's rows of P vol: out[C, m_pad, nv, nu] (rows beyond the rank's view count stay zero)."""
        import torch
        nv, nu = self.sino_shape[1:]
        if out is None:
            out = torch.zeros((channels, self.m_pad, nv, nu), device=vol.device, dtype=torch.float32)
        m = len(self.my_views)
        if m == self.m_pad:
            if m:
                self.part.fp(vol, out, channels, stream=stream)
        elif m:
            tmp = torch.empty((channels, m, nv, nu), device=vol.device, dtype=torch.float32)
            self.part.fp(vol, tmp, channels, stream=stream)
            out[:, :m].copy_(tmp)
        return out

    def gather_sinogram(self, local):
        """The one exchange step of a forward / backprojection pair: all-gather of the ranks' rows, reassembled in
        view order on every rank."""
        import torch
        import torch.distributed as dist
        if self.world == 1:
            return assemble_views([local], self.n_views)
        # output = the ranks' blocks concatenated along axis 0 (the layout both NCCL and gloo accept)
        gathered = torch.empty((self.world * local.shape[0],) + tuple(local.shape[1:]), device=local.device, dtype=local.dtype)
        dist.all_gather_into_tensor(gathered, local.contiguous(), group=self.group)
        return assemble_views(list(gathered.view((self.world,) + tuple(local.shape)).unbind(0)), self.n_views)

    def fp(self, vol, channels: int, stream=None):
        """P vol on every rank (replicated volume in, replicated sinogram out): local rows + all-gather."""
        return self.gather_sinogram(self.fp_local(vol, channels, stream=stream))

    # --- backprojection: this rank's planes ---------------------------------------------------------------------
    def _bp_local(self, which: str, sino, channels: int, out=None, stream=None):
        import torch
        ny, nx = self.vol_shape[1:]
        n = len(self.planes)
        if out is None:
            out = torch.empty((channels, n, ny, nx), device=sino.device, dtype=torch.float32)
        if n:
            fn = self.full.bp_adjoint_slab if which == "adjoint" else self.full.bp_fdk_slab
            fn(sino, out, self.z0, self.z1, channels, mirror_pair=self.mirror, stream=stream)
        return out

    def bp_adjoint_local(self, sino, channels: int, out=None, stream=None):
        """Planes `self.planes` of P^T sino (the whole sinogram in): out[C, len(planes), ny, nx]."""
        return self._bp_local("adjoint", sino, channels, out, stream)

    def bp_fdk_local(self, sino, channels: int, out=None, stream=None):
        return self._bp_local("fdk", sino, channels, out, stream)

    def gather_volume(self, local, channels: int):
        """Replicate a plane-sharded volume on every rank (needed before the NEXT view-sharded forward projection
        if nothing else -- e.g. a plane-sharded network block -- sits in between): all-gather of the padded shards."""
        import torch
        import torch.distributed as dist
        nz, ny, nx = self.vol_shape
        counts = [len(owned_planes(nz, r, self.world, self.mirror)) for r in range(self.world)]
        pad = max(counts)
        mine = torch.zeros((channels, pad, ny, nx), device=local.device, dtype=local.dtype)
        mine[:, :counts[self.rank]].copy_(local)
        if self.world == 1:
            shards = [mine]
        else:
            gathered = torch.empty((self.world * mine.shape[0],) + tuple(mine.shape[1:]), device=local.device, dtype=local.dtype)
            dist.all_gather_into_tensor(gathered, mine, group=self.group)
            shards = list(gathered.view((self.world,) + tuple(mine.shape)).unbind(0))
        return scatter_planes(shards, nz, self.world, self.mirror)


def scatter_planes(shards: Sequence, nz: int, world: int, mirror: bool):
    """shards[r][C, >= len(owned_planes(r)), ny, nx] -> the volume [C, nz, ny, nx]."""
    import torch
    C, _, ny, nx = shards[0].shape
    vol = torch.empty((C, nz, ny, nx), device=shards[0].device, dtype=shards[0].dtype)
    for r in range(world):
        planes = owned_planes(nz, r, world, mirror)
        if planes:
            vol[:, torch.as_tensor(planes, device=vol.device)] = shards[r][:, :len(planes)]
    return vol
