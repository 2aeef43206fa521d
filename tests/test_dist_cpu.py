"""N > 1 plumbing on CPU: world_size-2 gloo processes exercise the rank-side logic
bench.py uses under torchrun (channel partition, max / sum over ranks, barrier)."""
import os
import socket

import pytest

from paper_2512_21180_b200 import dist as cdist

torch = pytest.importorskip("torch")


def test_channel_shard_partitions():
    for channels in (0, 1, 4, 5, 8, 13):
        for world in (1, 2, 3, 8):
            seen = []
            for rank in range(world):
                first, count = cdist.channel_shard(channels, rank, world)
                seen += list(range(first, first + count))
            assert seen == list(range(channels))
            counts = [cdist.channel_shard(channels, r, world)[1] for r in range(world)]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        cdist.channel_shard(4, 2, 2)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert cdist.env_world() == (rank, rank, world)
        first, count = cdist.channel_shard(5, rank, world)
        # each rank "times" its shard: the job time is the max, the work the sum
        t = cdist.max_over_ranks([10.0 + rank, 3.0 - rank])
        w = cdist.sum_over_ranks([float(count), float(first)])
        cdist.barrier()
        out.put((rank, t, w))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_reductions():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, w in res:
        assert t == [11.0, 3.0]      # max over ranks, element-wise
        assert w == [5.0, 3.0]       # 3 + 2 channels; firsts 0 + 3


# ---------------------------------------------------------------------------------------------------------------
# sharded.py: partition arithmetic and the exchange step under world_size-2 gloo
# ---------------------------------------------------------------------------------------------------------------
def test_view_and_plane_partitions_tile_exactly():
    from paper_2512_21180_b200 import sharded
    for n_views in (1, 7, 400, 402, 720):
        for world in (1, 2, 3, 8):
            seen = sorted(v for r in range(world) for v in sharded.view_shard(n_views, r, world))
            assert seen == list(range(n_views))
            assert max(len(sharded.view_shard(n_views, r, world)) for r in range(world)) == \
                sharded.views_per_rank_padded(n_views, world)
    for nz in (1, 2, 27, 32, 255, 256):
        for world in (1, 2, 3, 8):
            for mirror in (False, True):
                seen = sorted(z for r in range(world) for z in sharded.owned_planes(nz, r, world, mirror))
                assert seen == list(range(nz)), (nz, world, mirror, seen)
                for r in range(world):
                    z0, z1 = sharded.plane_shard(nz, r, world, mirror)
                    assert 0 <= z0 <= z1 <= ((nz + 1) // 2 if mirror else nz)
    # a strided share of equispaced views keeps the quarter-turn symmetry when n / world is a multiple of 4
    mine = sharded.view_shard(400, 1, 2)
    assert len(mine) % 4 == 0 and all(mine[k + len(mine) // 4] - mine[k] == 100 for k in range(len(mine) // 4))


def _sharded_worker(rank, world, port, out):
    import numpy as np
    import torch.distributed as dist
    from paper_2512_21180_b200 import sharded
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        C, n_views, nv, nu, nz, ny, nx = 3, 9, 4, 5, 7, 3, 4
        full_s = torch.arange(C * n_views * nv * nu, dtype=torch.float32).reshape(C, n_views, nv, nu)
        full_v = torch.arange(C * nz * ny * nx, dtype=torch.float32).reshape(C, nz, ny, nx) + 0.5

        class Fake(sharded.ShardedGeometry):           # the collectives and the reassembly, without a GPU library
            def __init__(self):
                self.rank, self.world, self.group, self.n_views = rank, world, None, n_views
                self.my_views = sharded.view_shard(n_views, rank, world)
                self.m_pad = sharded.views_per_rank_padded(n_views, world)
                self.mirror = True
                self.vol_shape, self.sino_shape = (nz, ny, nx), (n_views, nv, nu)
                self.z0, self.z1 = sharded.plane_shard(nz, rank, world, True)
                self.planes = sharded.owned_planes(nz, rank, world, True)
        sg = Fake()
        local = torch.zeros((C, sg.m_pad, nv, nu))
        local[:, :len(sg.my_views)] = full_s[:, sg.my_views]          # "this rank's rows of P vol"
        got_s = sg.gather_sinogram(local)
        shard = full_v[:, sg.planes].contiguous()                      # "this rank's planes of P^T y"
        got_v = sg.gather_volume(shard, C)
        first, count = sharded.cdist.channel_shard(C, rank, world)
        out.put((rank, bool(torch.equal(got_s, full_s)), bool(torch.equal(got_v, full_v)), first, count))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_exchange_reassembles_sinogram_and_volume():
    """Every row of the gathered sinogram and every plane of the gathered volume exactly once, in place, on both
    ranks (uneven shares: 9 views and 7 planes over 2 ranks, z-mirror pairs with a middle plane)."""
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_sharded_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1:3] for r in res] == [(True, True), (True, True)]
    assert [(r[3], r[4]) for r in res] == [(0, 2), (2, 1)]
