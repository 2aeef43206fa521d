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
