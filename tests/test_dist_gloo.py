"""World-size-2 gloo test (CPU) of the multi-GPU bookkeeping: batch sharding and the
max-over-ranks timing reduction that bench.py reports.  The data path itself has no collective."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1806_06467_b200 import sharding


def test_shard_batch_partitions_the_batch():
    for total in (0, 1, 2, 7, 16, 33):
        for world in (1, 2, 3, 8):
            pieces = [sharding.shard_batch(total, r, world) for r in range(world)]
            assert pieces[0][0] == 0 and pieces[-1][1] == total
            for (a0, a1), (b0, b1) in zip(pieces, pieces[1:]):
                assert a1 == b0
            sizes = [b - a for a, b in pieces]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_batch(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lo, hi = sharding.shard_batch(16, rank, world)          # config-5 style: 16 wavelengths
        units = (hi - lo) * 10                                   # 10 planes each
        seconds = 0.5 + 0.25 * rank                              # rank 1 is the slow one
        rate = sharding.whole_job_rate(units, seconds)
        mx = sharding.max_over_ranks([seconds, float(rank)])
        # broadband image: every rank sums its own wavelengths, one all-reduce finishes the image
        g = torch.Generator().manual_seed(5)
        fields = torch.randn(16, 32, 32, dtype=torch.float64, generator=g)      # same on both ranks
        weights = torch.linspace(0.5, 2.0, 16, dtype=torch.float64)
        mine = (weights[lo:hi, None, None] * fields[lo:hi] ** 2).sum(0)
        full = sharding.reduce_image(mine.clone())
        img_err = float((full - (weights[:, None, None] * fields ** 2).sum(0)).abs().max())
        dist.barrier()
        q.put((rank, lo, hi, rate, mx, img_err))
    finally:
        dist.destroy_process_group()


def test_two_rank_timing_reduction_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(o[1], o[2]) for o in out] == [(0, 8), (8, 16)]
    for o in out:
        assert o[3] == pytest.approx(160 / 0.75)                 # all units / slowest rank
        assert o[4] == [0.75, 1.0]
        assert o[5] <= 1e-12                                     # sharded broadband image == unsharded


def test_single_process_is_identity():
    assert sharding.max_over_ranks([1.5, 2.0]) == [1.5, 2.0]
    assert sharding.whole_job_rate(20, 0.5) == 40
    t = torch.ones(4, 4)
    assert sharding.reduce_image(t) is t and bool((t == 1).all())
