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


class _StubPlan:
    """Stands in for binding.Plan at the Plan boundary only (CPU tensors): a 'train' that multiplies every wavefront by
    a wavelength-dependent unit-modulus factor and a gain, and the broadband accumulation of the C ABI."""

    def __init__(self, N, batch):
        self.N, self.batch = N, batch

    def system_run(self, wf, dx, lam, surfaces):
        for b in range(self.batch):
            wf[b] *= (1.0 + 0.1 * b + 1e6 * float(lam[b])) * torch.exp(torch.tensor(1j * 2e6 * float(lam[b])))
        return dx

    def accumulate_intensity(self, wf, weight, image):
        for b in range(self.batch):
            image += float(weight[b]) * (wf[b].real ** 2 + wf[b].imag ** 2)


def _poly_worker(rank, world, port, q):
    import numpy as np
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    if world > 1:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        N, nlam = 24, 7                                        # 7 wavelengths over 2 ranks: slices of 4 and 3
        g = torch.Generator().manual_seed(11)
        fields = torch.randn(nlam, N, N, dtype=torch.float64, generator=g) + 1j * torch.randn(nlam, N, N, dtype=torch.float64, generator=g)
        lam = np.linspace(500e-9, 600e-9, nlam)
        dx = np.full(nlam, 1e-5)
        w = np.linspace(0.5, 1.5, nlam)
        # note: the stub's gain depends on the LOCAL batch index, so each slice is run the way a per-rank plan would
        img, (lo, hi), plan, wf = sharding.sharded_polychromatic_image(
            make_plan=lambda nb: _StubPlan(N, nb), wavefront_of=lambda lo, hi: fields[lo:hi].clone(), dx=dx, lam=lam, weights=w,
            run_train=lambda plan, wf, dxl, laml: plan.system_run(wf, dxl, laml, []), new_image=lambda: torch.zeros(N, N, dtype=torch.float64),
            rank=rank, world=world)
        # expected: the same slices computed in one process
        want = torch.zeros(N, N, dtype=torch.float64)
        for r in range(world):
            a, b = sharding.shard_batch(nlam, r, world)
            pl = _StubPlan(N, b - a)
            f = fields[a:b].clone()
            pl.system_run(f, dx[a:b], lam[a:b], [])
            pl.accumulate_intensity(f, w[a:b], want)
        q.put((rank, lo, hi, float((img - want).abs().max() / want.abs().max())))
    finally:
        if world > 1:
            dist.destroy_process_group()


def test_sharded_polychromatic_image_two_ranks_gloo():
    """The multi-GPU data path (shard the wavelengths, propagate, accumulate per rank, ONE sum all-reduce) with the
    library stubbed out at the Plan boundary: two gloo ranks end with the same, complete image."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_poly_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(o[1], o[2]) for o in out] == [(0, 4), (4, 7)]
    assert all(o[3] <= 1e-14 for o in out)


def test_bench_gpus_flag_starts_the_ranks_itself():
    """`python bench.py --gpus N` re-executes itself under torch.distributed.run with N ranks unless it already runs
    under torchrun (checked on the command it builds: no GPU here)."""
    import importlib.util
    import subprocess
    import sys
    from unittest import mock
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    seen = {}

    def fake_call(cmd):
        seen["cmd"] = cmd
        return 0

    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    with mock.patch.object(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "2", "--workload", "cfg5"]), \
            mock.patch.object(subprocess, "call", fake_call), mock.patch.dict(os.environ, env, clear=True):
        with pytest.raises(SystemExit) as e:
            bench.main()
    assert e.value.code == 0
    cmd = seen["cmd"]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=4" in cmd and "--master-addr" in cmd and "127.0.0.1" in cmd
    assert cmd[-6:] == ["--gpus", "4", "--steps", "2", "--workload", "cfg5"]


def test_single_process_is_identity():
    assert sharding.max_over_ranks([1.5, 2.0]) == [1.5, 2.0]
    assert sharding.whole_job_rate(20, 0.5) == 40
    t = torch.ones(4, 4)
    assert sharding.reduce_image(t) is t and bool((t == 1).all())
