"""Host-side multi-GPU bookkeeping: the path shards along `batch` only (independent wavelengths /
realisations) -- contiguous slices per rank, no collective during propagation.  The only
communication is the timing reduction (max over ranks) that bench.py reports and, when a broadband image is
wanted, one sum all-reduce of the N x N intensity image at the very end (reduce_image); both work with any
torch.distributed backend (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

from typing import Tuple


def shard_batch(batch_total: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [start, stop) slice of the batch owned by `rank`; sizes differ by at most one."""
    if world <= 0 or not (0 <= rank < world) or batch_total < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(batch_total, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def max_over_ranks(values, device=None):
    """Element-wise max of a list of floats over all ranks (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def sum_over_ranks(values, device=None):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t]


def reduce_image(image):
    """Finish a broadband image whose wavelengths are sharded over ranks: every
    rank has accumulated sum_b w_b |U_b|^2 over ITS slice of the batch with fresnel_accumulate_intensity; one
    sum all-reduce of the N x N real image (NCCL over NVLink on GPUs, gloo in the CPU tests) gives every
    rank the full image.  In place; identity when not distributed.  This is the path's only data collective."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(image, op=dist.ReduceOp.SUM)
    return image


def whole_job_rate(units_this_rank: float, seconds_this_rank: float, device=None) -> float:
    """Throughput of the whole job: all ranks' units / the slowest rank's time."""
    total = sum_over_ranks([units_this_rank], device)[0]
    slowest = max_over_ranks([seconds_this_rank], device)[0]
    return total / slowest


def sharded_polychromatic_image(make_plan, wavefront_of, dx, lam, weights, run_train, new_image, rank: int, world: int):
    """The multi-GPU data path of a broadband image (PAPER.md:51 "repeated for all of the wavelengths", :63 one process
    per wavelength): the `len(lam)` wavelengths are split into contiguous slices, one per rank;
    every rank propagates ITS wavelengths through the train, accumulates sum_b w_b |U_b|^2 over them
    (fresnel_accumulate_intensity) and ONE sum all-reduce of the N x N image finishes the job on every rank.  No
    communication happens during propagation.

    The caller supplies the pieces that touch the device, so the same code runs on GPUs (bench.py, NCCL) and in the
    CPU test with the library stubbed out at the Plan boundary (gloo):
        make_plan(batch_local)            -> plan with .accumulate_intensity(wf, weights, image)
        wavefront_of(lo, hi)              -> this rank's wavefronts [hi-lo][N][N] (device tensor)
        run_train(plan, wf, dx_l, lam_l)  -> propagate in place (e.g. plan.system_run)
        new_image()                       -> zeroed real [N][N] tensor on the device
    Returns (image, (lo, hi), plan, wf)."""
    lo, hi = shard_batch(len(lam), rank, world)
    if hi == lo:
        raise ValueError(f"rank {rank}: no wavelength left ({len(lam)} wavelengths over {world} ranks)")
    plan = make_plan(hi - lo)
    wf = wavefront_of(lo, hi)
    run_train(plan, wf, dx[lo:hi], lam[lo:hi])
    image = new_image()
    plan.accumulate_intensity(wf, weights[lo:hi], image)
    reduce_image(image)
    return image, (lo, hi), plan, wf
