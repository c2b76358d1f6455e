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
