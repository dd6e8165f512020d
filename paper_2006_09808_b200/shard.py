"""Batch sharding for more than one GPU: one process per GPU, one plan per process, NO data-path collective.

Slices and coil field maps are independent ("the tasks of different slices are irrelevant, there is no data
dependency among them"), so a stack is split contiguously over the ranks and every rank runs pd_solve on its own part.
The only communication is the scalar bookkeeping of a benchmark or a caller that wants global statistics
(max of a time, sum of slice-iterations), done with torch.distributed on whatever backend the group uses
(nccl on GPUs, gloo in the CPU tests).  This module holds host logic only; it never touches the solver's arithmetic.
"""


def shard_bounds(batch, rank, world):
    """Contiguous [lo, hi) of `batch` entries owned by `rank` of `world`; sizes differ by at most one, in rank order."""
    if world < 1 or not (0 <= rank < world) or batch < 0:
        raise ValueError("bad shard request: batch=%r rank=%r world=%r" % (batch, rank, world))
    base, rem = divmod(batch, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def weak_first_slice(nslices_per_rank, rank):
    """Weak scaling (bench.py): rank r reconstructs its own stack, slices [r*n, (r+1)*n) of the synthetic generator."""
    return rank * nslices_per_rank


def _reduce(value, op, device):
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(value, device="cpu"):
    """Max of a per-rank scalar (device time of the timed region: the job is as slow as its slowest rank)."""
    import torch.distributed as dist
    return _reduce(value, dist.ReduceOp.MAX, device)


def sum_over_ranks(value, device="cpu"):
    """Sum of a per-rank scalar (slice-iterations done: whole-job throughput = sum / max time)."""
    import torch.distributed as dist
    return _reduce(value, dist.ReduceOp.SUM, device)


def job_throughput(units_local, ms_local, device="cpu"):
    """Whole-job units/s of a sharded run: all ranks' units divided by the slowest rank's time."""
    units = sum_over_ranks(units_local, device)
    ms = max_over_ranks(ms_local, device)
    return units / (ms * 1e-3), units, ms
