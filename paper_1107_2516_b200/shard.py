"""Host-side logic of the multi-GPU path (one process per GPU, no data-path collective).

The paper splits the DM list across GPUs, every GPU working on the same input buffer
(PAPER.md:74, :78); beams are the other independent axis (BASELINE.json cfg 5).  Neither needs an
exchange step, so the only collectives are the barrier and the max-over-ranks of the device time
that bench.py reports.  This module holds no arithmetic of the method.
"""
import numpy as np


def dm_slice(ndm, world, rank, multiple=1):
    """Contiguous DM-trial range [lo, hi) of `rank`: ranges are disjoint, cover [0, ndm) in rank
    order and differ in length by at most `multiple` (subband plans pass nfine so that coarse
    groups stay whole)."""
    if world <= 0 or not 0 <= rank < world or ndm < 0 or multiple <= 0 or ndm % multiple:
        raise ValueError("bad shard arguments")
    units = ndm // multiple
    base, extra = divmod(units, world)
    lo = rank * base + min(rank, extra)
    hi = lo + base + (1 if rank < extra else 0)
    return lo * multiple, hi * multiple


def beam_of(rank, nbeams_per_rank, b):
    """Global beam index of local beam b on `rank` (weak scaling: every rank has its own beams)."""
    return rank * nbeams_per_rank + b


def max_over_ranks(value, dist=None, device="cpu"):
    """Max of a scalar over all ranks (the contract's timing rule); identity without a group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, dist=None, device="cpu"):
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_this_rank, ms_this_rank, dist=None, device="cpu"):
    """Whole-job units per second: units of all ranks / max over ranks of the device time."""
    total = sum_over_ranks(units_this_rank, dist, device)
    ms = max_over_ranks(ms_this_rank, dist, device)
    return total / (ms * 1e-3), ms


def gather_rows(local_rows, dist=None):
    """All ranks' DM rows in rank order (CPU tensors / arrays; used by tests and by callers that
    want the full [ndm][n] array on every rank -- the product path leaves outputs sharded)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return np.asarray(local_rows)
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, np.asarray(local_rows))
    return np.concatenate(parts, axis=0)
