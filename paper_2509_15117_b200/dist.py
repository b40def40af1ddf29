"""Multi-GPU plumbing (one process per GPU, torch.distributed).

Trajectories are independent (the paper's eight K80s ran independent batches), so the path
shards by contiguous index ranges with NO data-path collective: every rank runs its own persistent
kernel with its own work counter on ``first_index + [0, n)``; the only exchange is the sum of the
~0.5 KB ensemble summaries and the max of the device times, done once after the timed region.
Host logic only -- nothing here computes the method.
"""
from __future__ import annotations

import dataclasses
from typing import Tuple

import numpy as np


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [first, first+count) of `rank`: no overlap, no gap, sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("need 0 <= rank < world")
    base, rem = divmod(int(n), world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def shard_launch(launch, rank: int, world: int):
    """The rank's share of a GRID / PHILOX launch (a dataclass with n and first_index): the generator is
    counter-based (index -> initial condition), so a shard is just another index range."""
    first, count = shard_range(launch.n, rank, world)
    return dataclasses.replace(launch, n=count, first_index=launch.first_index + first)


_SUM_FIELDS = ("n_done", "n_status", "n_complex", "steps_acc", "steps_rej", "steps_loc", "sum_ke", "sum_ke2",
               "hist_ncoll", "hist_tlife", "slots_bulk", "n_handoff", "steps_coop", "steps_kernel")


def summary_to_vector(summary) -> np.ndarray:
    """Additive fields of an ia_summary as one float64 vector (counts < 2^53 are exact in float64)."""
    return np.concatenate([np.atleast_1d(np.asarray(summary[f], dtype=np.float64)).ravel() for f in _SUM_FIELDS])


def vector_to_dict(vec: np.ndarray, like) -> dict:
    out, k = {}, 0
    for f in _SUM_FIELDS:
        size = int(np.atleast_1d(like[f]).size)
        chunk = vec[k:k + size]
        k += size
        if f in ("sum_ke", "sum_ke2"):
            out[f] = float(chunk[0])
        elif size == 1:
            out[f] = int(round(chunk[0]))
        else:
            out[f] = [int(round(c)) for c in chunk]
    return out


def all_reduce_summary(summary, device=None) -> dict:
    """Sum of the ranks' summaries (a dict), via one all_reduce of ~45 doubles; identity when not distributed."""
    import torch
    import torch.distributed as dist
    vec = summary_to_vector(summary)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.from_numpy(vec.copy())
        if device is not None:
            t = t.to(device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        vec = t.cpu().numpy()
    return vector_to_dict(vec, summary)


def all_reduce_max(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([float(value)], dtype=torch.float64)
        if device is not None:
            t = t.to(device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())
    return float(value)


def all_reduce_sum(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([float(value)], dtype=torch.float64)
        if device is not None:
            t = t.to(device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())
    return float(value)


def sum_summaries(arr: np.ndarray) -> np.ndarray:
    """Field-wise sum of an array of ia_summary records (host arithmetic on counters, for reporting)."""
    out = np.zeros((), dtype=arr.dtype)
    for f in arr.dtype.names:
        out[f] = arr[f].sum(axis=0)
    return out
