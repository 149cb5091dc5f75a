"""Multi-GPU plumbing for the sink-sharded path.

Every sink's result is an independent reduction over the sources, so the path shards over
SINKS: each rank holds all particles, evaluates its contiguous slice of the sink list, and the
only exchange is one all-gather of the accelerations (24 B x N) between the acceleration pass
and the gradient pass, because Eq. 9/13 need a_j of every source.  The paper
itself scales this way with MPI.  This module holds only that host logic; it
works on any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import List, Tuple


def sink_slice(n_sink: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of rank's contiguous share of n_sink sinks (sizes differ by at most 1)."""
    base, rem = divmod(n_sink, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def slice_counts(n_sink: int, world: int) -> List[int]:
    return [sink_slice(n_sink, r, world)[1] - sink_slice(n_sink, r, world)[0] for r in range(world)]


def allgather_rows(local_rows, n_total: int, group=None):
    """All-gather row blocks of unequal length along dim 0: rank r contributes the rows of
    sink_slice(n_total, r, world); every rank returns the full [n_total, ...] tensor."""
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    counts = slice_counts(n_total, world)
    rank = dist.get_rank(group)
    assert local_rows.shape[0] == counts[rank]
    tail = tuple(local_rows.shape[1:])
    if len(set(counts)) == 1:
        full = torch.empty((n_total,) + tail, dtype=local_rows.dtype, device=local_rows.device)
        dist.all_gather_into_tensor(full, local_rows.contiguous(), group=group)
        return full
    # unequal slices: pad every contribution to the longest slice, gather, strip the padding
    cmax = max(counts)
    padded = torch.zeros((cmax,) + tail, dtype=local_rows.dtype, device=local_rows.device)
    padded[: counts[rank]] = local_rows
    gathered = torch.empty((world * cmax,) + tail, dtype=local_rows.dtype, device=local_rows.device)
    dist.all_gather_into_tensor(gathered, padded, group=group)
    return torch.cat([gathered[r * cmax: r * cmax + counts[r]] for r in range(world)], dim=0)
