"""Multi-GPU plumbing.

Two ways to shard, both with every rank holding all particles:
  * over SINKS (any call): disjoint sink slices per rank, results are final, one all-gather assembles them;
  * over PAIRS (all-active acc / grad through the symmetric kernels, Context.set_shard): every rank evaluates its
    blocks of the unordered pairs and produces a partial sum for EVERY particle; one all-reduce (sum) of
    double[n][3] per pass yields the result - `allreduce_sum` below.  Half the arithmetic of the sink-sharded
    form, at the price of exchanging 24 B x N per pass instead of once.

Sink sharding needs ONE exchange per force evaluation: an all-gather of the accelerations (24 B x N)
between the acceleration pass and the gradient pass, because Eq. 9/13 need a_j of every source
(PAPER.md:L99).  The paper itself scales over particles with MPI.  This module holds only
host logic; it works on any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests).
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


def pair_block_owner(b: int, world: int) -> int:
    """Rank that evaluates block b of the symmetric kernels when the pair work is sharded (mirrors sym_owner in
    csrc/sym_kernels.cuh): blocks are dealt in snake order 0 1 .. w-1, w-1 .. 1 0, ... because a block's work
    (the pairs with every later block) falls linearly with b."""
    q, r = divmod(b, world)
    return world - 1 - r if q & 1 else r


def allreduce_sum(partial, group=None):
    """In-place sum over ranks of the partial sums the pair-sharded symmetric kernels write (the path's exchange
    step in that mode); returns `partial`.  The reduction order is NCCL's (fixed for a fixed communicator)."""
    import torch.distributed as dist

    dist.all_reduce(partial, op=dist.ReduceOp.SUM, group=group)
    return partial


def sharded_force(ctx, pos, mass, G, eps, acc, grad, group=None):
    """One force evaluation of the FSI cycle - bifrost_acc, then bifrost_grad on the new accelerations -
    with the pair work sharded over the ranks of `group`.  `ctx` is this rank's Context after
    ctx.set_shard(rank, world); `acc`, `grad` are [n, 3] outputs.  Exactly what bench.py times under torchrun:
    partial sums on every rank, one all-reduce after each pass.  Returns (acc, grad), complete on every rank."""
    ctx.acc(pos, mass, G, eps, out=acc)
    allreduce_sum(acc, group)
    ctx.grad(pos, mass, acc, G, eps, out=grad)
    allreduce_sum(grad, group)
    return acc, grad


def sharded_dtmin(ctx, pos, vel, mass, G, eta_ff, eta_fb, out, group=None):
    """bifrost_dtmin sharded over SINKS: this rank evaluates its contiguous slice of the particles against all
    sources; the four result arrays are assembled with all-gathers (unequal slices are padded).  `out` =
    (dt_ff, dt_fb, j_ff, j_fb), each [n]; returns them complete on every rank."""
    import torch
    import torch.distributed as dist

    n = mass.shape[0]
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    b, e = sink_slice(n, rank, world)
    sinks = torch.arange(b, e, dtype=torch.int32, device=mass.device)
    ctx.dtmin(pos, vel, mass, G, eta_ff, eta_fb, sinks, None, out=out)
    for t in out:
        t.copy_(allgather_rows(t[b:e], n, group))
    return out
