"""world_size-2 gloo test (CPU) of the sink-sharded multi-GPU plumbing: each rank evaluates its
slice of the sinks (with the oracle standing in for the kernels, which need a GPU), the
accelerations are all-gathered, the gradient pass runs on the slice, and the assembled result
must equal the single-process result bit for bit."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2210_02472_b200 import sharding


def test_sink_slices_partition():
    for n in (0, 1, 7, 1024, 1000003):
        for world in (1, 2, 3, 8):
            edges = [sharding.sink_slice(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [e - b for b, e in edges]
            assert max(sizes) - min(sizes) <= 1 and sizes == sharding.slice_counts(n, world)


def _worker(rank, world, port, n, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    rng = np.random.default_rng(123)
    pos = rng.normal(size=(n, 3))
    mass = rng.uniform(0.5, 1.5, n) / n
    b, e = sharding.sink_slice(n, rank, world)
    sinks = np.arange(b, e, dtype=np.int32)
    a_loc = torch.from_numpy(oracle.acc(pos, mass, 1.0, 1e-3, sink_idx=sinks))
    a_full = sharding.allgather_rows(a_loc, n)                      # the path's only exchange
    c_loc = torch.from_numpy(oracle.grad(pos, mass, a_full.numpy(), 1.0, 1e-3, sink_idx=sinks))
    c_full = sharding.allgather_rows(c_loc, n)
    if rank == 0:
        ret["a"], ret["c"] = a_full.numpy().copy(), c_full.numpy().copy()
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sink_sharding_matches_single_process():
    import oracle
    n = 333                                                         # odd: unequal slices
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, n, ret), nprocs=2, join=True)
    rng = np.random.default_rng(123)
    pos = rng.normal(size=(n, 3))
    mass = rng.uniform(0.5, 1.5, n) / n
    a = oracle.acc(pos, mass, 1.0, 1e-3)
    c = oracle.grad(pos, mass, a, 1.0, 1e-3)
    assert np.array_equal(ret["a"], a) and np.array_equal(ret["c"], c)


# ---- pair sharding (Context.set_shard): every rank holds a partial sum for every particle, one all-reduce ----------

def test_pair_block_owner_snake_is_balanced():
    for world in (1, 2, 3, 8):
        for nb in (1, 5, 64, 683):
            owners = [sharding.pair_block_owner(b, world) for b in range(nb)]
            assert all(0 <= o < world for o in owners)
            work = [0] * world                                   # block b pairs with nb - b blocks (itself included)
            for b, o in enumerate(owners):
                work[o] += nb - b
            assert max(work) - min(work) <= max(world, nb % (2 * world) * world)   # no rank is a whole column ahead
            if nb % (2 * world) == 0:
                assert max(work) == min(work)                    # whole snakes: exactly equal shares


def _pair_worker(rank, world, port, n, bs, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    rng = np.random.default_rng(321)
    pos = rng.normal(size=(n, 3))
    mass = rng.uniform(0.5, 1.5, n) / n
    blk = np.arange(n) // bs
    nb = int(blk.max()) + 1
    own = np.array([sharding.pair_block_owner(b, world) for b in range(nb)])
    # the rank's partial sums, with the oracle standing in for the kernels: particle k in block B receives the pairs
    # with every particle of blocks >= B if this rank owns B, and with the particles of earlier blocks this rank owns
    part = np.zeros((n, 3))
    for B in range(nb):
        sinks = np.flatnonzero(blk == B).astype(np.int32)
        srcs = np.flatnonzero(((blk >= B) & (own[B] == rank)) | ((blk < B) & (own[blk] == rank))).astype(np.int32)
        if srcs.size:
            part[sinks] = oracle.acc(pos, mass, 1.0, 1e-3, sink_idx=sinks, src_idx=srcs)
    total = sharding.allreduce_sum(torch.from_numpy(part))       # the path's exchange in this mode
    if rank == 0:
        ret["a"] = total.numpy().copy()
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_pair_sharding_sums_to_the_full_result():
    import oracle
    n, bs = 301, 16
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_pair_worker, args=(2, port, n, bs, ret), nprocs=2, join=True)
    rng = np.random.default_rng(321)
    pos = rng.normal(size=(n, 3))
    mass = rng.uniform(0.5, 1.5, n) / n
    a = oracle.acc(pos, mass, 1.0, 1e-3)
    assert np.abs(ret["a"] - a).max() <= 1e-13 * np.abs(a).max()


class _OracleContext:
    """Stands in for binding.Context on CPU (the kernels need a GPU): the same calls, answered by the oracle with the
    pair-sharding rule of the symmetric kernels (blocks of `bs` list positions, snake ownership)."""

    def __init__(self, bs=32):
        self.bs, self.rank, self.world = bs, 0, 1

    def set_shard(self, rank, world):
        self.rank, self.world = rank, world

    def _partial(self, fn, n):
        blk = np.arange(n) // self.bs
        own = np.array([sharding.pair_block_owner(b, self.world) for b in range(int(blk.max()) + 1)])
        part = np.zeros((n, 3))
        for B in range(own.size):
            sinks = np.flatnonzero(blk == B).astype(np.int32)
            srcs = np.flatnonzero(((blk >= B) & (own[B] == self.rank)) | ((blk < B) & (own[blk] == self.rank))).astype(np.int32)
            if srcs.size:
                part[sinks] = fn(sinks, srcs)
        return part

    def acc(self, pos, mass, G, eps, out=None):
        import oracle
        p, m = pos.numpy(), mass.numpy()
        out.copy_(torch.from_numpy(self._partial(lambda si, sj: oracle.acc(p, m, G, eps, si, sj), m.shape[0])))
        return out

    def grad(self, pos, mass, acc, G, eps, out=None):
        import oracle
        p, m, a = pos.numpy(), mass.numpy(), acc.numpy()
        out.copy_(torch.from_numpy(self._partial(lambda si, sj: oracle.grad(p, m, a, G, eps, si, sj), m.shape[0])))
        return out

    def dtmin(self, pos, vel, mass, G, eta_ff, eta_fb, sink_idx, src_idx, out=None):
        import oracle
        si = sink_idx.numpy()
        r = oracle.dtmin(pos.numpy(), vel.numpy(), mass.numpy(), G, eta_ff, eta_fb, sink_idx=si)
        for t, key in zip(out, ("dt_ff", "dt_fb", "j_ff", "j_fb")):
            t[torch.from_numpy(si.astype(np.int64))] = torch.from_numpy(r[key])
        return out


def _force_worker(rank, world, port, n, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(55)
    pos, vel = torch.from_numpy(rng.normal(size=(n, 3))), torch.from_numpy(rng.normal(size=(n, 3)))
    mass = torch.from_numpy(rng.uniform(0.5, 1.5, n) / n)
    ctx = _OracleContext()
    ctx.set_shard(rank, world)
    acc, grad = torch.zeros((n, 3), dtype=torch.float64), torch.zeros((n, 3), dtype=torch.float64)
    sharding.sharded_force(ctx, pos, mass, 1.0, 1e-3, acc, grad)
    dts = (torch.full((n,), np.inf, dtype=torch.float64), torch.full((n,), np.inf, dtype=torch.float64),
           torch.full((n,), -1, dtype=torch.int32), torch.full((n,), -1, dtype=torch.int32))
    sharding.sharded_dtmin(ctx, pos, vel, mass, 1.0, 0.02, 0.03, dts)
    ret[rank] = [t.numpy().copy() for t in (acc, grad, *dts)]
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_force_and_dtmin_control_flow_with_a_stub_context():
    """The multi-rank step bench.py times (pair-sharded acc / grad with an all-reduce each, sink-sharded dtmin with
    padded all-gathers, n not a multiple of the world size) on two gloo ranks, the oracle standing in for the
    kernels: every rank ends with the complete, correct arrays."""
    import oracle
    n = 203
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_force_worker, args=(2, port, n, ret), nprocs=2, join=True)
    rng = np.random.default_rng(55)
    pos, vel = rng.normal(size=(n, 3)), rng.normal(size=(n, 3))
    mass = rng.uniform(0.5, 1.5, n) / n
    a = oracle.acc(pos, mass, 1.0, 1e-3)
    for r in (0, 1):
        acc, grad, dff, dfb, jff, jfb = ret[r]
        assert np.abs(acc - a).max() <= 1e-13 * np.abs(a).max()
        c = oracle.grad(pos, mass, acc, 1.0, 1e-3)
        assert np.abs(grad - c).max() <= 1e-12 * np.abs(c).max()
        d = oracle.dtmin(pos, vel, mass, 1.0, 0.02, 0.03)
        assert np.array_equal(dff, d["dt_ff"]) and np.array_equal(dfb, d["dt_fb"])
        assert np.array_equal(jff, d["j_ff"]) and np.array_equal(jfb, d["j_fb"])
    assert all(np.array_equal(x, y) for x, y in zip(ret[0], ret[1]))      # both ranks hold the same bits
