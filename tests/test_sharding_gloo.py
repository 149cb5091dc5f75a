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
