"""oracle/cpu_fast.c (bench.py's `cpu_fast` timing baseline) is pinned TO the parity oracle: same sums
within 1e-12, self pair dropped by id, index lists honoured.  CPU only."""
import numpy as np

import oracle
from conftest import normwise_rel_err, workload
from oracle import cpu_fast


def test_cpu_fast_matches_the_oracle():
    w = workload(2)
    rng = np.random.default_rng(1)
    sinks = np.sort(rng.choice(w.n, 300, replace=False)).astype(np.int32)
    srcs = rng.permutation(w.n)[: w.n - 100].astype(np.int32)
    for eps in (0.0, 1e-3):
        for si, sj in ((sinks, None), (sinks, srcs)):
            a = cpu_fast.acc(w.pos, w.mass, w.G, eps, si, sj)
            a_ref = oracle.acc(w.pos, w.mass, w.G, eps, si, sj)
            assert np.isfinite(a).all() and (normwise_rel_err(a, a_ref) <= 1e-12).all()
            a_full = oracle.acc(w.pos, w.mass, w.G, eps)
            c = cpu_fast.grad(w.pos, w.mass, a_full, w.G, eps, si, sj)
            c_ref = oracle.grad(w.pos, w.mass, a_full, w.G, eps, si, sj)
            assert np.isfinite(c).all() and (normwise_rel_err(c, c_ref) <= 1e-12).all()


def test_cpu_fast_small_all_active_and_self_pair():
    w = workload(1)
    a = cpu_fast.acc(w.pos, w.mass, w.G, 0.0)
    assert (normwise_rel_err(a, oracle.acc(w.pos, w.mass, w.G, 0.0)) <= 1e-12).all()
    tot = np.abs((w.mass[:, None] * a).sum(0))
    assert (tot <= 1e-13 * (w.mass[:, None] * np.abs(a)).sum(0)).all()
