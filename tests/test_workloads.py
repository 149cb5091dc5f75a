"""Checks of the seeded synthetic input generators (CPU only): distributions the
recipes in DESIGN.md promise, and determinism."""
import numpy as np

from conftest import workload
from paper_2210_02472_b200 import workloads as W


def test_kroupa_imf_statistics():
    """Two-segment Kroupa IMF on [0.08, 100] Msun (reading C4): 76.07 % of stars below
    0.5 Msun, mean mass 0.57386 Msun, 1.176 % above 5 Msun (analytic values)."""
    m = W.kroupa_masses(np.random.default_rng(0), 2_000_000)
    assert m.min() >= 0.08 and m.max() <= 100.0
    assert abs((m < 0.5).mean() - 0.7607) < 2e-3
    assert abs(m.mean() / 0.57386 - 1) < 0.02
    assert abs((m > 5).mean() - 0.01176) < 5e-4


def test_plummer_phase_space_statistics():
    """Half-mass radius r_h = 1.30477 a_p; <v^2> = 3 pi / 32 G M / a_p."""
    pos, vel = W.plummer_phase_space(np.random.default_rng(1), 400_000)
    r = np.linalg.norm(pos, axis=1)
    assert abs(np.median(r) / W.R_HALF - 1) < 0.01
    assert r.max() <= 100.0 * (1 + 1e-12)
    assert abs((vel ** 2).sum(axis=1).mean() / (3 * np.pi / 32) - 1) < 0.01
    # speeds never exceed the local escape speed
    vesc2 = 2.0 / np.sqrt(1 + r * r)
    assert ((vel ** 2).sum(axis=1) <= vesc2 * (1 + 1e-12)).all()
    assert np.abs(pos.mean(axis=0)).max() < 0.05


def test_kepler_solver_residual():
    rng = np.random.default_rng(2)
    M = rng.uniform(0, 2 * np.pi, 100000)
    e = np.minimum(np.sqrt(rng.uniform(0, 1, 100000)), 0.999)
    E = W._kepler_E(M, e)
    assert np.abs(E - e * np.sin(E) - M).max() < 1e-12


def test_configs_shapes_and_determinism():
    w1 = W.config1()
    assert w1.n == 1024 and w1.pos.shape == (1024, 3) and np.all(w1.mass == 1.0 / 1024) and w1.eps == 1e-4
    assert np.array_equal(w1.pos, W.config1().pos)
    w3 = workload(3)
    assert w3.n == 131072 and w3.eps == 0.0 and abs(w3.mass.sum() - 1) < 1e-12
    # N/4 binaries: that many particles have a neighbour far closer than the mean spacing
    sub = np.random.default_rng(0).choice(w3.n, 2000, replace=False)
    d = np.linalg.norm(w3.pos[sub, None, :] - w3.pos[None, :, :], axis=2)
    d[np.arange(2000), sub] = np.inf
    # (binaries with a < 1e-3 r_h are half of the log-uniform range; chance neighbours are ~1e-3)
    frac_close = (d.min(axis=1) < 2.0 * 1e-3 * W.R_HALF).mean()
    assert 0.20 < frac_close < 0.35
    assert d.min() > 1e-4 * W.R_HALF * (1 - 0.999) * 0.99
    w4 = W.config4(n=4096)
    assert w4.mass[0] == 1e-3 and np.all(w4.pos[0] == 0) and w4.bh_idx.shape == (101,) and w4.bh_idx[0] == 0
    assert abs(w4.mass.sum() - 1) < 1e-12 and w4.c == 1e4 and w4.eps == 0.0
    assert len(set(w4.bh_idx.tolist())) == 101
    ratio = w4.mass[w4.bh_idx[1:]] / np.median(w4.mass)
    assert ratio.min() > 10
    for k in range(0, 15):
        s = W.config2_sink_list(k)
        assert s.shape == (2 ** k,) and s.dtype == np.int32 and np.all(np.diff(s) > 0) and s.max() < 16384
    assert W.config3_sink_list(10).shape == (128,) and W.config3_sink_list(0).shape == (131072,)


def test_config2_is_virialised():
    w = workload(2)
    assert w.n == 16384 and abs(w.mass.sum() - 1) < 1e-12
    t = 0.5 * (w.mass * (w.vel ** 2).sum(axis=1)).sum()
    pot = W._virial_potential_energy(w.pos, w.mass)
    assert abs(2 * t / -pot - 1) < 1e-12
    assert np.abs((w.mass[:, None] * w.vel).sum(axis=0)).max() < 1e-15
