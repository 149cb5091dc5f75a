"""Pins for the oracle's acceleration and gradient routines (CPU only).

Each test checks oracle/bifrost_oracle.cpp against something other than itself:
closed forms, a hand-computed fixture, invariants, finite differences, a
higher-precision instance, the Plummer model's analytic values.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from conftest import normwise_rel_err
from paper_2210_02472_b200 import workloads as W

U = 2.0 ** -53
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _random_cluster(n, seed, kroupa=True):
    rng = np.random.default_rng(seed)
    pos, vel = W.plummer_phase_space(rng, n)
    mass = W.kroupa_masses(rng, n) if kroupa else np.ones(n)
    mass /= mass.sum()
    return pos, vel, mass


# --- acc: formula, sign, softening (Eq. 6; readings A1, A2) -----------------

@pytest.mark.parametrize("eps", [0.0, 0.3, 2.0])
def test_acc_two_body_closed_form(eps):
    rng = np.random.default_rng(11)
    for _ in range(20):
        pos = rng.normal(size=(2, 3))
        mass = rng.uniform(0.1, 3.0, 2)
        G = rng.uniform(0.5, 2.0)
        a = oracle.acc(pos, mass, G, eps)
        r21 = pos[1] - pos[0]
        s2 = r21 @ r21 + eps * eps
        a0 = G * mass[1] * r21 / s2 ** 1.5          # towards particle 1 (attractive)
        a1 = -G * mass[0] * r21 / s2 ** 1.5
        assert np.allclose(a[0], a0, rtol=8 * U, atol=0)
        assert np.allclose(a[1], a1, rtol=8 * U, atol=0)
        assert (a[0] @ r21) > 0 and (a[1] @ r21) < 0


def _load_golden():
    rows = []
    for line in open(os.path.join(GOLDEN, "three_body_collinear.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        rows.append((int(t[0]), Fraction(int(t[1]), int(t[2])), Fraction(int(t[3]), int(t[4]))))
    return rows


def test_acc_grad_three_body_golden():
    """tests/golden/three_body_collinear.txt: exact rationals worked out by hand from Eq. 6 / Eq. 9."""
    pos = np.array([[0.0, 0, 0], [1.0, 0, 0], [3.0, 0, 0]])
    mass = np.array([1.0, 2.0, 3.0])
    a = oracle.acc(pos, mass, 1.0, 0.0)
    c = oracle.grad(pos, mass, a, 1.0, 0.0)
    for i, ax, cx in _load_golden():
        assert abs(a[i, 0] - float(ax)) <= 4 * U * abs(float(ax))
        assert abs(c[i, 0] - float(cx)) <= 16 * U * abs(float(cx))
        assert a[i, 1] == 0 and a[i, 2] == 0 and c[i, 1] == 0 and c[i, 2] == 0
    # the same fixture rotated into a general direction (exercises all components)
    rot = np.linalg.qr(np.random.default_rng(3).normal(size=(3, 3)))[0]
    pr = pos @ rot.T
    ar = oracle.acc(pr, mass, 1.0, 0.0)
    cr = oracle.grad(pr, mass, ar, 1.0, 0.0)
    assert np.allclose(ar, a @ rot.T, rtol=0, atol=1e-15 * np.abs(a).max())
    assert np.allclose(cr, c @ rot.T, rtol=0, atol=1e-14 * np.abs(c).max())


def test_acc_self_pair_skipped_by_id():
    """eps = 0: the j == i term would be 0/0; Eq. 6's sum excludes it (reading A3)."""
    pos, _, mass = _random_cluster(64, 5)
    a = oracle.acc(pos, mass, 1.0, 0.0)
    assert np.isfinite(a).all()
    # sink 3 against sources {3, 7}: only particle 7 contributes
    a37 = oracle.acc(pos, mass, 1.0, 0.0, sink_idx=[3], src_idx=[3, 7])
    r = pos[7] - pos[3]
    assert np.allclose(a37[0], mass[7] * r / (r @ r) ** 1.5, rtol=8 * U)


def test_acc_momentum_conservation():
    """Pairwise kicks conserve momentum: sum_i m_i a_i = 0 to round-off."""
    for eps in (0.0, 1e-3):
        pos, _, mass = _random_cluster(700, 6)
        a = oracle.acc(pos, mass, 1.0, eps)
        tot = np.abs((mass[:, None] * a).sum(axis=0))
        scale = (mass[:, None] * np.abs(a)).sum(axis=0)
        assert (tot <= 1e-15 * scale).all()


def test_acc_index_lists_are_partial_sums():
    """Eq. 12: the inter-level sums over disjoint source sets add up to the full sum."""
    pos, _, mass = _random_cluster(300, 7)
    ids = np.random.default_rng(0).permutation(300).astype(np.int32)
    S, F = np.sort(ids[:120]), np.sort(ids[120:])
    sinks = np.sort(ids[50:200])
    full = oracle.acc(pos, mass, 1.0, 1e-4, sink_idx=sinks)
    part = oracle.acc(pos, mass, 1.0, 1e-4, sink_idx=sinks, src_idx=S) + \
        oracle.acc(pos, mass, 1.0, 1e-4, sink_idx=sinks, src_idx=F)
    assert np.allclose(full, part, rtol=0, atol=1e-14 * np.abs(full).max())
    # compact output rows follow the sink list order
    allacc = oracle.acc(pos, mass, 1.0, 1e-4)
    assert np.array_equal(full, allacc[sinks])
    # source order only changes rounding
    rev = oracle.acc(pos, mass, 1.0, 1e-4, sink_idx=sinks, src_idx=np.arange(299, -1, -1))
    assert (normwise_rel_err(rev, full) < 4 * U).all()


def test_acc_grad_double_vs_long_double():
    """The binary64 instance agrees with the x87 80-bit instance to <= 5e-16 normwise,
    so the oracle's own rounding error is far below the 1e-12 parity gate."""
    pos, _, mass = _random_cluster(2048, 8)
    for eps in (0.0, 1e-4):
        a = oracle.acc(pos, mass, 1.0, eps)
        al = oracle.acc(pos, mass, 1.0, eps, long_double=True)
        assert (normwise_rel_err(a, al) < 5e-16).all()
        g = oracle.grad(pos, mass, al, 1.0, eps)
        gl = oracle.grad(pos, mass, al, 1.0, eps, long_double=True)
        assert (normwise_rel_err(g, gl) < 5e-16).all()


def test_plummer_potential_energy_and_mean_field():
    """W -> -3 pi G M^2 / (32 a) and a(r) -> -G M r / (r^2 + a^2)^(3/2) for a sampled
    Plummer sphere (statistical: pins generator + oracle at large N, ~1/sqrt(N))."""
    n = 16384
    pos, _, _ = _random_cluster(n, 9, kroupa=False)
    mass = np.full(n, 1.0 / n)
    w = oracle.potential(pos, mass, 1.0)
    assert abs(w / (-3 * np.pi / 32) - 1) < 0.03
    assert abs(oracle.potential(pos, mass, 1.0, long_double=True) / w - 1) < 1e-14
    a = oracle.acc(pos, mass, 1.0, 0.0)
    r = np.linalg.norm(pos, axis=1)
    a_rad = (a * pos).sum(axis=1) / r
    edges = [0.3, 0.6, 1.0, 1.5, 2.5, 5.0]
    for lo, hi in zip(edges[:-1], edges[1:]):
        sel = (r >= lo) & (r < hi)
        model = -(r[sel]) / (r[sel] ** 2 + 1) ** 1.5
        assert abs(np.median(a_rad[sel] / model) - 1) < 0.08


# --- grad: formula, sign, factor, softened form (Eq. 9; readings G1-G4) -----

@pytest.mark.parametrize("eps", [0.0, 0.4, 1.5])
def test_grad_two_body_closed_form(eps):
    """C_1 = -G^2 m_2 (m_1+m_2) (s^2 - 3 r^2) r_21 / s^8; at eps = 0: +2 G^2 m_2 M r_21 / r^6."""
    rng = np.random.default_rng(21)
    for _ in range(20):
        pos = rng.normal(size=(2, 3))
        mass = rng.uniform(0.1, 3.0, 2)
        G = rng.uniform(0.5, 2.0)
        a = oracle.acc(pos, mass, G, eps)
        c = oracle.grad(pos, mass, a, G, eps)
        r21 = pos[1] - pos[0]
        r2 = r21 @ r21
        s2 = r2 + eps * eps
        M = mass.sum()
        c0 = -G * G * mass[1] * M * (s2 - 3 * r2) * r21 / s2 ** 4
        c1 = +G * G * mass[0] * M * (s2 - 3 * r2) * r21 / s2 ** 4
        assert np.allclose(c[0], c0, rtol=64 * U, atol=0)
        assert np.allclose(c[1], c1, rtol=64 * U, atol=0)
        if eps == 0.0:
            assert (c[0] @ r21) > 0      # extra attraction (reading G4)


@pytest.mark.parametrize("eps_frac", [0.0, 1.0])
def test_grad_is_half_gradient_of_sum_m_a2(eps_frac):
    """"gradient potential grad |a|^2 = 2 a grad a":
    C_i = (1 / (2 m_i)) d/dr_i  sum_k m_k |a_k|^2, checked by central differences on
    N = 6, at eps = 0 and at eps ~ typical separation (discriminates reading G1)."""
    rng = np.random.default_rng(31)
    n = 6
    pos = rng.normal(size=(n, 3))
    mass = rng.uniform(0.2, 2.0, n)
    G = 1.3
    eps = eps_frac * 0.8

    def phi(p):
        a = oracle.acc(p, mass, G, eps, long_double=True)
        return float((mass * (a * a).sum(axis=1)).sum())

    a = oracle.acc(pos, mass, G, eps)
    c = oracle.grad(pos, mass, a, G, eps)
    h = 1e-5
    fd = np.zeros_like(c)
    for i in range(n):
        for k in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[i, k] += h
            pm[i, k] -= h
            fd[i, k] = (phi(pp) - phi(pm)) / (2 * h) / (2 * mass[i])
    assert np.abs(fd - c).max() <= 1e-7 * np.abs(c).max()
    if eps > 0:
        # the alternative reading (softening only the denominator r^5, keeping |r|^2 a_ji) is far off
        d = pos[None, :, :] - pos[:, None, :]
        r2 = (d * d).sum(-1)
        s2 = r2 + eps * eps
        np.fill_diagonal(s2, 1.0)
        da = a[None, :, :] - a[:, None, :]
        q = (da * d).sum(-1)
        alt = G * ((mass[None, :] * r2 / s2 ** 2.5)[:, :, None] * da
                   - (3 * mass[None, :] * q / s2 ** 2.5)[:, :, None] * d).sum(axis=1)
        assert np.abs(alt - fd).max() > 1e-2 * np.abs(fd).max()


def test_grad_momentum_conservation():
    """sum_i m_i C_i = 0 when sinks = sources = all and acc is the matching all-active result."""
    pos, _, mass = _random_cluster(600, 12)
    for eps in (0.0, 1e-3):
        a = oracle.acc(pos, mass, 1.0, eps)
        c = oracle.grad(pos, mass, a, 1.0, eps)
        tot = np.abs((mass[:, None] * c).sum(axis=0))
        scale = (mass[:, None] * np.abs(c)).sum(axis=0)
        assert (tot <= 1e-14 * scale).all()


def test_grad_hierarchical_slow_fast_antisymmetry():
    """Eq. 12 + Eq. 13 for disjoint S and F: with the inter-level accelerations, the
    slow<-fast and fast<-slow gradient kicks are pairwise antisymmetric, so
    sum over S and F of m_i C_i vanishes ("manifestly momentum-conserving")."""
    pos, _, mass = _random_cluster(400, 13)
    ids = np.random.default_rng(1).permutation(400).astype(np.int32)
    S, F = np.sort(ids[:300]), np.sort(ids[300:])
    a = np.zeros((400, 3))
    a[S] = oracle.acc(pos, mass, 1.0, 0.0, sink_idx=S, src_idx=F)
    a[F] = oracle.acc(pos, mass, 1.0, 0.0, sink_idx=F, src_idx=S)
    cS = oracle.grad(pos, mass, a, 1.0, 0.0, sink_idx=S, src_idx=F)
    cF = oracle.grad(pos, mass, a, 1.0, 0.0, sink_idx=F, src_idx=S)
    tot = (mass[S, None] * cS).sum(axis=0) + (mass[F, None] * cF).sum(axis=0)
    scale = (mass[S, None] * np.abs(cS)).sum(axis=0) + (mass[F, None] * np.abs(cF)).sum(axis=0)
    assert (np.abs(tot) <= 1e-14 * scale).all()


def test_grad_uses_supplied_accelerations_linearly():
    """C is linear in acc[] and vanishes for a uniform acceleration field (only a_j - a_i enters)."""
    pos, _, mass = _random_cluster(200, 14)
    rng = np.random.default_rng(2)
    a1, a2 = rng.normal(size=(200, 3)), rng.normal(size=(200, 3))
    c1 = oracle.grad(pos, mass, a1, 1.0, 1e-2)
    c2 = oracle.grad(pos, mass, a2, 1.0, 1e-2)
    c12 = oracle.grad(pos, mass, 2 * a1 - 0.5 * a2, 1.0, 1e-2)
    assert np.allclose(c12, 2 * c1 - 0.5 * c2, rtol=0, atol=1e-13 * np.abs(c12).max())
    cu = oracle.grad(pos, mass, np.tile([1.0, -2.0, 3.0], (200, 1)), 1.0, 1e-2)
    assert np.abs(cu).max() == 0.0
