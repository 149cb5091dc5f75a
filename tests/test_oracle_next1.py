"""Pins for the oracle's NEXT-1 routines (CPU only): jerk (Eq. 28), the per-particle
potential (Eq. 4, L724 Eq. 68) and the O(N) time-step criteria (Eq. 24, 26, 27, 29).

Each test checks the oracle against something other than itself: finite differences of the
already-pinned acceleration / potential routines, closed forms, invariants, hand-worked numbers.
"""
import numpy as np
import pytest

import oracle
from paper_2210_02472_b200 import workloads as W

U = 2.0 ** -53


def _cluster(n, seed):
    rng = np.random.default_rng(seed)
    pos, vel = W.plummer_phase_space(rng, n)
    mass = W.kroupa_masses(rng, n)
    mass /= mass.sum()
    return pos, vel, mass


# --- jerk ------------------------------------------------------------------------------

@pytest.mark.parametrize("eps", [0.0, 0.5])
def test_jerk_is_time_derivative_of_acc(eps):
    """j_i = d a_i / dt along the flow dr/dt = v ("just as in the Hermite codes"):
    central difference of the pinned O-acc at r +- v h.  Pins sign, the factor 3, v_ji vs v_ij,
    and (eps > 0) the softened form."""
    pos, vel, mass = _cluster(7, 21)
    pos *= 0.5
    h = 1e-5
    ap = oracle.acc(pos + h * vel, mass, 1.3, eps, long_double=True)
    am = oracle.acc(pos - h * vel, mass, 1.3, eps, long_double=True)
    fd = (ap - am) / (2 * h)
    j = oracle.jerk(pos, vel, mass, 1.3, eps)
    assert np.abs(j - fd).max() <= 2e-8 * np.abs(j).max()


@pytest.mark.parametrize("eps", [0.0, 0.7])
def test_jerk_two_body_closed_form(eps):
    rng = np.random.default_rng(22)
    for _ in range(10):
        pos, vel = rng.normal(size=(2, 3)), rng.normal(size=(2, 3))
        mass = rng.uniform(0.2, 2.0, 2)
        G = 0.8
        r, v = pos[1] - pos[0], vel[1] - vel[0]
        s2 = r @ r + eps * eps
        expect0 = G * mass[1] * (v / s2 ** 1.5 - 3 * (r @ v) * r / s2 ** 2.5)
        j = oracle.jerk(pos, vel, mass, G, eps)
        assert np.allclose(j[0], expect0, rtol=0, atol=16 * U * np.abs(expect0).max() + 1e-300)
        assert np.allclose(mass[0] * j[0] + mass[1] * j[1], 0, atol=16 * U * np.abs(mass[0] * j[0]).max())


def test_jerk_momentum_and_lists():
    pos, vel, mass = _cluster(300, 23)
    j = oracle.jerk(pos, vel, mass, 1.0, 1e-3)
    tot = np.abs((mass[:, None] * j).sum(axis=0))
    assert (tot <= 1e-14 * (mass[:, None] * np.abs(j)).sum(axis=0)).all()
    jl = oracle.jerk(pos, vel, mass, 1.0, 1e-3, long_double=True)
    assert np.abs(j - jl).max() <= 1e-15 * np.abs(jl).max()
    sinks = np.array([5, 17, 250], dtype=np.int32)
    srcs = np.arange(100, 300, dtype=np.int32)
    rest = np.arange(0, 100, dtype=np.int32)
    part = oracle.jerk(pos, vel, mass, 1.0, 1e-3, sinks, srcs) + oracle.jerk(pos, vel, mass, 1.0, 1e-3, sinks, rest)
    assert np.allclose(part, j[sinks], rtol=1e-13, atol=0)


# --- per-particle potential ---------------------------------------------------------------

def test_phi_two_body_and_total():
    pos = np.array([[0.0, 0, 0], [3.0, 4.0, 0]])
    mass = np.array([2.0, 5.0])
    phi = oracle.phi(pos, mass, 2.0, 0.0)
    assert phi[0] == -2.0 * 5.0 / 5.0 and phi[1] == -2.0 * 2.0 / 5.0      # -G m_j / r, r = 5 exactly
    phis = oracle.phi(pos, mass, 2.0, 12.0)                               # s = sqrt(25 + 144) = 13
    assert np.allclose(phis, [-10.0 / 13.0, -4.0 / 13.0], rtol=4 * U)
    pos, _, mass = _cluster(500, 24)
    w = 0.5 * float((mass * oracle.phi(pos, mass, 1.0, 1e-2)).sum())
    assert abs(w / oracle.potential(pos, mass, 1.0, 1e-2) - 1) < 1e-14


def test_acc_is_minus_gradient_of_potential():
    """m_i a_i = -dW/dr_i with W = 1/2 sum m_i phi_i: ties phi to the pinned acceleration."""
    pos, _, mass = _cluster(6, 25)
    eps, h = 0.3, 1e-6
    a = oracle.acc(pos, mass, 1.0, eps)
    for i in (0, 3):
        for c in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[i, c] += h
            pm[i, c] -= h
            wp = 0.5 * (mass * oracle.phi(pp, mass, 1.0, eps)).sum()
            wm = 0.5 * (mass * oracle.phi(pm, mass, 1.0, eps)).sum()
            assert abs(-(wp - wm) / (2 * h) - mass[i] * a[i, c]) <= 1e-8 * np.abs(mass[i] * a[i]).max()


# --- O(N) criteria -------------------------------------------------------------------------

def test_criteria_hand_worked():
    """Integer-norm vectors: |v| = 5, |a| = 10, |C| = 24*13 -> |g'| = 13, |j| = 25.
    Eq. 24: eta 5/10; Eq. 26: eta_g (5/13)^(1/3); Eq. 27: eta_g (10/13)^(1/2); Eq. 29: eta_j 10/25."""
    vel = np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 0.0]])
    acc = np.array([[0.0, 6.0, 8.0], [0.0, 0.0, 0.0]])
    grad = np.array([[24 * 5.0, 0.0, 24 * 12.0], [0.0, 0.0, 0.0]])
    jerk = np.array([[7.0, 0.0, 24.0], [0.0, 0.0, 0.0]])
    r = oracle.criteria(vel, acc, grad, jerk, 0.02, 0.1, 0.2)
    assert np.isclose(r["dt_va"][0], 0.02 * 0.5, rtol=4 * U)
    assert np.isclose(r["dt_gradv"][0], 0.1 * (5.0 / 13.0) ** (1.0 / 3.0), rtol=8 * U)
    assert np.isclose(r["dt_grada"][0], 0.1 * (10.0 / 13.0) ** 0.5, rtol=8 * U)
    assert np.isclose(r["dt_jerk"][0], 0.2 * 0.4, rtol=4 * U)
    assert all(np.isinf(r[k][1]) for k in r)                             # zero denominators -> +inf
    only = oracle.criteria(vel, acc, grad, jerk, 0.02, 0.1, 0.2, sink_idx=np.array([1, 0], dtype=np.int32))
    assert np.isinf(only["dt_va"][0]) and only["dt_va"][1] == r["dt_va"][0]
