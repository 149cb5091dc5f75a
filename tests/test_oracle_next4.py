"""Pins for the NEXT-4 oracle (oracle/integrator.py): FSI (§2.1, Eq. 5-10) and HHS-FSI
(§2.2, Eq. 11-13) against what the paper and the mathematics fix - the analytic Kepler orbit,
the order of convergence (fourth with the gradient term, second without: "the final acceleration
term proportional to eps^2 in Eq. (9) cancels the leading second-order error terms", L96), Eq. 73's
eta^4 energy-error scaling, time reversibility, momentum conservation ("manifestly
momentum-conserving", L131) and the structure of the hierarchy."""
import numpy as np
import pytest

import oracle
from oracle import integrator as I
from paper_2210_02472_b200 import workloads as W

G = 1.0


def two_body(m1, m2, a, e):
    """Periapsis of a Kepler orbit in the centre-of-mass frame; returns pos, vel, mass, period."""
    M = m1 + m2
    rp = a * (1 - e)
    vp = np.sqrt(G * M * (1 + e) / (a * (1 - e)))
    pos = np.array([[-m2 / M * rp, 0, 0], [m1 / M * rp, 0, 0]], dtype=float)
    vel = np.array([[0, -m2 / M * vp, 0], [0, m1 / M * vp, 0]], dtype=float)
    return pos, vel, np.array([m1, m2], dtype=float), 2 * np.pi * np.sqrt(a ** 3 / (G * M))


def kepler_relative(a, e, M, t):
    """Analytic relative position at time t after periapsis (Kepler's equation by bisection)."""
    n = np.sqrt(G * M / a ** 3)
    Mm = n * t
    lo, hi = Mm - 1.0, Mm + 1.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if mid - e * np.sin(mid) < Mm:
            lo = mid
        else:
            hi = mid
    E = 0.5 * (lo + hi)
    return np.array([a * (np.cos(E) - e), a * np.sqrt(1 - e * e) * np.sin(E), 0.0])


def orbit_error(steps, t_end, gradient_term=True):
    pos, vel, mass, period = two_body(0.7, 0.3, 1.0, 0.5)
    idx = np.arange(2, dtype=np.int32)
    h = t_end * period / steps
    for _ in range(steps):
        I.fsi_step(pos, vel, mass, idx, G, 0.0, h, gradient_term=gradient_term)
    exact = kepler_relative(1.0, 0.5, 1.0, t_end * period)
    return float(np.linalg.norm((pos[1] - pos[0]) - exact))


def test_fsi_is_fourth_order_against_the_analytic_kepler_orbit():
    e1, e2, e3 = orbit_error(150, 0.37), orbit_error(300, 0.37), orbit_error(600, 0.37)
    assert e3 < 2e-7                                              # and it converges to the analytic orbit
    assert 13.0 < e1 / e2 < 19.0 and 13.0 < e2 / e3 < 19.0        # halving eps: error / 2^4


def test_without_the_gradient_term_only_second_order():
    """Pins the gradient term and the 1/6, 2/3, 1/24 coefficients: any other weight leaves an O(eps^2) error."""
    e1, e2 = orbit_error(300, 0.37, False), orbit_error(600, 0.37, False)
    assert 3.5 < e1 / e2 < 4.5
    assert e2 > 50 * orbit_error(600, 0.37)


@pytest.mark.parametrize("c24", [12.0, 48.0])
def test_wrong_gradient_coefficient_breaks_fourth_order(c24, monkeypatch):
    """eps^2/24 (Eq. 9): with eps^2/12 or eps^2/48 (the g_i = 2 C_i mix-up of Eq. 23) the order drops to 2."""
    real_kick = I.kick

    def bad_kick(vel, acc, idx, h, grad=None, c=0.0):
        real_kick(vel, acc, idx, h, grad, c * 24.0 / c24)
    monkeypatch.setattr(I, "kick", bad_kick)
    e1, e2 = orbit_error(300, 0.37), orbit_error(600, 0.37)
    assert 3.0 < e1 / e2 < 6.0


def small_cluster(n=48, seed=11):
    rng = np.random.default_rng(seed)
    pos, vel = W.plummer_phase_space(rng, n)
    mass = np.full(n, 1.0 / n)
    W.recentre(pos, vel, mass)
    return pos, vel, mass


def test_energy_error_scales_with_the_fourth_power_eq73():
    eps_soft = 0.2
    errs = []
    for steps in (8, 16, 32):
        pos, vel, mass = small_cluster()
        e0 = I.total_energy(pos, vel, mass, G, eps_soft)
        idx = np.arange(mass.shape[0], dtype=np.int32)
        for _ in range(steps):
            I.fsi_step(pos, vel, mass, idx, G, eps_soft, 0.4 / steps)
        errs.append(abs(I.total_energy(pos, vel, mass, G, eps_soft) / e0 - 1.0))
    assert errs[2] < 1e-8
    assert 15.0 < errs[0] / errs[1] < 18.0 and 15.5 < errs[1] / errs[2] < 16.5          # 2^4


def test_fsi_is_time_reversible_and_conserves_momentum():
    pos, vel, mass = small_cluster(32, 3)
    p0, v0 = pos.copy(), vel.copy()
    idx = np.arange(32, dtype=np.int32)
    mom0 = (mass[:, None] * vel).sum(0)
    for _ in range(3):
        I.fsi_step(pos, vel, mass, idx, G, 0.05, 0.01)
    assert np.abs((mass[:, None] * vel).sum(0) - mom0).max() < 1e-16
    vel *= -1.0
    for _ in range(3):
        I.fsi_step(pos, vel, mass, idx, G, 0.05, 0.01)
    vel *= -1.0
    assert np.abs(pos - p0).max() < 1e-13 and np.abs(vel - v0).max() < 1e-13


def test_fsi_on_a_subset_leaves_the_rest_alone():
    pos, vel, mass = small_cluster(20, 5)
    p0, v0 = pos.copy(), vel.copy()
    idx = np.array([3, 4, 9, 17], dtype=np.int32)
    I.fsi_step(pos, vel, mass, idx, G, 0.0, 0.01)
    rest = np.setdiff1d(np.arange(20), idx)
    assert np.array_equal(pos[rest], p0[rest]) and np.array_equal(vel[rest], v0[rest])
    sp, sv, sm = p0[idx].copy(), v0[idx].copy(), mass[idx].copy()
    I.fsi_step(sp, sv, sm, np.arange(4, dtype=np.int32), G, 0.0, 0.01)     # the subset as a system of its own
    assert np.array_equal(pos[idx], sp) and np.array_equal(vel[idx], sv)


def binary_in_cluster():
    """A loose cluster of 30 particles plus a hard binary (a = 2e-3) near the centre."""
    pos, vel, mass = small_cluster(30, 7)
    bp, bv, bm, period = two_body(0.02, 0.03, 2e-3, 0.3)
    pos = np.vstack([pos, bp + np.array([0.05, 0.02, -0.01])])
    vel = np.vstack([vel, bv + np.array([0.1, -0.05, 0.02])])
    mass = np.concatenate([mass, bm])
    return pos, vel, mass, period


def test_hhs_all_slow_level_is_one_fsi_step_bit_for_bit():
    pos, vel, mass = small_cluster(24, 2)
    p1, v1 = pos.copy(), vel.copy()
    stats = {}
    I.hhs_fsi(pos, vel, mass, G, 0.05, 0.5, 0.5, 1e-4, stats=stats)
    assert stats["levels"] == [(0, 24, 0, 1e-4)]
    I.fsi_step(p1, v1, mass, np.arange(24, dtype=np.int32), G, 0.05, 1e-4)
    assert np.array_equal(pos, p1) and np.array_equal(vel, v1)


def test_hhs_puts_the_hard_binary_alone_on_the_fast_levels_and_conserves_momentum_and_energy():
    pos, vel, mass, period = binary_in_cluster()
    n = mass.shape[0]
    e0 = I.total_energy(pos, vel, mass, G, 0.0)
    mom0 = (mass[:, None] * vel).sum(0)
    stats = {}
    tau = 2e-3
    I.hhs_fsi(pos, vel, mass, G, 0.0, 0.02, 0.02, tau, stats=stats)
    levels = stats["levels"]
    assert levels[0][0] == 0 and levels[0][1] + levels[0][2] == n
    deepest = max(d for d, _, _, _ in levels)
    assert deepest >= 4                                                   # eta * period/(2 pi) << tau
    assert all(s + f == 2 for d, s, f, _ in levels if d >= 2)            # only the binary goes deep
    assert sum(1 for d, *_ in levels if d == 1) == 2 and sum(1 for d, *_ in levels if d == 2) <= 4
    assert np.abs((mass[:, None] * vel).sum(0) - mom0).max() < 1e-15     # round-off only: pairwise synchronous kicks (L131)
    e_hhs = abs(I.total_energy(pos, vel, mass, G, 0.0) / e0 - 1.0)
    assert e_hhs < 2e-6            # a hard binary (period ~ tau) without regularisation, eta = 0.02: ~300 steps per orbit
    # one plain FSI step of the same length cannot resolve the binary at all
    pos2, vel2, mass2, _ = binary_in_cluster()
    I.fsi_step(pos2, vel2, mass2, np.arange(n, dtype=np.int32), G, 0.0, tau)
    assert abs(I.total_energy(pos2, vel2, mass2, G, 0.0) / e0 - 1.0) > 1e4 * e_hhs


def test_hhs_energy_error_follows_eta_to_the_fourth_eq73():
    """Eq. 73: |dE/E|_1 = (eta_1/eta_0)^4 |dE/E|_0 for the hierarchical integrator (softened cluster)."""
    errs = []
    for eta in (0.2, 0.1):
        pos, vel, mass = small_cluster(40, 13)
        e0 = I.total_energy(pos, vel, mass, G, 0.02)
        for _ in range(2):
            I.hhs_fsi(pos, vel, mass, G, 0.02, eta, eta, 0.05)
        errs.append(abs(I.total_energy(pos, vel, mass, G, 0.02) / e0 - 1.0))
    assert errs[1] < errs[0] / 4.0            # block time-steps quantise eps_i to tau/2^k: between 2^2 and 2^6
    assert errs[1] > errs[0] / 200.0


def test_hhs_max_depth_bounds_the_recursion():
    pos, vel, mass, _ = binary_in_cluster()
    stats = {}
    I.hhs_fsi(pos, vel, mass, G, 0.0, 0.02, 0.02, 2e-3, max_depth=2, stats=stats)
    assert max(d for d, *_ in stats["levels"]) == 2
    assert all(f == 0 for d, s, f, _ in stats["levels"] if d == 2)


def test_hhs_dt_cap_is_minned_into_the_level0_timestep():
    """"The final time-step of a particle is the minimum of the set of its different time-steps" (L293):
    a further criterion handed in as dt_cap sends exactly the capped particles to the fast levels."""
    pos, vel, mass = small_cluster(24, 2)
    tau = 1e-4                                              # all slow by the pairwise criteria (see above)
    cap = np.full(24, np.inf)
    cap[[5, 17]] = 0.3 * tau                                # tau/4 <= cap < tau/2: fast at depths 0 and 1, slow at 2
    stats = {}
    I.hhs_fsi(pos, vel, mass, G, 0.05, 0.5, 0.5, tau, stats=stats, dt_cap=cap)
    lv = [(d, s, f) for d, s, f, _ in stats["levels"]]
    assert lv[0] == (0, 22, 2) and lv[1] == (1, 0, 2) and lv[2] == (2, 2, 0)
    assert sorted(lv) == sorted([(0, 22, 2), (1, 0, 2), (1, 0, 2), (2, 2, 0), (2, 2, 0), (2, 2, 0), (2, 2, 0)])
    # an infinite cap changes nothing
    p1, v1 = small_cluster(24, 2)[:2]
    p2, v2 = p1.copy(), v1.copy()
    I.hhs_fsi(p1, v1, mass, G, 0.05, 0.5, 0.5, tau)
    I.hhs_fsi(p2, v2, mass, G, 0.05, 0.5, 0.5, tau, dt_cap=np.full(24, np.inf))
    assert np.array_equal(p1, p2) and np.array_equal(v1, v2)


# --- the inter-level kicks of Eq. 11-13: fourth order as a whole -------------
# With the partition held fixed (dt_cap = 0.75 tau sends five chosen particles to level 1 and no
# further; eta so large that the pairwise criteria never split), HHS-FSI is a composition of FSI
# operators and must converge with tau^4 to the fine-step solution.  A wrong inter-level
# gradient coefficient in Eq. 13 (or a missing S<->F gradient kick) leaves an O(tau^2) error.

def _hhs_fixed_partition_error(steps, reference, grad_scale=1.0, monkeypatch=None):
    pos, vel, mass = small_cluster(12, 21)
    T, eps_soft = 0.4, 0.3
    tau = T / steps
    cap = np.full(12, np.inf)
    cap[[1, 4, 6, 9, 10]] = 0.75 * tau
    if monkeypatch is not None:
        real = oracle.grad

        def scaled(pos_, mass_, acc_, G_, eps_, sink_idx=None, src_idx=None, **kw):
            out = real(pos_, mass_, acc_, G_, eps_, sink_idx, src_idx, **kw)
            inter_level = sink_idx is not None and src_idx is not None and not np.array_equal(sink_idx, src_idx)
            return out * grad_scale if inter_level else out
        monkeypatch.setattr(oracle, "grad", scaled)
    stats = {}
    for _ in range(steps):
        I.hhs_fsi(pos, vel, mass, G, eps_soft, 1e3, 1e3, tau, dt_cap=cap, stats=stats)
    assert [(d, s, f) for d, s, f, _ in stats["levels"]] == [(0, 7, 5), (1, 5, 0), (1, 5, 0)]
    return float(np.abs(pos - reference).max())


@pytest.fixture(scope="module")
def fine_reference():
    pos, vel, mass = small_cluster(12, 21)
    idx = np.arange(12, dtype=np.int32)
    for _ in range(2048):
        I.fsi_step(pos, vel, mass, idx, G, 0.3, 0.4 / 2048)
    return pos


def test_hhs_two_level_scheme_is_fourth_order(fine_reference):
    e = [_hhs_fixed_partition_error(s, fine_reference) for s in (4, 8, 16)]
    assert e[2] < 2e-9
    assert 15.0 < e[0] / e[1] < 17.0 and 15.0 < e[1] / e[2] < 17.0


@pytest.mark.parametrize("scale", [0.0, 0.5, 1.1, 2.0])
def test_wrong_inter_level_gradient_coefficient_breaks_fourth_order(scale, fine_reference, monkeypatch):
    """Eq. 13's gradient kick between S and F with 0, 1/2, 1.1 or 2 times its weight: order 2."""
    e = [_hhs_fixed_partition_error(s, fine_reference, scale, monkeypatch) for s in (8, 16)]
    assert e[0] / e[1] < 6.0


def test_hhs_level_criteria_enter_every_level_and_stay_under_the_level0_cap():
    """with level_criteria the acceleration-based time-steps (Eq. 24-29) of the level's own particles
    are min'd into the level's time-steps.  Pins: (i) criteria that never bind (huge eta) change nothing, bit for bit;
    (ii) at level 0 the fast set is exactly {min(pairwise, criteria) < tau}, recomputed here from the pinned routines;
    (iii) a particle that is slow by its level-0 value can only get FASTER at depth (the cap of L295), so the level
    structure refines the one without criteria; (iv) momentum is still conserved to round-off."""
    tau = 2e-3
    base, with_c, huge = {}, {}, {}
    pos0, vel0, mass, _ = binary_in_cluster()
    p, v = pos0.copy(), vel0.copy()
    I.hhs_fsi(p, v, mass, G, 0.0, 0.02, 0.02, tau, stats=base)
    p2, v2 = pos0.copy(), vel0.copy()
    I.hhs_fsi(p2, v2, mass, G, 0.0, 0.02, 0.02, tau, stats=huge, level_criteria=(1e30, 1e30, 1e30))
    assert huge["levels"] == base["levels"] and np.array_equal(p, p2) and np.array_equal(v, v2)
    eta = (0.01, 0.01, 0.01)
    p3, v3 = pos0.copy(), vel0.copy()
    mom0 = (mass[:, None] * v3).sum(0)
    I.hhs_fsi(p3, v3, mass, G, 0.0, 0.02, 0.02, tau, stats=with_c, level_criteria=eta)
    n = mass.shape[0]
    idx = np.arange(n, dtype=np.int32)
    d = oracle.dtmin(pos0, vel0, mass, G, 0.02, 0.02)
    a = oracle.acc(pos0, mass, G, 0.0)
    cr = oracle.criteria(vel0, a, oracle.grad(pos0, mass, a, G, 0.0), oracle.jerk(pos0, vel0, mass, G, 0.0), *eta)
    dt = np.minimum.reduce([d["dt_ff"], d["dt_fb"], cr["dt_va"], cr["dt_gradv"], cr["dt_grada"], cr["dt_jerk"]])
    assert with_c["levels"][0][:3] == (0, int((dt >= tau).sum()), int((dt < tau).sum()))
    assert with_c["levels"][0][2] > base["levels"][0][2]                 # the criteria bind for some particles here
    assert max(x[0] for x in with_c["levels"]) >= max(x[0] for x in base["levels"])
    assert np.abs((mass[:, None] * v3).sum(0) - mom0).max() < 1e-15
    assert np.array_equal(I.level_criteria_timesteps(pos0, vel0, mass, idx, G, 0.0, *eta),
                          np.minimum.reduce([cr["dt_va"], cr["dt_gradv"], cr["dt_grada"], cr["dt_jerk"]]))
