"""Oracle for NEXT-4: the FSI cycle (§2.1, Eq. 5-10) and the hierarchical
HHS-FSI cycle (§2.2, Eq. 11-13), step by step in the paper's order.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): plain numpy for the O(N) operators, the pinned
O(N^2) routines of bifrost_oracle.cpp (acc, grad, dtmin, potential) for the sums.  Shares no code
with the CUDA path and does not import it.

What is computed
  kick        v_i <- v_i + h a_i                                   (Eq. 5)
  drift       r_i <- r_i + h v_i                                   (Eq. 7)
  gradient    v_i <- v_i + (2 eps/3) (a_i + (eps^2/24) C_i)        (Eq. 8-9; C_i = oracle.grad)
  fsi_step    kick(eps/6) drift(eps/2) gradient-kick(2 eps/3) drift(eps/2) kick(eps/6)   (Eq. 10)
              over a set `idx` of particles interacting only among themselves: four O(N^2) sums
              (acc, acc + grad, acc).
  hhs_fsi     Eq. 11: at each level, time-steps eps_i = min(eps_ff, eps_fb) (Eq. 21-22; FROST's
              criteria) over the level's particles, never above the particle's
              level-0 value ("eps_i = min(eps_i, eps_i^{level=0})"); fast F = {eps_i < tau},
              slow S = {eps_i >= tau}; then
                  U_SF(tau/6)  H_S(tau/2)  H_F(tau/2)  U~_SF(2 tau/3)  H_F(tau/2)  H_S(tau/2)  U_SF(tau/6)
              with the inter-level accelerations of Eq. 12 and gradient accelerations of Eq. 13,
              H_S = one fsi_step of tau/2 over S, H_F = this routine again over F with tau/2.
              "The process is repeated until no fast particles remain" (L105): a level without
              fast particles is one fsi_step of tau.

Readings (H1-H4)
  H1  Eq. 11 is palindromic, so the order of application is unambiguous.
  H2  The level's particle list is kept as one array: a STABLE partition puts S first, then F,
      both in their previous relative order; the recursion reorders only F's segment.  (Order
      only fixes the summation order.)
  H3  max_depth bounds the recursion: at that depth every particle is treated as slow.
  H4  Level 0 (depth 0) time-steps are the ones taken at the start of the interval over all
      particles; deeper levels recompute them over their own set at the moment they are entered.

Pins (tests/test_oracle_next4.py): fourth-order convergence of the two-body orbit against the
analytic Kepler solution, and second order only when the gradient term is dropped (pins the 1/6,
1/2, 2/3 and 1/24 coefficients); Eq. 73's eta^4 energy-error scaling on a softened cluster;
time reversibility; exact momentum conservation of HHS-FSI; the all-slow level reduces to
fsi_step bit for bit; a hard binary in a loose cluster lands alone on the fast levels.
"""
from __future__ import annotations

import numpy as np

import oracle


def kick(vel, acc, idx, h, grad=None, c=0.0):
    """Eq. 5 / Eq. 8-9: v_i += h (a_i + c C_i) for i in idx."""
    if grad is None:
        vel[idx] += h * acc[idx]
    else:
        vel[idx] += h * (acc[idx] + c * grad[idx])


def drift(pos, vel, idx, h):
    """Eq. 7: r_i += h v_i for i in idx."""
    pos[idx] += h * vel[idx]


def _acc_into(acc, pos, mass, G, eps_soft, sinks, srcs):
    acc[sinks] = oracle.acc(pos, mass, G, eps_soft, sinks, srcs)


def fsi_step(pos, vel, mass, idx, G, eps_soft, eps, gradient_term=True):
    """One FSI cycle (Eq. 10) of length eps over the particles idx, in place."""
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    n = mass.shape[0]
    acc = np.zeros((n, 3))
    grad = np.zeros((n, 3))
    _acc_into(acc, pos, mass, G, eps_soft, idx, idx)
    kick(vel, acc, idx, eps / 6.0)
    drift(pos, vel, idx, eps / 2.0)
    _acc_into(acc, pos, mass, G, eps_soft, idx, idx)
    if gradient_term:
        grad[idx] = oracle.grad(pos, mass, acc, G, eps_soft, idx, idx)
        kick(vel, acc, idx, 2.0 * eps / 3.0, grad, eps * eps / 24.0)
    else:
        kick(vel, acc, idx, 2.0 * eps / 3.0)
    drift(pos, vel, idx, eps / 2.0)
    _acc_into(acc, pos, mass, G, eps_soft, idx, idx)
    kick(vel, acc, idx, eps / 6.0)


def level_timesteps(pos, vel, mass, idx, G, eta_ff, eta_fb):
    """eps_i = min(eps_ff, eps_fb) (Eq. 21-22) of the particles idx among themselves."""
    d = oracle.dtmin(pos, vel, mass, G, eta_ff, eta_fb, idx, idx)
    return np.minimum(d["dt_ff"], d["dt_fb"])


def level_criteria_timesteps(pos, vel, mass, idx, G, eps_soft, eta, eta_grad, eta_jerk):
    """PAPER.md:L293-295, per level: the acceleration-based criteria of Eq. 24, 26, 27, 29 of the
    particles idx with the accelerations, gradient sums and jerks of the particles idx AMONG THEMSELVES (the sums of
    a sparse faster level - the "pathological situations" L295 guards against with the level-0 cap); returns their
    minimum per particle.  Built from the pinned routines only."""
    n = mass.shape[0]
    a = np.zeros((n, 3)); a[idx] = oracle.acc(pos, mass, G, eps_soft, idx, idx)
    j = np.zeros((n, 3)); j[idx] = oracle.jerk(pos, vel, mass, G, eps_soft, idx, idx)
    c = np.zeros((n, 3)); c[idx] = oracle.grad(pos, mass, a, G, eps_soft, idx, idx)
    cr = oracle.criteria(vel, a, c, j, eta, eta_grad, eta_jerk, idx)
    return np.minimum(np.minimum(cr["dt_va"], cr["dt_gradv"]), np.minimum(cr["dt_grada"], cr["dt_jerk"]))


def hhs_fsi(pos, vel, mass, G, eps_soft, eta_ff, eta_fb, tau, max_depth=32, stats=None, dt_cap=None, level_criteria=None):
    """One HHS-FSI integration interval of length tau (Eq. 11), in place.  stats (a dict, optional)
    receives 'levels' (list of (depth, n_slow, n_fast, tau)) in the order the levels are entered.
    dt_cap (optional, [n]): further per-particle time-steps (e.g. Eq. 24-29) min'd into the level-0 value.
    level_criteria (optional, (eta, eta_grad, eta_jerk)): Eq. 24-29 are ALSO evaluated at every level over the level's
    own particles and min'd into the level's time-steps ("the final time-step of a particle is the minimum of the set
    of its different time-steps"), still capped by the level-0 value (L295)."""
    n = mass.shape[0]
    order = np.arange(n, dtype=np.int32)
    dt0 = np.full(n, np.inf) if dt_cap is None else np.array(dt_cap, dtype=np.float64)   # further criteria (L293)
    if stats is not None:
        stats["levels"] = []
    _hhs_level(pos, vel, mass, G, eps_soft, eta_ff, eta_fb, order, 0, n, tau, 0, max_depth, dt0, stats, level_criteria)


def _hhs_level(pos, vel, mass, G, eps_soft, eta_ff, eta_fb, order, lo, hi, tau, depth, max_depth, dt0, stats,
               level_criteria=None):
    idx = order[lo:hi].copy()
    if idx.size == 0:
        return
    if depth < max_depth:
        dt = level_timesteps(pos, vel, mass, idx, G, eta_ff, eta_fb)
        if level_criteria is not None:
            dt = np.minimum(dt, level_criteria_timesteps(pos, vel, mass, idx, G, eps_soft, *level_criteria))
        if depth == 0:
            dt0[idx] = np.minimum(dt, dt0[idx])             # level-0 value = minimum of all criteria
        dt = np.minimum(dt, dt0[idx])
        fast = dt < tau
    else:
        fast = np.zeros(idx.size, dtype=bool)
    S, F = idx[~fast], idx[fast]                            # stable partition (reading H2)
    order[lo:hi] = np.concatenate([S, F])
    mid = lo + S.size
    if stats is not None:
        stats["levels"].append((depth, int(S.size), int(F.size), float(tau)))
    if F.size == 0:
        fsi_step(pos, vel, mass, S, G, eps_soft, tau)
        return
    n = mass.shape[0]
    acc = np.zeros((n, 3))
    grad = np.zeros((n, 3))

    def inter_level_acc():                                  # Eq. 12
        Fn = order[mid:hi].copy()
        if S.size:
            _acc_into(acc, pos, mass, G, eps_soft, S, Fn)
            _acc_into(acc, pos, mass, G, eps_soft, Fn, S)
        return Fn

    def H_S():
        if S.size:
            fsi_step(pos, vel, mass, S, G, eps_soft, tau / 2.0)

    def H_F():
        _hhs_level(pos, vel, mass, G, eps_soft, eta_ff, eta_fb, order, mid, hi, tau / 2.0, depth + 1, max_depth, dt0,
                   stats, level_criteria)

    Fn = inter_level_acc()
    if S.size:
        kick(vel, acc, np.concatenate([S, Fn]), tau / 6.0)
    H_S()
    H_F()
    Fn = inter_level_acc()
    if S.size:
        grad[S] = oracle.grad(pos, mass, acc, G, eps_soft, S, Fn)      # Eq. 13
        grad[Fn] = oracle.grad(pos, mass, acc, G, eps_soft, Fn, S)
        kick(vel, acc, np.concatenate([S, Fn]), 2.0 * tau / 3.0, grad, tau * tau / 24.0)
    H_F()
    H_S()
    Fn = inter_level_acc()
    if S.size:
        kick(vel, acc, np.concatenate([S, Fn]), tau / 6.0)


def total_energy(pos, vel, mass, G, eps_soft):
    """Eq. 4: H = sum 1/2 m v^2 + W, W from the pinned potential routine."""
    return 0.5 * float((mass * (vel * vel).sum(1)).sum()) + oracle.potential(pos, mass, G, eps_soft)
