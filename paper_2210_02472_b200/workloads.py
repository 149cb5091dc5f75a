"""Seeded synthetic star-cluster inputs for the five BASELINE.json configurations.

This module is the ONLY code shared between the CPU oracle's tests and the CUDA
path's tests / bench: it produces particle arrays (positions, velocities,
masses) and index lists.  None of the method's routines (acceleration, gradient,
time-step, PN) lives here and nothing here is called by the library or the
oracle.  One input-preparation helper does evaluate a pair sum: config 2 asks for
"virialised velocities", so `_virial_potential_energy` computes the cluster's
potential energy W once, in numpy, to rescale the sampled speeds to 2T = -W; it
feeds the INPUTS only and is never compared with, or used by, either side.  The recipes are
stated in DESIGN.md §"Input recipe"; they stand in for the paper's SCIC
initial-conditions generator (App. A), whose output is
not available.

Units: G = 1, total mass M = 1, Plummer scale radius a_p = 1
(BASELINE.json config 1 "G=M=a=1", taken literally - SURVEY.md §8c reading C1).

Everything is numpy on the host, float64 / int32, C-contiguous.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

G_NBODY = 1.0
A_PLUMMER = 1.0
#: r_h = (2^(2/3) - 1)^(-1/2) a_p  (App. A2)
R_HALF = (2.0 ** (2.0 / 3.0) - 1.0) ** -0.5 * A_PLUMMER


@dataclasses.dataclass
class Workload:
    """One configuration's particle data and parameters (host numpy arrays)."""

    name: str
    pos: np.ndarray            # float64 [n][3]
    vel: np.ndarray            # float64 [n][3]
    mass: np.ndarray           # float64 [n]
    G: float
    eps: float                 # Plummer softening length (0 = unsoftened)
    eta_ff: float
    eta_fb: float
    c: Optional[float] = None          # speed of light (config 4 only)
    bh_idx: Optional[np.ndarray] = None  # int32 ids of PN particles (config 4 only)
    seed: int = 0
    subsys: Optional[np.ndarray] = None  # int32 [n]: binary (subsystem) index of each star, -1 = single (config 3)

    @property
    def n(self) -> int:
        return int(self.mass.shape[0])


# ---------------------------------------------------------------------------
# building blocks
# ---------------------------------------------------------------------------

def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """n unit vectors, uniform on the sphere ("two random angles")."""
    cos_t = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    sin_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t * cos_t))
    return np.stack([sin_t * np.cos(phi), sin_t * np.sin(phi), cos_t], axis=1)


def plummer_radii(rng: np.random.Generator, n: int, r_max: float = 100.0) -> np.ndarray:
    """Inversion sampling of the Plummer cumulative mass profile:
    M(<r)/M = r^3 (r^2 + a^2)^(-3/2) = X  =>  r = a (X^(-2/3) - 1)^(-1/2).
    X is capped so that r <= r_max * a_p (the profile is truncated, as every
    practical Plummer sampler does)."""
    x_cap = r_max ** 3 / (r_max * r_max + 1.0) ** 1.5
    x = rng.uniform(0.0, 1.0, n) * x_cap
    x = np.maximum(x, 1e-300)
    return A_PLUMMER / np.sqrt(x ** (-2.0 / 3.0) - 1.0)


def plummer_speeds(rng: np.random.Generator, r: np.ndarray) -> np.ndarray:
    """von Neumann rejection sampling of the speed from the Plummer distribution
    function f(E) ~ E^(7/2) (Eq. A4-A5): with q = v / v_esc,
    p(q) ~ q^2 (1 - q^2)^(7/2), v_esc = sqrt(2 G M / a) (1 + r^2/a^2)^(-1/4)."""
    n = r.shape[0]
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        qq = rng.uniform(0.0, 1.0, todo.size)
        yy = rng.uniform(0.0, 0.1, todo.size)       # max of q^2 (1-q^2)^3.5 is 0.0922
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    v_esc = np.sqrt(2.0 * G_NBODY * 1.0 / A_PLUMMER) * (1.0 + (r / A_PLUMMER) ** 2) ** -0.25
    return q * v_esc


def plummer_phase_space(rng: np.random.Generator, n: int):
    r = plummer_radii(rng, n)
    pos = r[:, None] * _isotropic(rng, n)
    v = plummer_speeds(rng, r)
    vel = v[:, None] * _isotropic(rng, n)
    return np.ascontiguousarray(pos), np.ascontiguousarray(vel)


# Kroupa (2001) two-segment IMF on [0.08, 100] Msun (SURVEY.md §8c reading C4;
# the paper names the IMF, without printing its segments):
#   xi(m) ~ m^-1.3 on [0.08, 0.5),  m^-2.3 on [0.5, 100], continuous at 0.5.
_K_LO, _K_BREAK, _K_HI = 0.08, 0.5, 100.0
_K_A1, _K_A2 = 1.3, 2.3


def _kroupa_segment_numbers():
    n1 = (_K_LO ** (1 - _K_A1) - _K_BREAK ** (1 - _K_A1)) / (_K_A1 - 1)
    # continuity: A2 = A1 * break^(a2 - a1)
    a2 = _K_BREAK ** (_K_A2 - _K_A1)
    n2 = a2 * (_K_BREAK ** (1 - _K_A2) - _K_HI ** (1 - _K_A2)) / (_K_A2 - 1)
    return n1, n2


def kroupa_masses(rng: np.random.Generator, n: int) -> np.ndarray:
    """n stellar masses in Msun by inverse-CDF sampling of the two-segment IMF."""
    n1, n2 = _kroupa_segment_numbers()
    f1 = n1 / (n1 + n2)
    u = rng.uniform(0.0, 1.0, n)
    x = rng.uniform(0.0, 1.0, n)
    m = np.empty(n)
    lo = u < f1

    def inv(xx, a, m0, m1):
        e = 1.0 - a
        return (m0 ** e + xx * (m1 ** e - m0 ** e)) ** (1.0 / e)

    m[lo] = inv(x[lo], _K_A1, _K_LO, _K_BREAK)
    m[~lo] = inv(x[~lo], _K_A2, _K_BREAK, _K_HI)
    return m


def recentre(pos: np.ndarray, vel: np.ndarray, mass: np.ndarray) -> None:
    """Shift to the centre-of-mass frame in place."""
    mt = mass.sum()
    pos -= (mass[:, None] * pos).sum(axis=0) / mt
    vel -= (mass[:, None] * vel).sum(axis=0) / mt


def active_subset(seed: int, n: int, size: int) -> np.ndarray:
    """`size` distinct particle ids, uniform without replacement, sorted ascending
    (the sink list of one hierarchical time-bin level; "faster
    hierarchy levels ... contain fewer particles")."""
    rng = np.random.default_rng(seed)
    if size >= n:
        return np.arange(n, dtype=np.int32)
    ids = rng.choice(n, size=size, replace=False)
    ids.sort()
    return ids.astype(np.int32)


def _virial_potential_energy(pos: np.ndarray, mass: np.ndarray, chunk: int = 512) -> float:
    """W = -G sum_{i<j} m_i m_j / r_ij by chunked numpy direct summation.  INPUT PREPARATION ONLY:
    used once to virialise config 2's velocities (see the module docstring); not a routine of the
    method, not shared with the library or the oracle."""
    n = mass.shape[0]
    w = 0.0
    x, y, z = (np.ascontiguousarray(pos[:, c]) for c in range(3))
    for s in range(0, n, chunk):
        e = min(s + chunk, n)
        r2 = np.square(x[s:e, None] - x[None, :])
        r2 += np.square(y[s:e, None] - y[None, :])
        r2 += np.square(z[s:e, None] - z[None, :])
        idx = np.arange(s, e)
        r2[idx - s, idx] = np.inf
        np.sqrt(r2, out=r2)
        np.divide(mass[None, :], r2, out=r2)
        w += float(mass[s:e] @ r2.sum(axis=1))
    return -0.5 * G_NBODY * w


def _kepler_E(mean_anom: np.ndarray, ecc: np.ndarray) -> np.ndarray:
    """Eccentric anomaly from Kepler's equation M = E - e sin E (PAPER.md:L564,
    Eq. 50) by bracketed Newton iteration; input preparation for config 3's binaries."""
    lo, hi = mean_anom - ecc, mean_anom + ecc          # f is increasing; the root lies in between
    E = mean_anom + ecc * np.sin(mean_anom)
    for _ in range(80):
        f = E - ecc * np.sin(E) - mean_anom
        lo = np.where(f < 0, E, lo)
        hi = np.where(f > 0, E, hi)
        En = E - f / (1.0 - ecc * np.cos(E))
        bad = ~((En > lo) & (En < hi))
        E = np.where(bad, 0.5 * (lo + hi), En)
    return E


def _binary_relative_orbit(rng, m_tot, n_b):
    """Relative position and velocity of n_b Kepler binaries: semi-major axis
    log-uniform in [1e-4, 1e-2] r_h (BASELINE.json config 3; PAPER.md:L1221
    "flat in logarithmic space"), thermal eccentricities f(e) = 2e
    (PAPER.md:L1223), random i, Omega, omega and mean anomaly."""
    a = R_HALF * 10.0 ** rng.uniform(-4.0, -2.0, n_b)
    e = np.sqrt(rng.uniform(0.0, 1.0, n_b))
    e = np.minimum(e, 0.999)
    mean_anom = rng.uniform(0.0, 2.0 * np.pi, n_b)
    E = _kepler_E(mean_anom, e)
    cosE, sinE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    x = a * (cosE - e)
    y = a * b * sinE
    rr = a * (1.0 - e * cosE)
    nmot = np.sqrt(G_NBODY * m_tot / a ** 3)
    vx = -a * a * nmot * sinE / rr
    vy = a * a * nmot * b * cosE / rr
    cos_i = rng.uniform(-1.0, 1.0, n_b)
    sin_i = np.sqrt(1.0 - cos_i * cos_i)
    Om = rng.uniform(0.0, 2.0 * np.pi, n_b)
    om = rng.uniform(0.0, 2.0 * np.pi, n_b)
    cO, sO, co, so = np.cos(Om), np.sin(Om), np.cos(om), np.sin(om)
    # rotation R = Rz(Om) Rx(i) Rz(om) applied to (x, y, 0)
    px = np.stack([cO * co - sO * so * cos_i, sO * co + cO * so * cos_i, so * sin_i], axis=1)
    qx = np.stack([-cO * so - sO * co * cos_i, -sO * so + cO * co * cos_i, co * sin_i], axis=1)
    rel_pos = x[:, None] * px + y[:, None] * qx
    rel_vel = vx[:, None] * px + vy[:, None] * qx
    return rel_pos, rel_vel, a, e


# ---------------------------------------------------------------------------
# the five configurations (BASELINE.json "configs"; seeds: config k -> seed k-1)
# ---------------------------------------------------------------------------

def config1(n: int = 1024, seed: int = 0) -> Workload:
    """Plummer sphere, equal masses, eps = 1e-4, eta = 0.01, all active."""
    rng = np.random.default_rng(seed)
    pos, vel = plummer_phase_space(rng, n)
    mass = np.full(n, 1.0 / n)
    return Workload("config1", pos, vel, mass, G_NBODY, 1e-4, 0.01, 0.01, seed=seed)


def config2(n: int = 16384, seed: int = 1) -> Workload:
    """Plummer, Kroupa masses rescaled to M = 1, virialised velocities (2T = -W,
    centre-of-mass frame), eps = 1e-5.  Sink lists: active_subset(2000 + k, n, 2**k)."""
    rng = np.random.default_rng(seed)
    pos, vel = plummer_phase_space(rng, n)
    mass = kroupa_masses(rng, n)
    mass /= mass.sum()
    recentre(pos, vel, mass)
    w = _virial_potential_energy(pos, mass)
    t = 0.5 * float((mass * (vel * vel).sum(axis=1)).sum())
    vel *= np.sqrt(-0.5 * w / t)
    return Workload("config2", pos, vel, mass, G_NBODY, 1e-5, 0.01, 0.01, seed=seed)


def config2_sink_list(k: int, n: int = 16384) -> np.ndarray:
    return active_subset(2000 + k, n, 2 ** k)


def config3(n: int = 131072, seed: int = 2) -> Workload:
    """Plummer with 50 % of the stars in binaries treated as point particles
    (N_b = N/4 binaries), Kroupa masses, eps = 0.
    Pairing is random among the mass-sampled stars (the paper's mass-ratio
    pairing above 5 Msun, is simplified; DESIGN.md says so)."""
    rng = np.random.default_rng(seed)
    n_b = n // 4
    n_s = n - 2 * n_b
    mass = kroupa_masses(rng, n)
    mass /= mass.sum()
    m1, m2 = mass[:n_b], mass[n_b:2 * n_b]
    com_pos, com_vel = plummer_phase_space(rng, n_b + n_s)
    rel_pos, rel_vel, _, _ = _binary_relative_orbit(rng, m1 + m2, n_b)
    f1 = (m2 / (m1 + m2))[:, None]
    f2 = (m1 / (m1 + m2))[:, None]
    pos = np.empty((n, 3))
    vel = np.empty((n, 3))
    # r_rel = r_2 - r_1
    pos[:n_b] = com_pos[:n_b] - f1 * rel_pos
    vel[:n_b] = com_vel[:n_b] - f1 * rel_vel
    pos[n_b:2 * n_b] = com_pos[:n_b] + f2 * rel_pos
    vel[n_b:2 * n_b] = com_vel[:n_b] + f2 * rel_vel
    pos[2 * n_b:] = com_pos[n_b:]
    vel[2 * n_b:] = com_vel[n_b:]
    perm = rng.permutation(n)           # binary members are not neighbours in memory
    pos, vel, mass = pos[perm], vel[perm], mass[perm]
    # the binaries double as the subsystems of the NEXT-2 (subsystem-aware) parity cases
    subsys = np.concatenate([np.arange(n_b), np.arange(n_b), np.full(n_s, -1)]).astype(np.int32)[perm]
    recentre(pos, vel, mass)
    return Workload("config3", np.ascontiguousarray(pos), np.ascontiguousarray(vel),
                    np.ascontiguousarray(mass), G_NBODY, 0.0, 0.01, 0.01, seed=seed,
                    subsys=np.ascontiguousarray(subsys))


def config3_sink_list(frac_log2: int, n: int = 131072) -> np.ndarray:
    """Active fraction 2**-frac_log2, frac_log2 = 0..10 (1 ... 1/1024)."""
    return active_subset(3000 + frac_log2, n, n >> frac_log2)


def config4(n: int = 1 << 20, seed: int = 3, n_sbh: int = 100) -> Workload:
    """Plummer, Kroupa masses plus one central IMBH of 1e-3 M (id 0, at rest at
    the origin) and n_sbh stellar BHs of 10-30 Msun at Plummer-sampled
    phase-space points; all active; eps = 0 (reading C2); c = 1e4."""
    rng = np.random.default_rng(seed)
    pos, vel = plummer_phase_space(rng, n)
    m_msun = kroupa_masses(rng, n)
    bh = np.sort(rng.choice(np.arange(1, n), size=n_sbh, replace=False))
    m_msun[bh] = rng.uniform(10.0, 30.0, n_sbh)
    m_msun[0] = 0.0
    mass = m_msun / m_msun.sum() * (1.0 - 1e-3)
    mass[0] = 1e-3
    pos[0] = 0.0
    vel[0] = 0.0
    bh_idx = np.concatenate([[0], bh]).astype(np.int32)
    return Workload("config4", pos, vel, mass, G_NBODY, 0.0, 0.01, 0.01, c=1e4,
                    bh_idx=bh_idx, seed=seed)


def config5(n: int = 1 << 21, seed: int = 4) -> Workload:
    """Plummer, Kroupa masses, eps = 1e-5, all active (peak-throughput case)."""
    rng = np.random.default_rng(seed)
    pos, vel = plummer_phase_space(rng, n)
    mass = kroupa_masses(rng, n)
    mass /= mass.sum()
    return Workload("config5", pos, vel, mass, G_NBODY, 1e-5, 0.01, 0.01, seed=seed)


#: §5.2 / Fig. 8 in N-body units (G = M = a_p = 1): r_h = 3.1 pc fixes a_p = 3.1 pc / R_HALF,
#: M = 161000 x 0.5 Msun fixes the time unit sqrt(a_p^3 / (G M)) with G = 4.30091e-3 pc (km/s)^2 / Msun
#: and 1 pc / (km/s) = 0.977792 Myr.
FIG8_PC = 3.1 / R_HALF                                            # parsecs per length unit
FIG8_MYR = (FIG8_PC ** 3 / (4.30091e-3 * 161000 * 0.5)) ** 0.5 * 0.977792   # Myr per time unit


def fig8(n: int = 161000, seed: int = 8) -> Workload:
    """The softened equal-mass cluster of PAPER.md:L816-824 (§5.2, Fig. 8, "FROST-like" run): Plummer sphere of
    N = 161000 equal masses, r_h = 3.1 pc, Plummer softening eps_soft = 1e-3 pc, eta_ff = eta_fb = 0.2 (the
    gradient / jerk criteria use eta = 0.1), integration interval tau = 1e-3 Myr = `fig8_tau()`.  Centre-of-mass
    frame.  A smaller n keeps the physical scales (same r_h, same softening) with heavier particles."""
    rng = np.random.default_rng(seed)
    pos, vel = plummer_phase_space(rng, n)
    mass = np.full(n, 1.0 / n)
    recentre(pos, vel, mass)
    return Workload("fig8", pos, vel, mass, G_NBODY, 1e-3 / FIG8_PC, 0.2, 0.2, seed=seed)


def fig8_tau() -> float:
    """The integration interval of PAPER.md:L822 (1e-3 Myr) in N-body time units."""
    return 1e-3 / FIG8_MYR


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
