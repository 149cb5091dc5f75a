"""Pins for the oracle's time-step minima and PN1.0 routines (CPU only)."""
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


# --- dtmin (Eq. 21, L317 Eq. 22) --------------------------------------------

def _brute_dt(pos, vel, mass, G, eta_ff, eta_fb, sinks, srcs):
    """Independent brute force: dense numpy pair matrices, sources visited in REVERSE
    order, argmin by explicit scan with the smaller-id tie rule."""
    n_s = len(sinks)
    out = dict(dt_ff=np.full(n_s, np.inf), dt_fb=np.full(n_s, np.inf),
               j_ff=np.full(n_s, -1, np.int32), j_fb=np.full(n_s, -1, np.int32))
    for k, i in enumerate(sinks):
        for j in srcs[::-1]:
            if j == i:
                continue
            d = pos[j] - pos[i]
            r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2]
            r = np.sqrt(r2)
            tff = eta_ff * np.sqrt(r2 * r / (G * (mass[i] + mass[j])))
            dv = vel[j] - vel[i]
            v2 = dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]
            tfb = np.inf if v2 == 0 else eta_fb * r / np.sqrt(v2)
            if tff < out["dt_ff"][k] or (tff == out["dt_ff"][k] and j < out["j_ff"][k]):
                out["dt_ff"][k], out["j_ff"][k] = tff, j
            if tfb < out["dt_fb"][k] or (tfb == out["dt_fb"][k] and j < out["j_fb"][k]):
                out["dt_fb"][k], out["j_fb"][k] = tfb, j
    return out


def test_dtmin_matches_reverse_order_brute_force():
    pos, vel, mass = _cluster(150, 41)
    rng = np.random.default_rng(0)
    sinks = np.sort(rng.choice(150, 40, replace=False)).astype(np.int32)
    srcs = rng.permutation(150)[:120].astype(np.int32)
    got = oracle.dtmin(pos, vel, mass, 1.0, 0.02, 0.03, sink_idx=sinks, src_idx=srcs)
    ref = _brute_dt(pos, vel, mass, 1.0, 0.02, 0.03, sinks, srcs)
    for key in ("dt_ff", "dt_fb", "j_ff", "j_fb"):
        assert np.array_equal(got[key], ref[key]), key
    assert (got["margin_ff"] >= 0).all() and (got["margin_fb"] >= 0).all()


def test_dtmin_two_body_and_circular_binary():
    """Closed forms; and "the two time-step criteria are equal for a bound binary on a
    circular orbit" when eta_ff = eta_fb."""
    rng = np.random.default_rng(42)
    for _ in range(10):
        m = rng.uniform(0.1, 2.0, 2)
        G = rng.uniform(0.5, 2.0)
        r = rng.uniform(0.1, 3.0)
        v_circ = np.sqrt(G * m.sum() / r)
        rot = np.linalg.qr(rng.normal(size=(3, 3)))[0]
        pos = np.array([[0, 0, 0], [r, 0, 0]]) @ rot.T
        vel = np.array([[0, -v_circ * m[1] / m.sum(), 0], [0, v_circ * m[0] / m.sum(), 0]]) @ rot.T
        shift = rng.normal(size=3)
        d = oracle.dtmin(pos + shift, vel + 0.3 * shift, m, G, 0.01, 0.01)
        want = 0.01 * np.sqrt(r ** 3 / (G * m.sum()))
        assert np.allclose(d["dt_ff"], want, rtol=32 * U)
        assert np.allclose(d["dt_fb"], d["dt_ff"], rtol=64 * U)
        assert list(d["j_ff"]) == [1, 0] and list(d["j_fb"]) == [1, 0]
        # generic (non-circular) velocities: dt_fb = eta r / |v_rel|
        vel2 = rng.normal(size=(2, 3))
        d2 = oracle.dtmin(pos, vel2, m, G, 0.2, 0.1)
        assert np.allclose(d2["dt_fb"], 0.1 * r / np.linalg.norm(vel2[1] - vel2[0]), rtol=32 * U)
        assert np.allclose(d2["dt_ff"], 0.2 * np.sqrt(r ** 3 / (G * m.sum())), rtol=32 * U)


def test_dtmin_exact_ties_pick_smaller_id():
    """Cubic lattice, equal masses, coordinates and velocities small-integer multiples of
    a power of two: r^2 and v^2 are exact, so nearest-neighbour ties are exact (reading T4)."""
    g = np.arange(4)
    pos = np.array([[x, y, z] for x in g for y in g for z in g], dtype=np.float64) * 0.25
    n = pos.shape[0]
    rng = np.random.default_rng(5)
    perm = rng.permutation(n)
    pos = pos[perm]
    vel = pos[:, ::-1] * 0.5                      # |v_ij| = 0.5 |r_ij| for every pair: all fb ties
    mass = np.full(n, 0.125)
    d = oracle.dtmin(pos, vel, mass, 1.0, 0.5, 0.25)
    ip = np.rint(pos * 4).astype(np.int64)
    for i in range(n):
        dist2 = ((ip - ip[i]) ** 2).sum(axis=1)
        dist2[i] = 10 ** 9
        assert d["j_ff"][i] == np.flatnonzero(dist2 == dist2.min())[0]
        assert d["j_fb"][i] == (0 if i != 0 else 1)          # every source ties: smallest id wins
        assert d["margin_ff"][i] == 0.0
    assert np.all(d["dt_fb"] == 0.25 / 0.5)
    assert np.all(d["dt_ff"] == 0.5 * np.sqrt(0.25 ** 3 / 0.25))


def test_dtmin_degenerate_cases():
    pos, vel, mass = _cluster(8, 43)
    d = oracle.dtmin(pos, vel, mass, 1.0, 0.1, 0.1, sink_idx=[2], src_idx=[2])     # only itself
    assert np.isinf(d["dt_ff"][0]) and np.isinf(d["dt_fb"][0]) and d["j_ff"][0] == -1 and d["j_fb"][0] == -1
    vel0 = np.zeros_like(vel)                                                     # no relative motion
    d = oracle.dtmin(pos, vel0, mass, 1.0, 0.1, 0.1)
    assert np.isinf(d["dt_fb"]).all() and (d["j_fb"] == -1).all() and np.isfinite(d["dt_ff"]).all()


# --- pn1 (§3.8; reading P1) ---------------------------------------------

def _bodies(n, seed):
    rng = np.random.default_rng(seed)
    return rng.normal(size=(n, 3)), 0.3 * rng.normal(size=(n, 3)), rng.uniform(0.1, 1.0, n)


def test_pn1_c_scaling_is_exact():
    """The term is proportional to 1/c^2: c -> 2c divides it by exactly 4 (power of two)."""
    pos, vel, mass = _bodies(12, 51)
    bh = [1, 4]
    f1 = oracle.pn1(pos, vel, mass, bh, 1.0, 50.0)
    f2 = oracle.pn1(pos, vel, mass, bh, 1.0, 100.0)
    assert np.array_equal(f1, 4.0 * f2) and np.abs(f1).max() > 0


def test_pn1_pair_selection_and_additivity():
    """Every ordered pair with >= 1 member in the BH list exactly once; star-star pairs never."""
    pos, vel, mass = _bodies(5, 52)
    bh = [0, 3]
    full = oracle.pn1(pos, vel, mass, bh, 1.0, 30.0)

    def pair(i, j):   # force on i from j via a two-particle call
        sub = [i, j]
        return oracle.pn1(pos[sub], vel[sub], mass[sub], [0, 1], 1.0, 30.0)[0]

    for i in range(5):
        want = np.zeros(3)
        for j in range(5):
            if j != i and (i in bh or j in bh):
                want += pair(i, j)
        assert np.allclose(full[i], want, rtol=0, atol=1e-15 * np.abs(full).max())
    # label swap: permuting particle labels permutes the result
    perm = np.array([3, 1, 4, 0, 2])
    inv = np.argsort(perm)
    fp = oracle.pn1(pos[perm], vel[perm], mass[perm], [int(inv[b]) for b in bh], 1.0, 30.0)
    assert np.allclose(fp, full[perm], rtol=0, atol=1e-15 * np.abs(full).max())
    # no BHs -> nothing
    assert np.abs(oracle.pn1(pos, vel, mass, [], 1.0, 30.0)).max() == 0.0


def test_pn1_test_particle_limit():
    """m_i -> 0 around a mass M at rest: f = (G M / c^2 r^2) [ (4 G M / r - v^2) n + 4 (n.v) v ]."""
    rng = np.random.default_rng(53)
    for _ in range(10):
        G, M, c = 1.7, 2.5, 40.0
        r = rng.normal(size=3)
        v = rng.normal(size=3)
        pos = np.array([[0, 0, 0], r])
        vel = np.array([[0, 0, 0], v])
        mass = np.array([M, 1e-30])
        f = oracle.pn1(pos, vel, mass, [0], G, c)[1]
        rr = np.linalg.norm(r)
        n = r / rr
        want = G * M / (c * c * rr * rr) * ((4 * G * M / rr - v @ v) * n + 4 * (n @ v) * v)
        assert np.allclose(f, want, rtol=1e-14, atol=0)


@pytest.mark.parametrize("q", [1e-6, 0.5, 1.0])
def test_pn1_relative_acceleration_identity(q):
    """In the centre-of-mass frame f(1<-2) - f(2<-1) equals the textbook 1PN relative acceleration
    -(G M / c^2 r^2) { [ (1+3 nu) v^2 - 2 (2+nu) G M / r - 3/2 nu rdot^2 ] n - 2 (2-nu) rdot v }."""
    rng = np.random.default_rng(54)
    G, c = 1.3, 25.0
    m1 = 1.0
    m2 = q
    M = m1 + m2
    nu = m1 * m2 / M ** 2
    for _ in range(10):
        x = rng.normal(size=3)
        v = rng.normal(size=3)
        pos = np.array([m2 / M * x, -m1 / M * x])
        vel = np.array([m2 / M * v, -m1 / M * v])
        f = oracle.pn1(pos, vel, np.array([m1, m2]), [0, 1], G, c, long_double=True)
        rel = f[0] - f[1]
        r = np.linalg.norm(x)
        n = x / r
        rdot = n @ v
        want = -(G * M / (c * c * r * r)) * (((1 + 3 * nu) * (v @ v) - 2 * (2 + nu) * G * M / r
                                              - 1.5 * nu * rdot ** 2) * n - 2 * (2 - nu) * rdot * v)
        assert np.allclose(rel, want, rtol=0, atol=1e-13 * np.abs(want).max())


@pytest.mark.parametrize("q", [1e-6, 0.5, 1.0])
def test_pn1_periapsis_advance(q):
    """Integrate one radial period of an eccentric binary under Newtonian + PN1.0 pair
    accelerations (both from the oracle) and compare the periapsis advance with
    PAPER.md:L534 Eq. 46 (first term): Delta omega = 6 pi G M / (c^2 a (1 - e^2)) per orbit."""
    G, c = 1.0, 50.0
    m = np.array([1.0, q]) / (1.0 + q)
    M = m.sum()
    a_sma, ecc = 1.0, 0.5
    rp = a_sma * (1 - ecc)
    vp = np.sqrt(G * M * (1 + ecc) / (a_sma * (1 - ecc)))
    pos = np.array([[-m[1] / M * rp, 0, 0], [m[0] / M * rp, 0, 0]])
    vel = np.array([[0, -m[1] / M * vp, 0], [0, m[0] / M * vp, 0]])

    def rhs(p, v):
        return oracle.acc(p, m, G, 0.0) + oracle.pn1(p, v, m, [0, 1], G, c)

    period = 2 * np.pi * np.sqrt(a_sma ** 3 / (G * M))
    steps = 6000
    h = 1.12 * period / steps

    def rdot(p, v):
        d = p[1] - p[0]
        return (d @ (v[1] - v[0])) / np.linalg.norm(d)

    # t = 0 is a periapsis of the PN orbit too (rdot = 0 there); integrate to the next one
    peri_angles = [0.0]
    prev = 0.0
    for _ in range(steps):
        k1p, k1v = vel, rhs(pos, vel)
        k2p, k2v = vel + 0.5 * h * k1v, rhs(pos + 0.5 * h * k1p, vel + 0.5 * h * k1v)
        k3p, k3v = vel + 0.5 * h * k2v, rhs(pos + 0.5 * h * k2p, vel + 0.5 * h * k2v)
        k4p, k4v = vel + h * k3v, rhs(pos + h * k3p, vel + h * k3v)
        npos = pos + h / 6 * (k1p + 2 * k2p + 2 * k3p + k4p)
        nvel = vel + h / 6 * (k1v + 2 * k2v + 2 * k3v + k4v)
        cur = rdot(npos, nvel)
        if prev < 0 <= cur:                       # periapsis between the two states
            w = -prev / (cur - prev)              # rdot ~ linear in time near periapsis
            d0, d1 = pos[1] - pos[0], npos[1] - npos[0]
            ang0, ang1 = np.arctan2(d0[1], d0[0]), np.arctan2(d1[1], d1[0])
            dang = (ang1 - ang0 + np.pi) % (2 * np.pi) - np.pi
            peri_angles.append(ang0 + w * dang)   # theta'' = 0 at periapsis: linear is enough
            break
        pos, vel, prev = npos, nvel, cur
    assert len(peri_angles) == 2
    # a, e of the PN orbit differ from the Newtonian values used in `want` at O(v^2/c^2) ~ 1e-3
    advance = (peri_angles[1] - peri_angles[0]) % (2 * np.pi)
    want = 6 * np.pi * G * M / (c * c * a_sma * (1 - ecc * ecc))
    assert abs(advance / want - 1) < 0.01


# --- the per-body split of the PN1.0 pair term (reading P1) --------
# In the centre-of-mass frame `+4 v_i.v_j` and `-2 v_j.v_j` enter the relative acceleration only
# through their difference, so the pins above cannot tell (4, -2) from (6, 0).  A BOOSTED frame can:
# the 1PN (EIH) equations of motion conserve the 1PN total momentum and energy (Landau & Lifshitz,
# Classical Theory of Fields, §106)
#   P = sum_a m_a v_a [1 + v_a^2/2c^2 - sum_b G m_b/(2 c^2 r_ab)] - sum_a sum_b G m_a m_b/(2 c^2 r_ab) (n_ab.v_a) n_ab
#   E = sum_a m_a v_a^2/2 + 3/(8c^2) sum_a m_a v_a^4 - 1/2 sum_ab G m_a m_b/r_ab
#       + sum_ab G m_a m_b/(4 c^2 r_ab) [6 v_a^2 - 7 v_a.v_b - (n_ab.v_a)(n_ab.v_b)] + sum_abc G^2 m_a m_b m_c/(2 c^2 r_ab r_ac)
# up to O(c^-4): along an orbit integrated with acc + pn1, their drift must fall 16-fold when c doubles.
# Any other split of the velocity terms between the two bodies leaves an O(c^-2) drift (ratio 4).

def _eih_momentum(pos, vel, m, G, c):
    P = np.zeros(3)
    for a in range(len(m)):
        s = 1 + vel[a] @ vel[a] / (2 * c * c)
        for b in range(len(m)):
            if b == a:
                continue
            d = pos[a] - pos[b]
            r = np.linalg.norm(d)
            s -= G * m[b] / (2 * c * c * r)
            P -= G * m[a] * m[b] / (2 * c * c * r) * ((d / r) @ vel[a]) * (d / r)
        P += m[a] * vel[a] * s
    return P


def _eih_energy(pos, vel, m, G, c):
    E = 0.0
    for a in range(len(m)):
        va2 = vel[a] @ vel[a]
        E += 0.5 * m[a] * va2 + 3.0 / (8 * c * c) * m[a] * va2 * va2
        for b in range(len(m)):
            if b == a:
                continue
            d = pos[a] - pos[b]
            r = np.linalg.norm(d)
            nab = d / r
            E -= 0.5 * G * m[a] * m[b] / r
            E += G * m[a] * m[b] / (4 * c * c * r) * (6 * va2 - 7 * (vel[a] @ vel[b]) - (nab @ vel[a]) * (nab @ vel[b]))
            for k in range(len(m)):
                if k != a:
                    E += G * G * m[a] * m[b] * m[k] / (2 * c * c * r * np.linalg.norm(pos[a] - pos[k]))
    return E


def _pn1_split(ca, cb):
    """numpy restatement of the pair term with the coefficients of v_i.v_j and v_j.v_j left free
    (negative control only: (4, -2) is reading P1)."""
    def f(pos, vel, m, G, c):
        out = np.zeros_like(pos)
        for i in range(len(m)):
            for j in range(len(m)):
                if i == j:
                    continue
                d = pos[i] - pos[j]
                r = np.linalg.norm(d)
                n = d / r
                vi, vj = vel[i], vel[j]
                A = 5 * G * m[i] / r + 4 * G * m[j] / r + 1.5 * (n @ vj) ** 2 - vi @ vi + ca * (vi @ vj) + cb * (vj @ vj)
                out[i] += G * m[j] / (c * c * r * r) * (n * A + (4 * (n @ vi) - 3 * (n @ vj)) * (vi - vj))
        return out
    return f


def _boosted_drift(pn, c, invariant):
    G = 1.0
    m = np.array([1.0, 0.4])
    pos = np.array([[0.6, 0.1, -0.2], [-0.5, 0.3, 0.4]])
    vel = np.array([[0.3, 0.5, 0.1], [0.2, -0.6, 0.35]])       # total momentum far from zero

    def rhs(p, v):
        return oracle.acc(p, m, G, 0.0) + pn(p, v, m, G, c)

    q0 = invariant(pos, vel, m, G, c)
    steps = 400
    h = 1.0 / steps
    for _ in range(steps):                                      # RK4, test-only
        k1p, k1v = vel, rhs(pos, vel)
        k2p, k2v = vel + 0.5 * h * k1v, rhs(pos + 0.5 * h * k1p, vel + 0.5 * h * k1v)
        k3p, k3v = vel + 0.5 * h * k2v, rhs(pos + 0.5 * h * k2p, vel + 0.5 * h * k2v)
        k4p, k4v = vel + h * k3v, rhs(pos + h * k3p, vel + h * k3v)
        pos = pos + h / 6 * (k1p + 2 * k2p + 2 * k3p + k4p)
        vel = vel + h / 6 * (k1v + 2 * k2v + 2 * k3v + k4v)
    return float(np.linalg.norm(np.atleast_1d(invariant(pos, vel, m, G, c) - q0)))


def _oracle_pn(pos, vel, m, G, c):
    return oracle.pn1(pos, vel, m, [0, 1], G, c)


@pytest.mark.parametrize("invariant", [_eih_momentum, _eih_energy], ids=["momentum", "energy"])
def test_pn1_per_body_split_conserves_eih_invariants_in_a_boosted_frame(invariant):
    d = [_boosted_drift(_oracle_pn, c, invariant) for c in (20.0, 40.0, 80.0)]
    assert d[2] > 1e-10                                         # well above rounding: the ratios mean something
    assert abs(d[0] / d[1] - 16) < 1 and abs(d[1] / d[2] - 16) < 1
    # the restatement with reading P1's (4, -2) is the oracle's formula ...
    pos, vel, mass = _bodies(6, 57)
    assert np.allclose(_pn1_split(4, -2)(pos, vel, mass, 1.3, 30.0), oracle.pn1(pos, vel, mass, list(range(6)), 1.3, 30.0),
                       rtol=0, atol=1e-14 * 1e-3)


@pytest.mark.parametrize("split", [(6, 0), (2, -4), (5, -1), (4, -2.1)])
@pytest.mark.parametrize("invariant", [_eih_momentum, _eih_energy], ids=["momentum", "energy"])
def test_pn1_wrong_split_is_caught(split, invariant):
    """Negative control: splits that pass every centre-of-mass pin (same -a + b) leave a c^-2 drift."""
    d = [_boosted_drift(_pn1_split(*split), c, invariant) for c in (20.0, 40.0, 80.0)]
    assert d[1] / d[2] < 8
