"""Pins for the NEXT-3 oracle routines: neighbour search (§3.4, Eq. 18-19) and the
construction of subsystems as connected components of the neighbour graph (L279).  No GPU.

The pairs are BUILT from chosen orbital elements (a, e, true anomaly), so the expected answer of
every branch of Eq. 18-19 is known by construction; a second pin re-derives a and e with formulas the
oracle does not use (vis-viva and the Laplace-Runge-Lenz vector) on a random dense cluster."""
import numpy as np
import pytest

import oracle

G = 1.0
R_NGB, R_MAX = 1e-3, 0.1


def rot(rng):
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    return q


def two_body(rng, m1, m2, a, e, f, com_pos, com_vel):
    """Relative orbit with semi-major axis a (negative for a hyperbola), eccentricity e, true anomaly f."""
    mu = G * (m1 + m2)
    p = a * (1.0 - e * e)
    r = p / (1.0 + e * np.cos(f))
    rel = np.array([r * np.cos(f), r * np.sin(f), 0.0])
    s = np.sqrt(mu / p)
    vel = np.array([-s * np.sin(f), s * (e + np.cos(f)), 0.0])
    R = rot(rng)
    rel, vel = R @ rel, R @ vel
    pos = np.array([com_pos - m2 / (m1 + m2) * rel, com_pos + m1 / (m1 + m2) * rel])
    v = np.array([com_vel - m2 / (m1 + m2) * vel, com_vel + m1 / (m1 + m2) * vel])
    return pos, v, np.array([m1, m2]), r, np.linalg.norm(vel)


CASES = [
    # name, a, e, f, tau, expect
    ("close binary at apoapsis, r > r_ngb but a < r_ngb (particle A)", 8e-4, 0.9, np.pi, 1.0, True),
    ("distant binary near periapsis, a >= r_ngb and r < r_ngb (particle B)", 5e-3, 0.9, 0.0, 1.0, True),
    ("distant binary near apoapsis (particle C)", 5e-3, 0.9, np.pi, 1.0, False),
    ("circular binary wider than r_ngb", 3e-3, 0.0, 1.0, 1.0, False),
    ("close fly-by, r < r_ngb", -2e-3, 1.2, 0.3, 1e-12, True),
    ("distant fly-by entering r_ngb within tau (particle D)", -5e-3, 1.1, -2.2, 1e9, True),
    ("distant fly-by, too far for this tau (particle E)", -5e-3, 1.1, -2.2, 1e-9, False),
    ("fly-by whose periapsis stays outside r_ngb", -5e-3, 1.5, 0.1, 1e9, False),
]


@pytest.mark.parametrize("name,a,e,f,tau,expect", CASES)
def test_eq18_eq19_branches_on_constructed_orbits(name, a, e, f, tau, expect):
    rng = np.random.default_rng(100 + [c[0] for c in CASES].index(name))
    pos, vel, mass, r, v = two_body(rng, 0.7, 0.4, a, e, f, rng.normal(size=3), rng.normal(size=3))
    assert r < R_MAX
    # far bystanders that must never be neighbours of anything
    pos = np.vstack([pos, [[50.0, 0, 0], [0, 60.0, 0]]]); vel = np.vstack([vel, np.zeros((2, 3))])
    mass = np.concatenate([mass, [1.0, 1.0]])
    count, lst = oracle.ngb(pos, vel, mass, G, R_NGB, R_MAX, tau, 0.5)
    assert list(count) == ([1, 1, 0, 0] if expect else [0, 0, 0, 0]), name
    if expect:
        assert lst[0, 0] == 1 and lst[1, 0] == 0                      # symmetric
    # sanity of the construction itself: the chosen branch is the one the name says
    if a > 0:
        assert (a < R_NGB) or (r < R_NGB) or not expect
    else:
        assert (a * (1 - e) < R_NGB) or not expect


def test_distant_flyby_threshold_is_C_r_over_v():
    """Eq. 19: C r/|v| < tau.  Bracket the threshold by +-1e-9 relative."""
    rng = np.random.default_rng(3)
    pos, vel, mass, r, v = two_body(rng, 1.0, 1.0, -5e-3, 1.1, -2.0, np.zeros(3), np.zeros(3))
    assert r >= R_NGB and -5e-3 * (1 - 1.1) < R_NGB
    C = 0.3
    t = C * r / v
    assert oracle.ngb(pos, vel, mass, G, R_NGB, R_MAX, t * (1 + 1e-9), C)[0].tolist() == [1, 1]
    assert oracle.ngb(pos, vel, mass, G, R_NGB, R_MAX, t * (1 - 1e-9), C)[0].tolist() == [0, 0]


def test_r_ngb_max_cutoff_and_index_lists():
    rng = np.random.default_rng(4)
    # a very tight binary (a << r_ngb) is found; stretching the separation beyond r_ngb_max is impossible
    # for a bound pair with a < r_ngb, so test the cutoff with an unbound pair
    pos, vel, mass, r, v = two_body(rng, 1.0, 1.0, -5e-3, 1.1, -2.2, np.zeros(3), np.zeros(3))
    assert oracle.ngb(pos, vel, mass, G, R_NGB, r * 0.999, 1e9, 0.5)[0].tolist() == [0, 0]
    assert oracle.ngb(pos, vel, mass, G, R_NGB, r * 1.001, 1e9, 0.5)[0].tolist() == [1, 1]
    # sink / source lists: only listed sources are reported, in list order
    p3 = np.vstack([pos, pos[1] + [1e-5, 0, 0]]); v3 = np.vstack([vel, vel[1]]); m3 = np.array([1.0, 1.0, 1e-3])
    c, l = oracle.ngb(p3, v3, m3, G, R_NGB, R_MAX, 1e9, 0.5, sink_idx=np.array([1], np.int32),
                      src_idx=np.array([2, 0], np.int32))
    assert c.tolist() == [2] and l[0, :2].tolist() == [2, 0]
    c, l = oracle.ngb(p3, v3, m3, G, R_NGB, R_MAX, 1e9, 0.5, cap=1)
    assert c[1] == 2 and l.shape == (3, 1)                            # count is not truncated by the capacity


def test_against_vis_viva_and_runge_lenz_on_a_dense_cluster():
    """Independent formulas: a = 1/(2/r - v^2/mu), e = |((v^2 - mu/r) r - (r.v) v)/mu|."""
    rng = np.random.default_rng(5)
    n = 300
    pos = rng.normal(size=(n, 3)) * 4e-3
    vel = rng.normal(size=(n, 3)) * 8.0
    mass = rng.uniform(0.05, 0.5, n)
    r_ngb, r_max, tau, C = 1.5e-3, 8e-3, 2e-4, 0.5
    count, lst = oracle.ngb(pos, vel, mass, G, r_ngb, r_max, tau, C, cap=64)
    got = {(i, int(j)) for i in range(n) for j in lst[i, :count[i]]}
    expect, border = set(), set()
    branches = {"bound_a": 0, "bound_r": 0, "close": 0, "distant": 0}
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            d, u = pos[j] - pos[i], vel[j] - vel[i]
            r, v2 = np.linalg.norm(d), u @ u
            mu = G * (mass[i] + mass[j])
            a = 1.0 / (2.0 / r - v2 / mu)
            e = np.linalg.norm(((v2 - mu / r) * d - (d @ u) * u) / mu)
            rp = a * (1 - e)
            near = lambda x, y: abs(x / y - 1) < 1e-9
            if near(r, r_max) or near(abs(a), r_ngb) or near(r, r_ngb) or near(rp, r_ngb) or near(C * r / np.sqrt(v2), tau) \
                    or abs(2.0 / r - v2 / mu) * r < 1e-9:
                border.add((i, j))
            if r >= r_max:
                continue
            if a > 0:                                    # bound
                if a < r_ngb: expect.add((i, j)); branches["bound_a"] += 1
                elif r < r_ngb: expect.add((i, j)); branches["bound_r"] += 1
            else:
                if rp >= r_ngb: continue
                if r < r_ngb: expect.add((i, j)); branches["close"] += 1
                elif C * r / np.sqrt(v2) < tau: expect.add((i, j)); branches["distant"] += 1
    assert all(v > 0 for v in branches.values()), branches          # every branch of Eq. 18-19 is exercised
    assert (got ^ expect) <= border
    assert got == {(j, i) for (i, j) in got}                          # exactly symmetric relation


def test_components_figure1_chain_and_brute_force():
    # Fig. 1, bottom panel: target(0) - F(1) - G(2) chained; H(3) single; a separate pair (5, 4)
    sub = oracle.components(7, [0, 1, 5], [1, 2, 4])
    assert sub.tolist() == [0, 0, 0, -1, 4, 4, -1]
    rng = np.random.default_rng(6)
    n, m = 400, 150
    ei, ej = rng.integers(0, n, m), rng.integers(0, n, m)
    keep = ei != ej
    ei, ej = ei[keep], ej[keep]
    sub = oracle.components(n, ei, ej)
    lab = np.arange(n)
    for _ in range(n):                                                # brute force: relax to the fixed point
        new = lab.copy()
        np.minimum.at(new, ei, lab[ej]); np.minimum.at(new, ej, lab[ei])
        if np.array_equal(new, lab):
            break
        lab = new
    has_edge = np.zeros(n, bool); has_edge[ei] = True; has_edge[ej] = True
    assert np.array_equal(sub[has_edge], lab[has_edge]) and (sub[~has_edge] == -1).all()


def test_edges_from_lists_round_trip():
    rng = np.random.default_rng(7)
    pos, vel, mass, r, v = two_body(rng, 1.0, 0.5, 4e-4, 0.3, 1.0, np.zeros(3), np.zeros(3))
    count, lst = oracle.ngb(pos, vel, mass, G, R_NGB, R_MAX, 1.0, 0.5)
    ei, ej = oracle.edges_from_lists(None, count, lst)
    assert sorted(zip(ei.tolist(), ej.tolist())) == [(0, 1), (1, 0)]
    assert oracle.components(2, ei, ej).tolist() == [0, 0]
