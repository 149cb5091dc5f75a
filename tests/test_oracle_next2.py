"""Pins for the NEXT-2 oracle routines: subsystem-aware sums (Alg. 1 "Acceleration
calculations ignore intra-subsystem contributions", L299 §3.5.2, L488 §3.8) and the shared subsystem
time-step of Eq. 20 (L303).  No GPU.

Each pin uses something other than the routine under test: the already-pinned plain routines through
index lists (partial sums), closed degenerate cases, or an independent numpy brute force."""
import numpy as np
import pytest

import oracle


def cluster(n, seed, n_sub=4, sub_size=3):
    rng = np.random.default_rng(seed)
    pos = rng.normal(size=(n, 3))
    vel = rng.normal(size=(n, 3)) * 0.3
    mass = rng.uniform(0.2, 2.0, n)
    subsys = np.full(n, -1, np.int32)
    ids = rng.permutation(n)[: n_sub * sub_size].reshape(n_sub, sub_size)
    for s, members in enumerate(ids):
        subsys[members] = s
        # make the members close, like a real compact subsystem
        pos[members] = pos[members[0]] + 1e-3 * rng.normal(size=(sub_size, 3))
    return pos, vel, mass, subsys


def members_of(subsys, i):
    return np.flatnonzero((subsys == subsys[i]) & (subsys[i] >= 0)).astype(np.int32)


def test_no_subsystems_reproduces_the_plain_routines_bit_for_bit():
    pos, vel, mass, _ = cluster(60, 1)
    none = np.full(60, -1, np.int32)
    a = oracle.acc(pos, mass, 1.3, 0.01)
    assert np.array_equal(oracle.acc_sub(pos, mass, 1.3, 0.01, none), a)
    assert np.array_equal(oracle.grad_sub(pos, mass, a, 1.3, 0.01, none), oracle.grad(pos, mass, a, 1.3, 0.01))
    assert np.array_equal(oracle.jerk_sub(pos, vel, mass, 1.3, 0.01, none), oracle.jerk(pos, vel, mass, 1.3, 0.01))
    assert np.array_equal(oracle.phi_sub(pos, mass, 1.3, 0.01, none), oracle.phi(pos, mass, 1.3, 0.01))
    d0, d1 = oracle.dtmin(pos, vel, mass, 1.3, 0.02, 0.03), oracle.dtmin_sub(pos, vel, mass, 1.3, 0.02, 0.03, none)
    assert all(np.array_equal(d0[k], d1[k]) for k in d0)
    bh = np.array([3, 17], np.int32)
    assert np.array_equal(oracle.pn1_sub(pos, vel, mass, bh, 1.3, 50.0, none), oracle.pn1(pos, vel, mass, bh, 1.3, 50.0))


@pytest.mark.parametrize("eps", [0.0, 0.05])
def test_excluded_plus_intra_subsystem_partial_sum_is_the_full_sum(eps):
    """a_i(all) = a_i(excluding S_i) + a_i(sources = S_i): the last term through the pinned plain
    routine with an index list.  The intra-subsystem term is ~1e6 times larger than the rest, so a
    wrong mask cannot hide in the tolerance."""
    pos, vel, mass, subsys = cluster(80, 2)
    G = 0.7
    full = oracle.acc(pos, mass, G, eps)
    excl = oracle.acc_sub(pos, mass, G, eps, subsys)
    jfull, jexcl = oracle.jerk(pos, vel, mass, G, eps), oracle.jerk_sub(pos, vel, mass, G, eps, subsys)
    pfull, pexcl = oracle.phi(pos, mass, G, eps), oracle.phi_sub(pos, mass, G, eps, subsys)
    gfull, gexcl = oracle.grad(pos, mass, full, G, eps), oracle.grad_sub(pos, mass, full, G, eps, subsys)
    for i in range(80):
        mem = members_of(subsys, i)
        one = np.array([i], np.int32)
        if mem.size == 0:
            assert np.array_equal(excl[i], full[i]) and np.array_equal(gexcl[i], gfull[i])
            continue
        intra = oracle.acc(pos, mass, G, eps, sink_idx=one, src_idx=mem)[0]
        scale = np.abs(intra).max()
        if eps == 0.0:
            assert scale > 1e3 * np.abs(excl[i]).max()
        scale = max(scale, np.abs(full[i]).max())
        assert np.abs(excl[i] + intra - full[i]).max() <= 8e-16 * scale
        intra_j = oracle.jerk(pos, vel, mass, G, eps, sink_idx=one, src_idx=mem)[0]
        assert np.abs(jexcl[i] + intra_j - jfull[i]).max() <= 8e-16 * max(np.abs(intra_j).max(), np.abs(jfull[i]).max())
        intra_p = oracle.phi(pos, mass, G, eps, sink_idx=one, src_idx=mem)[0]
        assert abs(pexcl[i] + intra_p - pfull[i]) <= 8e-16 * max(abs(intra_p), abs(pfull[i]))
        intra_g = oracle.grad(pos, mass, full, G, eps, sink_idx=one, src_idx=mem)[0]
        assert np.abs(gexcl[i] + intra_g - gfull[i]).max() <= 8e-16 * max(np.abs(intra_g).max(), np.abs(gfull[i]).max())


def test_one_all_embracing_subsystem_gives_nothing():
    """"If all particles on a single hierarchy level end up in the same subsystem":
    no pair survives: zero sums, +inf time-steps with id -1."""
    pos, vel, mass, _ = cluster(20, 3)
    one = np.zeros(20, np.int32)
    assert np.all(oracle.acc_sub(pos, mass, 1.0, 0.0, one) == 0)
    assert np.all(oracle.grad_sub(pos, mass, vel, 1.0, 0.0, one) == 0)
    assert np.all(oracle.phi_sub(pos, mass, 1.0, 0.0, one) == 0)
    assert np.all(oracle.pn1_sub(pos, vel, mass, np.array([0, 5], np.int32), 1.0, 30.0, one) == 0)
    d = oracle.dtmin_sub(pos, vel, mass, 1.0, 0.01, 0.01, one)
    assert np.isinf(d["dt_ff"]).all() and np.isinf(d["dt_fb"]).all()
    assert (d["j_ff"] == -1).all() and (d["j_fb"] == -1).all()


def test_dtmin_sub_against_masked_numpy_brute_force():
    pos, vel, mass, subsys = cluster(70, 4)
    G, eff, efb = 1.1, 0.02, 0.05
    sinks = np.arange(0, 70, 3, dtype=np.int32)
    srcs = np.random.default_rng(9).permutation(70).astype(np.int32)[:60]
    d = oracle.dtmin_sub(pos, vel, mass, G, eff, efb, subsys, sink_idx=sinks, src_idx=srcs)
    for k, i in enumerate(sinks):
        ok = np.array([(j != i) and not (subsys[i] >= 0 and subsys[i] == subsys[j]) for j in srcs])
        js = srcs[ok]
        r = np.sqrt(((pos[js] - pos[i]) ** 2).sum(1))
        v = np.sqrt(((vel[js] - vel[i]) ** 2).sum(1))
        tff = eff * np.sqrt(r ** 3 / (G * (mass[i] + mass[js])))
        tfb = efb * r / v
        assert d["j_ff"][k] == js[np.argmin(tff)] and d["j_fb"][k] == js[np.argmin(tfb)]
        assert abs(d["dt_ff"][k] / tff.min() - 1) < 1e-14 and abs(d["dt_fb"][k] / tfb.min() - 1) < 1e-14
        # the excluded partner would otherwise have won: the exclusion is doing something
    plain = oracle.dtmin(pos, vel, mass, G, eff, efb, sink_idx=sinks, src_idx=srcs)
    in_sub = subsys[sinks] >= 0
    assert (plain["dt_ff"][in_sub] < d["dt_ff"][in_sub]).any()
    assert np.array_equal(plain["dt_ff"][~in_sub], d["dt_ff"][~in_sub])


def test_pn1_sub_additivity_and_partner_exclusion():
    """A BH and its subsystem partners exchange no PN kick; everything else is the
    plain routine's.  out_excl + (pairs inside subsystems, from the pinned pn1 on the sub-cluster) = out_full."""
    pos, vel, mass, subsys = cluster(40, 5, n_sub=3, sub_size=3)
    G, c = 1.0, 40.0
    bh = np.array([int(np.flatnonzero(subsys == 0)[0]), int(np.flatnonzero(subsys == -1)[0])], np.int32)
    full = oracle.pn1(pos, vel, mass, bh, G, c)
    excl = oracle.pn1_sub(pos, vel, mass, bh, G, c, subsys)
    mem = np.flatnonzero(subsys == 0)
    # intra-subsystem PN terms: the plain routine on the 3-body sub-cluster with its BH
    sub_out = oracle.pn1(pos[mem], vel[mem], mass[mem], np.array([0], np.int32), G, c)
    expect = full.copy()
    expect[mem] -= sub_out
    scale = np.abs(full).max(axis=1, keepdims=True) + np.abs(expect).max(axis=1, keepdims=True)
    assert (np.abs(excl - expect) <= 1e-14 * scale + 1e-300).all()
    assert np.abs(sub_out).max() > 0


def test_subsys_min_is_the_segment_minimum():
    rng = np.random.default_rng(6)
    n = 200
    subsys = rng.integers(-1, 12, n).astype(np.int32)
    dt = rng.uniform(1e-6, 1e-2, n)
    out = oracle.subsys_min(subsys, dt)
    single = subsys < 0
    assert np.array_equal(out[single], dt[single])
    for s in range(12):
        m = subsys == s
        if m.any():
            assert np.all(out[m] == dt[m].min())
    # idempotent, never increases
    assert np.array_equal(oracle.subsys_min(subsys, out), out) and np.all(out <= dt)
