"""Structure of the production schedule S1 and of the oracle's sweep driver (-m "not gpu").

Validity conditions: every site in exactly one pair per sweep; within a phase no site
of one pair equals or neighbours a site of another pair (the paper's map rule), so the
parallel result equals the sequential one in any order.
"""
import numpy as np
import pytest

import oracle


def neighbours(i, L):
    x, y = i % L, i // L
    return [y * L + (x + 1) % L, y * L + (x - 1) % L, ((y + 1) % L) * L + x, ((y - 1) % L) * L + x]


@pytest.mark.parametrize("L", [4, 8, 16, 32])
def test_s1_exact_cover_and_conflict_freeness(L):
    N = L * L
    kinds = set()
    for sweep in range(48):
        par = oracle.schedule_params(L, 77, sweep)
        kinds.add(par[:3] if par[0] else (0,))
        count = np.zeros(N, dtype=int)
        addr = set()
        for phase in (0, 1):
            ia, ib, c0, c1, wd = oracle.schedule_s1(L, 77, sweep, phase)
            assert len(ia) == N // 4
            owner = -np.ones(N, dtype=int)
            for k, (a, b) in enumerate(zip(ia, ib)):
                assert a != b and owner[a] < 0 and owner[b] < 0
                owner[a] = owner[b] = k
            for k, (a, b) in enumerate(zip(ia, ib)):
                for s in (a, b):
                    for t in neighbours(int(s), L):
                        assert owner[t] in (-1, k)               # V2: neighbours are inactive or the partner
            np.add.at(count, ia, 1); np.add.at(count, ib, 1)
            # ascending order of a-sites, unique random-number address per pair
            assert (np.diff(ia) > 0).all()
            for t in zip(c0.tolist(), c1.tolist(), wd.tolist()):
                t = t + (phase,)                                 # the phase is part of the counter (c2 = 2*sweep+phase)
                assert t not in addr and t[2] < 4 and t[0] < max(L // 4, 4) and t[1] < L
                addr.add(t)
            if par[0] == 0:   # FAR: partner by XOR with odd masks, same colour, a-sites at even x
                mx, my = par[1], par[2]
                assert mx % 2 == 1 and my % 2 == 1 and 0 < mx < L and 0 < my < L
                xa, ya, xb, yb = ia % L, ia // L, ib % L, ib // L
                assert ((xa ^ mx) == xb).all() and ((ya ^ my) == yb).all() and (xa % 2 == 0).all()
                assert (((xa + ya) & 1) == phase).all() and (((xb + yb) & 1) == phase).all()
            else:             # NEAR: dominoes, b = a + 1 along the axis
                xa, ya, xb, yb = ia % L, ia // L, ib % L, ib // L
                if par[1] == 0:
                    assert (ya == yb).all() and (((xa + 1) % L) == xb).all()
                else:
                    assert (xa == xb).all() and (((ya + 1) % L) == yb).all()
        assert (count == 1).all()                                # every site in exactly one pair per sweep
    if L >= 8:
        assert len(kinds) >= 6                                   # far sweeps and several domino patterns occur


def test_schedule_is_shared_by_replicas_and_changes_with_sweep_and_seed():
    a = [oracle.schedule_params(64, 5, s) for s in range(40)]
    assert [p[0] for p in a] == [s & 1 for s in range(40)]       # even sweeps far, odd sweeps near
    assert len(set(a[0::2])) > 10
    assert a != [oracle.schedule_params(64, 6, s) for s in range(40)]


def make(L, seed, T=1.0, q=None):
    q = L * L // 8 if q is None else q
    return oracle.Lattice(oracle.init_state(L, L, q, 0, seed), 0.5, 1.0, 1.0, seed=seed)


@pytest.mark.parametrize("L", [4, 8, 16, 64])
def test_order_independence_within_a_phase(L):
    """Pin P10: ascending, descending and threaded execution of a phase give identical lattices (V2)."""
    a, b, c = make(L, 5), make(L, 5), make(L, 5)
    ta = a.sweep_s1(0.9, 12, order=0, trace=True)
    tb = b.sweep_s1(0.9, 12, order=1, trace=True)
    tc = c.sweep_s1(0.9, 12, trace=True, threads=3)
    assert (a.code == b.code).all() and (ta == tb).all()
    assert (a.code == c.code).all() and (ta == tc).all()
    assert a.st.sumE == b.st.sumE == c.st.sumE and a.st.n_accept == c.st.n_accept > 0


def test_call_splitting_invariance():
    """Pin P11: the sweep counter is global: 10 sweeps == 3 + 7 sweeps."""
    a, b = make(16, 8), make(16, 8)
    a.sweep_s1(1.1, 10)
    b.sweep_s1(1.1, 3); b.sweep_s1(1.1, 7)
    assert (a.code == b.code).all() and a.st.sumE2 == b.st.sumE2 and a.st.sweep == b.st.sweep == 10


def test_replicas_and_seeds_decorrelate():
    a = make(16, 8); b = make(16, 8); b.st.replica = 1; c = make(16, 9)
    for l in (a, b, c):
        l.sweep_s1(1.0, 3)
    assert (a.code != b.code).any() and (a.code != c.code).any()


def test_trace_and_accumulators_follow_the_definition():
    """U5: E = Delta n2 + V bV + (J/4) bJ per sweep, sums in sweep order; C and chi from the sums."""
    lat = make(8, 3)
    tr = lat.sweep_s1(1.3, 200, trace=True).astype(float)
    E = (0.5 * tr[:, 0] + 1.0 * tr[:, 1]) + 0.25 * tr[:, 2]
    o = lat.observables(1.3)
    assert o["nmeas"] == 200
    np.testing.assert_allclose(o["sumE"], E.sum(), rtol=1e-12)
    np.testing.assert_allclose(o["sumE2"], (E * E).sum(), rtol=1e-12)
    np.testing.assert_allclose(o["sumM2"], (tr[:, 3] ** 2).sum(), rtol=1e-12)
    np.testing.assert_allclose(o["sumAbsMs"], np.abs(tr[:, 4]).sum(), rtol=1e-12)
    np.testing.assert_allclose(o["C"], (np.mean(E * E) - np.mean(E) ** 2) / (64 * 1.3 ** 2), rtol=1e-9)
    np.testing.assert_allclose(o["chi_u"], (np.mean(tr[:, 3] ** 2) - np.mean(tr[:, 3]) ** 2) / (64 * 1.3), rtol=1e-9)
    assert (tr[-1] == lat.ints()).all()


def test_ising_limit_orders_antiferromagnetically():
    """Pin P9 (qualitative): no charges, J > 0 -> 2-D Ising antiferromagnet with coupling J/4; well below
    T_c = (J/4) 2/ln(1+sqrt 2) = 0.567 J the staggered magnetisation saturates and bJ -> -2N."""
    L = 16
    neel = np.fromfunction(lambda y, x: (x + y) % 2, (L, L)).astype(np.int8)
    lat = oracle.Lattice(neel, 50.0, 0.0, 1.0, seed=4)                               # Delta large: no charges
    tr = lat.sweep_s1(0.3, 300, trace=True)
    assert (tr[:, 0] == 0).all()
    assert np.abs(tr[:, 4]).mean() > 0.9 * L * L and tr[:, 2].mean() < -1.8 * L * L   # stays ordered below T_c
    hot = oracle.Lattice(neel, 50.0, 0.0, 1.0, seed=4)
    hot.sweep_s1(5.0, 100)
    tr = hot.sweep_s1(5.0, 200, trace=True)
    assert np.abs(tr[:, 4]).mean() < 0.3 * L * L                                      # melts above T_c


@pytest.mark.parametrize("L", [64, 256, 1024])
def test_random_word_address_is_the_stated_function_of_the_slot_site(L):
    """DESIGN.md U3 "Random-word address": the pair whose slot site is (x, y) -- its a-site, or its b-site for horizontal
    dominoes -- uses word (x >> 2) & 3 of the Philox block with counter c0 = 4 (x >> 4) + (x & 3), c1 = y.  Stated here
    as a plain function of (x, y) and checked for every pair of FAR, NEAR-H and NEAR-V sweeps at sizes where x >> 4 > 0
    (the sampling pins run at L = 4, where it is always 0); addresses are unique within a phase."""
    seen_types = set()
    sweep = 0
    while len(seen_types) < 3 and sweep < 64:
        par = oracle.schedule_params(L, 31, sweep)
        kind = "far" if par[0] == 0 else ("near_h" if par[1] == 0 else "near_v")
        if kind in seen_types:
            sweep += 1
            continue
        seen_types.add(kind)
        for phase in (0, 1):
            ia, ib, c0, c1, wd = oracle.schedule_s1(L, 31, sweep, phase)
            assert len(ia) == L * L // 4
            slot = ib if kind == "near_h" else ia
            x, y = slot % L, slot // L
            assert (c0 == 4 * (x >> 4) + (x & 3)).all() and (c1 == y).all() and (wd == ((x >> 2) & 3)).all()
            assert (c0 >= 4).any() and c0.max() < L // 4                  # blocks beyond the first 16 columns occur
            key = (c1.astype(np.int64) * (L // 4) + c0.astype(np.int64)) * 4 + wd.astype(np.int64)
            assert len(np.unique(key)) == len(key)
        sweep += 1
    assert seen_types == {"far", "near_h", "near_v"}
