"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded inputs.

Bar (BASELINE.json north_star): lattices bit-exact, exact integers (n2,bV,bJ,M,Ms,Q) bit-exact, fp64 sums within 1e-6
relative (they are in fact computed with the same operations in the same order, so the tests also check for equality
where that holds).  Sum S = Q is checked after every run.
"""
import ctypes as C
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import ic_inputs
import oracle

pytestmark = pytest.mark.gpu

NCPU = os.cpu_count() or 1
S_OF = np.array([0, 0, 1, -1])
_ORACLE_RUNS = {}     # oracle results shared by the two state widths of a config (identical inputs, identical expected lattices)


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2301_11735_b200 as p
    return p


def oracle_run(codes, delta, V, J, seed, Ts, nsweeps, trace=False, threads=1):
    """One oracle lattice per replica (replica index = counter field), run in parallel host threads."""
    lats = [oracle.Lattice(codes[r], delta, V, J, seed, replica=r) for r in range(len(Ts))]

    def go(r):
        return lats[r].sweep_s1(Ts[r], nsweeps, trace=trace, threads=threads)

    if len(Ts) > 1 and threads == 1:
        with ThreadPoolExecutor(max_workers=min(NCPU, len(Ts))) as ex:
            traces = list(ex.map(go, range(len(Ts))))
    else:
        traces = [go(r) for r in range(len(Ts))]
    return lats, traces


def check_against_oracle(sim, lats, Ts, rtol=1e-6, exact_sums=True):
    obs = sim.observables()
    for r, lat in enumerate(lats):
        got = sim.state(r)
        assert np.array_equal(got, lat.code), f"replica {r}: lattice differs at {np.argwhere(got != lat.code)[:5]}"
        o, ref = obs[r], lat.observables(Ts[r])
        for k in ("n2", "bV", "bJ", "M", "Ms", "Q", "nmeas"):
            assert o[k] == ref[k], (r, k, o[k], ref[k])
        assert int(S_OF[got].sum()) == sim.Q                              # eq. (2)
        assert np.array_equal(sim.debug_recompute(r), lat.ints())         # incremental == full recomputation
        for k in ("sumE", "sumE2", "sumM", "sumM2", "sumAbsM", "sumMs", "sumMs2", "sumAbsMs", "C", "chi_u", "chi_s"):
            if exact_sums and k.startswith("sum"):
                assert o[k] == ref[k], (r, k, o[k], ref[k])
            assert abs(o[k] - ref[k]) <= rtol * max(1.0, abs(ref[k])), (r, k, o[k], ref[k])


# ------------------------------------------------------------------------------------------------ host logic
def test_threshold_table_matches_oracle(pkg):
    sim = pkg.Sim(16, 0.25, 0.5, 1.0, 1.0, seed=1)
    for (d, V, J) in [(0.5, 1.0, 1.0), (-0.5, 1.0, 2.0), (0.0, 0.5, 1.0), (1.0, 0.25, 1.0), (0.2, 1.0, 1.0)]:
        s = pkg.Sim(16, 0.25, d, V, J, seed=1)
        for T in (0.05, 0.1, 0.8, 1.0, 2.0, 3.2, 4.0):
            tab = s.thresholds(T)
            k = 0
            for dn2 in (-2, 0, 2):
                for dV in range(-16, 17):
                    for dJ in range(-16, 17):
                        assert int(tab[k]) == oracle.threshold(d, V, J, dn2, dV, dJ, T), (d, V, J, T, dn2, dV, dJ)
                        k += 1
        s.close()
    sim.close()


def test_schedule_matches_oracle(pkg):
    for L in (4, 16, 64, 1024):
        sim = pkg.Sim(L, 0.0, 0, 0, 0, seed=1234567890123)
        for s in list(range(40)) + [10 ** 6, 2 ** 31 - 2]:
            assert tuple(sim.schedule(s)) == oracle.schedule_params(L, 1234567890123, s)
        sim.close()


def test_stage1_init_matches_oracle(pkg):
    for (L, n, seed, reps) in [(16, 0.25, 1, 3), (64, 0.1, 2, 2), (64, -0.3, 9, 1), (256, 0.05, 5, 1), (128, -0.1, 6, 2), (2048, 0.2, 7, 1), (8, 1.0, 3, 1), (8, 0.0, 3, 1)]:
        for bits in (8, 2):
            sim = pkg.Sim(L, n, 0.5, 1.0, 1.0, seed=seed, replicas=reps, bits_per_site=bits)
            Q = sim.Q
            assert Q == int(np.floor(abs(n) * L * L + 0.5)) * (1 if n >= 0 else -1)
            for r in range(reps):
                ref = oracle.init_state(L, L, max(Q, 0), max(-Q, 0), seed, r)
                got = sim.state(r)
                assert np.array_equal(got, ref)
                assert np.array_equal(sim.debug_recompute(r), oracle.recompute(ref))
                o = sim.observables()[r]
                assert [o[k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")] == list(oracle.recompute(ref))
            sim.close()
    sim = pkg.Sim(64, 0.0, 0.5, 1.0, 1.0, seed=3)
    sim.init_charges(0, 700, 700)
    assert np.array_equal(sim.state(0), oracle.init_state(64, 64, 700, 700, 3, 0))
    with pytest.raises(pkg.IcError):
        sim.init_charges(0, 10, 9)
    sim.close()


def test_set_state_validation(pkg):
    sim = pkg.Sim(16, 0.25, 0.5, 1.0, 1.0, seed=1)
    good = ic_inputs.random_state(16, 64, 0, seed=5)
    sim.set_state(0, good)
    before = sim.state(0).copy()
    bad = good.copy(); bad[3, 3] = 4
    with pytest.raises(pkg.IcError) as e:
        sim.set_state(0, bad)
    assert e.value.code == pkg.IC_ERR_CHARGE
    wrongq = ic_inputs.random_state(16, 63, 0, seed=5)
    with pytest.raises(pkg.IcError):
        sim.set_state(0, wrongq)
    assert np.array_equal(sim.state(0), before)             # unchanged on error
    with pytest.raises(pkg.IcError):
        sim.sweep(0.0, 1)
    with pytest.raises(pkg.IcError):
        sim.sweep(1.0, -1)
    assert sim.sweep_count == 0
    sim.close()


# ------------------------------------------------------------------------------------------------ trajectories
PARITY_CASES = [
    # L, bits, replicas, (nplus, nminus), (delta, V, J), Ts, nsweeps
    (4, 8, 2, (4, 0), (0.5, 1.0, 1.0), [0.6, 2.0], 200),
    (4, 2, 1, (2, 2), (-0.5, 1.0, 2.0), [1.5], 200),
    (8, 8, 3, (6, 0), (0.5, 1.0, 1.0), [0.3, 1.0, 4.0], 150),
    (8, 2, 2, (0, 10), (0.0, 0.5, 1.0), [0.4, 1.0], 150),
    (16, 8, 4, (64, 0), (0.5, 1.0, 1.0), [0.1, 0.5, 1.0, 4.0], 120),
    (16, 2, 2, (64, 0), (0.5, 1.0, 1.0), [0.1, 2.0], 120),
    (32, 8, 2, (100, 100), (-0.5, 1.0, 2.0), [0.8, 1.6], 80),
    (64, 8, 5, (410, 0), (0.0, 0.5, 1.0), [0.05, 0.5, 1.0, 2.0, 3.2], 60),
    (64, 2, 3, (410, 0), (0.0, 0.5, 1.0), [0.05, 1.0, 3.2], 60),
    (128, 8, 2, (2000, 1000), (1.0, 0.25, 1.0), [0.2, 2.0], 40),
    (128, 2, 2, (2000, 1000), (1.0, 0.25, 1.0), [0.2, 2.0], 40),   # tiled 2-bit layout: two words per plane row
    (256, 8, 1, (0, 0), (0.2, 1.0, 1.0), [1.0], 30),            # no charges: plain Ising with coupling J/4
    (256, 2, 2, (20000, 20000), (-0.5, 1.0, 2.0), [0.8, 0.3], 30),
    (512, 8, 1, (13107, 0), (0.2, 1.0, 1.0), [1.0], 12),
    (512, 2, 1, (13107, 20000), (0.2, 1.0, 1.0), [0.9], 12),
]


@pytest.mark.parametrize("L,bits,reps,charges,par,Ts,nsweeps", PARITY_CASES)
def test_trajectory_parity(pkg, L, bits, reps, charges, par, Ts, nsweeps):
    nplus, nminus = charges
    delta, V, J = par
    seed = 1000 + L + bits
    n = (nplus - nminus) / (L * L)
    codes = [ic_inputs.random_state(L, nplus, nminus, seed, r) for r in range(reps)]
    sim = pkg.Sim(L, n, delta, V, J, seed=seed, replicas=reps, bits_per_site=bits)
    assert sim.Q == nplus - nminus
    for r in range(reps):
        sim.set_state(r, codes[r])
    tr = sim.sweep_trace(Ts, nsweeps)
    lats, traces = oracle_run(codes, delta, V, J, seed, Ts, nsweeps, trace=True)
    check_against_oracle(sim, lats, Ts)
    tr = tr.cpu().numpy()
    for r in range(reps):
        assert np.array_equal(tr[:, r, :], traces[r]), f"per-sweep integers differ, replica {r}"
        assert (tr[:, r, 5] == sim.Q).all()
    sim.close()


def test_call_splitting_and_reset(pkg):
    """The sweep counter is global: 30 sweeps == 7 + 0 + 23 sweeps; reset zeroes the sums only."""
    L, seed = 64, 42
    code = ic_inputs.random_state(L, 300, 110, seed)
    a = pkg.Sim(L, 190 / L / L, 0.5, 1.0, 1.0, seed=seed); a.set_state(0, code)
    b = pkg.Sim(L, 190 / L / L, 0.5, 1.0, 1.0, seed=seed); b.set_state(0, code)
    a.sweep(1.3, 30)
    b.sweep(1.3, 7); b.sweep(1.3, 0); b.sweep(1.3, 23)
    assert a.sweep_count == b.sweep_count == 30
    assert np.array_equal(a.state(0), b.state(0))
    assert a.observables()[0] == b.observables()[0]
    lat = oracle.Lattice(code, 0.5, 1.0, 1.0, seed)
    lat.sweep_s1(1.3, 30)
    check_against_oracle(a, [lat], [1.3])
    a.reset_observables(); lat.reset_observables()
    a.sweep(0.7, 5); lat.sweep_s1(0.7, 5)        # temperature change between calls
    check_against_oracle(a, [lat], [0.7])
    assert a.observables()[0]["nmeas"] == 5
    a.close(); b.close()


@pytest.mark.parametrize("L,bits,bits2", [(8, 8, 8), (64, 8, 2), (256, 2, 8), (1024, 8, 8), (2048, 8, 2)])
def test_resume_continues_the_same_trajectory(pkg, L, bits, bits2):
    """SURVEY sec. 5 (checkpoint / resume): lattice + sweep counter + seed determine the future.  40 sweeps in one context ==
    17 sweeps, save (ic_state, ic_sweep_count, ic_observables), a NEW context (other bits per site allowed), ic_set_state +
    ic_restore, 23 sweeps: lattices, exact integers and the fp64 sums equal with ==, for every kernel family."""
    seed, reps, Ts = 90 + L, 2, [0.8, 1.7]
    N = L * L
    nplus, nminus = N // 8, N // 16
    n = (nplus - nminus) / N
    codes = [ic_inputs.random_state(L, nplus, nminus, seed, r) for r in range(reps)]
    a = pkg.Sim(L, n, 0.4, 1.0, 1.2, seed=seed, replicas=reps, bits_per_site=bits)
    b = pkg.Sim(L, n, 0.4, 1.0, 1.2, seed=seed, replicas=reps, bits_per_site=bits)
    for r in range(reps):
        a.set_state(r, codes[r]); b.set_state(r, codes[r])
    a.sweep(Ts, 40)
    b.sweep(Ts, 17)
    saved = ([b.state(r).copy() for r in range(reps)], b.sweep_count, b.observables())
    b.close()
    c = pkg.Sim(L, n, 0.4, 1.0, 1.2, seed=seed, replicas=reps, bits_per_site=bits2)
    for r in range(reps):
        c.set_state(r, saved[0][r])
    for bad in (lambda: c.restore(-1, saved[2]), lambda: c.restore(1 << 31, saved[2]),
                lambda: c.restore(17, [dict(saved[2][0], sumE=float("nan")), saved[2][1]]),
                lambda: c.restore(17, [dict(saved[2][0], nmeas=-1), saved[2][1]])):
        with pytest.raises(pkg.IcError):
            bad()
    assert c.sweep_count == 0
    c.restore(saved[1], saved[2])
    assert c.sweep_count == 17
    c.sweep(Ts, 23)
    assert c.sweep_count == a.sweep_count == 40
    oa, oc = a.observables(), c.observables()
    for r in range(reps):
        assert np.array_equal(a.state(r), c.state(r)), r
        assert oa[r] == oc[r], (r, oa[r], oc[r])
        assert oa[r]["nmeas"] == 40
    a.close(); c.close()


def _pack_codes(code):
    """Public packing of ic.h: word i = sites 16 i .. 16 i + 15 of the row-major lattice, site k in bits 2k, 2k+1 (plain numpy)."""
    c = np.asarray(code, dtype=np.uint32).reshape(-1, 16)
    return (c << (2 * np.arange(16, dtype=np.uint32))).sum(axis=1, dtype=np.uint64).astype(np.uint32)


@pytest.mark.parametrize("L,bits", [(4, 8), (4, 2), (32, 8), (64, 2), (64, 8), (256, 2), (1024, 8), (2048, 8), (2048, 2)])
def test_packed_state_calls(pkg, L, bits):
    """ic_set_state_packed / ic_state_packed (2 bits per site on the host side) against the byte calls in every
    layout (ROW8, ROW2, P16, P2): the same lattice, the same integers, the same trajectory afterwards; a lattice with the
    wrong charge is refused and leaves the replica as it was."""
    N = L * L
    nplus, nminus = N // 4, N // 8
    n = (nplus - nminus) / N
    code = ic_inputs.random_state(L, nplus, nminus, 700 + L, 0)
    words = _pack_codes(code)
    a = pkg.Sim(L, n, 0.3, 1.0, 0.8, seed=9, replicas=2, bits_per_site=bits)
    b = pkg.Sim(L, n, 0.3, 1.0, 0.8, seed=9, replicas=2, bits_per_site=bits)
    before = b.state(1).copy()
    a.set_state(1, code); b.set_state_packed(1, words)
    assert np.array_equal(b.state(1), code) and np.array_equal(b.state_packed(1), words)
    assert np.array_equal(a.state_packed(1), words)
    assert np.array_equal(b.state(0), a.state(0))                        # the other replica is untouched
    assert list(b.debug_recompute(1)) == list(a.debug_recompute(1))
    oa, ob = a.observables(), b.observables()
    assert all(oa[1][k] == ob[1][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q"))
    bad = code.copy().reshape(-1)
    bad[np.flatnonzero(bad < 2)[0]] = 2                                  # one charge too many
    with pytest.raises(pkg.IcError) as e:
        b.set_state_packed(0, _pack_codes(bad))
    assert e.value.code == pkg.IC_ERR_CHARGE
    assert np.array_equal(b.state(0), a.state(0)) and np.array_equal(b.state(1), code)
    a.sweep([0.9, 1.4], 6); b.sweep([0.9, 1.4], 6)
    for r in range(2):
        assert np.array_equal(a.state(r), b.state(r))
        assert np.array_equal(_pack_codes(a.state(r)), b.state_packed(r))
    assert a.observables() == b.observables()
    assert before.shape == (L, L)
    a.close(); b.close()


@pytest.mark.parametrize("L,bits,family", [(8, 8, 4), (8, 2, 4), (16, 8, 6), (64, 2, 6), (128, 8, 5), (1024, 2, 5), (2048, 8, 3), (2048, 2, 3)])
def test_automatic_selection_runs_the_documented_kernel_family(pkg, L, bits, family):
    """ic_kernel_family: with automatic selection every lattice size runs the family ic.h and DESIGN.md name for it (no silent
    fall-back to the one-thread-per-pair kernels), and an explicit variant is reported as such."""
    sim = pkg.Sim(L, 0.1, 0.2, 1.0, 1.0, seed=3, bits_per_site=bits)
    assert sim.kernel_family == 0
    sim.sweep(1.0, 2)
    assert sim.kernel_family == family
    sim.set_variant(1); sim.sweep(1.0, 1)
    assert sim.kernel_family == 1
    sim.set_variant(0); sim.sweep(1.0, 1)
    assert sim.kernel_family == family
    sim.close()


def test_frozen_and_degenerate_lattices(pkg):
    L = 32
    # n = +-1: every pair has q = +-2, nothing can move; E = N (Delta + 2V) exactly
    for kind, n in (("all_plus", 1.0), ("all_minus", -1.0)):
        sim = pkg.Sim(L, n, 0.5, 1.0, 1.0, seed=3)
        assert (sim.state(0) == (2 if n > 0 else 3)).all()
        sim.sweep(1.0, 6)
        o = sim.observables()[0]
        assert (sim.state(0) == (2 if n > 0 else 3)).all()
        assert o["sumE"] == 6 * L * L * (0.5 + 2 * 1.0)
        sim.close()
    for kind in ("neel", "ferro", "stripes"):
        code = ic_inputs.structured_state(L, kind)
        for T in (0.02, 50.0):
            sim = pkg.Sim(L, 0.0, 0.5, 1.0, 1.0, seed=8, bits_per_site=2); sim.set_state(0, code)
            lat = oracle.Lattice(code, 0.5, 1.0, 1.0, 8)
            sim.sweep(T, 20); lat.sweep_s1(T, 20)
            check_against_oracle(sim, [lat], [T])
            sim.close()


def test_config_c1_full_length(pkg):
    """BASELINE config 1 at full length: L=16, 41 temperatures, 2000 + 10000 sweeps, fp64 observables."""
    c = ic_inputs.CONFIGS["C1"]
    L, Ts = c["L"], c["T"]
    sim = pkg.Sim(L, c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], replicas=len(Ts), bits_per_site=8)
    codes = [sim.state(r).copy() for r in range(len(Ts))]       # stage-1 states (checked against the oracle above)
    for r in range(len(Ts)):
        assert np.array_equal(codes[r], oracle.init_state(L, L, c["nplus"], 0, c["seed"], r))
    lats = [oracle.Lattice(codes[r], c["delta"], c["V"], c["J"], c["seed"], replica=r) for r in range(len(Ts))]

    def go(r):
        lats[r].sweep_s1(Ts[r], c["equil"]); lats[r].reset_observables(); lats[r].sweep_s1(Ts[r], c["sweeps"])

    with ThreadPoolExecutor(max_workers=NCPU) as ex:
        list(ex.map(go, range(len(Ts))))
    sim.sweep(Ts, c["equil"]); sim.reset_observables(); sim.sweep(Ts, c["sweeps"])
    check_against_oracle(sim, lats, Ts)
    obs = sim.observables()
    assert all(o["nmeas"] == c["sweeps"] for o in obs)
    # with the exact constraint the heat capacity stays finite as T -> 0 (that it -> 0 in equilibrium is pinned
    # by the exact 4x4 solution, tests/test_oracle_exact.py and test_gpu_scan.py; a 16x16 lattice quenched from a random
    # state to T = 0.1 may still relax during the measured sweeps, so no bound on the value is asserted here)
    assert all(np.isfinite(o["C"]) and o["C"] >= 0.0 for o in obs)
    sim.close()


def test_config_c2_batched_replicas(pkg):
    """BASELINE config 2 at full length: L=64, 64 temperatures as 64 replicas in one launch, 10^4 sweeps,
    both state widths, every replica against the oracle."""
    c = ic_inputs.CONFIGS["C2"]
    L, Ts, nsw = c["L"], c["T"], c["sweeps"]
    codes = [ic_inputs.random_state(L, c["nplus"], 0, c["seed"], r) for r in range(len(Ts))]
    for bits in (8, 2):
        sim = pkg.Sim(L, c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], replicas=len(Ts), bits_per_site=bits)
        for r in range(len(Ts)):
            sim.set_state(r, codes[r])
        sim.sweep(Ts, nsw)
        if bits == 8:
            lats, _ = oracle_run(codes, c["delta"], c["V"], c["J"], c["seed"], Ts, nsw)
        check_against_oracle(sim, lats, Ts)
        sim.close()


def test_config_c3_packed_l1024(pkg):
    """BASELINE config 3 at full length: L=1024, neutral with both charge signs at density 0.3, 2-bit packed
    state, 10^3 sweeps."""
    c = ic_inputs.CONFIGS["C3"]
    L, nsw = c["L"], c["sweeps"]
    code = ic_inputs.random_state(L, c["nplus"], c["nminus"], c["seed"])
    sim = pkg.Sim(L, c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], bits_per_site=2); sim.set_state(0, code)
    lat = oracle.Lattice(code, c["delta"], c["V"], c["J"], c["seed"])
    sim.sweep(c["T"], nsw); lat.sweep_s1(c["T"][0], nsw, threads=NCPU)
    check_against_oracle(sim, [lat], c["T"])
    sim.close()


@pytest.mark.parametrize("bits", [8, 2])
def test_config_c4_trace_l4096(pkg, bits):
    """BASELINE config 4 in the launch shape bench.py --config C4 times (L=4096, all 16 replicas in one launch: grid
    (sm_count / 16, 16) for the staged kernels): per-sweep integers via ic_sweep_trace for the first 20 sweeps against the
    oracle, replica by replica, then on to 500 sweeps with eq. (2) and incremental == recomputed integers on every replica
    (SURVEY 8(d))."""
    c = ic_inputs.CONFIGS["C4"]
    L, Ts, reps, nsw = c["L"], c["T"], len(c["T"]), 20
    sim = pkg.Sim(L, c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], replicas=reps, bits_per_site=bits)
    codes = [sim.state(r).copy() for r in range(reps)]                   # stage-1 states of ic_create
    for r in (0, reps - 1):
        assert np.array_equal(codes[r], oracle.init_state(L, L, c["nplus"], 0, c["seed"], r))
    tr = sim.sweep_trace(Ts, nsw).cpu().numpy()
    per = max(1, NCPU // 4)

    def go(r):
        lat = oracle.Lattice(codes[r], c["delta"], c["V"], c["J"], c["seed"], replica=r)
        t = lat.sweep_s1(Ts[r], nsw, trace=True, threads=per)
        return lat, t

    if "C4" not in _ORACLE_RUNS:
        with ThreadPoolExecutor(max_workers=4) as ex:
            _ORACLE_RUNS["C4"] = (codes, list(ex.map(go, range(reps))))
    codes0, res = _ORACLE_RUNS["C4"]
    assert all(np.array_equal(a, b) for a, b in zip(codes, codes0))       # the oracle run started from these very states
    for r in range(reps):
        assert np.array_equal(tr[:, r, :], res[r][1]), f"per-sweep integers differ, replica {r}"
    check_against_oracle(sim, [lt for lt, _ in res], Ts)
    tr2 = sim.sweep_trace(Ts, c["sweeps"] - nsw).cpu().numpy()
    assert (tr2[:, :, 5] == sim.Q).all()                                  # eq. (2) after every sweep, every replica
    obs = sim.observables()
    for r in range(reps):
        assert obs[r]["nmeas"] == c["sweeps"]
        assert list(sim.debug_recompute(r)) == [obs[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
        assert list(tr2[-1, r, :]) == [obs[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    sim.close()


@pytest.mark.parametrize("bits", [8, 2])
def test_config_c5_full_size_sampled(pkg, bits):
    """BASELINE config 5 at its full size (L=16384, the launch configuration bench.py times): the first 5 sweeps against
    the multi-threaded oracle, whole lattice compared; then eq. (2) and incremental == recomputed integers after all 100
    sweeps; also at 2 bits per site."""
    c = ic_inputs.CONFIGS["C5"]
    L = c["L"]
    sim = pkg.Sim(L, c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], bits_per_site=bits)
    code = sim.state(0).copy()
    assert int(S_OF[code].sum()) == sim.Q == c["nplus"]
    kinds = {("FAR",) if k[0] == 0 else ("NEAR", k[1]) for k in (sim.schedule(s) for s in range(5))}
    assert kinds == {("FAR",), ("NEAR", 0), ("NEAR", 1)}, kinds     # the compared sweeps run all three kernels: FAR, NEAR-H, NEAR-V
    sim.sweep(c["T"], 5)
    assert sim.kernel_family == 3                                    # the TMA-staged kernels bench.py times
    if "C5" not in _ORACLE_RUNS:
        lat = oracle.Lattice(code, c["delta"], c["V"], c["J"], c["seed"])
        lat.sweep_s1(c["T"][0], 5, threads=NCPU)
        _ORACLE_RUNS["C5"] = (code, lat)
    code0, lat = _ORACLE_RUNS["C5"]
    assert np.array_equal(code, code0)
    got = sim.state(0)
    assert np.array_equal(got, lat.code)
    o = sim.observables()[0]; ref = lat.observables(c["T"][0])
    for k in ("n2", "bV", "bJ", "M", "Ms", "Q", "sumE", "sumE2", "sumM2", "sumMs2"):
        assert o[k] == ref[k], (k, o[k], ref[k])
    sim.sweep(c["T"], c["sweeps"] - 5)
    assert int(S_OF[sim.state(0)].sum()) == sim.Q
    o = sim.observables()[0]
    assert o["nmeas"] == c["sweeps"]
    assert list(sim.debug_recompute(0)) == [o[k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    sim.close()


@pytest.mark.skipif(os.environ.get("IC_LONG_TESTS") != "1", reason="whole-run comparison: about 3 minutes of oracle time; set IC_LONG_TESTS=1")
def test_config_c5_whole_run_against_the_oracle(pkg):
    """BASELINE config 5 for its WHOLE run (100 sweeps at L=16384, what one bench.py step executes), both state widths against the
    multi-threaded oracle: lattice, exact integers and every fp64 sum equal.  Opt-in (IC_LONG_TESTS=1); the default suite
    compares the first 5 sweeps (test_config_c5_full_size_sampled)."""
    c = ic_inputs.CONFIGS["C5"]
    sims = [pkg.Sim(c["L"], c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], bits_per_site=b) for b in (8, 2)]
    code = sims[0].state(0).copy()
    for sim in sims:
        sim.sweep(c["T"], c["sweeps"])
        assert sim.kernel_family == 3
    lat = oracle.Lattice(code, c["delta"], c["V"], c["J"], c["seed"])
    lat.sweep_s1(c["T"][0], c["sweeps"], threads=NCPU)
    ref = lat.observables(c["T"][0])
    for sim in sims:
        assert np.array_equal(sim.state(0), lat.code)
        o = sim.observables()[0]
        for k in ("nmeas", "n2", "bV", "bJ", "M", "Ms", "Q", "sumE", "sumE2", "sumM", "sumM2", "sumAbsM", "sumMs", "sumMs2", "sumAbsMs"):
            assert o[k] == ref[k], (k, o[k], ref[k])
        sim.close()


def test_one_launch_kernel_with_more_replicas_than_sms(pkg):
    """More lattice copies than SMs at L = 128 (2 bits/site): every row of blocks of the one-launch kernel runs several
    replicas one after the other.  Three replicas against the oracle, all against eq. (2) and the recount."""
    import torch
    L, reps, seed, nsw = 128, torch.cuda.get_device_properties(0).multi_processor_count + 9, 61, 12
    Ts = [0.4 + 0.01 * r for r in range(reps)]
    sim = pkg.Sim(L, 0.1, 0.5, 1.0, 1.0, seed=seed, replicas=reps, bits_per_site=2); sim.set_variant(5)
    picks = [0, reps - 10, reps - 1]
    codes = {r: sim.state(r).copy() for r in picks}
    sim.sweep(Ts, nsw)
    obs = sim.observables()
    for r in picks:
        lat = oracle.Lattice(codes[r], 0.5, 1.0, 1.0, seed, replica=r)
        lat.sweep_s1(Ts[r], nsw)
        assert np.array_equal(sim.state(r), lat.code), r
        ref = lat.observables(Ts[r])
        for k in ("n2", "bV", "bJ", "M", "Ms", "Q", "sumE", "sumE2", "nmeas"):
            assert obs[r][k] == ref[k], (r, k)
    for r in range(0, reps, 5):
        assert obs[r]["Q"] == sim.Q and obs[r]["nmeas"] == nsw
        assert list(sim.debug_recompute(r)) == [obs[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    sim.close()


def test_variant_and_block_bound_argument_checks(pkg):
    """ic_set_variant refuses a kernel family that cannot run the context's (L, bits); ic_set_max_blocks a negative bound."""
    small = pkg.Sim(64, 0.1, 0.5, 1.0, 1.0, seed=1)
    for bad in (2 + 1, 5, 7, -1):                  # staged and one-launch kernels need L >= 2048 / 128; 7 does not exist
        with pytest.raises(pkg.IcError) as e:
            small.set_variant(bad)
        assert e.value.code == pkg.IC_ERR_PARAM
    for ok in (0, 1, 2, 4, 6):
        small.set_variant(ok)
    with pytest.raises(pkg.IcError):
        small.set_max_blocks(-1)
    small.set_max_blocks(3); small.set_max_blocks(0)
    small.close()
    mid = pkg.Sim(256, 0.1, 0.5, 1.0, 1.0, seed=1, bits_per_site=2)
    for bad in (2, 3, 4, 6):                       # tiled kernels are 8 bits/site only; resident kernels need L <= 64
        with pytest.raises(pkg.IcError):
            mid.set_variant(bad)
    mid.set_variant(5); mid.set_variant(1); mid.set_variant(0)
    mid.close()


def test_staged_kernels_one_block_per_replica(pkg):
    """More replicas than SMs: the staged kernels run with gridDim.x = 1 (one persistent block per replica walks the whole
    lattice).  L=2048, 160 replicas; three replicas against the oracle, every replica against eq. (2) and the recount."""
    import torch
    L, reps, seed = 2048, torch.cuda.get_device_properties(0).multi_processor_count + 12, 31
    Ts = [0.3 + 0.01 * r for r in range(reps)]
    sim = pkg.Sim(L, 0.1, 0.5, 1.0, 1.0, seed=seed, replicas=reps); sim.set_variant(3)
    picks = [0, reps // 2, reps - 1]
    codes = {r: sim.state(r).copy() for r in picks}
    sim.sweep(Ts, 4)
    obs = sim.observables()
    for r in picks:
        lat = oracle.Lattice(codes[r], 0.5, 1.0, 1.0, seed, replica=r)
        lat.sweep_s1(Ts[r], 4, threads=NCPU)
        assert np.array_equal(sim.state(r), lat.code), r
        assert [obs[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")] == list(lat.ints())
    for r in range(0, reps, 7):
        assert obs[r]["Q"] == sim.Q
        assert list(sim.debug_recompute(r)) == [obs[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    sim.close()


# ------------------------------------------------------------------------------------------------ kernel variants
@pytest.mark.parametrize("L,reps,nsweeps,variant,bits", [(64, 3, 64, 2, 8), (128, 2, 64, 2, 8), (256, 2, 48, 2, 8), (1024, 1, 40, 2, 8),
                                                         (2048, 2, 32, 2, 8), (2048, 2, 48, 3, 8), (4096, 2, 32, 3, 8), (8192, 1, 12, 3, 8),
                                                         (2048, 2, 64, 3, 2), (4096, 2, 48, 3, 2), (8192, 1, 16, 3, 2),
                                                         (128, 3, 64, 5, 8), (128, 2, 64, 5, 2), (256, 2, 64, 5, 2), (512, 1, 48, 5, 8),
                                                         (1024, 1, 48, 5, 8), (1024, 2, 48, 5, 2)])
def test_tiled_kernels_equal_reference_kernels(pkg, L, reps, nsweeps, variant, bits):
    """Variant 2 (tiled, L <= 2048), variant 3 (TMA-staged, L >= 2048) and variant 5 (one cooperative launch for all the
    sweeps of a call, 128 <= L <= 1024) against variant 1 (one thread per pair) on the
    same device memory layout, sweep by sweep so that many (mx, my) masks, both domino orientations and all four offsets
    are exercised; the reference kernels are themselves compared with the oracle above and (at L <= 256) here."""
    seed = 4242 + L
    nplus, nminus = L * L // 10, L * L // 20
    n = (nplus - nminus) / (L * L)
    Ts = [0.4, 1.1, 2.5][:reps]
    codes = [ic_inputs.random_state(L, nplus, nminus, seed, r) for r in range(reps)]
    a = pkg.Sim(L, n, 0.3, 1.0, 1.5, seed=seed, replicas=reps, bits_per_site=bits); a.set_variant(variant)
    b = pkg.Sim(L, n, 0.3, 1.0, 1.5, seed=seed, replicas=reps, bits_per_site=bits); b.set_variant(1)
    for r in range(reps):
        a.set_state(r, codes[r]); b.set_state(r, codes[r])
    seen = set()
    for s in range(nsweeps):
        seen.add(a.schedule(s)[:2] if a.schedule(s)[0] else (0, (a.schedule(s)[1] >> 2) & 15))
        a.sweep(Ts, 1); b.sweep(Ts, 1)
        oa, ob = a.observables(), b.observables()
        for r in range(reps):
            assert oa[r] == ob[r], (s, r, a.schedule(s))
        if s % 8 == 7 or s == nsweeps - 1:
            for r in range(reps):
                assert np.array_equal(a.state(r), b.state(r)), (s, r, a.schedule(s))
    if L <= 256:
        lats, _ = oracle_run(codes, 0.3, 1.0, 1.5, seed, Ts, nsweeps)
        check_against_oracle(a, lats, Ts)
    if variant == 5:
        # many sweeps inside ONE launch (the barriers between phases and sweeps are what is new), with the per-sweep trace
        tra = a.sweep_trace(Ts, 40).cpu().numpy(); trb = b.sweep_trace(Ts, 40).cpu().numpy()
        assert np.array_equal(tra, trb)
        a.sweep(Ts, 25); a.sweep(Ts, 15); b.sweep(Ts, 40)
        assert a.observables() == b.observables()
        for r in range(reps):
            assert np.array_equal(a.state(r), b.state(r)), r
            assert list(a.debug_recompute(r)) == [a.observables()[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    a.close(); b.close()


@pytest.mark.parametrize("bits", [8, 2])
def test_staged_kernels_against_oracle_l2048(pkg, bits):
    """Variant 3 (TMA-staged regions) at its smallest size against the oracle: several FAR and NEAR sweeps, 2 replicas;
    both tiled layouts (one byte and two bits per site)."""
    L, seed, nsw = 2048, 77, 6
    nplus, nminus = L * L // 8, L * L // 16
    Ts = [0.7, 1.9]
    codes = [ic_inputs.random_state(L, nplus, nminus, seed, r) for r in range(2)]
    sim = pkg.Sim(L, (nplus - nminus) / (L * L), -0.5, 1.0, 2.0, seed=seed, replicas=2, bits_per_site=bits); sim.set_variant(3)
    for r in range(2):
        sim.set_state(r, codes[r])
    Ts2 = [1.3, 0.45]                                  # the temperatures change between the calls: new class tables
    sim.sweep(Ts, nsw // 2); sim.sweep(Ts2, nsw - nsw // 2)
    lats = [oracle.Lattice(codes[r], -0.5, 1.0, 2.0, seed, replica=r) for r in range(2)]
    for r in range(2):
        lats[r].sweep_s1(Ts[r], nsw // 2, threads=NCPU); lats[r].sweep_s1(Ts2[r], nsw - nsw // 2, threads=NCPU)
    check_against_oracle(sim, lats, Ts2)
    sim.close()


def test_staged_kernels_self_partnered_regions(pkg):
    """FAR sweep whose mask keeps every staged region its own partner (my < 4 and mx < 2048 at L = 2048): the seed is
    searched with the oracle's schedule function; one FAR + one NEAR sweep against the oracle and the reference kernels."""
    L = 2048
    seed = next(sd for sd in range(1, 200000) if oracle.schedule_params(L, sd, 0)[2] < 4)
    typ, mx, my, _ = oracle.schedule_params(L, seed, 0)
    assert typ == 0 and my < 4
    code = ic_inputs.random_state(L, L * L // 10, L * L // 10, seed)
    a = pkg.Sim(L, 0.0, 0.5, 1.0, 1.0, seed=seed); a.set_variant(3); a.set_state(0, code)
    b = pkg.Sim(L, 0.0, 0.5, 1.0, 1.0, seed=seed); b.set_variant(1); b.set_state(0, code)
    assert tuple(a.schedule(0)) == (typ, mx, my, 0)
    lat = oracle.Lattice(code, 0.5, 1.0, 1.0, seed)
    a.sweep(1.2, 2); b.sweep(1.2, 2); lat.sweep_s1(1.2, 2, threads=NCPU)
    assert np.array_equal(a.state(0), b.state(0))
    check_against_oracle(a, [lat], [1.2])
    a.close(); b.close()


@pytest.mark.parametrize("L,bits,variant", [(2048, 8, 3), (2048, 2, 3), (4096, 8, 3), (512, 8, 5), (512, 2, 5), (1024, 8, 2)])
def test_results_do_not_depend_on_the_number_of_blocks(pkg, L, bits, variant):
    """The persistent kernels with 1, 2, 3, 5, 37 blocks per replica and with the automatic grid: every block then walks
    many tasks (many laps of the staged kernels' shared-memory ring, many arrivals at the one-launch kernel's barrier) and
    the task-to-block assignment changes.  Lattices and observables must equal those of the one-thread-per-pair kernels
    after every sweep group.  (No sanitizer is available on the GPU pool; this is the race check the library offers.)"""
    seed, nsw = 555 + L, 12
    nplus, nminus = L * L // 10, L * L // 25
    code = ic_inputs.random_state(L, nplus, nminus, seed)
    ref = pkg.Sim(L, (nplus - nminus) / (L * L), 0.3, 1.0, 1.5, seed=seed, bits_per_site=bits); ref.set_variant(1); ref.set_state(0, code)
    ref.sweep(0.9, nsw)
    want, wobs = ref.state(0).copy(), ref.observables()[0]
    ref.close()
    for cap in (1, 2, 3, 5, 37, 0):
        sim = pkg.Sim(L, (nplus - nminus) / (L * L), 0.3, 1.0, 1.5, seed=seed, bits_per_site=bits)
        sim.set_variant(variant); sim.set_max_blocks(cap); sim.set_state(0, code)
        sim.sweep(0.9, nsw // 2); sim.sweep(0.9, nsw - nsw // 2)
        assert np.array_equal(sim.state(0), want), cap
        assert sim.observables()[0] == wobs, cap
        sim.close()


@pytest.mark.parametrize("L,bits,reps,variant", [(4, 8, 2, 4), (8, 2, 3, 4), (16, 8, 5, 4), (32, 2, 2, 4), (64, 8, 3, 4), (64, 2, 2, 4),
                                                 (16, 8, 5, 6), (16, 2, 3, 6), (32, 8, 2, 6), (32, 2, 2, 6), (64, 8, 3, 6), (64, 2, 2, 6)])
def test_resident_kernel_equals_reference_kernels(pkg, L, bits, reps, variant):
    """Variants 4 and 6 (one launch for all sweeps, lattice resident in shared memory: one thread per pair / four-pair items,
    the defaults for L < 16 / 16 <= L <= 64) against variant 1 (one thread per pair, three launches per sweep): lattices,
    integers, fp64 sums and the per-sweep trace, with the call split in two on one side and a temperature change in between."""
    seed = 900 + L + bits
    nplus, nminus = L * L // 8, L * L // 16
    n = (nplus - nminus) / (L * L)
    Ts = [0.3, 0.9, 1.7, 2.6, 3.9][:reps]
    codes = [ic_inputs.random_state(L, nplus, nminus, seed, r) for r in range(reps)]
    a = pkg.Sim(L, n, -0.5, 1.0, 2.0, seed=seed, replicas=reps, bits_per_site=bits); a.set_variant(variant)
    b = pkg.Sim(L, n, -0.5, 1.0, 2.0, seed=seed, replicas=reps, bits_per_site=bits); b.set_variant(1)
    for r in range(reps):
        a.set_state(r, codes[r]); b.set_state(r, codes[r])
    ta = a.sweep_trace(Ts, 37).cpu().numpy()
    tb = np.concatenate([b.sweep_trace(Ts, 20).cpu().numpy(), b.sweep_trace(Ts, 17).cpu().numpy()])
    assert np.array_equal(ta, tb)
    Ts2 = [t + 0.25 for t in Ts]
    a.sweep(Ts2, 11); b.sweep(Ts2, 11)
    assert a.sweep_count == b.sweep_count == 48
    oa, ob = a.observables(), b.observables()
    for r in range(reps):
        assert oa[r] == ob[r], (r, oa[r], ob[r])
        assert np.array_equal(a.state(r), b.state(r))
        assert list(a.debug_recompute(r)) == [oa[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    a.close(); b.close()


def test_large_lattice_invariants_l32768(pkg):
    """A lattice beyond BASELINE's sizes (L = 32768, 1 GiB at one byte per site: 8 segments per plane row, 2^19 staged
    regions): no oracle run at this size, but eq. (2) holds exactly and the incrementally tracked integers equal the full
    recomputation from eq. (3) after FAR and NEAR sweeps."""
    L = 32768
    sim = pkg.Sim(L, 0.05, 0.2, 1.0, 1.0, seed=9)
    assert sim.Q == int(np.floor(0.05 * L * L + 0.5))
    sim.sweep(1.0, 4)
    o = sim.observables()[0]
    assert o["Q"] == sim.Q and o["nmeas"] == 4
    assert list(sim.debug_recompute(0)) == [o[k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    sim.close()


@pytest.mark.parametrize("case", ["self_partnered", "paired_across_segments_only"])
def test_staged_kernels_rare_far_masks_l4096(pkg, case):
    """L = 4096 has two staged regions per row quad.  FAR masks with my < 4 keep the partner in the same row quad: with
    mx < 2048 every region is its own partner, with mx >= 2048 regions pair across the two segments only.  Such masks come
    up once in a thousand sweeps, so the seed is searched with the oracle's schedule function; the staged kernels are
    compared with the one-thread-per-pair kernels (themselves checked against the oracle) after a FAR and a NEAR sweep."""
    L = 4096
    want_low = case == "self_partnered"
    seed = next(sd for sd in range(1, 400000)
                if oracle.schedule_params(L, sd, 0)[2] < 4 and (oracle.schedule_params(L, sd, 0)[1] < 2048) == want_low)
    typ, mx, my, _ = oracle.schedule_params(L, seed, 0)
    assert typ == 0 and my < 4 and (mx < 2048) == want_low
    code = ic_inputs.random_state(L, L * L // 10, L * L // 12, seed)
    n = (L * L // 10 - L * L // 12) / (L * L)
    a = pkg.Sim(L, n, 0.5, 1.0, 1.0, seed=seed); a.set_variant(3); a.set_state(0, code)
    b = pkg.Sim(L, n, 0.5, 1.0, 1.0, seed=seed); b.set_variant(1); b.set_state(0, code)
    assert tuple(a.schedule(0)) == (typ, mx, my, 0)
    a.sweep(0.9, 2); b.sweep(0.9, 2)
    assert np.array_equal(a.state(0), b.state(0))
    assert a.observables()[0] == b.observables()[0]
    assert list(a.debug_recompute(0)) == [a.observables()[0][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")]
    a.close(); b.close()


def test_staged_kernels_equal_reference_kernels_at_bench_size(pkg):
    """The launch configuration bench.py times (L = 16384: 8192 tasks per phase over 148 persistent blocks, every ring slot
    reused ~9 times per launch) against the one-thread-per-pair kernels, lattices compared after every second sweep: a
    protocol error in the producer/consumer ring shows up here as sporadically wrong row quads."""
    L = 16384
    a = pkg.Sim(L, 0.05, 0.2, 1.0, 1.0, seed=5); a.set_variant(3)
    b = pkg.Sim(L, 0.05, 0.2, 1.0, 1.0, seed=5); b.set_variant(1)
    for s in range(4):
        a.sweep(1.0, 2); b.sweep(1.0, 2)
        assert np.array_equal(a.state(0), b.state(0)), (s, a.schedule(2 * s), a.schedule(2 * s + 1))
        assert a.observables()[0] == b.observables()[0]
    a.close(); b.close()
