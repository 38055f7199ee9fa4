"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

Every function of oracle/ic_oracle.c is checked against something other than itself: known-answer
vectors, closed forms, brute force on tiny inputs, exact enumeration.  See the pin list in the header of
oracle/ic_oracle.c and in DESIGN.md.
"""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import exact

S_OF = {0: 0, 1: 0, 2: 1, 3: -1}      # S=+-1 charge states, S=0 magnetic
SG_OF = {0: 1, 1: -1, 2: 0, 3: 0}     # sigma = 2(1-S^2)s


# ---------------------------------------------------------------- Philox (U3)
def test_philox_known_answers(golden_dir):
    rows = [ln.split() for ln in open(os.path.join(golden_dir, "philox_kat.txt")) if ln.strip() and ln[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_seven_rounds_by_inverting_the_known_answers(golden_dir):
    """The update stream uses Philox4x32-7 (G5).  Pin: ten rounds = three more rounds on top of seven, and a
    round is a bijection, so the seven-round output must equal the published ten-round answer with rounds 10, 9, 8
    undone.  The inverse round is written here from the definition (multiplicative inverses of the odd multipliers
    modulo 2^32), independently of the oracle's forward code."""
    M0, M1, W0, W1, MASK = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85, 0xFFFFFFFF
    I0, I1 = pow(M0, -1, 1 << 32), pow(M1, -1, 1 << 32)
    rows = [ln.split() for ln in open(os.path.join(golden_dir, "philox_kat.txt")) if ln.strip() and ln[0] != "#"]
    for r in rows:
        v = [int(t, 16) for t in r]
        ctr, key, n = v[0:4], v[4:6], v[6:10]
        for rnd in (9, 8, 7):                                   # undo round index rnd (key bumped rnd times)
            k0, k1 = (key[0] + rnd * W0) & MASK, (key[1] + rnd * W1) & MASK
            c2 = (n[1] * I1) & MASK; c0 = (n[3] * I0) & MASK    # lo words carry M * c mod 2^32
            c1 = n[0] ^ ((M1 * c2) >> 32) ^ k0; c3 = n[2] ^ ((M0 * c0) >> 32) ^ k1
            n = [c0, c1, c2, c3]
        assert [int(x) for x in oracle.philox4x32(ctr, key, 7)] == n
        assert [int(x) for x in oracle.philox4x32(ctr, key, 10)] == v[6:10]
    assert oracle.UPDATE_ROUNDS == 7


def test_philox_counter_sensitivity():
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    for i in range(4):
        c = [1, 2, 3, 4]; c[i] ^= 1
        assert (oracle.philox4x32_10(c, [5, 6]) != base).any()
    assert (oracle.philox4x32_10([1, 2, 3, 4], [5, 7]) != base).any()


# ---------------------------------------------------------------- proposal table
def test_pair_table_class_sizes_and_order():
    sizes = {q: sum(oracle.pair_table(q, i) is not None for i in range(8)) for q in (-2, -1, 0, 1, 2)}
    assert sizes == {-2: 1, -1: 4, 0: 6, 1: 4, 2: 1}          # "1 / 4 / 6 configurations"
    for q in (-2, -1, 0, 1, 2):
        seen = set()
        for i in range(sizes[q]):
            a, b = oracle.pair_table(q, i)
            assert S_OF[a] + S_OF[b] == q
            seen.add((a, b))
        assert len(seen) == sizes[q]
    # listing order of PAPER.md:69: (+-1, 1/2), (+-1, -1/2), (1/2, +-1), (-1/2, +-1)
    assert [oracle.pair_table(1, i) for i in range(4)] == [(2, 0), (2, 1), (0, 2), (1, 2)]
    assert [oracle.pair_table(-1, i) for i in range(4)] == [(3, 0), (3, 1), (0, 3), (1, 3)]
    # (+-1, -+1), (+-1/2, +-1/2), (+-1/2, -+1/2)
    assert [oracle.pair_table(0, i) for i in range(6)] == [(2, 3), (3, 2), (0, 0), (1, 1), (0, 1), (1, 0)]
    # all configurations with a given q are in the table (brute force over the 16 pair states)
    for q in (-2, -1, 0, 1, 2):
        allq = {(a, b) for a in range(4) for b in range(4) if S_OF[a] + S_OF[b] == q}
        assert allq == {oracle.pair_table(q, i) for i in range(sizes[q])}


# ---------------------------------------------------------------- threshold (U2)
def test_threshold_closed_form():
    rng = np.random.default_rng(0)
    for _ in range(2000):
        d, V, J = rng.uniform(-2, 2, 3)
        T = rng.uniform(0.05, 4.0)
        dn2, dV, dJ = int(rng.choice([-2, 0, 2])), int(rng.integers(-16, 17)), int(rng.integers(-16, 17))
        t = oracle.threshold(d, V, J, dn2, dV, dJ, T)
        dE = (d * dn2 + V * dV) + (0.25 * J) * dJ
        if dE <= 0:
            assert t == 2 ** 29
        else:
            p = math.exp(-dE / T)
            assert t == min(max(math.floor(p * 2 ** 29), 1), 2 ** 29 - 1)
            assert abs(t / 2 ** 29 - p) <= 2.0 ** -29 + 1e-18   # acceptance probability within one quantum
    # limits and monotonicity in dE
    assert oracle.threshold(0, 1, 0, 0, 0, 0, 1.0) == 2 ** 29
    assert oracle.threshold(0, 1, 0, 0, 16, 0, 0.01) == 1
    ts = [oracle.threshold(0.0, 1.0, 0.0, 0, k, 0, 1.0) for k in range(-3, 17)]
    assert all(a >= b for a, b in zip(ts, ts[1:]))
    # J enters with the prefactor 1/4 (eq. 3, reading G4): dJ=4 at J=1 equals dV=1 at V=1
    assert oracle.threshold(0, 1, 1, 0, 0, 4, 0.7) == oracle.threshold(0, 1, 1, 0, 1, 0, 0.7)


# ---------------------------------------------------------------- eq. (3) recomputation
def brute_ints(code):
    """eq. (3) by explicit loops: every site with its +x and +y neighbour."""
    Ly, Lx = code.shape
    n2 = bV = bJ = M = Ms = Q = 0
    for y in range(Ly):
        for x in range(Lx):
            c = int(code[y, x])
            n2 += S_OF[c] ** 2; M += SG_OF[c]; Ms += (-1) ** (x + y) * SG_OF[c]; Q += S_OF[c]
            for (xx, yy) in (((x + 1) % Lx, y), (x, (y + 1) % Ly)):
                d = int(code[yy, xx])
                bV += S_OF[c] * S_OF[d]; bJ += SG_OF[c] * SG_OF[d]
    return np.array([n2, bV, bJ, M, Ms, Q])


@pytest.mark.parametrize("shape", [(3, 3), (4, 2), (2, 4), (5, 5), (4, 4), (8, 8), (3, 7)])
def test_recompute_against_bruteforce(shape):
    rng = np.random.default_rng(1)
    for _ in range(20):
        code = rng.integers(0, 4, size=shape).astype(np.int8)
        assert (oracle.recompute(code) == brute_ints(code)).all()


def test_frozen_lattice_closed_form():
    # n = +-1: every site charged, E = N(Delta + 2V) exactly (SURVEY pin P9): n2 = N, bV = 2N, bJ = 0
    for c, q in ((2, 1), (3, -1)):
        code = np.full((8, 8), c, dtype=np.int8)
        assert list(oracle.recompute(code)) == [64, 128, 0, 0, 0, 64 * q]
        lat = oracle.Lattice(code, 0.5, 1.0, 1.0, seed=3)
        lat.sweep_s1(1.0, 5); lat.sweep_s0(1.0, 5)
        assert (lat.code == c).all() and lat.st.n_accept == 0        # q=+-2 pairs are never changed
    # Neel state of the pure magnet: bJ = -2N, Ms = N
    code = np.fromfunction(lambda y, x: (x + y) % 2, (6, 6)).astype(np.int8)
    assert list(oracle.recompute(code)) == [0, 0, -72, 0, 36, 0]


# ---------------------------------------------------------------- pair update (U1, eq. 4/5)
@pytest.mark.parametrize("shape", [(3, 3), (2, 4), (4, 2), (4, 4), (5, 5), (8, 8)])
def test_pair_update_matches_full_recomputation(shape):
    """Incrementally tracked (n2,bV,bJ,M,Ms) == full recomputation after every move; sum S conserved (eq. 2)."""
    rng = np.random.default_rng(2)
    Ly, Lx = shape
    code = rng.integers(0, 4, size=shape).astype(np.int8)
    lat = oracle.Lattice(code, 0.3, 1.0, 1.0, seed=1)
    Q = int(lat.st.Q)
    n_adj = n_far = n_changed = 0
    for it in range(3000):
        a = int(rng.integers(0, Lx * Ly))
        if it % 2:   # neighbouring pair (eq. 5)
            xa, ya = a % Lx, a // Lx
            dx, dy = [(1, 0), (-1, 0), (0, 1), (0, -1)][int(rng.integers(0, 4))]
            xb, yb = (xa + dx) % Lx, (ya + dy) % Ly
            n_adj += 1
        else:        # any other site (eq. 4 when distant)
            b = int(rng.integers(0, Lx * Ly - 1)); b += b >= a
            xa, ya, xb, yb = a % Lx, a // Lx, b % Lx, b // Lx
            n_far += 1
        if (xa, ya) == (xb, yb):
            continue
        n_changed += lat.pair_update(xa, ya, xb, yb, int(rng.integers(0, 2 ** 32)), 2.0)
        assert (brute_ints(lat.code) == lat.ints()).all()
        assert lat.st.Q == Q
    assert n_changed > 300


def test_printed_EJ_is_garbled_EV_is_right():
    """Reading G1: eq. (4)/(5) E_V as printed is exact; E_J as printed is not."""
    rng = np.random.default_rng(3)
    L = 5
    bad_J = bad_V = moves = 0
    for _ in range(4000):
        code = rng.integers(0, 4, size=(L, L)).astype(np.int8)
        a = int(rng.integers(0, L * L)); xa, ya = a % L, a // L
        if rng.integers(0, 2):
            dx, dy = [(1, 0), (-1, 0), (0, 1), (0, -1)][int(rng.integers(0, 4))]
            xb, yb = (xa + dx) % L, (ya + dy) % L; adj = 1
        else:
            xb, yb = (xa + 2) % L, (ya + 2) % L; adj = 0
        ca, cb = int(code[ya, xa]), int(code[yb, xb])
        q = S_OF[ca] + S_OF[cb]
        if abs(q) == 2:
            continue
        k = 4 if abs(q) == 1 else 6
        na, nb = oracle.pair_table(q, int(rng.integers(0, k)))
        before = brute_ints(code)
        nbr = lambda x, y: [code[y, (x + 1) % L], code[y, (x - 1) % L], code[(y + 1) % L, x], code[(y - 1) % L, x]]
        sSa = sum(S_OF[int(c)] for c in nbr(xa, ya)); sSb = sum(S_OF[int(c)] for c in nbr(xb, yb))
        sGa = sum(SG_OF[int(c)] for c in nbr(xa, ya)); sGb = sum(SG_OF[int(c)] for c in nbr(xb, yb))
        new = code.copy(); new[ya, xa] = na; new[yb, xb] = nb
        after = brute_ints(new)
        dSa = S_OF[na] - S_OF[ca]; dGa = SG_OF[na] - SG_OF[ca]; dGb = SG_OF[nb] - SG_OF[cb]
        EV_printed = dSa * (sSa - sSb) - adj * dSa ** 2
        EJ_printed = dGa * (sGa - sGb) + adj * dGa * dGb
        bad_V += EV_printed != after[1] - before[1]
        bad_J += EJ_printed != after[2] - before[2]
        moves += 1
    assert bad_V == 0
    assert bad_J > moves // 10


def test_uniform_sampling_at_zero_coupling():
    """Delta=V=J=0: every move accepted, the chain samples the fixed-Q space uniformly (pin P4):
    <n2> = sum_{p-m=Q} (p+m) w / sum w,  w = N!/(p! m! (N-p-m)!) 2^(N-p-m)."""
    Lx = Ly = 3; N = 9; Q = 2
    num = den = 0
    for p in range(N + 1):
        m = p - Q
        if m < 0 or p + m > N:
            continue
        w = math.factorial(N) // (math.factorial(p) * math.factorial(m) * math.factorial(N - p - m)) * 2 ** (N - p - m)
        num += (p + m) * w; den += w
    assert den == exact.n_states_closed_form(N, Q)
    code = oracle.init_state(Lx, Ly, Q, 0, seed=11)
    lat = oracle.Lattice(code, 0.0, 0.0, 0.0, seed=11)
    tr = lat.sweep_s0(1.0, 200000, trace=True)
    x = tr[:, 0].astype(float)
    nb = 50; b = x[: nb * (len(x) // nb)].reshape(nb, -1).mean(1)
    assert abs(b.mean() - num / den) < 3 * b.std(ddof=1) / math.sqrt(nb)
    assert lat.st.n_accept + lat.st.n_null == lat.st.n_attempt      # nothing is ever rejected at dE = 0


# ---------------------------------------------------------------- stage 1 (U0)
def test_init_state_exact_counts_and_determinism():
    for (L, p, m, seed) in [(16, 64, 0, 1), (64, 410, 0, 2), (32, 153, 153, 3), (8, 0, 0, 4), (8, 64, 0, 5), (8, 0, 64, 6)]:
        c = oracle.init_state(L, L, p, m, seed)
        assert (c == 2).sum() == p and (c == 3).sum() == m and ((c >= 0) & (c <= 3)).all()
        assert (oracle.init_state(L, L, p, m, seed) == c).all()
        if p + m < L * L:
            assert (oracle.init_state(L, L, p, m, seed, replica=1) != c).any()
    c = oracle.init_state(64, 64, 0, 0, 9)
    assert abs((c == 0).mean() - 0.5) < 0.05                                  # random sigma
    c = oracle.init_state(64, 64, 1000, 0, 9)
    rows = (c == 2).sum(1)
    assert rows.min() > 2 and rows.max() < 40                                 # spread over the lattice, not clumped


def test_init_state_is_uniform_over_sites_and_signs():
    """Stage 1 (reading U0) draws the charged sites uniformly without replacement and deals the signs among
    them at random: over 400 seeds on an 8 x 8 lattice with 10 S=+1 and 6 S=-1 sites, the number of times each site is charged
    (expected 100) and is S=+1 (expected 62.5) pass a chi-square test with 63 degrees of freedom -- a selection that is off by
    one (a site that can never be drawn, or drawn twice as often) fails it by a wide margin -- and the uncharged sites are
    sigma=+1 half of the time."""
    L, N, p, m, S = 8, 64, 10, 6, 400
    K = p + m
    charged = np.zeros(N); plus = np.zeros(N); up = 0
    for seed in range(1000, 1000 + S):
        c = oracle.init_state(L, L, p, m, seed).reshape(-1)
        assert (c == 2).sum() == p and (c == 3).sum() == m
        charged += c >= 2; plus += c == 2; up += int((c == 0).sum())
    for cnt, k in ((charged, K), (plus, p)):
        q = k / N
        var = S * q * (1 - q)                  # per lattice a site is chosen with probability q; the seeds are independent
        chi2 = ((cnt - S * q) ** 2).sum() / var * (N - 1) / N      # the N counts sum to S k exactly: N-1 degrees of freedom
        assert 30.0 < chi2 < 110.0, chi2       # chi-square(63): mean 63, sd 11.2; both tails beyond 3 sd are rejected
        assert cnt.min() > 0.5 * S * q and cnt.max() < 1.6 * S * q
    n_unch = S * (N - K)
    assert abs(up - 0.5 * n_unch) < 4 * math.sqrt(0.25 * n_unch)


@pytest.mark.parametrize("L,nsweeps", [(16, 12000), (32, 5000)])
def test_seven_round_update_stream_samples_the_same_ensemble_as_ten_rounds(L, nsweeps):
    """Reading G5 runs the update stream on Philox4x32-7, the member of the family with the fewest rounds its authors report
    as passing BigCrush.  Beyond the exact 4 x 4 ensemble of test_oracle_exact, this compares what the physics sees at larger
    sizes: <E>/N, C and <n2> of schedule S1 near the specific-heat maximum, 8 independent seeds per round count; the means at 7
    and at 10 rounds agree within 3.5 standard errors of their difference, and the 10-round runs leave the switch as found."""
    delta, V, J, T, n = 0.2, 1.0, 1.0, 1.3, 0.1          # C(T) is largest around T = 1.3 for these parameters
    N = L * L
    Q = round(n * N)
    res = {}
    assert oracle.UPDATE_ROUNDS == 7
    for rounds in (7, 10):
        old = oracle.set_update_rounds(rounds)
        try:
            rows = []
            for seed in range(8):
                code = oracle.init_state(L, L, Q, 0, 500 + seed)
                lat = oracle.Lattice(code, delta, V, J, 500 + seed)
                lat.sweep_s1(T, nsweeps // 2)
                lat.reset_observables()
                lat.sweep_s1(T, nsweeps)
                o = lat.observables(T)
                rows.append((o["sumE"] / o["nmeas"] / N, o["C"], float(lat.st.n2) / N))
            res[rounds] = np.array(rows)
        finally:
            assert oracle.set_update_rounds(old) == rounds
    assert oracle.lib().orc_get_update_rounds() == 7
    assert not np.array_equal(res[7], res[10])                    # the switch does something
    for k, name in enumerate(("E/N", "C", "n2/N")):
        a, b = res[7][:, k], res[10][:, k]
        err = math.sqrt(a.var(ddof=1) / len(a) + b.var(ddof=1) / len(b))
        assert abs(a.mean() - b.mean()) < 3.5 * err, (name, a.mean(), b.mean(), err)
    assert 1.0 < res[7][:, 1].mean() < 6.0                       # a real specific heat, not a frozen lattice
