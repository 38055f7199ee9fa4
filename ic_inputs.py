"""Seeded synthetic inputs shared by the oracle-side and the CUDA-side callers (tests, bench.py, smoke).

Holds none of the method's arithmetic: only the workload table (BASELINE.json's five configs, restated in
DESIGN.md "Inputs") and a numpy generator of lattices with an exact number of charges.  Neither oracle/ nor
paper_2301_11735_b200/ imports this module; their callers do.

The paper measures on no public dataset: its workloads are square lattices from 4x4 (test) over 64x64 (drops)
to 256x256 "and larger", one to several copies, at various charge densities n.
Site codes: 0 sigma=+1, 1 sigma=-1, 2 S=+1, 3 S=-1.
"""
import numpy as np

# name -> parameters.  T: list of temperatures, one lattice copy (replica) per temperature.
CONFIGS = {
    "C1": dict(L=16, n=0.25, delta=0.5, V=1.0, J=1.0, T=[0.1 + i * (3.9 / 40) for i in range(41)], nplus=64, nminus=0,
               sweeps=10000, equil=2000, bits=8, seed=1),
    "C2": dict(L=64, n=0.1, delta=0.0, V=0.5, J=1.0, T=[0.05 * (r + 1) for r in range(64)], nplus=410, nminus=0,
               sweeps=10000, equil=0, bits=8, seed=2),
    "C3": dict(L=1024, n=0.0, delta=-0.5, V=1.0, J=2.0, T=[0.8], nplus=157286, nminus=157286,
               sweeps=1000, equil=0, bits=2, seed=3),
    "C4": dict(L=4096, n=0.2, delta=1.0, V=0.25, J=1.0, T=[0.2 + r * 0.12 for r in range(16)], nplus=3355443, nminus=0,
               sweeps=500, equil=0, bits=8, seed=4),
    "C5": dict(L=16384, n=0.05, delta=0.2, V=1.0, J=1.0, T=[1.0], nplus=13421773, nminus=0,
               sweeps=100, equil=0, bits=8, seed=5),
    # second workload of the paper (Fig. 7): formation of a charge "drop" on a 64 x 64 lattice with a
    # strong magnetic exchange J >> V; the paper gives no parameters (figure only), these are ours: a quench from a random
    # state at four temperatures
    "C6": dict(L=64, n=0.1, delta=0.0, V=0.1, J=4.0, T=[0.2, 0.4, 0.8, 1.6], nplus=410, nminus=0,
               sweeps=4000, equil=0, bits=8, seed=6),
}


def random_state(L, nplus, nminus, seed, replica=0):
    """L x L int8 lattice: nplus sites S=+1 (code 2), nminus sites S=-1 (code 3) at distinct uniformly random sites,
    all other sites sigma=+-1 (codes 0/1) with probability 1/2 each.  numpy PCG64 seeded by (seed, replica)."""
    rng = np.random.default_rng([int(seed), int(replica), 0x1C])
    N = L * L
    code = rng.integers(0, 2, size=N, dtype=np.int8)
    k = int(nplus) + int(nminus)
    if k:
        pos = rng.choice(N, size=k, replace=False) if N <= (1 << 24) else _choice_large(rng, N, k)
        code[pos[:nplus]] = 2
        code[pos[nplus:]] = 3
    return code.reshape(L, L)


def _choice_large(rng, N, k):
    """k distinct positions out of N without materialising a permutation of N (k << N)."""
    got = np.unique(rng.integers(0, N, size=int(k * 1.1) + 16))
    while got.size < k:
        got = np.unique(np.concatenate([got, rng.integers(0, N, size=k - got.size + 16)]))
    rng.shuffle(got)
    return got[:k]


def structured_state(L, kind):
    """Deterministic edge-case lattices: 'all_plus' (frozen, n=+1), 'all_minus', 'neel' (staggered sigma),
    'ferro' (sigma=+1 everywhere), 'stripes' (alternating columns S=+1 / S=-1: neutral, fully charged)."""
    y, x = np.mgrid[0:L, 0:L]
    if kind == "all_plus":
        return np.full((L, L), 2, dtype=np.int8)
    if kind == "all_minus":
        return np.full((L, L), 3, dtype=np.int8)
    if kind == "neel":
        return ((x + y) & 1).astype(np.int8)
    if kind == "ferro":
        return np.zeros((L, L), dtype=np.int8)
    if kind == "stripes":
        return (2 + (x & 1)).astype(np.int8)
    raise ValueError(kind)
