"""Exact constrained canonical averages from an enumerated density of states.

TEST INFRASTRUCTURE (see oracle/ic_enum.c).  Weights exp(-E/T) with
E = Delta*n2 + V*bV + (J/4)*bJ (eq. 3) restricted to sum S = Q
(eq. 2); k_B = 1.
"""
import ctypes as C
import math

import numpy as np

from . import lib, _p


def enum_bruteforce(Lx, Ly, cap=1 << 20):
    """All 4^(Lx*Ly) states through orc_recompute.  Returns keys[:,6]=(n2,bV,bJ,M,Ms,Q), counts."""
    keys = np.zeros((cap, 6), dtype=np.int64); counts = np.zeros(cap, dtype=np.uint64)
    n = lib().orc_enum_bruteforce(int(Lx), int(Ly), _p(keys, C.c_int64), _p(counts, C.c_uint64), cap)
    if n < 0:
        raise RuntimeError("enumeration failed (cap too small or lattice too large)")
    return keys[:n].copy(), counts[:n].copy()


def enum_rows(Lx, Ly, threads=8, cap=1 << 22):
    """Row decomposition.  Returns keys[:,4]=(Q,n2,bV,bJ), counts, sumM2, sumMs2."""
    keys = np.zeros((cap, 4), dtype=np.int64)
    counts = np.zeros(cap, dtype=np.uint64); m2 = np.zeros(cap, dtype=np.uint64); ms2 = np.zeros(cap, dtype=np.uint64)
    n = lib().orc_enum_rows(int(Lx), int(Ly), int(threads), _p(keys, C.c_int64), _p(counts, C.c_uint64),
                            _p(m2, C.c_uint64), _p(ms2, C.c_uint64), cap)
    if n < 0:
        raise RuntimeError("enumeration failed")
    return keys[:n].copy(), counts[:n].copy(), m2[:n].copy(), ms2[:n].copy()


def averages(dos, Q, delta, V, J, T):
    """dos = (keys[:,4]=(Q,n2,bV,bJ), counts, sumM2, sumMs2).  Returns dict of exact averages in sector Q."""
    keys, counts, m2, ms2 = dos
    sel = keys[:, 0] == Q
    if not sel.any():
        raise ValueError("empty charge sector")
    k = keys[sel]
    E = (delta * k[:, 1].astype(float) + V * k[:, 2].astype(float)) + (0.25 * J) * k[:, 3].astype(float)
    lw = -(E - E.min()) / T
    w = np.exp(lw)
    cnt = counts[sel].astype(float)
    Z = float(np.sum(cnt * w))
    out = dict(E=float(np.sum(cnt * w * E)) / Z, E2=float(np.sum(cnt * w * E * E)) / Z,
               n2=float(np.sum(cnt * w * k[:, 1])) / Z,
               M2=float(np.sum(m2[sel].astype(float) * w)) / Z, Ms2=float(np.sum(ms2[sel].astype(float) * w)) / Z,
               nstates=int(counts[sel].sum()))
    return out


def averages_grand(dos, mu, delta, V, J, T):
    """Grand-canonical averages over ALL charge sectors with weights exp(-(E - mu Q)/T): what single-site Metropolis
    with the extra term -mu sum S samples at fixed mu.  Returns <E>, <E^2>, <Q>, <Q^2>."""
    keys, counts, _, _ = dos
    E = (delta * keys[:, 1].astype(float) + V * keys[:, 2].astype(float)) + (0.25 * J) * keys[:, 3].astype(float)
    Qs = keys[:, 0].astype(float)
    H = E - mu * Qs
    w = counts.astype(float) * np.exp(-(H - H.min()) / T)
    Z = float(w.sum())
    return dict(E=float((w * E).sum()) / Z, E2=float((w * E * E).sum()) / Z, Q=float((w * Qs).sum()) / Z,
                Q2=float((w * Qs * Qs).sum()) / Z)


def dos_from_bruteforce(keys6, counts):
    """Collapse brute-force keys (n2,bV,bJ,M,Ms,Q) to the (Q,n2,bV,bJ) form used by `averages`."""
    acc = {}
    for k, c in zip(keys6, counts):
        key = (int(k[5]), int(k[0]), int(k[1]), int(k[2]))
        a = acc.setdefault(key, [0, 0, 0])
        a[0] += int(c); a[1] += int(c) * int(k[3]) ** 2; a[2] += int(c) * int(k[4]) ** 2
    ks = sorted(acc)
    return (np.array(ks, dtype=np.int64).reshape(-1, 4), np.array([acc[k][0] for k in ks], dtype=np.uint64),
            np.array([acc[k][1] for k in ks], dtype=np.uint64), np.array([acc[k][2] for k in ks], dtype=np.uint64))


def save_dos(path, dos, header):
    keys, counts, m2, ms2 = dos
    with open(path, "w") as f:
        for line in header.strip().splitlines():
            f.write("# " + line + "\n")
        f.write("# Q n2 bV bJ count sumM2 sumMs2\n")
        for k, c, a, b in zip(keys, counts, m2, ms2):
            f.write(f"{k[0]} {k[1]} {k[2]} {k[3]} {int(c)} {int(a)} {int(b)}\n")


def load_dos(path):
    rows = [tuple(int(v) for v in ln.split()) for ln in open(path) if ln.strip() and not ln.startswith("#")]
    a = np.array(rows, dtype=object)
    keys = np.array([[r[0], r[1], r[2], r[3]] for r in rows], dtype=np.int64)
    return (keys, np.array([r[4] for r in rows], dtype=np.uint64), np.array([r[5] for r in rows], dtype=np.uint64),
            np.array([r[6] for r in rows], dtype=np.uint64))


def n_states_closed_form(N, Q):
    """Number of states with sum S = Q on N four-state sites: coefficient of x^Q in (x + 2 + 1/x)^N = C(2N, N+Q)."""
    return math.comb(2 * N, N + Q) if -N <= Q <= N else 0
