"""CPU oracle of the coupled-pair Metropolis sweep (arXiv:2301.11735).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
shares nothing with paper_2301_11735_b200 and never imports it.

Thin ctypes wrapper over oracle/ic_oracle.c and oracle/ic_enum.c (plain C, built
with gcc by oracle/build.py).  All arithmetic lives in the C files, each
function citing the passage of the paper it follows.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build


class OrcState(C.Structure):
    _fields_ = [
        ("Lx", C.c_int32), ("Ly", C.c_int32), ("replica", C.c_int32), ("pad_", C.c_int32),
        ("delta", C.c_double), ("V", C.c_double), ("J", C.c_double),
        ("seed", C.c_uint64), ("sweep", C.c_uint64),
        ("n2", C.c_int64), ("bV", C.c_int64), ("bJ", C.c_int64), ("M", C.c_int64), ("Ms", C.c_int64), ("Q", C.c_int64),
        ("nmeas", C.c_int64),
        ("sumE", C.c_double), ("sumE2", C.c_double), ("sumM", C.c_double), ("sumM2", C.c_double),
        ("sumAbsM", C.c_double), ("sumMs", C.c_double), ("sumMs2", C.c_double), ("sumAbsMs", C.c_double),
        ("n_attempt", C.c_int64), ("n_accept", C.c_int64), ("n_null", C.c_int64),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        u32p, i8p, i64p, u64p, i32p = (C.POINTER(C.c_uint32), C.POINTER(C.c_int8), C.POINTER(C.c_int64),
                                       C.POINTER(C.c_uint64), C.POINTER(C.c_int32))
        stp = C.POINTER(OrcState)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]; L.orc_philox4x32_10.restype = None
        L.orc_philox4x32.argtypes = [u32p, u32p, C.c_int, u32p]; L.orc_philox4x32.restype = None
        L.orc_set_update_rounds.argtypes = [C.c_int]; L.orc_set_update_rounds.restype = C.c_int
        L.orc_get_update_rounds.argtypes = []; L.orc_get_update_rounds.restype = C.c_int
        L.orc_threshold.argtypes = [C.c_double] * 3 + [C.c_int] * 3 + [C.c_double]; L.orc_threshold.restype = C.c_uint32
        L.orc_recompute.argtypes = [i8p, C.c_int, C.c_int, i64p]; L.orc_recompute.restype = None
        L.orc_pair_table.argtypes = [C.c_int, C.c_int, i8p]; L.orc_pair_table.restype = C.c_int
        L.orc_pair_update.argtypes = [stp, i8p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint32, C.c_double]
        L.orc_pair_update.restype = C.c_int
        L.orc_init_state.argtypes = [i8p, C.c_int, C.c_int, C.c_int64, C.c_int64, C.c_uint64, C.c_int]
        L.orc_init_state.restype = None
        L.orc_attach.argtypes = [stp, i8p]; L.orc_attach.restype = None
        L.orc_reset_observables.argtypes = [stp]; L.orc_reset_observables.restype = None
        L.orc_schedule_params.argtypes = [C.c_int, C.c_uint64, C.c_uint64, i32p]; L.orc_schedule_params.restype = None
        L.orc_schedule_s1.argtypes = [C.c_int, C.c_uint64, C.c_uint64, C.c_int, i64p, i64p, u32p, u32p, u32p]
        L.orc_schedule_s1.restype = C.c_int64
        L.orc_sweep_s1.argtypes = [stp, i8p, C.c_double, C.c_int64, C.c_int, i64p]; L.orc_sweep_s1.restype = C.c_int
        L.orc_sweep_s1_mt.argtypes = [stp, i8p, C.c_double, C.c_int64, C.c_int, i64p]; L.orc_sweep_s1_mt.restype = C.c_int
        L.orc_sweep_s0.argtypes = [stp, i8p, C.c_double, C.c_int64, i64p]; L.orc_sweep_s0.restype = C.c_int
        u8p, dblp = C.POINTER(C.c_uint8), C.POINTER(C.c_double)
        L.orc_sweep_nn.argtypes = [stp, i8p, C.c_double, C.c_int64, i64p]; L.orc_sweep_nn.restype = C.c_int
        L.orc_sweep_mu.argtypes = [stp, i8p, C.c_double, C.c_int64, dblp, C.c_double, C.c_int64, i64p]; L.orc_sweep_mu.restype = C.c_int
        L.orc_build_map_paper.argtypes = [C.c_int, C.c_int, C.c_uint64, C.c_uint64, C.c_int64, i64p, i64p]; L.orc_build_map_paper.restype = C.c_int64
        L.orc_build_map_luby.argtypes = [C.c_int, C.c_int, C.c_uint64, C.c_uint64, C.c_int64, i64p, i64p, u8p]; L.orc_build_map_luby.restype = C.c_int64
        L.orc_sweep_maps.argtypes = [stp, i8p, C.c_double, C.c_int64, C.c_int, C.c_int64, i64p, i64p]; L.orc_sweep_maps.restype = C.c_int
        L.orc_largest_cluster.argtypes = [i8p, C.c_int, C.c_int, C.c_int, i64p]; L.orc_largest_cluster.restype = C.c_int
        L.orc_enum_bruteforce.argtypes = [C.c_int, C.c_int, i64p, u64p, C.c_int64]; L.orc_enum_bruteforce.restype = C.c_int64
        L.orc_enum_rows.argtypes = [C.c_int, C.c_int, C.c_int, i64p, u64p, u64p, u64p, C.c_int64]
        L.orc_enum_rows.restype = C.c_int64
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy(); k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


UPDATE_ROUNDS = 7      # Philox rounds of the update stream (ORC_UPDATE_ROUNDS in ic_oracle.h; G5)


def philox4x32(ctr, key, rounds):
    c = np.asarray(ctr, dtype=np.uint32).copy(); k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32(_p(c, C.c_uint32), _p(k, C.c_uint32), int(rounds), _p(out, C.c_uint32))
    return out


def set_update_rounds(rounds):
    """Philox rounds of the update stream for the runs that follow (UPDATE_ROUNDS = 7 is the default and what the library
    uses); returns the previous value.  For the 7-versus-10-round ensemble comparison only."""
    old = lib().orc_get_update_rounds()
    if lib().orc_set_update_rounds(int(rounds)) != 0:
        raise ValueError("rounds must be in 1..16")
    return old


def threshold(delta, V, J, dn2, dV, dJ, T):
    """29-bit acceptance threshold t29: accept iff (w >> 3) < t29."""
    return int(lib().orc_threshold(float(delta), float(V), float(J), int(dn2), int(dV), int(dJ), float(T)))


def recompute(code, Lx=None, Ly=None):
    """(n2, bV, bJ, M, Ms, Q) of a lattice, straight from eq. (3)."""
    code = np.ascontiguousarray(code, dtype=np.int8)
    if Lx is None:
        Ly, Lx = code.shape
    out = np.zeros(6, dtype=np.int64)
    lib().orc_recompute(_p(code, C.c_int8), int(Lx), int(Ly), _p(out, C.c_int64))
    return out


def pair_table(q, idx):
    out = np.zeros(2, dtype=np.int8)
    ok = lib().orc_pair_table(int(q), int(idx), _p(out, C.c_int8))
    return (int(out[0]), int(out[1])) if ok else None


def init_state(Lx, Ly, nplus, nminus, seed, replica=0):
    """Stage 1: random sigma everywhere, then exactly nplus sites S=+1, nminus sites S=-1."""
    code = np.zeros((Ly, Lx), dtype=np.int8)
    lib().orc_init_state(_p(code, C.c_int8), int(Lx), int(Ly), int(nplus), int(nminus), int(seed), int(replica))
    return code


def schedule_params(L, seed, sweep):
    out = np.zeros(4, dtype=np.int32)
    lib().orc_schedule_params(int(L), int(seed), int(sweep), _p(out, C.c_int32))
    return tuple(int(v) for v in out)


def schedule_s1(L, seed, sweep, phase):
    """pairs(sweep, phase): arrays (ia, ib, c0, c1, word)."""
    n = L * L // 4
    ia = np.zeros(n, dtype=np.int64); ib = np.zeros(n, dtype=np.int64)
    c0 = np.zeros(n, dtype=np.uint32); c1 = np.zeros(n, dtype=np.uint32); wd = np.zeros(n, dtype=np.uint32)
    m = lib().orc_schedule_s1(int(L), int(seed), int(sweep), int(phase), _p(ia, C.c_int64), _p(ib, C.c_int64),
                              _p(c0, C.c_uint32), _p(c1, C.c_uint32), _p(wd, C.c_uint32))
    return ia[:m], ib[:m], c0[:m], c1[:m], wd[:m]


def build_map_paper(Lx, Ly, seed, map_index, npairs):
    """The paper's sequential map builder: arrays (ia, ib) of the pairs placed."""
    ia = np.zeros(int(npairs), dtype=np.int64); ib = np.zeros(int(npairs), dtype=np.int64)
    n = lib().orc_build_map_paper(int(Lx), int(Ly), int(seed), int(map_index), int(npairs), _p(ia, C.c_int64), _p(ib, C.c_int64))
    return ia[:n], ib[:n]


def build_map_luby(Lx, Ly, seed, map_index, K):
    """K random candidate pairs and which of them survive the one-round conflict resolution: (ia, ib, alive)."""
    ia = np.zeros(int(K), dtype=np.int64); ib = np.zeros(int(K), dtype=np.int64); alive = np.zeros(int(K), dtype=np.uint8)
    lib().orc_build_map_luby(int(Lx), int(Ly), int(seed), int(map_index), int(K), _p(ia, C.c_int64), _p(ib, C.c_int64), _p(alive, C.c_uint8))
    return ia, ib, alive.astype(bool)


def largest_cluster(code, which=0):
    """(size of the largest connected cluster of charged sites, number of clusters); which: 0 any charge, 1 S=+1, 2 S=-1."""
    code = np.ascontiguousarray(code, dtype=np.int8)
    Ly, Lx = code.shape
    out = np.zeros(2, dtype=np.int64)
    rc = lib().orc_largest_cluster(_p(code, C.c_int8), int(Lx), int(Ly), int(which), _p(out, C.c_int64))
    if rc != 0:
        raise MemoryError("orc_largest_cluster")
    return int(out[0]), int(out[1])


class Lattice:
    """One lattice copy driven by the oracle."""

    def __init__(self, code, delta, V, J, seed, replica=0):
        self.code = np.ascontiguousarray(code, dtype=np.int8).copy()
        Ly, Lx = self.code.shape
        self.st = OrcState()
        self.st.Lx, self.st.Ly, self.st.replica = Lx, Ly, int(replica)
        self.st.delta, self.st.V, self.st.J = float(delta), float(V), float(J)
        self.st.seed, self.st.sweep = int(seed), 0
        lib().orc_attach(C.byref(self.st), _p(self.code, C.c_int8))
        lib().orc_reset_observables(C.byref(self.st))

    @property
    def N(self):
        return self.st.Lx * self.st.Ly

    def ints(self):
        s = self.st
        return np.array([s.n2, s.bV, s.bJ, s.M, s.Ms, s.Q], dtype=np.int64)

    def reset_observables(self):
        lib().orc_reset_observables(C.byref(self.st))

    def pair_update(self, xa, ya, xb, yb, w, T):
        return lib().orc_pair_update(C.byref(self.st), _p(self.code, C.c_int8), int(xa), int(ya), int(xb), int(yb),
                                     int(w) & 0xFFFFFFFF, float(T))

    def sweep_s1(self, T, nsweeps, order=0, trace=False, threads=1):
        tr = np.zeros((int(nsweeps), 6), dtype=np.int64) if trace else None
        trp = _p(tr, C.c_int64) if trace else None
        if threads > 1:
            rc = lib().orc_sweep_s1_mt(C.byref(self.st), _p(self.code, C.c_int8), float(T), int(nsweeps), int(threads), trp)
        else:
            rc = lib().orc_sweep_s1(C.byref(self.st), _p(self.code, C.c_int8), float(T), int(nsweeps), int(order), trp)
        if rc != 0:
            raise ValueError(f"orc_sweep_s1 failed with {rc}")
        return tr

    def sweep_s0(self, T, nsweeps, trace=False):
        tr = np.zeros((int(nsweeps), 6), dtype=np.int64) if trace else None
        rc = lib().orc_sweep_s0(C.byref(self.st), _p(self.code, C.c_int8), float(T), int(nsweeps),
                                _p(tr, C.c_int64) if trace else None)
        if rc != 0:
            raise ValueError(f"orc_sweep_s0 failed with {rc}")
        return tr

    def sweep_nn(self, T, nsweeps, trace=False):
        """Nearest-neighbour-only coupled pairs: the paper's first, rejected version."""
        tr = np.zeros((int(nsweeps), 6), dtype=np.int64) if trace else None
        rc = lib().orc_sweep_nn(C.byref(self.st), _p(self.code, C.c_int8), float(T), int(nsweeps), _p(tr, C.c_int64) if trace else None)
        if rc != 0:
            raise ValueError(f"orc_sweep_nn failed with {rc}")
        return tr

    def sweep_mu(self, T, nsweeps, mu, kappa, q_target, trace=False):
        """Penalty / chemical-potential single-site Metropolis.  Returns (trace, mu after the run)."""
        tr = np.zeros((int(nsweeps), 6), dtype=np.int64) if trace else None
        m = C.c_double(float(mu))
        rc = lib().orc_sweep_mu(C.byref(self.st), _p(self.code, C.c_int8), float(T), int(nsweeps), C.byref(m), float(kappa),
                                int(q_target), _p(tr, C.c_int64) if trace else None)
        if rc != 0:
            raise ValueError(f"orc_sweep_mu failed with {rc}")
        return tr, m.value

    def sweep_maps(self, T, nmaps, mode, K, trace=False):
        """Sweeps made of maps: mode 0 the paper's sequential builder, 1 one-round conflict resolution.
        Returns (trace, number of attempted pair updates)."""
        tr = np.zeros((int(nmaps), 6), dtype=np.int64) if trace else None
        att = C.c_int64(0)
        rc = lib().orc_sweep_maps(C.byref(self.st), _p(self.code, C.c_int8), float(T), int(nmaps), int(mode), int(K),
                                  _p(tr, C.c_int64) if trace else None, C.byref(att))
        if rc != 0:
            raise ValueError(f"orc_sweep_maps failed with {rc}")
        return tr, att.value

    def observables(self, T):
        """U5: C = (<E^2>-<E>^2)/(N T^2) (k=1); chi = (<M^2>-<M>^2)/(N T) (reading G9)."""
        s = self.st
        n = max(int(s.nmeas), 1)
        mE, mE2 = s.sumE / n, s.sumE2 / n
        mM, mM2, mMs, mMs2 = s.sumM / n, s.sumM2 / n, s.sumMs / n, s.sumMs2 / n
        N = self.N
        return dict(nmeas=int(s.nmeas), n2=s.n2, bV=s.bV, bJ=s.bJ, M=s.M, Ms=s.Ms, Q=s.Q,
                    sumE=s.sumE, sumE2=s.sumE2, sumM=s.sumM, sumM2=s.sumM2, sumAbsM=s.sumAbsM,
                    sumMs=s.sumMs, sumMs2=s.sumMs2, sumAbsMs=s.sumAbsMs, T=float(T),
                    C=(mE2 - mE * mE) / (N * T * T), chi_u=(mM2 - mM * mM) / (N * T), chi_s=(mMs2 - mMs * mMs) / (N * T))
