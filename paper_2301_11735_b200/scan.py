"""Temperature scan: heat capacity C(T) and magnetic susceptibilities chi(T) with error bars.

The step after the hot path and the paper's main result (PAPER.md:49-53, 161, 188 / Fig. 6): all temperatures run as
replicas of one `Sim` (one launch per sweep phase, or one launch per call for L <= 64); E, E^2, M, M^2, ... are accumulated
per sweep by the library (`ic_observables`), read and reset once per block, and this module only does the statistics over
blocks on the host:

    E = Delta*n2 + V*bV + (J/4)*bJ                                   (eq. 3)
    C = (<E^2> - <E>^2) / (N T^2)                                    (k_B = 1)
    chi_u = (<M^2> - <M>^2) / (N T),  chi_s the same with Ms        (G9)

Errors are jackknife errors over `bins` consecutive blocks of the measured sweeps (blocks must be much longer than the
autocorrelation time: about 50 sweeps at T ~ 1 on a 4 x 4 lattice).

    python -m paper_2301_11735_b200.scan --L 16 --n 0.25 --delta 0.5 --V 1 --J 1 --T 0.1:4.0:41 --equil 2000 --sweeps 10000
"""
import argparse

import numpy as np

from .binding import Sim


def _jackknife(blocks, f):
    """blocks: array [bins, k] of per-block means of k quantities; f maps a k-vector of means to a scalar."""
    nb = blocks.shape[0]
    total = blocks.sum(axis=0)
    full = f(total / nb)
    loo = np.array([f((total - blocks[b]) / (nb - 1)) for b in range(nb)])
    err = np.sqrt((nb - 1) / nb * np.sum((loo - loo.mean()) ** 2))
    return full, err


def temperature_scan(L, n, delta, V, J, Ts, equil, sweeps, seed=1, bins=32, bits_per_site=8, init_charges=None):
    """Runs len(Ts) replicas at temperatures Ts: `equil` sweeps discarded, `sweeps` measured.  Returns a dict of numpy
    arrays over the temperatures: T, E, E_err, C, C_err, chi_u, chi_u_err, chi_s, chi_s_err, absM, absMs and the
    exact integer charge Q (eq. 2 is checked after every block)."""
    Ts = [float(t) for t in Ts]
    reps = len(Ts)
    if sweeps < bins or bins < 2:
        raise ValueError("need at least `bins` >= 2 measured sweeps")
    sim = Sim(L, n, delta, V, J, seed=seed, replicas=reps, bits_per_site=bits_per_site)
    try:
        if init_charges is not None:
            for r in range(reps):
                sim.init_charges(r, int(init_charges[0]), int(init_charges[1]))
        if equil:
            sim.sweep(Ts, int(equil))
        sim.reset_observables()
        N = float(L) * float(L)
        per_bin = sweeps // bins
        used = per_bin * bins
        # per-block means of (E, E^2, M, M^2, |M|, Ms, Ms^2, |Ms|): the library's own fp64 accumulators (A9), read and
        # reset once per block -- the host does statistics over blocks only
        acc = np.zeros((reps, bins, 8))
        keys = ("sumE", "sumE2", "sumM", "sumM2", "sumAbsM", "sumMs", "sumMs2", "sumAbsMs")
        for b in range(bins):
            sim.reset_observables()
            sim.sweep(Ts, per_bin)
            obs = sim.observables()
            for r in range(reps):
                if obs[r]["Q"] != sim.Q or obs[r]["nmeas"] != per_bin:
                    raise RuntimeError("charge not conserved (eq. 2) or sweeps lost")
                acc[r, b, :] = [obs[r][k] / per_bin for k in keys]
        out = {k: np.zeros(reps) for k in ("E", "E_err", "C", "C_err", "chi_u", "chi_u_err", "chi_s", "chi_s_err", "absM", "absMs")}
        for r, T in enumerate(Ts):
            blk = acc[r]
            out["E"][r], out["E_err"][r] = _jackknife(blk, lambda v: v[0])
            out["C"][r], out["C_err"][r] = _jackknife(blk, lambda v: (v[1] - v[0] * v[0]) / (N * T * T))
            out["chi_u"][r], out["chi_u_err"][r] = _jackknife(blk, lambda v: (v[3] - v[2] * v[2]) / (N * T))
            out["chi_s"][r], out["chi_s_err"][r] = _jackknife(blk, lambda v: (v[6] - v[5] * v[5]) / (N * T))
            out["absM"][r] = blk[:, 4].mean(); out["absMs"][r] = blk[:, 7].mean()
        out["T"] = np.array(Ts); out["Q"] = sim.Q; out["sweeps"] = used; out["bins"] = bins
        return out
    finally:
        sim.close()


def _parse_T(spec):
    if ":" in spec:
        lo, hi, cnt = spec.split(":")
        return list(np.linspace(float(lo), float(hi), int(cnt)))
    return [float(x) for x in spec.split(",")]


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--L", type=int, default=16)
    ap.add_argument("--n", type=float, default=0.25)
    ap.add_argument("--delta", type=float, default=0.5)
    ap.add_argument("--V", type=float, default=1.0)
    ap.add_argument("--J", type=float, default=1.0)
    ap.add_argument("--T", default="0.1:4.0:41", help="lo:hi:count or a comma-separated list")
    ap.add_argument("--equil", type=int, default=2000)
    ap.add_argument("--sweeps", type=int, default=10000)
    ap.add_argument("--bins", type=int, default=32)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--bits", type=int, default=8)
    a = ap.parse_args()
    res = temperature_scan(a.L, a.n, a.delta, a.V, a.J, _parse_T(a.T), a.equil, a.sweeps, seed=a.seed, bins=a.bins, bits_per_site=a.bits)
    print(f"# L={a.L} n={a.n} Q={res['Q']} Delta={a.delta} V={a.V} J={a.J}  {res['sweeps']} sweeps in {res['bins']} bins")
    print("#      T          E/N        err          C        err      chi_u        err      chi_s        err")
    N = a.L * a.L
    for i, T in enumerate(res["T"]):
        print(f"{T:8.4f} {res['E'][i] / N:12.6f} {res['E_err'][i] / N:10.6f} {res['C'][i]:10.5f} {res['C_err'][i]:10.5f} "
              f"{res['chi_u'][i]:10.5f} {res['chi_u_err'][i]:10.5f} {res['chi_s'][i]:10.5f} {res['chi_s_err'][i]:10.5f}")


if __name__ == "__main__":
    main()
