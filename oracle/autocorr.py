"""Integrated autocorrelation times of the update schemes, oracle only (test infrastructure, CPU).

    python -m oracle.autocorr [--quick]

Compares, at equal work, the schedules the oracle holds: S0 (the literal sequential algorithm with completely random
pairs), S1 (the production schedule: FAR and NEAR sweeps alternating, U4), the paper's maps
(N/10 mutually non-interacting random pairs per map, sequential builder) and the one-round device
maps (K candidates, survivors of the conflict resolution).  Work is counted in attempted pair updates per site, so that
a "sweep" of N/2 pairs and a map of N/10 pairs are comparable.  tau_int = 1/2 + sum_t rho(t) with Sokal's automatic
window (sum up to the first t >= 6 tau); errors are not attached: the figures are a qualitative record for DESIGN.md.
"""
import argparse
import sys

import numpy as np

import ic_inputs
import oracle


def tau_int(x, c=6.0):
    x = np.asarray(x, dtype=np.float64)
    x = x - x.mean()
    n = x.size
    var = float(x @ x) / n
    if var == 0.0:
        return 0.5
    f = np.fft.rfft(x, 2 * n)
    acf = np.fft.irfft(f * np.conj(f))[:n] / (n * var)
    tau = 0.5
    for t in range(1, n // 4):
        tau += acf[t]
        if t >= c * tau:
            break
    return max(tau, 0.5)


def energy(tr, delta, V, J):
    return delta * tr[:, 0] + V * tr[:, 1] + 0.25 * J * tr[:, 2]


def run(L, nplus, nminus, delta, V, J, T, seed, nsw, schemes):
    N = L * L
    out = []
    for name in schemes:
        code = ic_inputs.random_state(L, nplus, nminus, seed)
        lat = oracle.Lattice(code, delta, V, J, seed)
        if name == "S0":
            lat.sweep_s0(T, nsw // 10); tr = lat.sweep_s0(T, nsw, trace=True); per = 0.5
        elif name == "S1":
            lat.sweep_s1(T, nsw // 10); tr = lat.sweep_s1(T, nsw, trace=True); per = 0.5
            tr = tr[1::2]; per = 1.0                      # one FAR + one NEAR sweep is the period of the schedule
        elif name == "maps (paper, N/10)":
            K = max(1, N // 10)
            lat.sweep_maps(T, nsw // 2, 0, K); tr, att = lat.sweep_maps(T, 5 * nsw, 0, K, trace=True); per = att / (5 * nsw) / N
        else:                                             # one-round maps, K = N/5 candidates
            K = max(2, N // 5)
            lat.sweep_maps(T, nsw // 2, 1, K); tr, att = lat.sweep_maps(T, 5 * nsw, 1, K, trace=True); per = att / (5 * nsw) / N
        E = energy(tr, delta, V, J)
        acc = dict(scheme=name, work_per_step=per, tau_E=tau_int(E) * per, tau_Ms=tau_int(np.abs(tr[:, 4])) * per,
                   tau_n2=tau_int(tr[:, 0]) * per, mean_E=E.mean() / N)
        out.append(acc)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true")
    args = ap.parse_args()
    schemes = ["S0", "S1", "maps (paper, N/10)", "maps (one round, K=N/5)"]
    cases = [
        ("8x8, Q=6, Delta=0.5 V=1 J=1, T=1.0", 8, 6, 0, 0.5, 1.0, 1.0, 1.0, 200000),
        ("8x8, Q=6, Delta=0.5 V=1 J=1, T=0.5", 8, 6, 0, 0.5, 1.0, 1.0, 0.5, 200000),
        ("64x64, n=0.1, Delta=0 V=0.5 J=1 (C2), T=1.0", 64, 410, 0, 0.0, 0.5, 1.0, 1.0, 20000),
        ("64x64, n=0.1, Delta=0 V=0.5 J=1 (C2), T=0.4", 64, 410, 0, 0.0, 0.5, 1.0, 0.4, 20000),
    ]
    for title, L, npl, nmi, delta, V, J, T, nsw in cases:
        if args.quick:
            nsw //= 10
        print(f"## {title}   ({nsw} sweeps / {5 * nsw} maps measured)")
        print("| scheme | attempted pair updates per site and step | tau_int(E) | tau_int(abs Ms) | tau_int(n2) | <E>/N |")
        print("|---|---|---|---|---|---|")
        for r in run(L, npl, nmi, delta, V, J, T, 11, nsw, schemes):
            print(f"| {r['scheme']} | {r['work_per_step']:.3f} | {r['tau_E']:.2f} | {r['tau_Ms']:.2f} | {r['tau_n2']:.2f} | {r['mean_E']:.4f} |")
        print("(tau in attempted pair updates per site)\n")
        sys.stdout.flush()


if __name__ == "__main__":
    main()
