"""Writes the stored expected values under tests/golden/.  Calls only oracle/ (never the CUDA path).

    python tests/golden/make_golden.py

  dos_3x3.txt, dos_2x4.txt, dos_4x4.txt
      exact density of states g(Q, n2, bV, bJ) with sum M^2, sum Ms^2 per key, by enumeration
      (oracle/ic_enum.c): brute force through eq. (3) for 3x3 and 2x4, row decomposition for 4x4
      (2^32 states; the paper's own test lattice).
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))

from oracle import exact  # noqa: E402


def main():
    for (Lx, Ly) in [(3, 3), (2, 4)]:
        k, c = exact.enum_bruteforce(Lx, Ly)
        dos = exact.dos_from_bruteforce(k, c)
        exact.save_dos(os.path.join(HERE, f"dos_{Lx}x{Ly}.txt"), dos,
                       f"exact density of states of the {Lx}x{Ly} periodic lattice (Lx={Lx}, Ly={Ly}), 4 states per site\n"
                       "brute force over all states, each evaluated with eq. (3) (PAPER.md:37) by orc_recompute\n"
                       "written by tests/golden/make_golden.py (oracle only)")
    dos = exact.enum_rows(4, 4, threads=os.cpu_count() or 1)
    exact.save_dos(os.path.join(HERE, "dos_4x4.txt"), dos,
                   "exact density of states of the 4x4 periodic lattice (the paper's test lattice, PAPER.md:151)\n"
                   "row decomposition over 2^32 states (oracle/ic_enum.c: orc_enum_rows)\n"
                   "written by tests/golden/make_golden.py (oracle only)")


if __name__ == "__main__":
    main()
