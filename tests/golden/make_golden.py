"""Writes tests/golden/c0_exact_energies.txt: exact local energies (E_L, E1, E_J, E_K) of the 8 walkers of
config 0 (BASELINE.json:configs[0], seed gen.BASE_SEED) from the oracle's brute-force route (Eq. 8 + Eq. 10,
PAPER.md:91-100).  Calls only gen/ (inputs) and oracle/ (values).  The paper prints no local energy, so this
file is a regression anchor for the oracle's arithmetic, not an external pin (those are in
tests/test_oracle_pins.py).   Usage:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import gen      # noqa: E402
import oracle   # noqa: E402


def main():
    P = gen.make_problem(0)
    phis = gen.make_walkers(P)
    rows = []
    for w in range(P.n_w):
        e = oracle.local_energy_exact(P.h, P.L, P.psi, [phis[0][w]], "bruteforce")
        rows.append([x for z in e for x in (z.real, z.imag)])
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c0_exact_energies.txt")
    np.savetxt(out, np.array(rows), fmt="%.17e",
               header="config 0, seed %d, walkers 0..%d; columns: Re/Im of E_L, E1, E_J, E_K; oracle route "
                      "'bruteforce' (Eq. 8 + Eq. 10 of arxiv 2202.00832); written by tests/golden/make_golden.py"
                      % (P.seed, P.n_w - 1))
    print("wrote", out)


if __name__ == "__main__":
    main()
