"""Writes tests/golden/ideal_gas_energies.txt: exact canonical energies of N non-interacting xi-particles in the
d-dimensional harmonic trap at the BASELINE.json configurations, at finite P (what the sampled primitive / virial
estimators converge to) and at P = infinity.  Calls only oracle/ideal_gas.py (the finite-P partition-function
recursion written from Eq. 4 and Eq. 6 of arXiv 2404.02628).

    python tests/golden/make_ideal_gas_table.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import ideal_gas  # noqa: E402

ROWS = [
    # name, N, beta, d, xi, P
    ("cfg1", 4, 2.0, 2, 1.0, 16),
    ("cfg1_xi0", 4, 2.0, 2, 0.0, 16),
    ("cfg1_xi-0.5", 4, 2.0, 2, -0.5, 16),
    ("cfg2_g0", 100, 3.0, 2, 1.0, 32),
    ("cfg4_g0", 1000, 3.0, 2, 1.0, 32),
    ("cfg3_g0", 1600, 3.0, 2, 1.0, 32),
    ("cfg5_N2500", 2500, 3.0, 2, 1.0, 16),
    ("cfg5_N10000", 10000, 3.0, 2, 1.0, 16),
    ("cfg5_N20000", 20000, 3.0, 2, 1.0, 16),
    ("cfg5_N40000", 40000, 3.0, 2, 1.0, 16),
    ("paper_beta6_N1600", 1600, 6.0, 2, 1.0, 72),
]


def main():
    out = ["# name N beta d xi P  E(finite P)  E(P = infinity); omega = hbar = m = k_B = 1; written by make_ideal_gas_table.py"]
    for name, N, beta, d, xi, P in ROWS:
        ep = ideal_gas.exact_energy(N, beta, 1.0, d, xi, P)
        ei = ideal_gas.exact_energy(N, beta, 1.0, d, xi, None)
        out.append("%s %d %.17g %d %.17g %d %.15e %.15e" % (name, N, beta, d, xi, P, ep, ei))
    with open(os.path.join(HERE, "ideal_gas_energies.txt"), "w") as f:
        f.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
