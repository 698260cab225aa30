"""Writes tests/golden/saw_cubic_exact.txt from the oracle's brute-force enumerator only.

Usage:  python tests/golden/make_saw_exact.py [n_max]      (default 15; n=15 takes ~6 min)

For every n = 1..n_max: c_n, sum over all n-step cubic-lattice SAWs of Ree^2, sum of N^2*Rg^2
(N = n+1 monomers), and the exact survival probability P_alive(n) = sum_w 1/W(w) as a fraction
(Eq. 3). Calls nothing but oracle/ (saw_enum.cpp + the oracle's free-site routine).
"""
import os
import sys
from fractions import Fraction

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
import oracle  # noqa: E402


def main():
    n_max = int(sys.argv[1]) if len(sys.argv) > 1 else 15
    lines = [
        "# exact enumeration of n-step self-avoiding walks on the simple cubic lattice",
        "# written by tests/golden/make_saw_exact.py (oracle/saw_enum.cpp); c_n agrees with the",
        "# published series (tests/golden/saw_cubic_counts.txt)",
        "# n  c_n  sum_Ree2  sum_N2Rg2  P_alive_num/P_alive_den",
    ]
    for n in range(1, n_max + 1):
        e = oracle.saw_enumerate(n, fix_first=(n >= 9))
        pa = sum(Fraction(c, 2 ** a * 3 ** b * 5 ** cc) for (a, b, cc), c in e["hist"].items())
        lines.append(f"{n} {e['count']} {e['sum_ree2']} {e['sum_n2rg2']} {pa.numerator}/{pa.denominator}")
        print(lines[-1], flush=True)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "saw_cubic_exact.txt")
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
