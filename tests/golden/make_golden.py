"""Writes tests/golden/tiny_exact.json: exact likelihoods of tiny pairs.

Calls only oracle/ code: ``oracle.bruteforce.likelihood(..., exact=True)`` enumerates every alignment
path of the PairHMM of reference/PAPER.md Eq.1-4 in rational arithmetic (fractions.Fraction built
from the double values of the per-row probabilities), so each stored number is the exactly rounded
log10 of the model's likelihood -- no DP, no GPU value.  Run:  python tests/golden/make_golden.py
"""
import json
import math
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import bruteforce  # noqa: E402

CASES = [
    # read, hap, qb, qi, qd, qg  (scalars or per-base lists); shapes within north_star's brute-force box
    ("A", "A", 30, 45, 45, 10),
    ("A", "C", 30, 45, 45, 10),
    ("A", "ACGT", 20, 45, 45, 10),
    ("AC", "AC", 30, 40, 40, 10),
    ("AC", "ACGT", [30, 20], [40, 35], [45, 30], [10, 10]),
    ("ACG", "ACG", 30, 45, 45, 10),
    ("ACG", "ATCG", [10, 20, 30], [45, 40, 35], [30, 35, 40], [10, 10, 10]),
    ("ACGT", "ACGT", 35, 45, 45, 10),
    ("ACGT", "AGGTAC", [25, 30, 35, 40], [45, 45, 45, 45], [45, 45, 45, 45], [10, 10, 10, 10]),
    ("TTTT", "ACGACG", 30, 45, 45, 10),
    ("GATC", "GATTC", [30, 31, 32, 33], [20, 25, 30, 35], [35, 30, 25, 20], [10, 10, 10, 10]),
    ("ACGT", "TGCATG", [6, 40, 22, 13], [12, 50, 33, 21], [44, 15, 27, 38], [8, 12, 10, 15]),  # non-uniform GCP
]


def main():
    out = []
    for read, hap, qb, qi, qd, qg in CASES:
        L = bruteforce.likelihood(read, hap, qb, qi, qd, qg, exact=True)
        log10L = math.log10(float(L))  # float(Fraction) is correctly rounded; L > 1e-30 for these cases
        out.append({"read": read, "hap": hap, "qb": qb, "qi": qi, "qd": qd, "qg": qg,
                    "L": float(L), "log10L": log10L})
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_exact.json")
    with open(path, "w") as f:
        json.dump({"source": "oracle.bruteforce.likelihood(exact=True): exhaustive path sum of PAPER.md Eq.1-4 "
                             "(readings G1,G4-G8 of DESIGN.md); written by tests/golden/make_golden.py",
                   "cases": out}, f, indent=1)
    print("wrote", path, len(out), "cases")


if __name__ == "__main__":
    main()
