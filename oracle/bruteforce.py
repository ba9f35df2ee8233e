"""ORACLE COMPANION -- test infrastructure.  Brute-force enumeration of every alignment path.

Independent of ``pairhmm_oracle.c`` (no DP, no shared code): a recursive depth-first walk over the
PairHMM state graph that multiplies transition and emission probabilities along each complete
path and sums over paths.  Only usable for tiny inputs (read <= ~5, haplotype <= ~7).

Path model (equivalent to reference/PAPER.md Eq.1-2, readings G1, G6, G7 of DESIGN.md):
  * start: state D at row 0, column j0 in 0..k-1, weight 1/k each (Eq.1: D_{0,j} = C/k; C = 1);
    (a start at column k can never emit a base inside the haplotype and contributes 0);
  * (D,0,j0) -> (M,1,j0+1)                      weight T_DM_1 * P(r_1|h_{j0+1})
  * (M,i,j)  -> (M,i+1,j+1)  T_MM_{i+1} * P     (Eq.2, first line)
               (I,i+1,j)    T_MI_{i+1}          (Eq.2, second line)
               (D,i,j+1)    T_MD_i              (Eq.2, third line: same row i)
  * (I,i,j)  -> (M,i+1,j+1)  T_IM_{i+1} * P ;  (I,i+1,j)  T_II_{i+1}
  * (D,i,j)  -> (M,i+1,j+1)  T_DM_{i+1} * P ;  (D,i,j+1)  T_DD_i        (i >= 1)
  * no I <-> D moves; columns stay <= k; a path is accepted when it sits in M or I at row l (Eq.4).
``exact=True`` does the arithmetic in ``fractions.Fraction`` built from the double values of the
per-row probabilities, so the returned sum is the exact rational value of that model.
"""
from __future__ import annotations

import math
from fractions import Fraction


def row_probs(qb, qi, qd, qg, exact=False):
    """Per-row (p_match, p_mismatch, T_MM, T_MI, T_MD, gamma) from Phred values (Eq.3, G5-G7)."""
    rows = []
    for b, i, d, g in zip(qb, qi, qd, qg):
        eps, iota, dele, gam = (10.0 ** (-q / 10.0) for q in (b, i, d, g))
        if exact:
            eps, iota, dele, gam = Fraction(eps), Fraction(iota), Fraction(dele), Fraction(gam)
            rows.append((1 - eps, eps / 3, 1 - iota - dele, iota, dele, gam))
        else:
            rows.append((1.0 - eps, eps / 3.0, 1.0 - iota - dele, iota, dele, gam))
    return rows


def likelihood(read, hap, qb, qi, qd, qg, exact=False, n_wildcard=False):
    """L (not its log) by summing the weight of every alignment path.  n_wildcard: an ``N`` in either sequence
    matches anything (the compatibility switch of SURVEY 8(f) item 3; off by default = literal Eq.3)."""
    l, k = len(read), len(hap)
    read = read.encode() if isinstance(read, str) else bytes(read)
    hap = hap.encode() if isinstance(hap, str) else bytes(hap)
    sc = lambda v: [v] * l if not hasattr(v, "__len__") else list(v)
    rows = row_probs(sc(qb), sc(qi), sc(qd), sc(qg), exact)
    one = Fraction(1) if exact else 1.0
    zero = Fraction(0) if exact else 0.0

    def emit(i, j):  # P(r_i | h_j), 1-based
        pm, px = rows[i - 1][0], rows[i - 1][1]
        a, c = read[i - 1], hap[j - 1]
        return pm if (a == c or (n_wildcard and (a == 78 or c == 78))) else px

    def walk(state, i, j, w):
        """Sum of weights of all accepted completions of a path currently at (state,i,j) with weight w."""
        total = zero
        if i == l and state in ("M", "I"):
            total += w  # accepted here; (continuations would need row l+1)
        if state == "M" or state == "I" or state == "D":
            # moves that consume read base i+1
            if i < l:
                _, _, tmm, tmi, _, gam = rows[i]
                if j < k:
                    t = tmm if state == "M" else (one - gam)
                    total += walk("M", i + 1, j + 1, w * t * emit(i + 1, j + 1))
                if state == "M":
                    total += walk("I", i + 1, j, w * tmi)
                elif state == "I":
                    total += walk("I", i + 1, j, w * gam)
            # moves that skip haplotype base j+1 (deletion), row i >= 1 only
            if i >= 1 and j < k and state in ("M", "D") and i < l:
                _, _, _, _, tmd, gam = rows[i - 1]
                total += walk("D", i, j + 1, w * (tmd if state == "M" else gam))
        return total

    total = zero
    for j0 in range(k):
        total += walk("D", 0, j0, one / k)
    return total


def log10_likelihood(read, hap, qb, qi, qd, qg, n_wildcard=False):
    return math.log10(float(likelihood(read, hap, qb, qi, qd, qg, n_wildcard=n_wildcard)))
