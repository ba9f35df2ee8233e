"""ORACLE COMPANION -- test infrastructure.  A second, log-space implementation for large sizes.

Independent of ``pairhmm_oracle.c``: numpy, natural-log domain, and it evaluates the deletion
state through the *closed form* of reference/PAPER.md Eq.6,
    D_{i,j} = T_MD_i * sum_{b<j} M_{i,b} * T_DD_i^(j-1-b),
as a log-cumulative-sum per row, instead of the serial D recurrence of Eq.2.  Agreement with the
C oracle therefore also checks Eq.6.  Uniform or per-row GCP (reading G7).
"""
from __future__ import annotations

import numpy as np

_NEG = -np.inf


def log10_likelihood(read, hap, qb, qi, qd, qg) -> float:
    read = np.frombuffer(read.encode(), np.uint8) if isinstance(read, str) else np.asarray(read, np.uint8)
    hap = np.frombuffer(hap.encode(), np.uint8) if isinstance(hap, str) else np.asarray(hap, np.uint8)
    l, k = len(read), len(hap)
    arr = lambda v: np.full(l, v, dtype=np.float64) if np.isscalar(v) else np.asarray(v, dtype=np.float64)
    qb, qi, qd, qg = arr(qb), arr(qi), arr(qd), arr(qg)
    ln10 = np.log(10.0)
    eps, iota, dele, gam = (np.exp(-q / 10.0 * ln10) for q in (qb, qi, qd, qg))
    with np.errstate(divide="ignore"):
        l_pm, l_px = np.log1p(-eps), np.log(eps / 3.0)
        l_tmm, l_tmi, l_tmd = np.log(1.0 - iota - dele), np.log(iota), np.log(dele)
        l_g, l_1g = np.log(gam), np.log1p(-gam)
    jj = np.arange(k + 1, dtype=np.float64)
    # row 0 (Eq.1, reading G1): M = I = 0, D = 1/k in every column 0..k
    M = np.full(k + 1, _NEG)
    I = np.full(k + 1, _NEG)
    D = np.full(k + 1, -np.log(k))
    for i in range(1, l + 1):
        r = i - 1
        p = np.where(hap == read[r], l_pm[r], l_px[r])                       # Eq.3, columns 1..k
        with np.errstate(invalid="ignore"):
            inner = np.logaddexp(np.logaddexp(l_tmm[r] + M[:-1], l_1g[r] + I[:-1]), l_1g[r] + D[:-1])
            Mn = np.concatenate([[_NEG], p + inner])                          # Eq.2 (M), column 0 = 0
            In = np.logaddexp(l_tmi[r] + M, l_g[r] + I)                       # Eq.2 (I)
            In[0] = _NEG
            # Eq.6: D_{i,j} = T_MD_i * sum_{b<j} M_{i,b} gamma^(j-1-b)
            #             = T_MD_i * gamma^(j-1) * cumsum_{b<j}( M_{i,b} gamma^(-b) )
            t = Mn - jj * l_g[r]
            t[~np.isfinite(Mn)] = _NEG
            c = np.logaddexp.accumulate(t)
            Dn = np.full(k + 1, _NEG)
            Dn[1:] = l_tmd[r] + (jj[1:] - 1.0) * l_g[r] + c[:-1]
        M, I, D = Mn, In, Dn
    tot = np.logaddexp.reduce(np.logaddexp(M[1:], I[1:]))                     # Eq.4
    return float(tot / ln10)
