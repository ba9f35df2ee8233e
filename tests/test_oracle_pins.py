"""Pins for the CPU oracle (oracle/pairhmm_oracle.c): everything here checks it against something
other than itself -- exhaustive path sums, closed forms, the paper's own first-row formula and Eq.6,
bounds, invariants, stored exact values and a log-space second implementation.  CPU only."""
import json
import math
import os

import numpy as np
import pytest

import oracle
from oracle import bruteforce, logspace
from paper_2606_25738_b200 import workloads as W

LOG10_2 = math.log10(2.0)


def _rand_case(rng, l, k, uniform_gcp=False):
    read = "".join(rng.choice(list("ACGT"), l))
    hap = "".join(rng.choice(list("ACGT"), k))
    qb = rng.integers(3, 42, l)
    qi = rng.integers(8, 60, l)
    qd = rng.integers(8, 60, l)
    qg = np.full(l, 10) if uniform_gcp else rng.integers(4, 25, l)
    return read, hap, qb, qi, qd, qg


# ----------------------------------------------------------------------------- brute force
def test_bruteforce_all_small_shapes():
    """north_star: all alignment paths for reads <= 4 bp and haplotypes <= 6 bp (non-uniform GCP too)."""
    rng = np.random.default_rng(11)
    worst = 0.0
    for l in range(1, 5):
        for k in range(1, 7):
            for rep in range(4):
                read, hap, qb, qi, qd, qg = _rand_case(rng, l, k, uniform_gcp=(rep % 2 == 0))
                if rep == 3:  # make the read (nearly) a substring so match paths dominate
                    hap = (read + hap)[:k] if k >= l else hap
                got = oracle.forward_pair(read, qb, qi, qd, qg, hap)
                want = bruteforce.log10_likelihood(read, hap, qb, qi, qd, qg)
                worst = max(worst, abs(got - want))
    assert worst < 1e-12, worst


def test_bruteforce_n_bases_literal_and_wildcard():
    """Reading G17: Eq.3 compares bytes, so an N matches an N only; with the compatibility switch n_wildcard (SURVEY 8(f)
    item 3, off in every config) an N in either sequence matches anything.  Both against the path enumeration, which
    implements the two rules in its own emit()."""
    rng = np.random.default_rng(17)
    worst = 0.0
    differ = 0
    for l in range(1, 5):
        for k in range(1, 7):
            for rep in range(4):
                read, hap, qb, qi, qd, qg = _rand_case(rng, l, k, uniform_gcp=(rep % 2 == 0))
                read, hap = list(read), list(hap)
                read[int(rng.integers(0, l))] = "N"
                if rep >= 2:
                    hap[int(rng.integers(0, k))] = "N"
                read, hap = "".join(read), "".join(hap)
                vals = []
                for wild in (False, True):
                    got = oracle.forward_pair(read, qb, qi, qd, qg, hap, n_wildcard=wild)
                    want = bruteforce.log10_likelihood(read, hap, qb, qi, qd, qg, n_wildcard=wild)
                    worst = max(worst, abs(got - want))
                    vals.append(got)
                assert vals[1] >= vals[0] - 1e-12  # a wildcard can only add matches
                differ += vals[1] > vals[0] + 1e-9
    assert worst < 1e-12, worst
    assert differ > 50
    assert oracle.forward_pair("N", 30, 45, 45, 10, "N") == oracle.forward_pair("A", 30, 45, 45, 10, "A")  # literal N == N
    assert oracle.forward_pair("N", 30, 45, 45, 10, "A") < oracle.forward_pair("N", 30, 45, 45, 10, "A", n_wildcard=True)


def test_golden_exact_values():
    """tests/golden/tiny_exact.json: exact rational path sums (written by make_golden.py from oracle/bruteforce)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "tiny_exact.json")
    cases = json.load(open(path))["cases"]
    assert len(cases) >= 10
    for c in cases:
        got = oracle.forward_pair(c["read"], c["qb"], c["qi"], c["qd"], c["qg"], c["hap"])
        assert abs(got - c["log10L"]) < 1e-12, (c, got)


def test_golden_hand_values():
    """Values that can be checked by hand from Eq.1-3: read 'A' vs hap 'A' at Q30, GCP 10:
    L = T_DM * (1-eps) / k = 0.9 * 0.999; vs hap 'C': 0.9 * 0.001/3."""
    assert abs(oracle.forward_pair("A", 30, 45, 45, 10, "A") - math.log10(0.9 * 0.999)) < 1e-14
    assert abs(oracle.forward_pair("A", 30, 45, 45, 10, "C") - math.log10(0.9 * 0.001 / 3)) < 1e-14


# ----------------------------------------------------------------------------- closed forms
def test_closed_form_one_base_read():
    """l = 1: L = (1-gamma_1)/k * [n_match (1-eps) + (k-n_match) eps/3]   (Eq.1-4 by inspection)."""
    rng = np.random.default_rng(5)
    for _ in range(50):
        k = int(rng.integers(1, 200))
        hap = "".join(rng.choice(list("ACGT"), k))
        r = str(rng.choice(list("ACGT")))
        qb, qg = int(rng.integers(2, 60)), int(rng.integers(3, 30))
        eps, gam = 10 ** (-qb / 10), 10 ** (-qg / 10)
        nm = hap.count(r)
        want = math.log10((1 - gam) / k * (nm * (1 - eps) + (k - nm) * eps / 3))
        got = oracle.forward_pair(r, qb, int(rng.integers(5, 60)), int(rng.integers(5, 60)), qg, hap)
        assert abs(got - want) < 1e-13


def test_closed_form_one_base_haplotype():
    """k = 1, l >= 2: only 'match then insertions' survives:
    L = p_{1,1} (1-gamma_1) iota_2 prod_{i>=3} gamma_i."""
    rng = np.random.default_rng(6)
    for _ in range(50):
        l = int(rng.integers(2, 40))
        read, hap, qb, qi, qd, qg = _rand_case(rng, l, 1)
        eps1 = 10 ** (-qb[0] / 10)
        p11 = (1 - eps1) if read[0] == hap[0] else eps1 / 3
        want = math.log10(p11) + math.log10(1 - 10 ** (-qg[0] / 10)) + (-qi[1] / 10) + sum(-qg[i] / 10 for i in range(2, l))
        got = oracle.forward_pair(read, qb, qi, qd, qg, hap)
        assert abs(got - want) < 1e-12 * max(1.0, abs(want))


def test_gapless_limit():
    """With Qi = Qd = 93 every gapped path is ~1e-9 below the gapless mass, so for a read that is an
    exact substring L = sum_{j0} (1/k)(1-gamma) prod_i p(r_i|h_{j0+i}) prod_{i>=2} T_MM_i to ~1e-8."""
    rng = np.random.default_rng(7)
    for l, k in [(5, 9), (40, 90), (150, 300)]:
        hap = "".join(rng.choice(list("ACGT"), k))
        s = int(rng.integers(0, k - l + 1))
        read = list(hap[s:s + l])
        for pos in rng.choice(l, size=min(2, l), replace=False):   # <= 2 mismatches
            read[pos] = "ACGT"[("ACGT".index(read[pos]) + 1) % 4]
        read = "".join(read)
        qb = rng.integers(20, 41, l)
        eps = 10.0 ** (-qb / 10.0)
        tmm = 1.0 - 2 * 10.0 ** (-9.3)
        terms = []
        for j0 in range(0, k - l + 1):
            lp = math.log(0.9 / k) + (l - 1) * math.log(tmm)
            for i in range(l):
                lp += math.log(1 - eps[i]) if read[i] == hap[j0 + i] else math.log(eps[i] / 3)
            terms.append(lp)
        m = max(terms)
        want = (m + math.log(sum(math.exp(t - m) for t in terms))) / math.log(10)
        got = oracle.forward_pair(read, qb, 93, 93, 10, hap)
        assert abs(got - want) < 2e-7, (l, k, got, want)


# ----------------------------------------------------------------------------- the paper's own statements
def test_first_row_formula_of_the_paper():
    """M_{1,j} = p_{1,j} * T_DM * 2^1020 / k for every j (incl. j = 1, reading G1); I_{1,j} = 0."""
    rng = np.random.default_rng(8)
    read, hap, qb, qi, qd, qg = _rand_case(rng, 3, 17, uniform_gcp=True)
    _, M, I, D, ex = oracle.forward_pair(read, qb, qi, qd, qg, hap, log2C=1020, rescale=False, matrices=True)
    eps = 10 ** (-qb[0] / 10)
    for j in range(1, 18):
        p = (1 - eps) if read[0] == hap[j - 1] else eps / 3
        want = p * 0.9 * 2.0 ** 1020 / 17
        assert abs(M[1, j] - want) <= 4e-16 * want
        assert I[1, j] == 0.0
    assert np.all(M[:, 0] == 0) and np.all(I[:, 0] == 0) and np.all(D[1:, 0] == 0)   # Eq.1
    assert np.all(D[0, :] == 2.0 ** 1020 / 17) and np.all(ex == 0)


def test_eq6_identity_on_stored_rows():
    """PAPER.md:112-115 (Eq.6): D_{i,j} = T_MD_i sum_{b=1}^{j-1} M_{i,b} T_DD^(j-1-b) for i >= 1."""
    rng = np.random.default_rng(9)
    read, hap, qb, qi, qd, qg = _rand_case(rng, 12, 23)
    _, M, I, D, ex = oracle.forward_pair(read, qb, qi, qd, qg, hap, rescale=False, matrices=True)
    for i in range(1, 13):
        tmd, g = 10 ** (-qd[i - 1] / 10), 10 ** (-qg[i - 1] / 10)
        for j in range(1, 24):
            want = tmd * sum(M[i, b] * g ** (j - 1 - b) for b in range(1, j))
            assert abs(D[i, j] - want) <= 1e-13 * max(want, 1e-300)


def test_eq7_rowwise_form_and_eq9_tile_carry():
    """PAPER.md:119 (Eq.7) and :245-257 (Eq.8-9): M_{i,j} from row i-1 only, with the weighted prefix
    T = sum_{b<=tN} M_{i-1,b} g^(tN-b) carried into a tile that starts at column tN+1:
    cell tN+1 needs (T - M_{tN})/g, cell tN+2 needs T, cell tN+3 needs g*T + M_{tN+1}, ..."""
    rng = np.random.default_rng(10)
    read, hap, qb, qi, qd, qg = _rand_case(rng, 6, 16, uniform_gcp=True)
    _, M, I, D, _ = oracle.forward_pair(read, qb, qi, qd, qg, hap, rescale=False, matrices=True)
    g, N = 0.1, 4
    for i in range(2, 7):
        eps = 10 ** (-qb[i - 1] / 10)
        tmm = 1 - 10 ** (-qi[i - 1] / 10) - 10 ** (-qd[i - 1] / 10)
        tmd_prev = 10 ** (-qd[i - 2] / 10)
        for t in range(1, 4):
            T = sum(M[i - 1, b] * g ** (t * N - b) for b in range(1, t * N + 1))          # Eq.8
            sums = [(T - M[i - 1, t * N]) / g, T]                                          # Eq.9
            sums.append(g * sums[-1] + M[i - 1, t * N + 1])
            sums.append(g * sums[-1] + M[i - 1, t * N + 2])
            for c in range(N):
                j = t * N + 1 + c
                p = (1 - eps) if read[i - 1] == hap[j - 1] else eps / 3
                want = p * (tmm * M[i - 1, j - 1] + 0.9 * I[i - 1, j - 1] + 0.9 * tmd_prev * sums[c])   # Eq.7
                assert abs(M[i, j] - want) <= 1e-11 * max(M[i, j], 1e-300), (i, j)


# ----------------------------------------------------------------------------- bounds
def test_bounds():
    """With constant Qd and GCP the out-weights of every state sum to 1 and emissions to <= 1: L <= 1.
    Always: L >= weight of one gapless diagonal path."""
    rng = np.random.default_rng(12)
    for _ in range(30):
        l, k = int(rng.integers(1, 60)), int(rng.integers(1, 90))
        read, hap, qb, qi, _, _ = _rand_case(rng, l, k)
        got = oracle.forward_pair(read, qb, qi, 40, 10, hap)
        assert got <= 1e-12
        if k >= l:
            lp = math.log10(0.9 / k)
            for i in range(l):
                eps = 10 ** (-qb[i] / 10)
                lp += math.log10(1 - eps if read[i] == hap[i] else eps / 3)
                if i >= 1:
                    lp += math.log10(1 - 10 ** (-qi[i] / 10) - 1e-4)
            assert got >= lp - 1e-12


# ----------------------------------------------------------------------------- invariants
def test_mismatch_monotonicity():
    """Haplotype over {A,C}, read an exact substring; turning read bases into 'G' (matches nowhere)
    one at a time strictly lowers L every time."""
    rng = np.random.default_rng(13)
    hap = "".join(rng.choice(list("AC"), 80))
    read = list(hap[20:60])
    prev = oracle.forward_pair("".join(read), 30, 45, 45, 10, hap)
    for pos in rng.permutation(40)[:15]:
        read[pos] = "G"
        cur = oracle.forward_pair("".join(read), 30, 45, 45, 10, hap)
        assert cur < prev
        prev = cur


def test_pair_order_independence_bitwise():
    b = W.generate(0)
    base = oracle.forward_batch(b)
    perm = np.random.default_rng(14).permutation(b.n_pairs)
    again = oracle.forward_batch(b.select_pairs(perm))
    assert np.array_equal(again, base[perm])
    dup = oracle.forward_batch(b.select_pairs(np.concatenate([perm[:10], perm[:10]])))
    assert np.array_equal(dup[:10], dup[10:])
    one = oracle.forward_batch(b, n_threads=1)
    assert np.array_equal(one, base)


def test_scale_constant_and_rescaling_independence():
    """Result does not depend on C (Eq.1's 2^1020 vs 1) nor on whether rows are rescaled."""
    b = W.generate(1, n=1)
    idx = np.arange(0, b.n_pairs, 37)
    a = oracle.forward_batch(b, pairs=idx)                                  # C = 1, rescaled
    c = oracle.forward_batch(b, pairs=idx, log2C=1020, rescale=False)       # the paper's setting
    d = oracle.forward_batch(b, pairs=idx, log2C=1020, rescale=True)
    e = oracle.forward_batch(b, pairs=idx, log2C=0, rescale=False)
    assert np.max(np.abs(a - c)) < 1e-11 and np.max(np.abs(a - d)) < 1e-11 and np.max(np.abs(a - e)) < 1e-11


def test_appending_haplotype_bases():
    """Every path inside hap is a path inside hap+X with the same weight apart from the 1/k start
    factor, so (k+1) L(hap+X) >= k L(hap)."""
    rng = np.random.default_rng(15)
    for _ in range(20):
        l, k = int(rng.integers(1, 30)), int(rng.integers(1, 40))
        read, hap, qb, qi, qd, qg = _rand_case(rng, l, k)
        a = oracle.forward_pair(read, qb, qi, qd, qg, hap)
        c = oracle.forward_pair(read, qb, qi, qd, qg, hap + "ACGT"[int(rng.integers(4))])
        assert c + math.log10(k + 1) >= a + math.log10(k) - 1e-12


def test_never_underflows_and_is_finite():
    """Unrelated 3000-bp read: L ~ 1e-3000, far below double range; the exponent bookkeeping keeps it finite."""
    rng = np.random.default_rng(16)
    read, hap, qb, qi, qd, qg = _rand_case(rng, 3000, 3300, uniform_gcp=True)
    v = oracle.forward_pair(read, qb, qi, qd, qg, hap)
    assert math.isfinite(v) and -5000 < v < -1500
    w = oracle.forward_pair(read, qb, qi, qd, qg, hap, log2C=1020, rescale=False)
    assert w == -math.inf or not math.isfinite(w)      # the paper's constant alone does underflow here


# ----------------------------------------------------------------------------- second implementation
def test_logspace_second_implementation():
    b = W.generate(0)
    o = oracle.forward_batch(b)
    for p in range(0, b.n_pairs, 16):
        r, qb, qi, qd, qg, h = b.pair(p)
        assert abs(logspace.log10_likelihood(r, h, qb, qi, qd, qg) - o[p]) < 1e-9
    b3 = W.generate(3, n=2, len_lo=1800, len_hi=2200)
    o3 = oracle.forward_batch(b3)
    for p in range(2):
        r, qb, qi, qd, qg, h = b3.pair(p)
        assert abs(logspace.log10_likelihood(r, h, qb, qi, qd, qg) - o3[p]) < 1e-9


def test_nonuniform_gcp_logspace():
    rng = np.random.default_rng(17)
    read, hap, qb, qi, qd, qg = _rand_case(rng, 60, 90, uniform_gcp=False)
    assert abs(logspace.log10_likelihood(read, hap, qb, qi, qd, qg) - oracle.forward_pair(read, qb, qi, qd, qg, hap)) < 1e-10
