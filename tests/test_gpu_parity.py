"""Parity of the CUDA path (through the C ABI, include/pairhmm_b200.h) against the CPU oracle.

Element by element on seeded inputs shaped like BASELINE.json configs[0..4] at sizes the oracle
finishes in seconds, on sampled pairs at the full sizes bench.py times, plus the edge cases.
Tolerances (BASELINE.json north_star): |dlog10 L| <= 1e-3 for PHMM_FP32_RESCUE (rescued pairs
included), <= 1e-9 for PHMM_FP64; pair indexing and the rescue flag set exact (reading G16)."""
import math

import numpy as np
import pytest

import oracle
from paper_2606_25738_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL32, TOL64 = 1e-3, 1e-9
LOG10_2 = math.log10(2.0)
# G16: the fp32 pass runs with C = 2^120 and a pair is redone in fp64 iff its scaled sum < 2^-90
RESCUE_LOG10 = (-90 - 120) * LOG10_2
BORDER = 1e-3


@pytest.fixture(scope="module")
def B():
    from paper_2606_25738_b200 import binding
    return binding


@pytest.fixture(scope="module")
def ctx(B):
    c = B.Context(0)
    yield c
    c.close()


def run(B, ctx, batch, prec):
    db = B.DeviceBatch(batch)
    out, fl = ctx.forward_batch(db, prec)
    return out.cpu().numpy(), fl.cpu().numpy()


def check(B, ctx, batch, prec, ref=None, pairs=None):
    out, fl = run(B, ctx, batch, prec)
    assert np.all(np.isfinite(out)), "non-finite outputs at %s" % np.where(~np.isfinite(out))[0][:8]
    if ref is None:
        ref = oracle.forward_batch(batch, pairs=pairs)
    got = out if pairs is None else out[pairs]
    err = np.abs(got - ref)
    tol = TOL32 if prec == B.PHMM_FP32_RESCUE else TOL64
    bad = np.where(~(err <= tol))[0]
    assert len(bad) == 0, "max err %g at %s (got %s want %s)" % (err.max(), bad[:5], got[bad[:5]], ref[bad[:5]])
    return out, fl, ref


def check_flags(B, batch, fl, ref, pairs=None, long_may_fall_back=False):
    """Rescue flags must equal the oracle's prediction except within +-1e-3 of the threshold (G16).
    That criterion is the short path's; long-path pairs carry PHMM_FLAG_LONG, and PHMM_FLAG_RESCUED on top only where the
    fp32 long kernel handed the pair to fp64 (never on the GCP-10 data of the configs)."""
    f = fl if pairs is None else fl[pairs]
    is_long = (f & B.PHMM_FLAG_LONG) != 0
    want = ref < RESCUE_LOG10
    border = np.abs(ref - RESCUE_LOG10) <= BORDER
    sel = ~is_long & ~border
    got = (f & B.PHMM_FLAG_RESCUED) != 0
    assert np.array_equal(got[sel], want[sel]), "rescue flag mismatch at %s" % np.where(got[sel] != want[sel])[0][:8]
    assert long_may_fall_back or not np.any(got & is_long)
    return int(border.sum())


# ------------------------------------------------------------------ configs at oracle-sized scale
def test_config0_tiny_fp32_and_fp64(B, ctx):
    b = W.generate(0)
    assert b.n_pairs == 256
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert check_flags(B, b, fl, ref) == 0
    # 3 of 4 haplotypes are unrelated to each read: most pairs must have needed the fp64 rescue
    assert 150 <= int((fl & B.PHMM_FLAG_RESCUED).sum()) <= 200
    out64, fl64, _ = check(B, ctx, b, B.PHMM_FP64, ref=ref)
    assert not np.any(fl64 & B.PHMM_FLAG_RESCUED)


def test_config1_short_regions(B, ctx):
    b = W.generate(1, n=12)  # 12 regions x 1024 pairs; spans many warps / tasks and ragged lane groups
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    check_flags(B, b, fl, ref)
    check(B, ctx, b, B.PHMM_FP64, ref=ref)


def test_config2_mixed_stream(B, ctx):
    b = W.generate(2, n=30000)  # unsorted pairs, 5% unrelated reads, haplotypes up to 1200 (short and long path)
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    nb = check_flags(B, b, fl, ref)
    assert nb <= 3
    n_resc = int((fl & B.PHMM_FLAG_RESCUED).sum())
    assert 0.02 * b.n_pairs < n_resc < 0.25 * b.n_pairs  # >= the ~5% unrelated reads, plus reads overhanging their haplotype window
    st = ctx.stats()
    assert st["n_rescued"] == n_resc
    b64 = b.select_pairs(np.arange(0, b.n_pairs, 5))
    check(B, ctx, b64, B.PHMM_FP64, ref=ref[::5])


def test_config3_long_reads_scaled(B, ctx):
    b = W.generate(3, n=6, len_lo=1500, len_hi=2500)
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert np.all(fl & B.PHMM_FLAG_LONG)
    check(B, ctx, b, B.PHMM_FP64, ref=ref)


def test_config3_long_reads_full_length(B, ctx):
    b = W.generate(3, n=4)  # 5-15 kbp reads: thousands of bits of dynamic range, rescaling mandatory
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert ref.min() < -1000
    check(B, ctx, b, B.PHMM_FP64, ref=ref)


def test_config4_very_long_scaled(B, ctx):
    b = W.generate(4, n=2, len_lo=24000, len_hi=24000)  # same error model, 24 kbp x 25.2 kbp: ~25 strips per pair
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert np.all(fl & B.PHMM_FLAG_LONG)
    check(B, ctx, b, B.PHMM_FP64, ref=ref)


# ------------------------------------------------------------------ full sizes, sampled
def test_config1_full_size_sampled(B, ctx):
    """The batch and launch configuration bench.py times (2.05 M pairs); oracle on 1500 sampled pairs."""
    b = W.generate(1)
    assert b.n_pairs == 2000 * 128 * 8
    rng = np.random.default_rng(5)
    pairs = np.sort(rng.choice(b.n_pairs, 1500, replace=False))
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE, pairs=pairs)
    check_flags(B, b, fl, ref, pairs=pairs)
    assert np.all(out <= 0.5)  # L stays below a small constant


def test_config3_full_size_sampled(B, ctx):
    b = W.generate(3)
    rng = np.random.default_rng(6)
    pairs = np.sort(rng.choice(b.n_pairs, 3, replace=False))
    check(B, ctx, b, B.PHMM_FP32_RESCUE, pairs=pairs)


def test_config2_full_size_sampled(B, ctx):
    """BASELINE.json configs[2] at its stated size: 10 M unsorted pairs, 5 % unrelated reads (6.9e11 cells), in the
    launch configuration bench.py --workload mixed times.  Oracle on 20 000 uniformly sampled pairs (unrelated reads
    included at their natural rate): values element-wise, the rescue-flag set exactly (reading G16), the library's
    rescue count against the flags; then every 50th pair (200 000) through PHMM_FP64 at 1e-9."""
    b = W.generate(2)
    assert b.n_pairs == 10_000_000
    rng = np.random.default_rng(7)
    pairs = np.sort(rng.choice(b.n_pairs, 20000, replace=False))
    db = B.DeviceBatch(b)
    out_t, fl_t = ctx.forward_batch(db, B.PHMM_FP32_RESCUE)
    st = ctx.stats()
    out, fl = out_t.cpu().numpy(), fl_t.cpu().numpy()
    del out_t, fl_t
    assert np.all(np.isfinite(out))
    ref = oracle.forward_batch(b, pairs=pairs)
    err = np.abs(out[pairs] - ref)
    assert err.max() <= TOL32, "max err %g at pair %d" % (err.max(), pairs[int(err.argmax())])
    n_border = check_flags(B, b, fl, ref, pairs=pairs)
    print("configs[2] full: max |dlog10| %.2e on %d sampled pairs, %d borderline, %d rescued of %d, %d slices"
          % (err.max(), len(pairs), n_border, st["n_rescued"], b.n_pairs, st["n_slices"]))
    assert n_border <= 3
    n_resc = int((fl & B.PHMM_FLAG_RESCUED).sum())
    assert st["n_rescued"] == n_resc and st["n_pairs"] == b.n_pairs and st["cells"] == b.cells()
    assert 0.04 * b.n_pairs < n_resc < 0.25 * b.n_pairs
    assert int(((ref < RESCUE_LOG10) & (np.abs(ref - RESCUE_LOG10) > BORDER)).sum()) > 500  # the sample does exercise the rescue
    sub = np.arange(0, b.n_pairs, 50)
    del db
    b64 = b.select_pairs(sub)
    ref64 = oracle.forward_batch(b64)
    out64, fl64 = run(B, ctx, b64, B.PHMM_FP64)
    e64 = np.abs(out64 - ref64)
    assert e64.max() <= TOL64, "fp64 max err %g" % e64.max()
    assert np.max(np.abs(out[sub] - ref64)) <= TOL32  # and the fp32+rescue run of the full batch on those 200 000 pairs


def test_config4_full_size_all_pairs(B, ctx):
    """BASELINE.json configs[4] at its stated size: 16 pairs of 100 kbp x 105 kbp, every pair against the oracle in
    both precisions at north_star's tolerances (1e-3 after fp32, 1e-9 in fp64); about -0.8 bits per row."""
    b = W.generate(4)
    assert b.n_pairs == 16
    ref = oracle.forward_batch(b)
    o32, f32 = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    o64, f64 = run(B, ctx, b, B.PHMM_FP64)
    assert np.all(np.isfinite(o32)) and np.all(np.isfinite(o64))
    assert np.all((ref < -15000) & (ref > -40000))
    assert np.all(f32 & B.PHMM_FLAG_LONG) and np.all(f64 & B.PHMM_FLAG_LONG)
    e32, e64 = np.abs(o32 - ref), np.abs(o64 - ref)
    print("configs[4] full: max |dlog10| fp32 %.2e fp64 %.2e" % (e32.max(), e64.max()))
    assert e32.max() <= TOL32
    assert e64.max() <= TOL64


# ------------------------------------------------------------------ indexing / batching invariants
def test_pair_order_and_duplicates_bitwise(B, ctx):
    b = W.generate(2, n=6000)
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    rng = np.random.default_rng(9)
    perm = rng.permutation(b.n_pairs)
    out_p, fl_p = run(B, ctx, b.select_pairs(perm), B.PHMM_FP32_RESCUE)
    assert np.array_equal(out_p, out[perm]) and np.array_equal(fl_p, fl[perm])
    dup = np.concatenate([np.arange(100), np.arange(100), np.arange(50)])
    out_d, _ = run(B, ctx, b.select_pairs(dup), B.PHMM_FP32_RESCUE)
    assert np.array_equal(out_d, out[dup])


def test_equal_length_sweep_shape(B, ctx):
    """the paper's scalability-sweep shape (read length = haplotype length, noisy copies,
    PAPER.md:366), one length per kernel family: 32 and 512 (short kernel; 512-bp reads partly rescued), 1024 (short
    kernel + chain fallback of the rescued ones), 3000 (chain kernel, 3 strips)."""
    for L, n in ((32, 300), (512, 40), (1024, 12), (3000, 4)):
        b = W.generate(5, seed=40 + L, n=n, len_lo=L)
        out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
        check_flags(B, b, fl, ref)
        check(B, ctx, b, B.PHMM_FP64, ref=ref)


def test_equal_length_sweep_shape_long(B, ctx):
    """The upper end of the paper's scalability sweep (PAPER.md:378-392 runs to 131072 bp): one pair each of 16384 and
    65536 bp (16 and 64 strips chained through boundary records), both precisions, against the oracle."""
    for L in (16384, 65536):
        b = W.generate(5, seed=40 + L, n=1, len_lo=L)
        ref = oracle.forward_batch(b)
        out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
        assert fl[0] == B.PHMM_FLAG_LONG
        assert abs(out[0] - ref[0]) <= TOL32, (L, out[0], ref[0])
        out64, _ = run(B, ctx, b, B.PHMM_FP64)
        assert abs(out64[0] - ref[0]) <= TOL64, (L, out64[0], ref[0])


def test_long_kernel_stress_mixed_structure(B, ctx):
    """The fp32 long kernel's exponent scheme on inputs built to move the mass around: haplotypes of
    1.1-5 kbp, reads of 50-3000 bp that are related, unrelated, or related in one part and unrelated in the other, with
    deletions of up to 55 and insertions of up to 40 bases, per-base gap-continuation qualities between 5 and 30 (rows on
    which the running sum hardly decays next to rows on which it vanishes within a lane), base qualities 5-40."""
    rng = np.random.default_rng(77)
    cases = []
    for it in range(120):
        k = int(rng.integers(1100, 5000))
        hap = _rand_seq(rng, k)
        l = int(rng.integers(50, min(3000, k - 100)))
        kind = it % 4
        s0 = int(rng.integers(0, k - l - 60))
        rd = list(hap[s0:s0 + l + 60])
        if kind == 1:
            rd = list(_rand_seq(rng, l))                                   # unrelated
        elif kind == 2:
            cut = int(rng.integers(l // 4, 3 * l // 4))
            rd = rd[:cut] + list(_rand_seq(rng, l - cut))                  # related head, unrelated tail
        elif kind == 3:
            cut = int(rng.integers(l // 4, 3 * l // 4))
            d = int(rng.integers(5, 56))
            rd = rd[:cut] + rd[cut + d:]                                   # a deletion of d bases in the read
            if rng.random() < 0.5:
                c2 = int(rng.integers(10, max(11, cut - 5)))
                rd = rd[:c2] + list(_rand_seq(rng, int(rng.integers(3, 41)))) + rd[c2:]  # and an insertion
        rd = rd[:l]
        for i in rng.choice(len(rd), max(1, len(rd) // 30), replace=False):
            rd[i] = "ACGT"[int(rng.integers(0, 4))]
        n = len(rd)
        gcp = rng.integers(5, 31, n) if it % 3 else np.full(n, 10)
        cases.append(("".join(rd), hap, list(rng.integers(5, 41, n)), list(rng.integers(15, 50, n)), list(rng.integers(15, 50, n)), list(gcp)))
    b = W.from_strings(cases)
    ref = oracle.forward_batch(b)
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert np.all(np.isfinite(out))
    err = np.abs(out - ref)
    bad = np.where(~(err <= TOL32))[0]
    assert len(bad) == 0, "max err %g at %s (got %s want %s, flags %s)" % (err.max(), bad[:6], out[bad[:6]], ref[bad[:6]], fl[bad[:6]])
    assert np.all(fl & B.PHMM_FLAG_LONG)
    n_fb = int((fl & B.PHMM_FLAG_RESCUED).sum())
    print("long-kernel stress: max |dlog10| %.2e, %d of %d pairs fell back to the fp64 chain kernel" % (err.max(), n_fb, b.n_pairs))
    out64, _ = run(B, ctx, b, B.PHMM_FP64)
    assert np.max(np.abs(out64 - ref)) <= TOL64


def test_reads_with_a_long_deletion_against_the_haplotype(B, ctx):
    """A read made of two stretches of the haplotype that lie hundreds of columns apart (a long deletion in the read; also the
    reverse order, which no path can follow): the second stretch starts as a cell far below the lanes to its left and must
    not be flushed by their exponents -- the long kernel's constraint allows for what a path pays to cross a lane (DESIGN.md
    section 6; without that term these came out too small by up to 240 in log10, silently).  Reference: the log-space
    companion (the C oracle's 2^-1074-per-row limit bites on three of the eight)."""
    from oracle import logspace
    rng = np.random.default_rng(11)
    cases = []
    for (k, x0, xl, y0, yl) in ((2000, 100, 300, 1300, 300), (2000, 100, 150, 700, 400), (3000, 50, 600, 1500, 600),
                                (5000, 100, 1000, 3000, 1000), (2000, 1200, 300, 100, 300), (1500, 100, 300, 600, 300),
                                (4000, 200, 400, 500, 400), (2500, 100, 500, 1124, 500), (1030, 10, 200, 500, 300), (1100, 0, 120, 980, 120)):
        hap = _rand_seq(rng, k)
        cases.append((hap[x0:x0 + xl] + hap[y0:y0 + yl], hap))
    b = W.from_strings(cases, qb=30, qi=45, qd=45, qg=10)
    ref = np.array([logspace.log10_likelihood(*[b.pair(i)[j] for j in (0, 5, 1, 2, 3, 4)]) for i in range(b.n_pairs)])
    c_or = oracle.forward_batch(b)
    assert np.sum(np.abs(c_or - ref) > 1e-6) >= 2 and np.all(c_or <= ref + 1e-9)  # the C oracle loses mass on some of these, never gains
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert np.max(np.abs(out - ref)) <= TOL32, (out, ref)
    assert np.all(fl == B.PHMM_FLAG_LONG)  # computed by the fp32 long kernel itself, no fp64 fallback
    out64, _ = run(B, ctx, b, B.PHMM_FP64)
    assert np.max(np.abs(out64 - ref)) <= TOL64


def test_m_states_inside_a_long_deletion(B, ctx):
    """Where opening a gap costs about what extending one does (deletion quality 10), a long deletion can be split by an M
    state in any column whose base happens to match: together those paths carry percents of the likelihood, and each of their
    cells sits up to 103 bits below the largest cell of its 32-column lane.  The fp32 long kernel flushed the ones at the far
    end of the lanes inside the deletion (0.6 % of the likelihood, found by the randomized batches: generator seed 600227,
    a 2559-base read against a 4407-base haplotype) until what a lane proposes to its right neighbours became what can
    LEAVE it within an interval instead of its maximum (csrc/phmm_long.cu).  Reference: the log-space companion (the C
    oracle drops cells 2^-1074 below their row maximum and loses the second stretch altogether)."""
    from oracle import logspace
    rng = np.random.default_rng(600227)
    b = _fz_make(rng, 12, 6000, 3000)
    sel = [i for i in range(b.n_pairs) if b.read_len()[b.pair_read[i]] == 2559 and b.hap_len()[b.pair_hap[i]] == 4407]
    assert sel, "the generator no longer reproduces the batch of seed 600227"
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    out64, _ = run(B, ctx, b, B.PHMM_FP64)
    for i in sel:
        pp = b.pair(i)
        ref = logspace.log10_likelihood(pp[0], pp[5], pp[1], pp[2], pp[3], pp[4])
        assert abs(out64[i] - ref) <= TOL64 and abs(out[i] - ref) <= TOL32 / 10, (out[i], out64[i], ref, fl[i])
    rng = np.random.default_rng(52)
    hap = _rand_seq(rng, 4300)
    pairs, refs = [], []
    for gap in (150, 333, 597, 801, 1100, 2050):
        for a0 in (700, 711, 733):
            cut, l = 400 + int(rng.integers(0, 30)), 900
            read = hap[a0:a0 + cut] + hap[a0 + cut + gap:a0 + gap + l]
            qb = list(rng.integers(2, 42, l)) if a0 != 711 else [30] * l
            pairs.append((read, hap, qb, 40, 10, 10))
    b = W.from_strings(pairs)
    ref = np.array([logspace.log10_likelihood(*[b.pair(i)[j] for j in (0, 5, 1, 2, 3, 4)]) for i in range(b.n_pairs)])
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    out64, _ = run(B, ctx, b, B.PHMM_FP64)
    assert np.all(np.abs(out64 - ref) <= TOL64), np.abs(out64 - ref).max()
    assert np.all(np.abs(out - ref) <= TOL32 / 10), (np.abs(out - ref).max(), fl)
    assert np.all((fl & B.PHMM_FLAG_LONG) != 0)


def test_async_calls_back_to_back_bitwise(B, ctx):
    """The call only enqueues: different batches issued back to back on one stream (plan uploads of call s+1 run
    on the context's copy stream under the kernels of call s, two plan sets alternate) must give exactly what each
    batch gives alone, in both precisions, also on a side stream."""
    import torch
    batches = [W.generate(1, seed=11, n=3), W.generate(2, seed=12, n=6000), W.generate(1, seed=13, n=2),
               W.generate(3, seed=14, n=3, len_lo=1200, len_hi=2600), W.generate(0, seed=15), W.generate(2, seed=16, n=3000)]
    dbs = [B.DeviceBatch(b) for b in batches]
    for prec in (B.PHMM_FP32_RESCUE, B.PHMM_FP64):
        alone = []
        for db in dbs:
            o, f = ctx.forward_batch(db, prec)
            alone.append((o.cpu().numpy().copy(), f.cpu().numpy().copy()))
        for stream in (None, torch.cuda.Stream()):
            res = [ctx.forward_batch(db, prec, stream=stream, sync=False) for db in dbs for _ in range(2)]
            torch.cuda.synchronize()
            for i, (o, f) in enumerate(res):
                a = alone[i // 2]
                assert np.array_equal(o.cpu().numpy(), a[0]) and np.array_equal(f.cpu().numpy(), a[1]), "call %d differs" % i


def test_slices_of_reads_match_one_slice(B, ctx):
    """A batch whose row-constant table exceeds the workspace budget (phmm_options.max_table_bytes) is processed in slices
    of reads, each with its own table, plan and launches (stats.n_slices > 1): outputs and flags must be bitwise those of
    the one-slice run, through both entries and in both precisions; long pairs and rescued pairs included."""
    b = W.generate(2, n=40000)
    out1, fl1 = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert ctx.stats()["n_slices"] == 1
    n_resc = ctx.stats()["n_rescued"]
    c = B.Context(0, max_table_bytes=24 << 20)
    try:
        out2, fl2 = run(B, c, b, B.PHMM_FP32_RESCUE)
        st = c.stats()
        assert st["n_slices"] >= 5 and st["table_bytes"] <= 24 << 20
        assert np.array_equal(out1, out2) and np.array_equal(fl1, fl2)
        assert st["n_rescued"] == n_resc and st["n_pairs"] == b.n_pairs and st["cells"] == b.cells()
        oh, fh = c.forward_batch_host(b, B.PHMM_FP32_RESCUE)
        assert np.array_equal(oh, out1) and np.array_equal(fh, fl1)
        assert c.stats()["n_rescued"] == n_resc
    finally:
        c.close()


def test_host_entry_matches_device_entry(B, ctx):
    b = W.generate(1, n=3)
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    oh, fh = ctx.forward_batch_host(b, B.PHMM_FP32_RESCUE)
    assert np.array_equal(oh, out) and np.array_equal(fh, fl)
    hb = B.HostBatch(b)
    oh2, fh2 = ctx.forward_batch_host(hb, B.PHMM_FP32_RESCUE)
    assert np.array_equal(oh2, out) and np.array_equal(fh2, fl)
    assert hb.h2d_bytes() > 5 * len(b.read_bases) and hb.d2h_bytes() == 9 * b.n_pairs


def test_host_stream_two_calls_in_flight(B, ctx):
    """phmm_forward_batch_host_async / phmm_wait_host: a stream of different batches (short-read regions with rescued pairs,
    a long-read batch, a mixed one, in both precisions), two calls in flight, every result equal to the synchronous entry's
    and within tolerance of the oracle; sets are reused (5 calls on 2 sets), tickets can be waited for late, twice or never."""
    batches = [W.generate(1, n=6, seed=31), W.generate(3, n=3, seed=32), W.generate(2, n=3000, seed=33),
               W.generate(1, n=4, seed=34), W.generate(0, seed=35)]
    precs = [B.PHMM_FP32_RESCUE, B.PHMM_FP32_RESCUE, B.PHMM_FP32_RESCUE, B.PHMM_FP64, B.PHMM_FP32_RESCUE]
    want = []
    for b, pr in zip(batches, precs):
        o, f = ctx.forward_batch_host(b, pr)
        want.append((o.copy(), f.copy()))
    hbs = [B.HostBatch(b) for b in batches]
    for hb in hbs:
        hb.out.fill_(float("nan"))
    c = B.Context(0)
    try:
        tickets = []
        for i, (hb, pr) in enumerate(zip(hbs, precs)):
            tickets.append(c.forward_batch_host_async(hb, pr))
            if i >= 1 and i != 3:
                c.wait_host(tickets[i - 1])  # (ticket 2 is never waited for: the fifth call takes over its set)
        c.wait_host(tickets[-1])
        c.wait_host(tickets[0])   # long completed
        c.wait_host(tickets[-1])  # twice
        assert c.stats()["n_pairs"] == batches[-1].n_pairs
        for i, (hb, (o, f)) in enumerate(zip(hbs, want)):
            assert np.array_equal(hb.out.numpy(), o), "batch %d" % i
            assert np.array_equal(hb.flags.numpy(), f), "batch %d" % i
        ref = oracle.forward_batch(batches[4])
        assert np.all(np.abs(hbs[4].out.numpy() - ref) <= TOL32)
        assert (hbs[4].flags.numpy() & 1).sum() > 0 and (hbs[0].flags.numpy() & 1).sum() > 0
        # a bad batch is refused by the submitting call and leaves nothing in flight
        bad = B.HostBatch(batches[0])
        bad.pair_read[0] = 10 ** 6
        with pytest.raises(B.PhmmError) as ei:
            c.forward_batch_host_async(bad, B.PHMM_FP32_RESCUE)
        assert ei.value.code == B.PHMM_E_OFFSETS
        t = c.forward_batch_host_async(hbs[1], precs[1])
        c.wait_host(t)
        assert np.array_equal(hbs[1].out.numpy(), want[1][0])
    finally:
        c.close()


# ------------------------------------------------------------------ randomized batches (the fuzzer that found round 2's bugs)
def _fz_rs(rng, n): return "".join(rng.choice(list("ACGT"), n))
def _fz_make(rng, npairs, kmax, lmax):
    haps=[]; reads=[]; pr=[]; ph=[]
    nh = max(1, npairs // int(rng.integers(1, 12)))
    for h in range(nh):
        k = int(rng.integers(1, kmax)) if rng.random() < 0.9 else int(rng.choice([1,2,31,32,33,63,64,65,1023,1024,1025,2048]))
        s = list(_fz_rs(rng, k))
        if rng.random() < 0.2:
            for i in rng.choice(k, max(1, k // 40), replace=False): s[i] = 'N'
        haps.append("".join(s))
    for p in range(npairs):
        h = int(rng.integers(0, nh)); hap = haps[h]; k = len(hap)
        l = int(rng.integers(1, lmax))
        mode = rng.random()
        if mode < 0.12 and k > 200 and l > 60:  # two stretches of the haplotype, possibly far apart, in either order
            cut = int(rng.integers(20, l - 20))
            a0, b0 = int(rng.integers(0, k - 20)), int(rng.integers(0, k - 20))
            rd = list((hap[a0:a0 + cut] + _fz_rs(rng, cut))[:cut] + (hap[b0:b0 + l - cut] + _fz_rs(rng, l))[:l - cut])
        elif mode < 0.55 and k > 2:
            s0 = int(rng.integers(0, max(1, k - 1)))
            rd = list((hap[s0:s0 + l] + _fz_rs(rng, l))[:l])
            for i in rng.choice(l, max(0, l // 25), replace=False): rd[i] = "ACGTN"[int(rng.integers(0, 5))]
            if l > 20 and rng.random() < 0.3:
                c = int(rng.integers(5, l - 5)); d = int(rng.integers(1, 30)); rd = (rd[:c] + rd[c + d:] + list(_fz_rs(rng, d)))[:l]
        else:
            rd = list(_fz_rs(rng, l))
        qmode = rng.random()
        if qmode < 0.4:
            q = (rng.integers(2, 42, l), rng.integers(10, 61, l), rng.integers(10, 61, l), np.full(l, 10))
        elif qmode < 0.55:
            q = (rng.integers(2, 8, l), rng.integers(10, 61, l), rng.integers(10, 61, l), rng.integers(3, 11, l))
        elif qmode < 0.8:
            q = (rng.integers(2, 42, l), rng.integers(10, 61, l), rng.integers(10, 61, l), rng.integers(3, 41, l))
        else:
            q = (np.full(l, 30), np.full(l, 45), np.full(l, 45), np.full(l, 10))
        reads.append(("".join(rd),) + q); pr.append(len(reads) - 1); ph.append(h)
        if rng.random() < 0.3 and nh > 1:
            pr.append(len(reads) - 1); ph.append(int(rng.integers(0, nh)))
    cat = lambda i: np.concatenate([np.asarray(r[i], dtype=np.uint8) if i else np.frombuffer(r[0].encode(), dtype=np.uint8) for r in reads])
    b = W.Batch(np.concatenate([[0], np.cumsum([len(r[0]) for r in reads])]).astype(np.int64),
                np.concatenate([[0], np.cumsum([len(h) for h in haps])]).astype(np.int64),
                cat(0), cat(1), cat(2), cat(3), cat(4), np.frombuffer("".join(haps).encode(), dtype=np.uint8),
                np.asarray(pr, dtype=np.int32), np.asarray(ph, dtype=np.int32))
    return b.select_pairs(rng.permutation(b.n_pairs))


def test_randomized_batches_against_oracle(B, ctx):
    """Seeded random batches of every shape the entry points accept -- haplotypes of 1..6000 bases (tile-boundary lengths
    over-represented), reads of 1..3000, related / unrelated / with gaps, N bases, constant and per-base qualities with GCP
    between 3 and 40 -- through both precisions, one and many slices, and the host entry, element-wise against the oracle.
    For reads of 300 rows or more (100 with a GCP quality above 20) the log-space companion (oracle/logspace.py) is
    computed too and replaces the C oracle's value where they differ: the C oracle flushes cells 2^-1074 below a row's
    maximum (its documented limit), and on such reads a flushed cell can become the dominant one later.  That is decided from
    the two CPU implementations alone.
    This loop, run for minutes, found: -inf from the fp64 chain kernel for long reads against very short haplotypes at
    GCP 40 (padding lanes), and silent errors of up to 0.6 in the fp32 long kernel for GCP above 10 (now guarded)."""
    from oracle import logspace
    cs = B.Context(0, max_table_bytes=4 << 20)
    n_arb = n_long = n_fb = 0
    try:
        for it in range(24):
            rng = np.random.default_rng(7000 + it)
            kind = it % 3
            b = _fz_make(rng, [400, 60, 12][kind], [400, 1500, 6000][kind], [300, 700, 3000][kind])
            ref = oracle.forward_batch(b)
            # the C oracle keeps 1074 bits below a row's maximum (its documented limit).  A cell that far down can still matter later:
            # a read whose matching stretch runs off the haplotype's end pays a gap continuation per row from there on (3.3 bits at
            # GCP 10, 13 at GCP 40), the unrelated background about 2.5 -- after some hundred rows the background wins.  For
            # reads long enough for that the log-space companion is computed as well and takes over where the two differ
            # (decided on the CPU, before anything runs on the GPU)
            gmax = np.maximum.reduceat(b.qual_gcp, b.read_off[:-1])
            lp = b.read_len()[b.pair_read]
            for i in np.where((lp >= 300) | ((gmax[b.pair_read] > 20) & (lp >= 100)))[0]:  # (1074 bits take > 80 rows at GCP 40, > 320 at GCP 10)
                pp = b.pair(i)
                ls = logspace.log10_likelihood(pp[0], pp[5], pp[1], pp[2], pp[3], pp[4])
                if abs(ls - ref[i]) > 1e-10:
                    ref[i] = ls
                    n_arb += 1
            db = B.DeviceBatch(b)
            o64, _ = ctx.forward_batch(db, B.PHMM_FP64)
            o64 = o64.cpu().numpy()
            assert np.all(np.abs(o64 - ref) <= TOL64), "seed %d fp64: max err %g" % (7000 + it, np.nanmax(np.abs(o64 - ref)))
            for c in (ctx, cs):
                o, f = c.forward_batch(db, B.PHMM_FP32_RESCUE)
                o, f = o.cpu().numpy(), f.cpu().numpy()
                e = np.abs(o - ref)
                assert np.all(e <= TOL32), "seed %d fp32: pair %d got %r want %r flag %d" % (7000 + it, int(np.nanargmax(e)), o[int(np.nanargmax(e))], ref[int(np.nanargmax(e))], f[int(np.nanargmax(e))])
                n_long += int(((f & 2) == 2).sum()); n_fb += int(((f & 3) == 3).sum())
            oh, fh = ctx.forward_batch_host(b, B.PHMM_FP32_RESCUE)
            assert np.all(np.abs(oh - ref) <= TOL32), "seed %d host entry" % (7000 + it)
    finally:
        cs.close()
    print("randomized: %d long pairs, %d of them handed to fp64, %d arbitrations by the log-space companion" % (n_long, n_fb, n_arb))
    assert n_long > 150 and n_fb < n_long


# ------------------------------------------------------------------ edge cases
def _rand_seq(rng, n):
    return "".join(rng.choice(list("ACGT"), n))


def test_edge_lengths(B, ctx):
    """1-base reads / haplotypes, haplotype lengths at and around every tile boundary (32 columns per
    lane, 1024 per warp = short/long cut, 1024-column strips), reads longer than haplotypes."""
    rng = np.random.default_rng(21)
    pairs = []
    for k in (1, 2, 15, 16, 17, 31, 32, 33, 63, 64, 65, 255, 256, 257, 511, 512, 513, 1023, 1024, 1025, 2047, 2048, 2049, 3100):
        for l in (1, 2, 17, 130):
            hap = _rand_seq(rng, k)
            if l <= k and rng.random() < 0.7:
                s = int(rng.integers(0, k - l + 1))
                read = hap[s:s + l]
            else:
                read = _rand_seq(rng, l)
            pairs.append((read, hap, list(rng.integers(5, 41, l)), list(rng.integers(10, 50, l)),
                          list(rng.integers(10, 50, l)), 10))
    b = W.from_strings(pairs)
    check(B, ctx, b, B.PHMM_FP32_RESCUE)
    check(B, ctx, b, B.PHMM_FP64)


def test_nonuniform_gcp_and_streams(B, ctx):
    """Per-base gap-continuation qualities (reading G7) through every kernel: several reads streamed against
    one haplotype (short kernel), unrelated reads (fp64 sub-warp kernel), a haplotype > 1024 (chain kernel),
    reads around the fp64 sub-warp kernel's length limit (512)."""
    rng = np.random.default_rng(24)
    reads, haps, pr, ph = [], [], [], []
    for h, k in enumerate((40, 300, 500, 700, 1500)):
        haps.append(_rand_seq(rng, k))
        for l in (3, 60, 200, 511, 512, 513, 600):
            if l + 5 < k and rng.random() < 0.6:
                s = int(rng.integers(0, k - l))
                rd = haps[-1][s:s + l]
            else:
                rd = _rand_seq(rng, l)
            reads.append((rd, list(rng.integers(5, 41, l)), list(rng.integers(12, 50, l)), list(rng.integers(12, 50, l)),
                          list(rng.integers(5, 30, l))))
            pr.append(len(reads) - 1); ph.append(h)
    cat = lambda i: np.concatenate([np.asarray(r[i], dtype=np.uint8) if i else np.frombuffer(r[0].encode(), dtype=np.uint8)
                                    for r in reads])
    b = W.Batch(np.concatenate([[0], np.cumsum([len(r[0]) for r in reads])]).astype(np.int64),
                np.concatenate([[0], np.cumsum([len(h) for h in haps])]).astype(np.int64),
                cat(0), cat(1), cat(2), cat(3), cat(4), np.frombuffer("".join(haps).encode(), dtype=np.uint8),
                np.asarray(pr, dtype=np.int32), np.asarray(ph, dtype=np.int32))
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    check_flags(B, b, fl, ref, long_may_fall_back=True)  # (GCP above 10 on the 1500-base haplotype: the input guard sends those to fp64)
    assert np.all(fl[28:] & B.PHMM_FLAG_LONG)
    check(B, ctx, b, B.PHMM_FP64, ref=ref)


def test_read_longer_than_haplotype_and_unrelated(B, ctx):
    rng = np.random.default_rng(22)
    pairs = [(_rand_seq(rng, 300), _rand_seq(rng, 40)), (_rand_seq(rng, 250), _rand_seq(rng, 600)),
             (_rand_seq(rng, 36), _rand_seq(rng, 60)), (_rand_seq(rng, 1), _rand_seq(rng, 1200))]
    b = W.from_strings(pairs, qb=25, qi=40, qd=40)
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    check_flags(B, b, fl, ref)
    assert fl[0] & B.PHMM_FLAG_RESCUED and fl[1] & B.PHMM_FLAG_RESCUED and not (fl[2] & B.PHMM_FLAG_RESCUED)


def test_n_bases_literal_equality(B, ctx):
    """Reading G17: Eq.3 compares bytes literally, so an N matches an N and nothing else -- in the
    oracle and in every kernel.  Cases where N meets N on the alignment diagonal, N against a base, N in only one
    of the two sequences; through the short fp32 kernel, the fp64 sub-warp kernel and both chain kernels."""
    rng = np.random.default_rng(31)
    cases = [("ACGNTACG", "ACGNTACGGA"), ("ACGNTACG", "ACGTTACGGA"), ("ACGTTACG", "ACGNTACGGA"), ("ACGTTACG", "ACGTTACGGA"),
             ("NNNN", "ANNNNC"), ("N", "N"), ("N", "A"), ("A", "N")]
    for k in (70, 300, 1500):  # one lane group, several lanes, the chain path
        hap = list(_rand_seq(rng, k))
        for i in rng.choice(k, k // 10, replace=False):
            hap[i] = "N"
        hap = "".join(hap)
        for l in (40, 60):
            s = int(rng.integers(0, k - l))
            rd = list(hap[s:s + l])  # N meets N wherever the haplotype window has one
            rd[l // 2] = "N"
            for i in rng.choice(l, 3, replace=False):
                rd[i] = "ACGT"[int(rng.integers(0, 4))]
            cases.append(("".join(rd), hap))
    b = W.from_strings(cases)
    ref = oracle.forward_batch(b)
    out, _ = run(B, ctx, b, B.PHMM_FP64)
    assert np.max(np.abs(out - ref)) <= TOL64
    assert out[0] > out[1] and out[0] > out[2]  # N on N is a match, N on a base is not
    out32, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert np.max(np.abs(out32 - ref)) <= TOL32
    assert not np.any(fl[:8] & B.PHMM_FLAG_RESCUED)
    # a byte outside ACGTN is treated as N (include/pairhmm_b200.h)
    bx = W.from_strings([("ACGXTACG", "ACGNTACGGA"), ("ACGNTACG", "ACG*TACGGA")])
    ox, _ = run(B, ctx, bx, B.PHMM_FP64)
    assert abs(ox[0] - ref[0]) <= TOL64 and abs(ox[1] - ref[0]) <= TOL64


def _options_batch(rng, with_n):
    """Pairs through every kernel family: short related / unrelated (fp32 + rescue), haplotype > 1024 (long path)."""
    cases = []
    for k, l in ((60, 30), (300, 120), (700, 250), (1500, 400), (2500, 700)):
        hap = list(_rand_seq(rng, k))
        if with_n:
            for i in rng.choice(k, max(1, k // 25), replace=False):
                hap[i] = "N"
        hap = "".join(hap)
        for rel in (True, True, False):
            s0 = int(rng.integers(0, k - l))
            rd = list(hap[s0:s0 + l]) if rel else list(_rand_seq(rng, l))
            for i in rng.choice(l, max(1, l // 20), replace=False):
                rd[i] = "N" if with_n else "ACGT"[int(rng.integers(0, 4))]
            cases.append(("".join(rd), hap, list(rng.integers(2, 41, l)), list(rng.integers(12, 50, l)), list(rng.integers(12, 50, l)),
                          list(rng.integers(8, 30, l))))
    return cases


def test_option_n_is_wildcard(B):
    """phmm_options.n_is_wildcard: an N on either side matches every base -- the same switch in the oracle
    (pinned by the path enumeration, tests/test_oracle_pins.py); all kernel families, both precisions."""
    rng = np.random.default_rng(41)
    b = W.from_strings(_options_batch(rng, True))
    ref_w = oracle.forward_batch(b, n_wildcard=True)
    ref_l = oracle.forward_batch(b)
    assert np.max(ref_w - ref_l) > 1.0  # the switch matters on these inputs
    c = B.Context(0, n_is_wildcard=1)
    try:
        out, fl = run(B, c, b, B.PHMM_FP32_RESCUE)
        assert np.max(np.abs(out - ref_w)) <= TOL32
        out64, _ = run(B, c, b, B.PHMM_FP64)
        assert np.max(np.abs(out64 - ref_w)) <= TOL64
    finally:
        c.close()


def test_options_qual_offset_and_floor(B):
    """phmm_options.qual_offset (ASCII+33 qualities) and min_base_qual (a floor on the base quality): the
    library on encoded bytes == the oracle on the decoded / floored Phred values."""
    rng = np.random.default_rng(42)
    cases = _options_batch(rng, False)
    plain = W.from_strings(cases)
    floor = 10
    dec = W.from_strings([(r, h, np.maximum(np.asarray(qb), floor), qi, qd, qg) for r, h, qb, qi, qd, qg in cases])
    enc = W.from_strings([(r, h, np.asarray(qb) + 33, np.asarray(qi) + 33, np.asarray(qd) + 33, np.asarray(qg) + 33)
                          for r, h, qb, qi, qd, qg in cases])
    ref = oracle.forward_batch(dec)
    assert np.max(np.abs(ref - oracle.forward_batch(plain))) > 1e-3  # the floor matters on these inputs
    c = B.Context(0, qual_offset=33, min_base_qual=floor)
    try:
        out, fl = run(B, c, enc, B.PHMM_FP32_RESCUE)
        assert np.max(np.abs(out - ref)) <= TOL32
        out64, _ = run(B, c, enc, B.PHMM_FP64)
        assert np.max(np.abs(out64 - ref)) <= TOL64
    finally:
        c.close()


def test_pair_dump_through_the_library(B, ctx, tmp_path):
    """A pair dump in the text format of paper_2606_25738_b200/pairs_text.py (ASCII+33 qualities) through the library both
    ways -- decoded by the adaptor, or taken as it is by a context with qual_offset = 33 -- against the oracle."""
    from paper_2606_25738_b200 import pairs_text
    src = W.generate(2, n=300)
    path = str(tmp_path / "dump.txt")
    pairs_text.write_pairs(path, src)
    b = pairs_text.read_pairs(path)
    ref = oracle.forward_batch(src)
    out, fl = run(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert np.max(np.abs(out - ref)) <= TOL32
    c = B.Context(0, qual_offset=33, validate=1)
    try:
        out2, fl2 = run(B, c, pairs_text.read_pairs(path, decode=False), B.PHMM_FP32_RESCUE)
        assert np.array_equal(out2, out) and np.array_equal(fl2, fl)
    finally:
        c.close()


def test_option_validate_rejects_bad_payloads(B):
    """phmm_options.validate: a byte outside ACGTN, a quality below the offset, or iota + delta >= 1 make the call return
    PHMM_E_ARG before anything is launched: outputs untouched.  A clean batch passes and gives the usual result."""
    import torch
    rng = np.random.default_rng(43)
    good = W.from_strings(_options_batch(rng, True))
    c = B.Context(0, validate=1)
    try:
        out, fl, ref = check(B, c, good, B.PHMM_FP32_RESCUE)
        oh, fh = c.forward_batch_host(good, B.PHMM_FP32_RESCUE)
        assert np.array_equal(oh, out)
        bad_base = W.from_strings([("ACGT", "ACGTAC"), ("ACXT", "ACGTAC")])
        bad_hap = W.from_strings([("ACGT", "AC*TAC")])
        bad_gap = W.from_strings([("ACGT", "ACGTAC", 30, 2, 2, 10)])  # iota + delta = 1.26
        for bad in (bad_base, bad_hap, bad_gap):
            sentinel = torch.full((bad.n_pairs,), 7.0, dtype=torch.float64, device="cuda:0")
            with pytest.raises(B.PhmmError) as ei:
                c.forward_batch(B.DeviceBatch(bad), B.PHMM_FP32_RESCUE, out=sentinel)
            assert ei.value.code == B.PHMM_E_ARG
            torch.cuda.synchronize()
            assert torch.all(sentinel == 7.0)
            with pytest.raises(B.PhmmError) as ei:
                c.forward_batch_host(bad, B.PHMM_FP64)
            assert ei.value.code == B.PHMM_E_ARG
    finally:
        c.close()
    c2 = B.Context(0, validate=1, qual_offset=33)
    try:
        low = W.from_strings([("ACGT", "ACGTAC", 20, 45, 45, 10)])  # raw bytes below the offset of 33
        with pytest.raises(B.PhmmError) as ei:
            c2.forward_batch(B.DeviceBatch(low), B.PHMM_FP32_RESCUE)
        assert ei.value.code == B.PHMM_E_ARG
    finally:
        c2.close()


def test_few_reads_on_a_fresh_context_with_dirty_memory(B):
    """The zero run at the start of the row-constant table (what idle lanes walk before their stream starts) must be
    cleared whatever the batch size: 1-4 reads against haplotypes of more than 32 bases on a NEW context whose device
    memory was filled with 0xFF beforehand."""
    import torch
    rng = np.random.default_rng(33)
    for n_reads in (1, 2, 4):
        junk = torch.full((64 << 20,), 0xFF, dtype=torch.uint8, device="cuda:0")
        torch.cuda.synchronize()
        del junk
        torch.cuda.empty_cache()
        c = B.Context(0)
        try:
            hap = _rand_seq(rng, 700)
            pairs = []
            for _ in range(n_reads):
                s = int(rng.integers(0, 500))
                pairs.append((hap[s:s + int(rng.integers(30, 150))], hap))
            b = W.from_strings(pairs)
            b = b.select_pairs(np.arange(n_reads))
            b.pair_hap[:] = 0
            out, fl, ref = check(B, c, b, B.PHMM_FP32_RESCUE)
            assert not np.any(fl)
        finally:
            c.close()


def test_two_streams_on_one_context(B, ctx):
    """Calls issued on DIFFERENT streams of one context share its workspaces (table, counters, queues): the library
    orders them itself (each call's stream waits for the previous call's device work).  Results must be bitwise
    those of each batch alone."""
    import torch
    batches = [W.generate(1, seed=21, n=4), W.generate(2, seed=22, n=8000), W.generate(3, seed=23, n=3, len_lo=1200, len_hi=2000),
               W.generate(0, seed=24)]
    dbs = [B.DeviceBatch(b) for b in batches]
    alone = []
    for db in dbs:
        o, f = ctx.forward_batch(db, B.PHMM_FP32_RESCUE)
        alone.append((o.cpu().numpy().copy(), f.cpu().numpy().copy()))
    streams = [torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    res = []
    for rep in range(3):
        for i, db in enumerate(dbs):
            res.append((i, ctx.forward_batch(db, B.PHMM_FP32_RESCUE, stream=streams[(rep + i) % 3], sync=False)))
    torch.cuda.synchronize()
    for i, (o, f) in res:
        assert np.array_equal(o.cpu().numpy(), alone[i][0]) and np.array_equal(f.cpu().numpy(), alone[i][1]), "batch %d" % i


def test_sum_entry_column_codes(B, ctx):
    """The short kernel takes Eq.4 from the running-sum chain on a "sum entry" that selects columns by their base
    code (phmm_engine.cuh, SC): haplotypes that fill their last lane exactly (k = 32, 64, 96), that end one column
    short of it or one past it, with an N as last / first / middle column."""
    rng = np.random.default_rng(25)
    reads, haps, pairs = [], [], []
    for k in (31, 32, 33, 64, 95, 96, 97, 160):
        for variant in range(3):
            hap = list(_rand_seq(rng, k))
            if variant == 1:
                hap[-1] = "N"
            if variant == 2:
                hap[0] = "N"; hap[k // 2] = "N"
            hap = "".join(hap)
            for l in (1, 7, 30):
                s = int(rng.integers(0, k - l + 1))
                pairs.append((hap[s:s + l].replace("N", "A"), hap, list(rng.integers(8, 41, l)), list(rng.integers(20, 50, l)),
                              list(rng.integers(20, 50, l)), 10))
    b = W.from_strings(pairs)
    out, fl, ref = check(B, ctx, b, B.PHMM_FP32_RESCUE)
    assert not np.any(fl & B.PHMM_FLAG_RESCUED)  # all of these must have come out of the fp32 kernel itself
    check(B, ctx, b, B.PHMM_FP64, ref=ref)


def test_constant_quals_long_read_fp32_error(B, ctx):
    """SURVEY hard part 4: constant qualities make the fp32 rounding of the row constants systematic;
    the worst case for the 1e-3 bound.  8 kbp read with constant quals."""
    rng = np.random.default_rng(23)
    hap = _rand_seq(rng, 8400)
    read = list(hap[100:8100])
    for i in rng.choice(8000, 200, replace=False):
        read[i] = "ACGT"[("ACGT".index(read[i]) + 1) % 4]
    b = W.from_strings([("".join(read), hap)], qb=30, qi=40, qd=40)
    check(B, ctx, b, B.PHMM_FP32_RESCUE)
    check(B, ctx, b, B.PHMM_FP64)


def test_empty_batch_and_errors(B, ctx):
    import torch
    b = W.generate(0)
    e = b.select_pairs(np.zeros(0, dtype=np.int64))
    out, fl = ctx.forward_batch(B.DeviceBatch(e), B.PHMM_FP32_RESCUE)
    assert out.numel() == 0
    assert ctx.stats()["n_pairs"] == 0
    # pair index out of range -> PHMM_E_OFFSETS, output untouched
    db = B.DeviceBatch(b)
    bad = db.with_pairs(np.array([0, b.n_reads], dtype=np.int32), np.array([0, 0], dtype=np.int32))
    sentinel = torch.full((2,), 7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.PhmmError) as ei:
        ctx.forward_batch(bad, B.PHMM_FP32_RESCUE, out=sentinel)
    assert ei.value.code == B.PHMM_E_OFFSETS
    assert torch.all(sentinel == 7.0)
    # empty read -> PHMM_E_EMPTY
    z = W.from_strings([("ACGT", "ACGTAA"), ("", "ACGT")])
    with pytest.raises(B.PhmmError) as ei:
        ctx.forward_batch(B.DeviceBatch(z), B.PHMM_FP64)
    assert ei.value.code == B.PHMM_E_EMPTY
    with pytest.raises(B.PhmmError) as ei:
        ctx.forward_batch(db, 5)
    assert ei.value.code == B.PHMM_E_ARG


def test_measured_peaks_are_sane(B):
    f32, f32x2, f64 = B.measure_peak(0), B.measure_peak(1), B.measure_peak(2)
    assert 40 < f32 < 90 and 40 < f32x2 < 90 and 20 < f64 < 45
