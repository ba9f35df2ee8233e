"""Host-side logic without a GPU: the batcher's work plan (phmm_plan_host) and the
replica aggregation bench.py uses for N > 1 (world_size-2 gloo run on CPU)."""
import os
import sys

import numpy as np
import pytest

from paper_2606_25738_b200 import binding as B
from paper_2606_25738_b200 import replicas
from paper_2606_25738_b200 import workloads as W


def _check_plan(b, plan, long_min=1024):
    rl, hl = b.read_len(), b.hap_len()
    N2 = plan["cols_per_lane"]
    k = hl[b.pair_hap]; l = rl[b.pair_read]
    is_short = (k <= long_min) & (l <= 4096) & ~((k > long_min * 7 // 8) & (l >= 768))
    # every short pair exactly once, no long pair
    assert sorted(plan["sorted_pair"].tolist()) == np.where(is_short)[0].tolist()
    wf, tk, sp = plan["warp_first"], plan["tasks"], plan["sorted_pair"]
    assert wf[0] == 0 and wf[-1] == len(tk) and np.all(np.diff(wf) >= 1)
    # tasks partition the sorted pairs into contiguous, non-overlapping runs of one haplotype each
    covered = np.zeros(len(sp), dtype=np.int32)
    for hap, first, n, rows in tk:
        assert n >= 1
        idx = sp[first:first + n]
        covered[first:first + n] += 1
        assert np.all(b.pair_hap[idx] == hap)
        assert rows == int(rl[b.pair_read[idx]].sum())
    assert np.all(covered == 1)
    # lanes of a warp: sum over its tasks of ceil(k / cols_per_lane) <= 32
    for w in range(len(wf) - 1):
        lanes = sum(-(-int(hl[t[0]]) // N2) for t in tk[wf[w]:wf[w + 1]])
        assert 1 <= lanes <= 32


def test_plan_config1_shape():
    b = W.generate(1, n=6)
    _check_plan(b, B.plan_host(b))


def test_plan_mixed_unsorted_stream_and_long_pairs_left_out():
    b = W.generate(2, n=4000)
    p = B.plan_host(b)
    _check_plan(b, p)
    assert len(p["sorted_pair"]) < b.n_pairs  # some haplotypes exceed 1024 and go to the chain path


def test_plan_many_haplotypes_shuffled_and_grouped():
    """The three ways the batcher sorts pairs by haplotype (csrc/phmm_batcher.cpp, sort_ids_by_hap): a list that is grouped
    already (copied), many more haplotypes than pairs per thread (radix sort), else per-thread histograms; and the packing of
    many equal one-pair tasks (whole warps at once, several threads, merged class by class): same invariants for all."""
    rng = np.random.default_rng(3)
    n_h, n_r = 300_000, 1000
    hap_len = rng.integers(20, 90, n_h)
    read_len = rng.integers(10, 60, n_r)
    ho = np.concatenate([[0], np.cumsum(hap_len)]).astype(np.int64)
    ro = np.concatenate([[0], np.cumsum(read_len)]).astype(np.int64)
    z = np.zeros(int(ro[-1]), dtype=np.uint8)
    pair_hap = rng.choice(n_h, 40_000, replace=False).astype(np.int32)
    pair_hap = np.concatenate([pair_hap, pair_hap[:5000]])          # some haplotypes twice
    pair_read = rng.integers(0, n_r, len(pair_hap)).astype(np.int32)
    b = W.Batch(ro, ho, z, z, z, z, z, np.zeros(int(ho[-1]), dtype=np.uint8), pair_read, pair_hap)
    p = B.plan_host(b)                                                # shuffled, 300 000 haplotypes for 45 000 pairs: radix
    _check_plan(b, p)
    order = np.argsort(pair_hap, kind="stable")
    g = b.select_pairs(order)                                         # grouped already
    pg = B.plan_host(g)
    _check_plan(g, pg)
    assert np.array_equal(order[pg["sorted_pair"]], p["sorted_pair"])  # the same stable order either way
    # equal tasks: every pair its own haplotype of 32 bases -> one class, one lane count, whole warps of 32 tasks
    n = 70_000
    e = W.Batch(np.arange(n + 1, dtype=np.int64) * 32, np.arange(n + 1, dtype=np.int64) * 32, np.zeros(n * 32, np.uint8),
                np.zeros(n * 32, np.uint8), np.zeros(n * 32, np.uint8), np.zeros(n * 32, np.uint8), np.zeros(n * 32, np.uint8),
                np.zeros(n * 32, np.uint8), np.arange(n, dtype=np.int32), np.arange(n, dtype=np.int32))
    pe = B.plan_host(e)
    _check_plan(e, pe)
    assert pe["n_warps"] <= -(-n // 32) + 16


def test_plan_custom_cut_and_small_tasks():
    b = W.generate(1, n=2)
    p = B.plan_host(b, long_min_hap_len=300, task_rows=500)
    _check_plan(b, p, long_min=300)
    assert np.all(p["tasks"][:, 3] < 500 + 260)  # a task closes once it holds >= task_rows read rows


def test_plan_empty_and_invalid():
    b = W.from_strings([("ACGT", "ACGTACGT")])
    e = b.select_pairs(np.zeros(0, dtype=np.int64))
    assert B.plan_host(e)["n_warps"] == 0
    bad = W.Batch(b.read_off, b.hap_off, b.read_bases, b.qual_base, b.qual_ins, b.qual_del, b.qual_gcp, b.hap_bases,
                  np.array([0], dtype=np.int32), np.array([3], dtype=np.int32))
    with pytest.raises(B.PhmmError):
        B.plan_host(bad)


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, cells, pairs = replicas.aggregate(10.0 + 5.0 * rank, 1e9 * (rank + 1), 100 * (rank + 1), dist)
    q.put((rank, ms, cells, pairs, replicas.rank_seed(7, rank)))
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, cells, pairs, seed in res:
        assert ms == 15.0 and cells == 3e9 and pairs == 300  # max over ranks, sums over ranks
        assert seed == 7 + rank
    assert replicas.whole_job_gcups(15.0, 3e9, 3) == pytest.approx(3e9 / 5e-3 / 1e9)


def test_replica_aggregation_single_process():
    assert replicas.aggregate(4.0, 8.0, 2.0) == (4.0, 8.0, 2.0)


def test_slices_of_reads_respect_the_table_budget():
    """phmm_plan_slices_host: the cut of a batch into slices of consecutive reads: the slices cover
    all reads in order, every slice's table (64 bytes per entry: l + 3 rounded up to even per read, 4 slots of slack) stays
    within the budget up to one read, every pair lands in the slice of its read."""
    b = W.generate(2, n=60000)
    rl = b.read_len()
    for budget, min_slices in ((8 << 20, 1), (32 << 20, 1), (4 << 30, 1), (4 << 30, 6)):
        first, cnt = B.plan_slices_host(b, budget, min_slices)
        ns = len(cnt)
        assert first[0] == 0 and first[-1] == b.n_reads and np.all(np.diff(first) >= 0)
        assert ns >= min_slices and cnt.sum() == b.n_pairs
        sl = np.searchsorted(first, b.pair_read, side="right") - 1
        assert np.array_equal(np.bincount(sl, minlength=ns), cnt)
        entries = np.add.reduceat(rl + 5, first[:-1])[:ns] if ns > 1 else np.array([np.sum(rl + 5)])  # (at most l + 5 table slots per read)
        if budget < (4 << 30):
            assert ns > 1 and np.all(entries * 64 <= budget + 64 * (rl.max() + 5))
        else:
            assert ns == max(1, min_slices)


def test_pair_dump_text_adaptor_round_trip(tmp_path):
    """paper_2606_25738_b200/pairs_text.py: write a seeded batch as a six-column pair dump with ASCII+33
    qualities, read it back: the same pairs (sequences and qualities, pair by pair), shared reads / haplotypes stored once;
    decode=False keeps the encoded bytes; malformed lines are refused."""
    from paper_2606_25738_b200 import pairs_text
    b = W.generate(1, n=1)  # 128 reads x 8 haplotypes, 1024 pairs
    path = str(tmp_path / "pairs.txt")
    pairs_text.write_pairs(path, b)
    r = pairs_text.read_pairs(path)
    assert r.n_pairs == b.n_pairs and r.n_reads <= b.n_reads and r.n_haps <= b.n_haps
    for p in (0, 1, 7, 500, b.n_pairs - 1):
        for x, y in zip(b.pair(p), r.pair(p)):
            assert np.array_equal(x, y)
    assert r.cells() == b.cells()
    e = pairs_text.read_pairs(path, decode=False)
    assert np.array_equal(e.qual_base, r.qual_base + 33) and np.array_equal(e.qual_gcp, r.qual_gcp + 33)
    with open(path, "ab") as f:
        f.write(b"# a comment\n\nACGT ACG III III III\n")
    with pytest.raises(ValueError):
        pairs_text.read_pairs(path)
