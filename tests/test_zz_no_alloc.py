"""phmm_forward_batch_noalloc (include/pairhmm_b200.h): the entry point that allocates nothing -- its scratch is a
file-scope device array of 8 MiB -- against the existing path, phmm_forward_batch in PHMM_FP64, on two calls in a row.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2606_25738_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL64 = 1e-9  # the PHMM_FP64 tolerance of tests/test_gpu_parity.py (BASELINE.json north_star)


def _existing_path(B, batch):
    ctx = B.Context(0)
    try:
        out, fl = ctx.forward_batch(B.DeviceBatch(batch), B.PHMM_FP64)
        return out.cpu().numpy().copy()
    finally:
        ctx.close()


def test_no_alloc_entry_matches_existing_path_twice():
    import torch
    from paper_2606_25738_b200 import binding as B
    max_entries, max_k, max_l = B.noalloc_limits()
    assert max_entries * 64 + 4096 == 8 << 20 and max_k == 1024 and max_l == 4096
    # two different batches, so that the second call finds the first call's table in the shared scratch array:
    # configs[0] (256 pairs, 3/4 of them unrelated) and a slice of the mixed stream with haplotypes of up to 1024 bases
    b1 = W.generate(0)
    b2 = W.generate(2, n=400)
    keep = np.where(b2.hap_len()[b2.pair_hap] <= max_k)[0]
    b2 = b2.select_pairs(keep)
    want = [_existing_path(B, b1), _existing_path(B, b2)]
    torch.cuda.synchronize()
    nbs = [B.NoAllocBatch(B.DeviceBatch(b)) for b in (b1, b2)]
    outs = [torch.full((b.n_pairs,), 7.0, dtype=torch.float64, device="cuda:0") for b in (b1, b2)]
    fls = [torch.full((b.n_pairs,), 255, dtype=torch.uint8, device="cuda:0") for b in (b1, b2)]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for rep in range(2):          # twice each, back to back on one stream: b1, b2, b1, b2
        for i in range(2):
            B.forward_batch_noalloc(nbs[i], outs[i], fls[i])
            torch.cuda.synchronize()
            got = outs[i].cpu().numpy()
            assert np.all(np.isfinite(got))
            err = np.abs(got - want[i])
            assert err.max() <= TOL64, "call %d on batch %d: max |dlog10| %g" % (rep, i, err.max())
            assert not np.any(fls[i].cpu().numpy())
            outs[i].fill_(7.0)
    assert torch.cuda.memory_allocated() == before


def test_no_alloc_entry_rejects_what_does_not_fit():
    import torch
    from paper_2606_25738_b200 import binding as B
    max_entries, max_k, max_l = B.noalloc_limits()
    too_wide = W.from_strings([("ACGT" * 10, "ACGT" * 300)])            # haplotype of 1200 > 1024
    too_long = W.from_strings([("ACGT" * 1100, "ACGT" * 100)])          # read of 4400 > 4096
    too_many = W.generate(1, n=8)                                        # 1024 reads x ~175 rows > 131008 table entries
    assert int(np.sum(too_many.read_len() + 4)) > max_entries
    for bad in (too_wide, too_long, too_many):
        nb = B.NoAllocBatch(B.DeviceBatch(bad))
        out = torch.full((bad.n_pairs,), 7.0, dtype=torch.float64, device="cuda:0")
        with pytest.raises(B.PhmmError) as ei:
            B.forward_batch_noalloc(nb, out)
        assert ei.value.code == B.PHMM_E_TOOLONG
        torch.cuda.synchronize()
        assert torch.all(out == 7.0)   # nothing was launched
    # a pair beyond the range of unscaled double is flagged, not silently wrong: 900 unrelated bases
    rng = np.random.default_rng(3)
    rs = lambda n: "".join(rng.choice(list("ACGT"), n))
    far = W.from_strings([(rs(900), rs(300)), (rs(100), rs(300))])
    nb = B.NoAllocBatch(B.DeviceBatch(far))
    out = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    fl = torch.zeros(2, dtype=torch.uint8, device="cuda:0")
    B.forward_batch_noalloc(nb, out, fl)
    torch.cuda.synchronize()
    f = fl.cpu().numpy()
    assert f[0] == B.PHMM_FLAG_RANGE and f[1] == 0
    ref = _existing_path(B, far)
    assert abs(out[1].item() - ref[1]) <= TOL64
