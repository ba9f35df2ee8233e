"""Small driver for compute-sanitizer runs ("race detection"): every kernel family of the
library on tiny seeded batches, both precisions, checked against the oracle.  Not collected by pytest.

    compute-sanitizer --tool racecheck|memcheck|synccheck|initcheck python tests/sanitize_case.py

The batches: configs[0] (short kernel + fp64 rescue of 3/4 of the pairs), a mixed stream with haplotypes over
1024 bases (short + chain), config-3-shaped pairs of 1.2-2.6 kbp (2-3 strips chained through boundary blocks and
progress counters) and two 3 kbp pairs in the configs[4] shape.  The summaries are kept under profiles/.
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import oracle  # noqa: E402
from paper_2606_25738_b200 import binding as B, workloads as W  # noqa: E402


def main():
    ctx = B.Context(0)
    cases = [("configs[0]", W.generate(0)),
             ("configs[2] x 600 pairs", W.generate(2, n=600)),
             ("configs[3] shape, 3 pairs of 1.2-2.6 kbp", W.generate(3, n=3, len_lo=1200, len_hi=2600)),
             ("configs[4] shape, 2 pairs of 3 kbp", W.generate(4, n=2, len_lo=3000, len_hi=3000))]
    worst = 0.0
    for name, b in cases:
        ref = oracle.forward_batch(b)
        db = B.DeviceBatch(b)
        for prec, tol in ((B.PHMM_FP32_RESCUE, 1e-3), (B.PHMM_FP64, 1e-9)):
            out, fl = ctx.forward_batch(db, prec)
            err = float(np.max(np.abs(out.cpu().numpy() - ref)))
            st = ctx.stats()
            print("%-42s %s  pairs %5d  launches %d  rescued %4d  max|dlog10| %.2e" %
                  (name, "fp32+rescue" if prec == B.PHMM_FP32_RESCUE else "fp64       ", b.n_pairs,
                   st["n_kernel_launches"], st["n_rescued"], err), flush=True)
            assert err <= tol, (name, prec, err)
            worst = max(worst, err)
    ctx.close()
    print("sanitize_case: all results within tolerance")


if __name__ == "__main__":
    main()
