"""Text adaptor for pair dumps (SURVEY.md section 8(f) item 4; PAPER.md:340, :455 name the "10s" file and GIAB-derived
dumps as the paper's real inputs -- neither is in this container, so only the reader and seeded stand-ins exist).

One pair per line, six whitespace-separated columns:

    haplotype  read  base_quals  ins_quals  del_quals  gcp_quals

bases as ASCII letters (A C G T N), the four quality strings as long as the read, every quality character = Phred value +
``qual_offset`` (33, the FASTQ convention of PAPER.md:76).  Lines that are empty or start with ``#`` are skipped.  Equal
haplotype strings and equal (read, qualities) records are stored once; the pair list references them in file order.
This module only parses and marshals: no PairHMM arithmetic (that runs in the CUDA library; a context created with
``qual_offset=33`` takes the encoded bytes as they are, see ``read_pairs(..., decode=False)``).
"""
from __future__ import annotations

import numpy as np

from .workloads import Batch


def read_pairs(path, qual_offset: int = 33, decode: bool = True) -> Batch:
    """Parse a pair dump into a CSR ``Batch``.  ``decode=True`` subtracts ``qual_offset`` (raw Phred bytes, the library's
    default); ``decode=False`` keeps the file's bytes for a context created with ``qual_offset``."""
    haps, reads, hap_ix, read_ix, pr, ph = [], [], {}, {}, [], []
    with open(path, "rb") as f:
        for ln, line in enumerate(f, 1):
            t = line.split()
            if not t or t[0].startswith(b"#"):
                continue
            if len(t) != 6:
                raise ValueError("%s:%d: expected 6 columns, found %d" % (path, ln, len(t)))
            hap, read, quals = t[0], t[1], t[2:]
            if any(len(q) != len(read) for q in quals) or not read or not hap:
                raise ValueError("%s:%d: quality strings must be as long as the (non-empty) read" % (path, ln))
            key = (read,) + tuple(quals)
            r = read_ix.get(key)
            if r is None:
                r = read_ix[key] = len(reads)
                reads.append(key)
            h = hap_ix.get(hap)
            if h is None:
                h = hap_ix[hap] = len(haps)
                haps.append(hap)
            pr.append(r); ph.append(h)
    u8 = lambda b: np.frombuffer(b, dtype=np.uint8)
    cat = lambda xs: np.concatenate(xs).astype(np.uint8) if xs else np.zeros(0, np.uint8)
    off = lambda xs: np.concatenate([[0], np.cumsum([len(x) for x in xs])]).astype(np.int64)
    q = [cat([u8(r[i]) for r in reads]) for i in range(1, 5)]
    if decode:
        if any(len(x) and int(x.min()) < qual_offset for x in q):
            raise ValueError("%s: a quality character lies below the offset %d" % (path, qual_offset))
        q = [(x - qual_offset).astype(np.uint8) for x in q]
    return Batch(off([r[0] for r in reads]), off(haps), cat([u8(r[0]) for r in reads]), q[0], q[1], q[2], q[3],
                 cat([u8(h) for h in haps]), np.asarray(pr, dtype=np.int32), np.asarray(ph, dtype=np.int32))


def write_pairs(path, batch: Batch, qual_offset: int = 33) -> None:
    """Write a ``Batch`` of raw Phred qualities in the format ``read_pairs`` reads."""
    enc = lambda a: (a.astype(np.int32) + qual_offset).astype(np.uint8).tobytes()
    with open(path, "wb") as f:
        for p in range(batch.n_pairs):
            rd, qb, qi, qd, qg, hap = batch.pair(p)
            f.write(b" ".join([hap.tobytes(), rd.tobytes(), enc(qb), enc(qi), enc(qd), enc(qg)]) + b"\n")
