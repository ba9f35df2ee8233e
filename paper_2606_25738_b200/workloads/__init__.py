"""Seeded synthetic PairHMM workloads (inputs only -- no PairHMM arithmetic lives here).

The generator itself is plain C (``gen.c``, compiled on first use with gcc); this module only
marshals its output into numpy arrays.  Both the CPU oracle tests and the CUDA path (tests,
``bench.py``, ``__graft_entry__.smoke``) draw their inputs from here so that they see the same
bytes.  Shapes follow BASELINE.json ``configs[0..4]``; the recipe is written out in DESIGN.md.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libphmm_workloads.so")
_lock = threading.Lock()
_lib = None


class _WlBatch(ctypes.Structure):
    _fields_ = [
        ("n_reads", ctypes.c_int64), ("n_haps", ctypes.c_int64), ("n_pairs", ctypes.c_int64),
        ("read_off", ctypes.POINTER(ctypes.c_int64)), ("hap_off", ctypes.POINTER(ctypes.c_int64)),
        ("read_bases", ctypes.POINTER(ctypes.c_uint8)), ("qual_base", ctypes.POINTER(ctypes.c_uint8)),
        ("qual_ins", ctypes.POINTER(ctypes.c_uint8)), ("qual_del", ctypes.POINTER(ctypes.c_uint8)),
        ("qual_gcp", ctypes.POINTER(ctypes.c_uint8)), ("hap_bases", ctypes.POINTER(ctypes.c_uint8)),
        ("pair_read", ctypes.POINTER(ctypes.c_int32)), ("pair_hap", ctypes.POINTER(ctypes.c_int32)),
    ]


class _WlParams(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int64), ("len_lo", ctypes.c_int32), ("len_hi", ctypes.c_int32)]


def build(force: bool = False) -> str:
    """Compile gen.c into libphmm_workloads.so (gcc, OpenMP).  Returns the library path."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp%d" % os.getpid()
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.wl_generate.argtypes = [ctypes.c_int, ctypes.c_uint64, ctypes.POINTER(_WlParams), ctypes.POINTER(_WlBatch)]
        lib.wl_generate.restype = ctypes.c_int
        lib.wl_free.argtypes = [ctypes.POINTER(_WlBatch)]
        lib.wl_free.restype = None
        _lib = lib
    return _lib


@dataclass
class Batch:
    """CSR batch in the layout of ``phmm_batch`` (include/pairhmm_b200.h), all host numpy arrays.

    Bases are ASCII ``ACGT``; qualities are raw Phred bytes (not ASCII+33)."""
    read_off: np.ndarray   # int64 [n_reads+1]
    hap_off: np.ndarray    # int64 [n_haps+1]
    read_bases: np.ndarray  # uint8 [read_off[-1]]
    qual_base: np.ndarray
    qual_ins: np.ndarray
    qual_del: np.ndarray
    qual_gcp: np.ndarray
    hap_bases: np.ndarray  # uint8 [hap_off[-1]]
    pair_read: np.ndarray  # int32 [n_pairs]
    pair_hap: np.ndarray   # int32 [n_pairs]

    @property
    def n_reads(self) -> int:
        return len(self.read_off) - 1

    @property
    def n_haps(self) -> int:
        return len(self.hap_off) - 1

    @property
    def n_pairs(self) -> int:
        return len(self.pair_read)

    def read_len(self) -> np.ndarray:
        return np.diff(self.read_off)

    def hap_len(self) -> np.ndarray:
        return np.diff(self.hap_off)

    def cells(self) -> int:
        """Sum over pairs of read length x haplotype length (the TCUPS numerator)."""
        rl, hl = self.read_len(), self.hap_len()
        return int(np.sum(rl[self.pair_read].astype(np.int64) * hl[self.pair_hap].astype(np.int64)))

    def select_pairs(self, idx) -> "Batch":
        """Same payload, a subset / permutation of the pair list."""
        idx = np.asarray(idx)
        return Batch(self.read_off, self.hap_off, self.read_bases, self.qual_base, self.qual_ins, self.qual_del,
                     self.qual_gcp, self.hap_bases, np.ascontiguousarray(self.pair_read[idx]),
                     np.ascontiguousarray(self.pair_hap[idx]))

    def pair(self, p: int):
        """(read, qb, qi, qd, qg, hap) byte arrays of pair p."""
        r, h = int(self.pair_read[p]), int(self.pair_hap[p])
        a, b = int(self.read_off[r]), int(self.read_off[r + 1])
        c, d = int(self.hap_off[h]), int(self.hap_off[h + 1])
        return (self.read_bases[a:b], self.qual_base[a:b], self.qual_ins[a:b], self.qual_del[a:b],
                self.qual_gcp[a:b], self.hap_bases[c:d])


def _copy(ptr, n, dtype):
    if n == 0:
        return np.zeros(0, dtype=dtype)
    return np.ctypeslib.as_array(ptr, shape=(n,)).astype(dtype, copy=True)


def generate(cfg: int, seed: int | None = None, n: int = 0, len_lo: int = 0, len_hi: int = 0) -> Batch:
    """Generate BASELINE.json ``configs[cfg]`` (cfg 0..4) or the equal-length sweep shape (cfg 5).

    ``seed`` defaults to 1 + cfg.  ``n`` scales the batch (cfg1: regions, cfg2-5: pairs; 0 = the
    full size BASELINE.json names); ``len_lo/len_hi`` override the read-length range (tests use this
    to get config-3-shaped pairs the oracle finishes in seconds)."""
    lib = _load()
    if seed is None:
        seed = 1 + cfg
    wb = _WlBatch()
    prm = _WlParams(n, len_lo, len_hi)
    rc = lib.wl_generate(cfg, seed, ctypes.byref(prm), ctypes.byref(wb))
    if rc != 0:
        raise RuntimeError("wl_generate(cfg=%d) failed rc=%d" % (cfg, rc))
    try:
        nr, nh, npairs = wb.n_reads, wb.n_haps, wb.n_pairs
        read_off = _copy(wb.read_off, nr + 1, np.int64)
        hap_off = _copy(wb.hap_off, nh + 1, np.int64)
        rb, hb = int(read_off[-1]), int(hap_off[-1])
        out = Batch(read_off, hap_off, _copy(wb.read_bases, rb, np.uint8), _copy(wb.qual_base, rb, np.uint8),
                    _copy(wb.qual_ins, rb, np.uint8), _copy(wb.qual_del, rb, np.uint8),
                    _copy(wb.qual_gcp, rb, np.uint8), _copy(wb.hap_bases, hb, np.uint8),
                    _copy(wb.pair_read, npairs, np.int32), _copy(wb.pair_hap, npairs, np.int32))
    finally:
        lib.wl_free(ctypes.byref(wb))
    return out


def from_strings(pairs, qb=30, qi=45, qd=45, qg=10) -> Batch:
    """Small hand-made batches for tests: ``pairs`` = list of (read_str, hap_str) or
    (read_str, hap_str, qb, qi, qd, qg) with per-base lists or scalars for the qualities."""
    reads, haps, quals = [], [], []
    for item in pairs:
        r, h = item[0], item[1]
        q = list(item[2:]) + [None] * (4 - len(item[2:]))
        q = [d if v is None else v for v, d in zip(q, (qb, qi, qd, qg))]
        q = [np.full(len(r), v, dtype=np.uint8) if np.isscalar(v) else np.asarray(v, dtype=np.uint8) for v in q]
        reads.append(np.frombuffer(r.encode(), dtype=np.uint8))
        haps.append(np.frombuffer(h.encode(), dtype=np.uint8))
        quals.append(q)
    read_off = np.concatenate([[0], np.cumsum([len(r) for r in reads])]).astype(np.int64)
    hap_off = np.concatenate([[0], np.cumsum([len(h) for h in haps])]).astype(np.int64)
    cat = lambda xs: np.concatenate(xs).astype(np.uint8) if xs else np.zeros(0, np.uint8)
    n = len(pairs)
    return Batch(read_off, hap_off, cat(reads), cat([q[0] for q in quals]), cat([q[1] for q in quals]),
                 cat([q[2] for q in quals]), cat([q[3] for q in quals]), cat(haps),
                 np.arange(n, dtype=np.int32), np.arange(n, dtype=np.int32))
