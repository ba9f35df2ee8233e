"""ORACLE -- test infrastructure, not the product.

ctypes wrapper over ``pairhmm_oracle.c`` (the literal three-matrix PairHMM forward of
reference/PAPER.md Eq.1-4 in double precision with a separate power-of-two exponent), plus two
independent companions used to pin it: ``oracle.bruteforce`` (path enumeration) and
``oracle.logspace`` (a log-space row-wise implementation).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may import
this package; nothing under ``paper_2606_25738_b200/`` does.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pairhmm_oracle.c")
_LIB = os.path.join(_HERE, "libpairhmm_oracle.so")
_lock = threading.Lock()
_lib = None

_u8p = ctypes.POINTER(ctypes.c_uint8)
_i64p = ctypes.POINTER(ctypes.c_int64)
_i32p = ctypes.POINTER(ctypes.c_int32)
_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the C oracle (gcc -O2 -fopenmp; no fast-math).  Returns the library path."""
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
        lib.phmm_oracle_pair.argtypes = [_u8p, _u8p, _u8p, _u8p, _u8p, ctypes.c_int64, _u8p, ctypes.c_int64,
                                         ctypes.c_double, ctypes.c_int, _f64p, _f64p, _i32p]
        lib.phmm_oracle_pair.restype = ctypes.c_int
        lib.phmm_oracle_batch.argtypes = [ctypes.c_int64, _i32p, _i32p, _i64p, _i64p, _u8p, _u8p, _u8p, _u8p, _u8p,
                                          _u8p, ctypes.c_double, ctypes.c_int, ctypes.c_int, _f64p]
        lib.phmm_oracle_batch.restype = ctypes.c_int
        lib.phmm_oracle_num_threads.restype = ctypes.c_int
        lib.phmm_oracle_set_n_wildcard.argtypes = [ctypes.c_int]
        lib.phmm_oracle_set_n_wildcard.restype = None
        _lib = lib
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _u8(x):
    if isinstance(x, (bytes, str)):
        x = np.frombuffer(x.encode() if isinstance(x, str) else x, dtype=np.uint8)
    return np.ascontiguousarray(x, dtype=np.uint8)


def num_threads() -> int:
    return int(_load().phmm_oracle_num_threads())


def forward_pair(read, qb, qi, qd, qg, hap, log2C: float = 0.0, rescale: bool = True, matrices: bool = False,
                 n_wildcard: bool = False):
    """log10 L of one pair.  With ``matrices=True`` also returns (M, I, D, row_exp): arrays of shape
    (l+1, k+1) holding mantissas, true value = X[i] * 2**row_exp[i]."""
    lib = _load()
    read, hap = _u8(read), _u8(hap)
    l, k = len(read), len(hap)
    q = []
    for v in (qb, qi, qd, qg):
        q.append(np.full(l, v, dtype=np.uint8) if np.isscalar(v) else _u8(v))
        assert len(q[-1]) == l
    out = np.zeros(1, dtype=np.float64)
    dump = np.zeros((3, l + 1, k + 1), dtype=np.float64) if matrices else None
    dexp = np.zeros(l + 1, dtype=np.int32) if matrices else None
    lib.phmm_oracle_set_n_wildcard(int(bool(n_wildcard)))
    rc = lib.phmm_oracle_pair(_p(read, _u8p), _p(q[0], _u8p), _p(q[1], _u8p), _p(q[2], _u8p), _p(q[3], _u8p), l,
                              _p(hap, _u8p), k, float(log2C), int(bool(rescale)), _p(out, _f64p),
                              _p(dump, _f64p) if matrices else None, _p(dexp, _i32p) if matrices else None)
    if rc != 0:
        raise ValueError("phmm_oracle_pair rc=%d" % rc)
    if matrices:
        return float(out[0]), dump[0], dump[1], dump[2], dexp
    return float(out[0])


def forward_batch(batch, log2C: float = 0.0, rescale: bool = True, n_threads: int = 0, pairs=None,
                  n_wildcard: bool = False) -> np.ndarray:
    """log10 L for every pair of a workloads.Batch-like object (or for the pair indices ``pairs``)."""
    lib = _load()
    pr = np.ascontiguousarray(batch.pair_read if pairs is None else batch.pair_read[pairs], dtype=np.int32)
    ph = np.ascontiguousarray(batch.pair_hap if pairs is None else batch.pair_hap[pairs], dtype=np.int32)
    out = np.zeros(len(pr), dtype=np.float64)
    arrs = [np.ascontiguousarray(a) for a in (batch.read_off, batch.hap_off, batch.read_bases, batch.qual_base,
                                              batch.qual_ins, batch.qual_del, batch.qual_gcp, batch.hap_bases)]
    lib.phmm_oracle_set_n_wildcard(int(bool(n_wildcard)))
    rc = lib.phmm_oracle_batch(len(pr), _p(pr, _i32p), _p(ph, _i32p), _p(arrs[0], _i64p), _p(arrs[1], _i64p),
                               _p(arrs[2], _u8p), _p(arrs[3], _u8p), _p(arrs[4], _u8p), _p(arrs[5], _u8p),
                               _p(arrs[6], _u8p), _p(arrs[7], _u8p), float(log2C), int(bool(rescale)),
                               int(n_threads), _p(out, _f64p))
    if rc != 0:
        raise ValueError("phmm_oracle_batch rc=%d" % rc)
    return out
