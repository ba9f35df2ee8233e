"""Thin ctypes binding over libpairhmm_b200.so (include/pairhmm_b200.h).

Argument marshalling only: every step of the PairHMM forward path runs inside the library's CUDA
kernels.  PyTorch is used for device memory and streams.  There is NO CPU fallback: if the shared
library is missing or cannot be loaded, importing a symbol from here raises.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("PHMM_LIB", os.path.join(_HERE, "libpairhmm_b200.so"))  # PHMM_LIB: try another build of the same ABI

PHMM_OK = 0
PHMM_E_ARG, PHMM_E_OFFSETS, PHMM_E_EMPTY, PHMM_E_TOOLONG = -1, -2, -3, -4
PHMM_E_CUDA, PHMM_E_NOMEM, PHMM_E_UNSUPPORTED = -5, -6, -7
PHMM_FP32_RESCUE, PHMM_FP64 = 0, 1
PHMM_FLAG_RESCUED, PHMM_FLAG_LONG, PHMM_FLAG_RANGE = 1, 2, 4

EXPORTS = ["phmm_create", "phmm_destroy", "phmm_forward_batch", "phmm_forward_batch_host",
           "phmm_forward_batch_host_async", "phmm_wait_host", "phmm_get_stats",
           "phmm_strerror", "phmm_last_cuda_error", "phmm_measure_peak", "phmm_plan_host", "phmm_plan_slices_host",
           "phmm_noalloc_setup", "phmm_noalloc_limits", "phmm_forward_batch_noalloc"]


class phmm_options(ctypes.Structure):
    _fields_ = [("size", ctypes.c_uint32), ("rescue_log2_threshold", ctypes.c_int32),
                ("long_min_hap_len", ctypes.c_int32), ("task_rows", ctypes.c_int32),
                ("max_table_bytes", ctypes.c_int64), ("profile_events", ctypes.c_int32),
                ("validate", ctypes.c_int32), ("qual_offset", ctypes.c_int32), ("min_base_qual", ctypes.c_int32),
                ("n_is_wildcard", ctypes.c_int32)]


class phmm_batch(ctypes.Structure):
    _fields_ = [("n_reads", ctypes.c_int64), ("n_haps", ctypes.c_int64), ("n_pairs", ctypes.c_int64),
                ("h_read_off", ctypes.c_void_p), ("h_hap_off", ctypes.c_void_p),
                ("d_read_bases", ctypes.c_void_p), ("d_qual_base", ctypes.c_void_p), ("d_qual_ins", ctypes.c_void_p),
                ("d_qual_del", ctypes.c_void_p), ("d_qual_gcp", ctypes.c_void_p), ("d_hap_bases", ctypes.c_void_p),
                ("h_pair_read", ctypes.c_void_p), ("h_pair_hap", ctypes.c_void_p)]


class phmm_stats(ctypes.Structure):
    _fields_ = [("n_pairs", ctypes.c_int64), ("cells", ctypes.c_int64), ("n_short_pairs", ctypes.c_int64),
                ("n_long_pairs", ctypes.c_int64), ("n_rescued", ctypes.c_int64), ("short_cells", ctypes.c_int64),
                ("short_padded_cells", ctypes.c_int64), ("n_kernel_launches", ctypes.c_int64),
                ("table_bytes", ctypes.c_int64), ("host_batch_ms", ctypes.c_double),
                ("n_short_warps", ctypes.c_int32), ("n_slices", ctypes.c_int32),
                ("ms_table", ctypes.c_double), ("ms_short", ctypes.c_double), ("ms_rescue", ctypes.c_double),
                ("ms_long", ctypes.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def build(force: bool = False) -> str:
    """Compile the library in-tree with nvcc for sm_100a (csrc/build.sh)."""
    src_dir = os.path.join(_HERE, "csrc")
    srcs = [os.path.join(src_dir, f) for f in os.listdir(src_dir)] + [os.path.join(_HERE, "..", "include", "pairhmm_b200.h")]
    stale = (not os.path.exists(LIB_PATH)) or any(os.path.getmtime(s) > os.path.getmtime(LIB_PATH) for s in srcs)
    if force or stale:
        subprocess.check_call(["sh", os.path.join(src_dir, "build.sh")])
    return LIB_PATH


_lib = None


def lib() -> ctypes.CDLL:
    """The loaded C-ABI library.  Raises (loudly) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libpairhmm_b200.so is missing: run paper_2606_25738_b200.binding.build() "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        L.phmm_create.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.POINTER(phmm_options)]
        L.phmm_create.restype = ctypes.c_int
        L.phmm_destroy.argtypes = [ctypes.c_void_p]
        L.phmm_destroy.restype = ctypes.c_int
        L.phmm_forward_batch.argtypes = [ctypes.c_void_p, ctypes.POINTER(phmm_batch), ctypes.c_int, ctypes.c_void_p,
                                         ctypes.c_void_p, ctypes.c_void_p]
        L.phmm_forward_batch.restype = ctypes.c_int
        L.phmm_forward_batch_host.argtypes = [ctypes.c_void_p, ctypes.POINTER(phmm_batch), ctypes.c_int,
                                              ctypes.c_void_p, ctypes.c_void_p]
        L.phmm_forward_batch_host.restype = ctypes.c_int
        L.phmm_forward_batch_host_async.argtypes = [ctypes.c_void_p, ctypes.POINTER(phmm_batch), ctypes.c_int,
                                                    ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(ctypes.c_int)]
        L.phmm_forward_batch_host_async.restype = ctypes.c_int
        L.phmm_wait_host.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.phmm_wait_host.restype = ctypes.c_int
        L.phmm_get_stats.argtypes = [ctypes.c_void_p, ctypes.POINTER(phmm_stats)]
        L.phmm_get_stats.restype = ctypes.c_int
        L.phmm_strerror.argtypes = [ctypes.c_int]
        L.phmm_strerror.restype = ctypes.c_char_p
        L.phmm_last_cuda_error.argtypes = [ctypes.c_void_p]
        L.phmm_last_cuda_error.restype = ctypes.c_int
        L.phmm_measure_peak.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        L.phmm_plan_host.restype = ctypes.c_int
        L.phmm_plan_host.argtypes = [ctypes.POINTER(phmm_batch), ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                     ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64]
        L.phmm_measure_peak.restype = ctypes.c_int
        L.phmm_noalloc_setup.argtypes = [ctypes.c_int]
        L.phmm_noalloc_setup.restype = ctypes.c_int
        L.phmm_noalloc_limits.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.phmm_noalloc_limits.restype = ctypes.c_int
        L.phmm_forward_batch_noalloc.argtypes = [ctypes.c_int, ctypes.POINTER(phmm_batch)] + [ctypes.c_void_p] * 7
        L.phmm_forward_batch_noalloc.restype = ctypes.c_int
        L.phmm_plan_slices_host.restype = ctypes.c_int
        L.phmm_plan_slices_host.argtypes = [ctypes.POINTER(phmm_batch), ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                            ctypes.c_void_p, ctypes.c_int64]
        _lib = L
    return _lib


class PhmmError(RuntimeError):
    def __init__(self, code: int, cuda: int = 0):
        self.code = code
        msg = lib().phmm_strerror(code).decode()
        super().__init__("phmm error %d: %s%s" % (code, msg, (" (cudaError %d)" % cuda) if cuda else ""))


def _hp(a: np.ndarray) -> int:
    return a.ctypes.data


class DeviceBatch:
    """A workloads.Batch-like object with its payload uploaded to the GPU (torch uint8 tensors) and the
    offset / pair arrays kept on the host, i.e. exactly the phmm_batch layout."""

    def __init__(self, batch, device="cuda:0"):
        import torch
        self.host = batch
        self.device = torch.device(device)
        self.read_off = np.ascontiguousarray(batch.read_off, dtype=np.int64)
        self.hap_off = np.ascontiguousarray(batch.hap_off, dtype=np.int64)
        self.pair_read = np.ascontiguousarray(batch.pair_read, dtype=np.int32)
        self.pair_hap = np.ascontiguousarray(batch.pair_hap, dtype=np.int32)
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint8)).to(self.device)
        self.t = [up(batch.read_bases), up(batch.qual_base), up(batch.qual_ins), up(batch.qual_del),
                  up(batch.qual_gcp), up(batch.hap_bases)]

    def with_pairs(self, pair_read, pair_hap) -> "DeviceBatch":
        o = object.__new__(DeviceBatch)
        o.__dict__.update(self.__dict__)
        o.pair_read = np.ascontiguousarray(pair_read, dtype=np.int32)
        o.pair_hap = np.ascontiguousarray(pair_hap, dtype=np.int32)
        return o

    @property
    def n_pairs(self):
        return len(self.pair_read)

    def c_struct(self) -> phmm_batch:
        ptr = lambda t: t.data_ptr() if t.numel() else 0
        return phmm_batch(len(self.read_off) - 1, len(self.hap_off) - 1, len(self.pair_read), _hp(self.read_off),
                          _hp(self.hap_off), ptr(self.t[0]), ptr(self.t[1]), ptr(self.t[2]), ptr(self.t[3]),
                          ptr(self.t[4]), ptr(self.t[5]), _hp(self.pair_read), _hp(self.pair_hap))


def plan_host(batch, long_min_hap_len: int = 0, task_rows: int = 0):
    """phmm_plan_host: the host batcher's work plan for a workloads.Batch-like object (no device needed).
    Returns dict(n_warps, cols_per_lane, warp_first[n_warps+1], tasks[n_tasks,4] = (hap, first sorted pair,
    n pairs, read rows), sorted_pair[n_sorted])."""
    ro = np.ascontiguousarray(batch.read_off, dtype=np.int64); ho = np.ascontiguousarray(batch.hap_off, dtype=np.int64)
    pr = np.ascontiguousarray(batch.pair_read, dtype=np.int32); ph = np.ascontiguousarray(batch.pair_hap, dtype=np.int32)
    cb = phmm_batch(len(ro) - 1, len(ho) - 1, len(pr), _hp(ro), _hp(ho), 0, 0, 0, 0, 0, 0, _hp(pr), _hp(ph))
    counts = np.zeros(4, dtype=np.int64)
    L = lib()
    rc = L.phmm_plan_host(ctypes.byref(cb), long_min_hap_len, task_rows, counts.ctypes.data, None, 0, None, 0, None, 0)
    if rc != PHMM_OK:
        raise PhmmError(rc)
    nw, nt, ns = int(counts[0]), int(counts[1]), int(counts[2])
    wf = np.zeros(nw + 1, dtype=np.int32); tk = np.zeros((max(nt, 1), 4), dtype=np.int32); sp = np.zeros(max(ns, 1), dtype=np.int32)
    rc = L.phmm_plan_host(ctypes.byref(cb), long_min_hap_len, task_rows, counts.ctypes.data, wf.ctypes.data, nw,
                          tk.ctypes.data, nt, sp.ctypes.data, ns)
    if rc != PHMM_OK:
        raise PhmmError(rc)
    return {"n_warps": nw, "cols_per_lane": int(counts[3]), "warp_first": wf, "tasks": tk[:nt], "sorted_pair": sp[:ns]}


def plan_slices_host(batch, max_table_bytes: int = 0, min_slices: int = 1):
    """phmm_plan_slices_host: (read_first[n_slices+1], pair_count[n_slices]) -- the slices of reads phmm_forward_batch would
    process the batch in (no device needed)."""
    ro = np.ascontiguousarray(batch.read_off, dtype=np.int64); ho = np.ascontiguousarray(batch.hap_off, dtype=np.int64)
    pr = np.ascontiguousarray(batch.pair_read, dtype=np.int32); ph = np.ascontiguousarray(batch.pair_hap, dtype=np.int32)
    cb = phmm_batch(len(ro) - 1, len(ho) - 1, len(pr), _hp(ro), _hp(ho), 0, 0, 0, 0, 0, 0, _hp(pr), _hp(ph))
    n = np.zeros(1, dtype=np.int64)
    L = lib()
    rc = L.phmm_plan_slices_host(ctypes.byref(cb), max_table_bytes, min_slices, n.ctypes.data, None, None, 0)
    if rc != PHMM_OK:
        raise PhmmError(rc)
    ns = int(n[0])
    first = np.zeros(ns + 1, dtype=np.int64); cnt = np.zeros(max(ns, 1), dtype=np.int64)
    rc = L.phmm_plan_slices_host(ctypes.byref(cb), max_table_bytes, min_slices, n.ctypes.data, first.ctypes.data, cnt.ctypes.data, ns)
    if rc != PHMM_OK:
        raise PhmmError(rc)
    return first, cnt[:ns]


class HostBatch:
    """The phmm_batch layout with EVERY buffer in page-locked host memory (torch pinned tensors), plus
    pinned result buffers: the argument of phmm_forward_batch_host, the end-to-end entry."""

    def __init__(self, batch):
        import torch
        pin = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).pin_memory()
        self.read_off = np.ascontiguousarray(batch.read_off, dtype=np.int64)
        self.hap_off = np.ascontiguousarray(batch.hap_off, dtype=np.int64)
        self.pair_read = np.ascontiguousarray(batch.pair_read, dtype=np.int32)
        self.pair_hap = np.ascontiguousarray(batch.pair_hap, dtype=np.int32)
        self.t = [pin(a, np.uint8) for a in (batch.read_bases, batch.qual_base, batch.qual_ins, batch.qual_del,
                                             batch.qual_gcp, batch.hap_bases)]
        n = len(self.pair_read)
        self.out = torch.empty(n, dtype=torch.float64).pin_memory()
        self.flags = torch.zeros(n, dtype=torch.uint8).pin_memory()

    def h2d_bytes(self) -> int:
        """payload bytes + offset arrays + pair lists copied host->device by one call"""
        return (sum(int(t.numel()) for t in self.t) + self.read_off.nbytes + self.hap_off.nbytes +
                self.pair_read.nbytes + self.pair_hap.nbytes)

    def d2h_bytes(self) -> int:
        return int(self.out.numel()) * 8 + int(self.flags.numel())

    def c_struct(self) -> phmm_batch:
        ptr = lambda t: t.data_ptr() if t.numel() else 0
        return phmm_batch(len(self.read_off) - 1, len(self.hap_off) - 1, len(self.pair_read), _hp(self.read_off),
                          _hp(self.hap_off), ptr(self.t[0]), ptr(self.t[1]), ptr(self.t[2]), ptr(self.t[3]),
                          ptr(self.t[4]), ptr(self.t[5]), _hp(self.pair_read), _hp(self.pair_hap))


class Context:
    """phmm_ctx wrapper."""

    def __init__(self, device: int = 0, **opts):
        self._h = ctypes.c_void_p()
        o = phmm_options()
        o.size = ctypes.sizeof(phmm_options)
        for k, v in opts.items():
            setattr(o, k, v)
        rc = lib().phmm_create(ctypes.byref(self._h), device, ctypes.byref(o))
        if rc != PHMM_OK:
            raise PhmmError(rc)
        self.device = device

    def close(self):
        if self._h:
            lib().phmm_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def forward_batch(self, db: DeviceBatch, precision: int = PHMM_FP32_RESCUE, out=None, flags=None, stream=None,
                      sync: bool = True):
        """phmm_forward_batch: returns (log10 likelihoods [float64 cuda tensor], flags [uint8 cuda tensor])."""
        import torch
        n = db.n_pairs
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=db.device)
        if flags is None:
            flags = torch.zeros(n, dtype=torch.uint8, device=db.device)
        st = torch.cuda.current_stream(db.device) if stream is None else stream
        cb = db.c_struct()
        rc = lib().phmm_forward_batch(self._h, ctypes.byref(cb), precision, out.data_ptr() if n else 0,
                                      flags.data_ptr() if n else 0, st.cuda_stream)
        if rc != PHMM_OK:
            raise PhmmError(rc, lib().phmm_last_cuda_error(self._h))
        if sync:
            st.synchronize()
        return out, flags

    def forward_batch_host(self, batch, precision: int = PHMM_FP32_RESCUE):
        """phmm_forward_batch_host: everything on the host; copies are inside the call.  ``batch`` is a
        HostBatch (pinned buffers; returns its pinned result tensors as numpy views) or any
        workloads.Batch-like object of numpy arrays (pageable)."""
        if isinstance(batch, HostBatch):
            cb = batch.c_struct()
            rc = lib().phmm_forward_batch_host(self._h, ctypes.byref(cb), precision, batch.out.data_ptr(),
                                               batch.flags.data_ptr())
            if rc != PHMM_OK:
                raise PhmmError(rc, lib().phmm_last_cuda_error(self._h))
            return batch.out.numpy(), batch.flags.numpy()
        arrs = [np.ascontiguousarray(a, dtype=np.uint8) for a in (batch.read_bases, batch.qual_base, batch.qual_ins,
                                                                  batch.qual_del, batch.qual_gcp, batch.hap_bases)]
        ro = np.ascontiguousarray(batch.read_off, dtype=np.int64)
        ho = np.ascontiguousarray(batch.hap_off, dtype=np.int64)
        pr = np.ascontiguousarray(batch.pair_read, dtype=np.int32)
        ph = np.ascontiguousarray(batch.pair_hap, dtype=np.int32)
        n = len(pr)
        out = np.empty(n, dtype=np.float64)
        flags = np.zeros(n, dtype=np.uint8)
        cb = phmm_batch(len(ro) - 1, len(ho) - 1, n, _hp(ro), _hp(ho), *[_hp(a) for a in arrs], _hp(pr), _hp(ph))
        rc = lib().phmm_forward_batch_host(self._h, ctypes.byref(cb), precision, _hp(out), _hp(flags))
        if rc != PHMM_OK:
            raise PhmmError(rc, lib().phmm_last_cuda_error(self._h))
        return out, flags

    def forward_batch_host_async(self, batch: "HostBatch", precision: int = PHMM_FP32_RESCUE) -> int:
        """phmm_forward_batch_host_async: enqueue one HostBatch (pinned buffers) and return its ticket; the results are
        in ``batch.out`` / ``batch.flags`` after ``wait_host(ticket)``.  Up to two calls in flight; the batch object must
        stay alive and untouched until then."""
        cb = batch.c_struct()
        t = ctypes.c_int(-1)
        rc = lib().phmm_forward_batch_host_async(self._h, ctypes.byref(cb), precision, batch.out.data_ptr(),
                                                 batch.flags.data_ptr(), ctypes.byref(t))
        if rc != PHMM_OK:
            raise PhmmError(rc, lib().phmm_last_cuda_error(self._h))
        return t.value

    def wait_host(self, ticket: int) -> None:
        rc = lib().phmm_wait_host(self._h, ticket)
        if rc != PHMM_OK:
            raise PhmmError(rc, lib().phmm_last_cuda_error(self._h))

    def stats(self) -> dict:
        s = phmm_stats()
        rc = lib().phmm_get_stats(self._h, ctypes.byref(s))
        if rc != PHMM_OK:
            raise PhmmError(rc)
        return s.as_dict()


def noalloc_limits():
    """phmm_noalloc_limits: (max table entries, max haplotype length, max read length) of the no-alloc entry point."""
    e = ctypes.c_int64(); k = ctypes.c_int32(); l = ctypes.c_int32()
    lib().phmm_noalloc_limits(ctypes.byref(e), ctypes.byref(k), ctypes.byref(l))
    return int(e.value), int(k.value), int(l.value)


class NoAllocBatch:
    """What phmm_forward_batch_noalloc takes besides a DeviceBatch: device copies of the offset arrays and of the pair list
    (made here, once, by torch; the entry point itself allocates nothing)."""

    def __init__(self, db: DeviceBatch):
        import torch
        self.db = db
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(db.device)
        self.d_read_off, self.d_hap_off = up(db.read_off), up(db.hap_off)
        self.d_pair_read, self.d_pair_hap = up(db.pair_read), up(db.pair_hap)


def forward_batch_noalloc(nb: NoAllocBatch, out, flags=None, stream=None, device: int = 0):
    """phmm_forward_batch_noalloc into the caller's `out` (float64 cuda tensor, n_pairs) and `flags` (uint8, optional);
    asynchronous on `stream` (default: torch's current stream)."""
    import torch
    st = torch.cuda.current_stream(nb.db.device) if stream is None else stream
    cb = nb.db.c_struct()
    ptr = lambda t: t.data_ptr() if t is not None and t.numel() else 0
    rc = lib().phmm_forward_batch_noalloc(device, ctypes.byref(cb), ptr(nb.d_read_off), ptr(nb.d_hap_off), ptr(nb.d_pair_read),
                                          ptr(nb.d_pair_hap), ptr(out), ptr(flags), st.cuda_stream)
    if rc != PHMM_OK:
        raise PhmmError(rc)
    return out, flags


def measure_peak(kind: int, device: int = 0, reps: int = 5) -> float:
    """TFLOP/s of independent FMA chains: kind 0 FFMA, 1 FFMA2, 2 DFMA."""
    v = ctypes.c_double()
    rc = lib().phmm_measure_peak(device, kind, reps, ctypes.byref(v))
    if rc != PHMM_OK:
        raise PhmmError(rc)
    return v.value
