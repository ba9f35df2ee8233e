"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol that
include/pairhmm_b200.h declares; the ctypes structs of the binding have the C layout; calls that need
no device return the documented error codes.  CPU only (no compute calls)."""
import ctypes
import os
import re
import subprocess
import tempfile

import pytest

from paper_2606_25738_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "pairhmm_b200.h")


@pytest.fixture(scope="module")
def lib():
    binding.build()
    return binding.lib()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(phmm_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 8
    for n in names:
        assert hasattr(lib, n), "libpairhmm_b200.so does not export %s" % n
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and the header disagree"


def test_struct_layouts_match_the_header():
    """Compile a tiny C program against the header and compare sizeof/offsetof with ctypes."""
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "pairhmm_b200.h"
int main(void) {
  printf("%zu %zu %zu\n", sizeof(phmm_options), sizeof(phmm_batch), sizeof(phmm_stats));
  printf("%zu %zu %zu\n", offsetof(phmm_options, max_table_bytes), offsetof(phmm_batch, h_pair_hap), offsetof(phmm_stats, ms_long));
  printf("%d %d %d %d\n", PHMM_E_UNSUPPORTED, PHMM_FP64, PHMM_FLAG_LONG, PHMM_VERSION);
  return 0;
}'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "t.c")
        open(c, "w").write(prog)
        exe = os.path.join(d, "t")
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", exe, c])
        out = subprocess.check_output([exe], text=True).split()
    got = list(map(int, out))
    want = [ctypes.sizeof(binding.phmm_options), ctypes.sizeof(binding.phmm_batch), ctypes.sizeof(binding.phmm_stats),
            binding.phmm_options.max_table_bytes.offset, binding.phmm_batch.h_pair_hap.offset,
            binding.phmm_stats.ms_long.offset, binding.PHMM_E_UNSUPPORTED, binding.PHMM_FP64, binding.PHMM_FLAG_LONG, 1]
    assert got == want


def test_strerror_and_null_arguments(lib):
    assert lib.phmm_strerror(0) == b"ok"
    for code in range(-7, 0):
        assert lib.phmm_strerror(code) not in (b"ok", b"unknown error")
    assert lib.phmm_strerror(-99) == b"unknown error"
    assert lib.phmm_create(None, 0, None) == binding.PHMM_E_ARG
    assert lib.phmm_destroy(None) == binding.PHMM_E_ARG
    assert lib.phmm_forward_batch(None, None, 0, None, None, None) == binding.PHMM_E_ARG
    assert lib.phmm_forward_batch_host(None, None, 0, None, None) == binding.PHMM_E_ARG
    assert lib.phmm_get_stats(None, None) == binding.PHMM_E_ARG
    assert lib.phmm_last_cuda_error(None) == 0
    assert lib.phmm_measure_peak(0, 7, 1, None) == binding.PHMM_E_ARG


def test_create_fails_cleanly_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    h = ctypes.c_void_p()
    rc = lib.phmm_create(ctypes.byref(h), 0, None)
    assert rc in (binding.PHMM_E_CUDA, binding.PHMM_E_UNSUPPORTED) and not h.value
    with pytest.raises(binding.PhmmError):
        binding.Context(0)


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", os.path.join(ROOT, "does_not_exist.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lib()
