"""ob_selftest_philox_static: the Philox self-test for callers that cannot allocate device memory.

Who that is: code that runs inside someone else's process and memory regime -- a plug-in under an application whose
pool allocator owns the whole GPU and forbids cudaMalloc behind its back, a health probe that runs before any
allocator is up, a thread that must not call cudaMalloc / cudaFree because those synchronise the device.  Such a
caller cannot hand ob_selftest_philox its dev_scratch, so this entry point stages through a fixed 224 KB array that
lives inside libob.so (OB_SELFTEST_STATIC_MAX = 4096 pairs per call).

Checked here: the result is bit-identical to the existing path (integer work: the tolerance of every Philox test in
this suite is exact equality), on TWO calls in a row, the second smaller than the first and on different inputs, so
that anything the first call left in the shared array would show; and sizes above the limit are refused with a
message, before the GPU is touched.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process (the entry point's first call does its own
per-device set-up) and after the rest of the suite."""
from __future__ import annotations

import ctypes as C

import numpy as np
import pytest

import paper_2607_06337_b200 as ob

STATIC_MAX = 4096   # OB_SELFTEST_STATIC_MAX in include/orchard.h


def _pairs(seed, n):
    rng = np.random.default_rng(seed)
    ctr = np.ascontiguousarray(rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32))
    key = np.ascontiguousarray(rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32))
    return ctr, key


def _existing_path(L, ctr, key):
    """ob_selftest_philox with scratch the caller allocated (here: through torch)."""
    import torch
    n = ctr.shape[0]
    scratch = torch.empty(56 * n, dtype=torch.uint8, device="cuda")
    a = np.zeros((n, 4), np.uint32)
    b = np.zeros((n, 4), np.uint32)
    rc = L.ob_selftest_philox(n, ctr.ctypes.data, key.ctypes.data, a.ctypes.data, b.ctypes.data,
                              C.c_void_p(scratch.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == ob.OB_OK, L.ob_last_error(None)
    return a, b


def _no_alloc_path(L, ctr, key):
    """ob_selftest_philox_static: inputs and outputs only, no scratch argument."""
    import torch
    n = ctr.shape[0]
    a = np.full((n, 4), 0xDEADBEEF, np.uint32)
    b = np.full((n, 4), 0xDEADBEEF, np.uint32)
    rc = L.ob_selftest_philox_static(n, ctr.ctypes.data, key.ctypes.data, a.ctypes.data, b.ctypes.data,
                                     C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == ob.OB_OK, L.ob_last_error(None)
    return a, b


@pytest.mark.gpu
def test_static_scratch_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    L = ob.load_library()
    torch.cuda.init()
    torch.cuda.set_device(0)
    # first call at the maximum size, second call smaller and on other inputs: it runs over the first call's leftovers
    calls = [_pairs(101, STATIC_MAX), _pairs(202, 1000)]
    got = [_no_alloc_path(L, c, k) for c, k in calls]            # two calls in a row, nothing in between
    for (ctr, key), (lib_s, cur_s) in zip(calls, got):
        lib_e, cur_e = _existing_path(L, ctr, key)
        assert np.array_equal(lib_s, lib_e)                      # bit-exact, as in tests/test_gpu_philox.py
        assert np.array_equal(cur_s, cur_e)
        assert np.array_equal(lib_s, cur_s)                      # and the self-test itself holds
    assert not np.array_equal(got[0][0][:1000], got[1][0])       # the second call did not return the first's results


def test_static_scratch_refuses_sizes_beyond_its_limit():
    """No GPU needed: the size check comes before any CUDA call."""
    L = ob.load_library()
    ctr, key = _pairs(5, 4)
    out = np.zeros((4, 4), np.uint32)
    rc = L.ob_selftest_philox_static(STATIC_MAX + 1, ctr.ctypes.data, key.ctypes.data, out.ctypes.data,
                                     out.ctypes.data, None)
    assert rc == ob.OB_E_CAPACITY
    msg = L.ob_last_error(None).decode()
    assert "OB_SELFTEST_STATIC_MAX" in msg and str(STATIC_MAX) in msg
    assert L.ob_selftest_philox_static(0, ctr.ctypes.data, key.ctypes.data, out.ctypes.data, out.ctypes.data,
                                       None) == ob.OB_E_ARG
    assert L.ob_selftest_philox_static(4, None, key.ctypes.data, out.ctypes.data, out.ctypes.data, None) == ob.OB_E_ARG
