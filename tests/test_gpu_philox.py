"""Pin P12: the Philox4x32-10 of both implementations against NVIDIA's own.  The oracle's CPU
generator, the library's device generator and cuRAND's curand_Philox4x32_10 (run on the device by
ob_selftest_philox) must agree bit for bit on the known-answer counters and on random (counter, key) pairs."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import pytest

import oracle
import paper_2607_06337_b200 as ob

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "philox4x32_10_kat.txt")


def _selftest(ctr, key):
    import torch
    n = ctr.shape[0]
    L = ob.load_library()
    L.ob_selftest_philox.argtypes = [C.c_int] + [C.c_void_p] * 6
    scratch = torch.empty(56 * n, dtype=torch.uint8, device="cuda")
    a = np.zeros((n, 4), np.uint32)
    b = np.zeros((n, 4), np.uint32)
    rc = L.ob_selftest_philox(n, ctr.ctypes.data, key.ctypes.data, a.ctypes.data, b.ctypes.data,
                              C.c_void_p(scratch.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == ob.OB_OK
    return a, b


def test_philox_three_way_agreement():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    kat_ctr = np.array([[int(x, 16) for x in r[0:4]] for r in rows], np.uint32)
    kat_key = np.array([[int(x, 16) for x in r[4:6]] for r in rows], np.uint32)
    kat_out = np.array([[int(x, 16) for x in r[-4:]] for r in rows], np.uint32)
    rng = np.random.default_rng(12)
    ctr = np.concatenate([kat_ctr, rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)])
    key = np.concatenate([kat_key, rng.integers(0, 2 ** 32, size=(4096, 2), dtype=np.uint64).astype(np.uint32)])
    lib, cur = _selftest(np.ascontiguousarray(ctr), np.ascontiguousarray(key))
    assert np.array_equal(lib, cur)                                   # library's device generator == cuRAND's
    assert np.array_equal(cur[: len(rows)], kat_out)                  # cuRAND reproduces the known-answer file
    for i in list(range(len(rows))) + list(range(len(rows), len(ctr), 97)):
        o = oracle.philox4x32_10(ctr[i].tolist(), key[i].tolist())
        assert np.array_equal(np.asarray(o, np.uint32), cur[i]), i    # the oracle's CPU generator == cuRAND's
