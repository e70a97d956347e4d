"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol the
header declares, rejects bad arguments LAPACK-style, its host draw equals the oracle's, and its
compute entry points fail loudly (code 4) when there is no device -- there is no CPU fallback."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

from paper_2606_18411_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    txt = open(os.path.join(ROOT, "include", "mrcqr.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(mrcqr_[a-z_0-9]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    L = B.lib()
    syms = header_symbols()
    assert set(syms) == set(B.EXPORTS)
    for name in syms:
        assert getattr(L, name) is not None


def test_host_draw_equals_oracle(orc):
    for m, s, seed in [(4096, 32, 2), (1 << 20, 128, 12), (64, 33, 5), (100, 7, 1)]:
        signs, idx = B.mrcqr_draw(m, s, seed)
        osigns, oidx = orc.draw(m, s, seed)
        assert np.array_equal(signs.numpy().view(np.uint64), osigns)
        assert np.array_equal(idx.numpy(), oidx)


def test_draw_argument_errors():
    L = B.lib()
    buf = (C.c_uint64 * 4)()
    ibuf = (C.c_int64 * 4)()
    assert L.mrcqr_draw(0, 1, 0, buf, ibuf) == -1
    assert L.mrcqr_draw(64, 34, 0, buf, ibuf) == -2
    assert L.mrcqr_draw(64, 2, 0, None, ibuf) == -4
    assert L.mrcqr_draw(64, 2, 0, buf, None) == -5


def test_argument_errors_before_any_device_work():
    L = B.lib()
    p = C.c_void_p(16)            # never dereferenced: argument checks come first
    # mrcqr_factor: -1 m, -2 n, -3 lda, -4 A, -5 Q, -6 R, -7 prec, -8 s
    assert L.mrcqr_factor(1000, 8, 1000, p, p, p, 32, 16, 0, None) == -1       # not a power of two
    assert L.mrcqr_factor(64, 128, 64, p, p, p, 32, 16, 0, None) == -1         # m < n
    assert L.mrcqr_factor(1024, 0, 1024, p, p, p, 32, 16, 0, None) == -2
    assert L.mrcqr_factor(1024, 513, 1024, p, p, p, 32, 16, 0, None) == -2
    assert L.mrcqr_factor(1024, 8, 1000, p, p, p, 32, 16, 0, None) == -3
    assert L.mrcqr_factor(1024, 8, 1024, None, p, p, 32, 16, 0, None) == -4
    assert L.mrcqr_factor(1024, 8, 1024, p, None, p, 32, 16, 0, None) == -5
    assert L.mrcqr_factor(1024, 8, 1024, p, p, None, 32, 16, 0, None) == -6
    assert L.mrcqr_factor(1024, 8, 1024, p, p, p, 8, 16, 0, None) == -7
    assert L.mrcqr_factor(1024, 8, 1024, p, p, p, 32, 4, 0, None) == -8        # s < n
    assert L.mrcqr_factor(1024, 8, 1024, p, p, p, 32, 600, 0, None) == -8      # s > m/2+1
    assert L.mrcqr_precondition_gram(4, 8, 4, p, p, None, p, None) == -1
    assert L.mrcqr_precondition_gram(64, 8, 32, p, p, None, p, None) == -3
    assert L.mrcqr_form_q(64, 8, 64, p, p, p, 32, p, p, None) == -7
    assert L.mrcqr_sketch(1024, 8, 1024, p, 32, 16, None, p, None, p, None) == -7


def test_batched_argument_errors():
    L = B.lib()
    p = C.c_void_p(16)            # never dereferenced
    assert L.mrcqr_factor_batched(0, 1024, 8, 1024, 8192, p, 8192, p, p, 32, 16, 0, None, None) == -1
    assert L.mrcqr_factor_batched(2, 1000, 8, 1000, 8000, p, 8000, p, p, 32, 16, 0, None, None) == -2
    assert L.mrcqr_factor_batched(2, 1024, 0, 1024, 8192, p, 8192, p, p, 32, 16, 0, None, None) == -3
    assert L.mrcqr_factor_batched(2, 1024, 8, 1000, 8192, p, 8192, p, p, 32, 16, 0, None, None) == -4
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 100, p, 8192, p, p, 32, 16, 0, None, None) == -5
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 8192, None, 8192, p, p, 32, 16, 0, None, None) == -6
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 8192, p, 100, p, p, 32, 16, 0, None, None) == -7
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 8192, p, 8192, None, p, 32, 16, 0, None, None) == -8
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 8192, p, 8192, p, None, 32, 16, 0, None, None) == -9
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 8192, p, 8192, p, p, 8, 16, 0, None, None) == -10
    assert L.mrcqr_factor_batched(2, 1024, 8, 1024, 8192, p, 8192, p, p, 32, 4, 0, None, None) == -11


def test_async_argument_errors():
    # mrcqr_factor_async checks its arguments like mrcqr_factor and reports them at once (include/mrcqr.h)
    L = B.lib()
    p = C.c_void_p(16)            # never dereferenced
    assert L.mrcqr_factor_async(1000, 8, 1000, p, p, p, 32, 16, 0, None) == -1
    assert L.mrcqr_factor_async(1024, 0, 1024, p, p, p, 32, 16, 0, None) == -2
    assert L.mrcqr_factor_async(1024, 8, 1000, p, p, p, 32, 16, 0, None) == -3
    assert L.mrcqr_factor_async(1024, 8, 1024, None, p, p, 32, 16, 0, None) == -4
    assert L.mrcqr_factor_async(1024, 8, 1024, p, None, p, 32, 16, 0, None) == -5
    assert L.mrcqr_factor_async(1024, 8, 1024, p, p, None, 32, 16, 0, None) == -6
    assert L.mrcqr_factor_async(1024, 8, 1024, p, p, p, 8, 16, 0, None) == -7
    assert L.mrcqr_factor_async(1024, 8, 1024, p, p, p, 32, 4, 0, None) == -8
    if not torch.cuda.is_available():
        assert L.mrcqr_factor_async(1024, 8, 1024, p, p, p, 32, 16, 0, None) == 4     # no device: no fallback
        assert L.mrcqr_wait(None) == 4


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_cpu_fallback_without_device():
    L = B.lib()
    a = np.zeros((1024, 8), order="F")
    q = np.zeros((1024, 8), order="F")
    r = np.zeros((8, 8), order="F")
    rc = L.mrcqr_factor_host(1024, 8, 1024, a.ctypes.data, q.ctypes.data, r.ctypes.data, 32, 16, 0)
    assert rc == 4                      # MRCQR_ERR_CUDA: the product path needs the GPU
    assert B.mrcqr_workspace_bytes(1024, 8, 16, 32) == 0
