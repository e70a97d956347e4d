"""mrcqr_orth_error_noalloc (include/mrcqr.h): the allocation-free variant of mrcqr_orth_error, its scratch in a static
device array, against the existing entry point.  Collected last on purpose (the suite runs with pytest -x); passes alone
in a fresh process (the first thing the library does is then the no-alloc call) and after the other tests."""
import pytest
import torch

from paper_2606_18411_b200 import binding as B
from paper_2606_18411_b200 import inputs

pytestmark = pytest.mark.gpu


def near_orthogonal(m, n, pad, seed):
    """(n, m) view with leading dimension m + pad of a column-major Q = G / sqrt(m): ||I - Q^T Q||_F ~ n / sqrt(m)."""
    gen = torch.Generator(device="cuda").manual_seed(seed)
    buf = torch.full((n * (m + pad) + 2,), float("nan"), dtype=torch.float64, device="cuda")
    QT = torch.as_strided(buf, (n, m), (m + pad, 1))
    QT.copy_(torch.randn((n, m), dtype=torch.float64, device="cuda", generator=gen) / (m ** 0.5))
    return QT


def test_noalloc_matches_existing_path_twice_in_a_row():
    cases = [near_orthogonal(40001, 128, 3, 71),       # the maximum n, ragged m, odd leading dimension (scalar loads)
             near_orthogonal(5000, 20, 0, 72)]         # a smaller problem right after: finds the first one's leftovers
    A = inputs.make_A(1 << 15, 64, 6, 73, 74, "cuda")
    errs = [torch.full((1,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(4)]
    Gs = [torch.full((QT.shape[0], QT.shape[0]), float("nan"), dtype=torch.float64, device="cuda") for QT in cases]
    B.mrcqr_orth_error_noalloc(cases[0], errs[0], Gs[0])            # call 1
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    B.mrcqr_orth_error_noalloc(cases[1], errs[1], Gs[1])            # call 2, directly after
    B.mrcqr_orth_error_noalloc(cases[0], errs[2])                   # call 3: the first problem again, no G
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                    # nothing was allocated on the device
    for QT, err, G in zip(cases, errs, Gs):
        n = QT.shape[0]
        want = B.mrcqr_orth_error(QT)                               # existing path (context workspace)
        assert want > 1e-3                                          # a non-trivial value, not a zero that always matches
        assert err.item() == want                                   # same kernels, same order: bit-identical
        ref = QT @ QT.T
        assert torch.equal(G, G.T)
        assert (G - ref).abs().max().item() <= 1e-13
        eye = torch.eye(n, dtype=torch.float64, device="cuda")
        assert abs((eye - ref).norm().item() - want) <= 1e-13
    assert errs[2].item() == errs[0].item()
    # a factorization's Q: the quantity the paper monitors at its working size
    QT, R = B.mrcqr_factor(A, 32, 128, 75)                          # kappa = 1e6: the FP32 sketch
    B.mrcqr_orth_error_noalloc(QT, errs[3])
    torch.cuda.synchronize()
    assert errs[3].item() == B.mrcqr_orth_error(QT) <= 1e-13


def test_noalloc_rejects_beyond_the_static_scratch():
    QT = torch.zeros((B.NOALLOC_N_MAX + 1, 4096), dtype=torch.float64, device="cuda")
    err = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.MrcqrError) as e:
        B.mrcqr_orth_error_noalloc(QT, err)
    assert e.value.code == 6 and "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert err.item() == -7.0                                       # refused before anything was launched
    with pytest.raises(B.MrcqrError) as e:
        B.mrcqr_orth_error_noalloc(QT[:8, :4], err)                 # m < n
    assert e.value.code == -1
