"""mrcqr_factor_async / mrcqr_wait (include/mrcqr.h, "calls in flight"; the QR inside a loop):
the same kernels as mrcqr_factor without the per-call synchronisation.  Checked against the oracle once and, bit for
bit, against the synchronous call on every shape family; the status of the calls in flight is the first error."""
import numpy as np
import pytest
import torch

from helpers import U, colmajor_to_dev, to_np
from paper_2606_18411_b200 import binding as B
from paper_2606_18411_b200 import inputs

pytestmark = pytest.mark.gpu


def _sync_results(ATs, prec, s, seeds):
    out = []
    for AT, seed in zip(ATs, seeds):
        QT, R = B.mrcqr_factor(AT, prec, s, seed)
        out.append((QT.clone(), R.clone()))
    return out


@pytest.mark.parametrize("m,n,s,prec", [(4096, 16, 32, 32),          # C0's shape: fused form
                                        (8192, 72, 150, 16),         # Y dumped by K3 (48 <= n16 <= 112)
                                        (16384, 136, 272, 64),       # panel solves + SYRK, ragged first panel
                                        (2048, 7, 0, 64)])           # odd n, s <= 0 -> 3n, radix-4 form of K1
def test_async_calls_equal_the_synchronous_ones(orc, m, n, s, prec):
    rng = np.random.default_rng(100 + n)
    K = 5
    ATs = [colmajor_to_dev(rng.standard_normal((m, n)) @ np.diag(np.logspace(0, -3, n))) for _ in range(K)]
    seeds = [7 + 3 * k for k in range(K)]
    ref = _sync_results(ATs, prec, s, seeds)
    stream = torch.cuda.Stream()
    outs = [(torch.empty_like(AT), torch.empty((n, n), dtype=torch.float64, device="cuda")) for AT in ATs]
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        for AT, seed, (QT, R) in zip(ATs, seeds, outs):
            B.mrcqr_factor_async(AT, prec, s, seed, QT, R, stream)
        assert B.mrcqr_wait() == (0, 0)
    for (QT, R), (Qs, Rs_) in zip(outs, ref):
        assert torch.equal(QT, Qs) and torch.equal(R, Rs_)
    # ... and the oracle once (the synchronous call is compared with it everywhere else)
    A = to_np(ATs[0])
    o = orc.factor(A, s if s > 0 else 3 * n, seeds[0])
    assert o["rc"] == 0
    kappa = np.linalg.cond(A)
    assert np.linalg.norm(to_np(outs[0][0]) - o["Q"]) <= 10 * kappa * n * U
    assert np.linalg.norm(to_np(outs[0][1]) - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
    assert B.mrcqr_wait() == (0, 0)                       # nothing pending: returns at once


def test_async_status_is_the_first_error_and_later_calls_still_run():
    rng = np.random.default_rng(5)
    m, n, s = 4096, 8, 16
    good = [colmajor_to_dev(rng.standard_normal((m, n))) for _ in range(3)]
    bad5 = np.asfortranarray(rng.standard_normal((m, n))); bad5[:, 5] = 0.0      # R_s[5, 5] = 0: code 2, column 5
    bad2 = np.asfortranarray(rng.standard_normal((m, n))); bad2[:, 2] = 0.0
    ATs = [good[0], colmajor_to_dev(bad5), good[1], colmajor_to_dev(bad2), good[2]]
    ref = _sync_results([good[0], good[1], good[2]], 64, s, [1, 3, 5])
    outs = [(torch.empty_like(AT), torch.empty((n, n), dtype=torch.float64, device="cuda")) for AT in ATs]
    for k, (AT, (QT, R)) in enumerate(zip(ATs, outs)):
        B.mrcqr_factor_async(AT, 64, s, 1 + k, QT, R)
    assert B.mrcqr_wait(check=False) == (2, 5)            # the FIRST error, with its column
    assert B.mrcqr_last_info() == 5
    for i, k in enumerate((0, 2, 4)):                     # the clean calls around the failing ones are complete
        assert torch.equal(outs[k][0], ref[i][0]) and torch.equal(outs[k][1], ref[i][1])
    assert B.mrcqr_wait(check=False) == (0, 0)            # cleared
    B.mrcqr_factor_async(good[0], 64, s, 1, *outs[0])
    assert B.mrcqr_wait() == (0, 0)
    with pytest.raises(B.MrcqrError) as e:                # argument errors come back at once
        B.mrcqr_factor_async(good[0], 64, m, 1, *outs[0])
    assert e.value.code == -8


def test_async_more_calls_than_ring_slots_and_a_change_of_stream():
    rng = np.random.default_rng(6)
    m, n, s = 4096, 16, 40
    AT = colmajor_to_dev(rng.standard_normal((m, n)))
    K = 21                                                # the ring of pinned bin buffers has 8 slots
    ref = _sync_results([AT] * K, 32, s, list(range(50, 50 + K)))
    outs = [(torch.empty_like(AT), torch.empty((n, n), dtype=torch.float64, device="cuda")) for _ in range(K)]
    for k in range(K):
        B.mrcqr_factor_async(AT, 32, s, 50 + k, *outs[k])
    assert B.mrcqr_wait() == (0, 0)
    for k in range(K):
        assert torch.equal(outs[k][0], ref[k][0]) and torch.equal(outs[k][1], ref[k][1])
    # a failing call on one stream, a clean one on another: the first is drained, its status carried over
    bad = np.asfortranarray(rng.standard_normal((m, n))); bad[:, 9] = 0.0
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    B.mrcqr_factor_async(colmajor_to_dev(bad), 32, s, 1, *outs[0], stream=s1)
    B.mrcqr_factor_async(AT, 32, s, 50, *outs[1], stream=s2)
    assert B.mrcqr_wait(check=False) == (2, 9)
    assert torch.equal(outs[1][0], ref[0][0])
    # a larger shape while calls are pending (the workspace grows): drained first, results intact
    big = colmajor_to_dev(rng.standard_normal((1 << 15, 40)))
    Qb, Rb = B.mrcqr_factor(big, 64, 80, 3)
    Qb, Rb = Qb.clone(), Rb.clone()
    B.mrcqr_shutdown()                                    # back to no workspace at all
    B.mrcqr_factor_async(AT, 32, s, 51, *outs[2])
    Qa, Ra = torch.empty_like(big), torch.empty((40, 40), dtype=torch.float64, device="cuda")
    B.mrcqr_factor_async(big, 64, 80, 3, Qa, Ra)
    assert B.mrcqr_wait() == (0, 0)
    assert torch.equal(outs[2][0], ref[1][0]) and torch.equal(Qa, Qb) and torch.equal(Ra, Rb)


def test_async_honours_the_switches_of_the_context():
    # the Re+Im sketch (draw kernel + radix-4 K1) and the forced forms of stage 2 take the same path in flight
    rng = np.random.default_rng(8)
    m, n, s = 16384, 48, 96
    AT = colmajor_to_dev(rng.standard_normal((m, n)))
    outs = [(torch.empty_like(AT), torch.empty((n, n), dtype=torch.float64, device="cuda")) for _ in range(3)]
    try:
        for reim, store in ((True, None), (False, False), (False, True)):
            B.mrcqr_set_sketch_reim(reim)
            B.mrcqr_set_store_y(store)
            Qs, Rs_ = B.mrcqr_factor(AT, 32, s, 11)
            Qs, Rs_ = Qs.clone(), Rs_.clone()
            for k in range(3):
                B.mrcqr_factor_async(AT, 32, s, 11, *outs[k])
            assert B.mrcqr_wait() == (0, 0)
            for k in range(3):
                assert torch.equal(outs[k][0], Qs) and torch.equal(outs[k][1], Rs_)
    finally:
        B.mrcqr_set_sketch_reim(False)
        B.mrcqr_set_store_y(None)
