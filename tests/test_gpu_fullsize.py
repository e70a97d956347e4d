"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(mrcqr_factor on device buffers).  C1 and C2: the oracle runs the whole factorization (seconds to
tens of seconds on the box's host cores) and every element of Q and R is compared.  C3 and the
m = 2^21 column sweep: invariants that hold at any size, computed on the device with tree
summation, plus oracle-computed sampled rows of Q where kappa makes the bound meaningful."""
import numpy as np
import pytest
import torch

from helpers import U, colmajor_to_dev, draw_to_dev, gpu_orth_error_fro, gpu_residual_fro, to_np
from paper_2606_18411_b200 import binding as B
from paper_2606_18411_b200 import inputs

pytestmark = pytest.mark.gpu
SKETCH_TOL = {16: 1e-2, 32: 1e-5, 64: 1e-12}


def check_invariants(AT, QT, R):
    n = AT.shape[0]
    assert gpu_orth_error_fro(QT) <= 1e-13
    assert gpu_residual_fro(AT, QT, R) <= 1e-13
    Rn = to_np(R)
    assert np.all(np.diag(Rn) > 0) and np.array_equal(np.tril(Rn, -1), np.zeros((n, n)))


@pytest.mark.parametrize("name", ["C1", "C2"])
def test_full_config_elementwise(orc, name):
    cfg = inputs.CONFIGS[name]
    AT = inputs.make_config(cfg, "cuda")
    A = to_np(AT)
    m, n, s, prec = cfg["m"], cfg["n"], cfg["s"], cfg["prec"]
    signs, idx = orc.draw(m, s, cfg["seed_draw"])
    o = orc.factor_from_draw(A, signs, idx, want_intermediates=True)
    assert o["rc"] == 0
    dsigns, didx = draw_to_dev(signs, idx)
    _, As = B.mrcqr_sketch(AT, prec, dsigns, didx, want_As=True)
    assert np.linalg.norm(to_np(As) - o["As"]) / np.linalg.norm(o["As"]) <= SKETCH_TOL[prec]
    QT, R = B.mrcqr_factor(AT, prec, s, cfg["seed_draw"])
    check_invariants(AT, QT, R)
    Q = to_np(QT)
    assert orc.orth_error_fro(Q) <= 1e-13                     # the oracle's own checker agrees
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(Q - o["Q"]) <= 10 * kappa * n * U
    assert np.linalg.norm(to_np(R) - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
    if B.mrcqr_last_used_store_y():                            # C2: the default stored Y; north_star's fused form as well
        B.mrcqr_set_store_y(False)
        try:
            QF, RF = B.mrcqr_factor(AT, prec, s, cfg["seed_draw"])
            assert not B.mrcqr_last_used_store_y()
        finally:
            B.mrcqr_set_store_y(None)
        check_invariants(AT, QF, RF)
        assert np.linalg.norm(to_np(QF) - o["Q"]) <= 10 * kappa * n * U
        assert np.linalg.norm(to_np(RF) - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
        del QF
    else:
        assert name == "C1"
    # kappa(A Rs^-1) = O(1) for the GPU's own reduced-precision R_s
    Rs, _ = B.mrcqr_sketch(AT, prec, dsigns, didx)
    Rc, _ = B.mrcqr_precondition_gram(AT, Rs)
    sv = np.linalg.svd(to_np(Rc), compute_uv=False)            # singular values of A Rs^-1 = those of Rc
    assert sv[0] / sv[-1] < 50


def test_config3_invariants_and_sampled_rows(orc):
    cfg = inputs.CONFIGS["C3"]
    AT = inputs.make_config(cfg, "cuda")
    m, n, s, prec = cfg["m"], cfg["n"], cfg["s"], cfg["prec"]
    QT, R = B.mrcqr_factor(AT, prec, s, cfg["seed_draw"])
    check_invariants(AT, QT, R)
    # sketch parity at full size against the oracle (FFT of 256 columns of length 2^21)
    signs, idx = orc.draw(m, s, cfg["seed_draw"])
    dsigns, didx = draw_to_dev(signs, idx)
    Rs, As = B.mrcqr_sketch(AT, prec, dsigns, didx, want_As=True)
    cols = [0, 1, 100, 255]                                    # the oracle transforms these columns
    A_cols = np.asfortranarray(to_np(AT[cols]))
    As_o = orc.sketch(A_cols, signs, idx)
    As_g = to_np(As)[:, cols]
    assert np.linalg.norm(As_g - As_o) / np.linalg.norm(As_o) <= SKETCH_TOL[prec]
    # sampled rows of Q: q = (a Rs^-1) Rc^-1 computed by the oracle's row solves from the GPU's Rs, Rc.
    # kappa ~ 1e15 makes the comparison with an independent QR vacuous; rows computed
    # from the SAME triangular factors are comparable to kappa(Rs) u per row in the A Rs^-1 step only
    # through the residual, so check the defining equations instead: q Rc Rs = a row by row.
    rows = np.array([0, 1, 12345, m // 2, m - 1])
    a = to_np(AT[:, rows].contiguous())                        # (5, n) rows of A
    q = to_np(QT[:, rows].contiguous())
    Rn = to_np(R)
    for r in range(len(rows)):
        assert np.linalg.norm(q[r] @ Rn - a[r]) <= 1e-13 * np.linalg.norm(a[r]) * n
    Rc, _ = B.mrcqr_precondition_gram(AT, Rs)
    sv = np.linalg.svd(to_np(Rc), compute_uv=False)
    assert sv[0] / sv[-1] < 50


@pytest.mark.parametrize("n", [16, 32, 64, 128, 256, 512])
@pytest.mark.parametrize("prec", [16, 32, 64])
def test_column_sweep_invariants(orc, n, prec):
    """Every (n, precision) point of BASELINE.json configs[4] (m = 2^21, s = 2n, kappa ~ 1e4): the invariants, and the
    sketch of four columns against the oracle's transform of those columns at full length."""
    cfg = inputs.sweep_config(n, prec)
    AT = inputs.make_config(cfg, "cuda")
    m, s = cfg["m"], cfg["s"]
    QT, R = B.mrcqr_factor(AT, prec, s, cfg["seed_draw"])
    check_invariants(AT, QT, R)
    del QT
    signs, idx = orc.draw(m, s, cfg["seed_draw"])
    dsigns, didx = draw_to_dev(signs, idx)
    _, As = B.mrcqr_sketch(AT, prec, dsigns, didx, want_As=True)
    cols = [0, 1, n // 2, n - 1]
    As_o = orc.sketch(np.asfortranarray(to_np(AT[cols])), signs, idx)
    assert np.linalg.norm(to_np(As)[:, cols] - As_o) / np.linalg.norm(As_o) <= SKETCH_TOL[prec]
    del AT
    torch.cuda.empty_cache()


@pytest.mark.slow
@pytest.mark.parametrize("n", [16, 32, 64, 128])
def test_column_sweep_elementwise(orc, n):
    """The FP16-sketch sweep points the oracle finishes in seconds to a minute (n <= 128 at m = 2^21, kappa ~ 1e4, where
    10 kappa n u is a meaningful bound): every element of Q and R against the oracle's factorization."""
    cfg = inputs.sweep_config(n, 16)
    AT = inputs.make_config(cfg, "cuda")
    A = to_np(AT)
    o = orc.factor(A, cfg["s"], cfg["seed_draw"])
    assert o["rc"] == 0
    QT, R = B.mrcqr_factor(AT, 16, cfg["s"], cfg["seed_draw"])
    check_invariants(AT, QT, R)
    Q = to_np(QT)
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(Q - o["Q"]) <= 10 * kappa * n * U
    assert np.linalg.norm(to_np(R) - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
    del AT, QT
    torch.cuda.empty_cache()
