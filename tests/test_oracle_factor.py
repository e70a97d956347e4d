"""Pins for the oracle's whole Algorithm 2: invariants, planted factors, closed
forms, metamorphic relations, the paper's stated accuracy levels.  CPU only."""
import numpy as np
import pytest
import torch

from paper_2606_18411_b200 import inputs

U = 1.1e-16


def as_np(AT):
    """(n, m) C-contiguous tensor -> m x n Fortran-ordered numpy view (no copy)."""
    return AT.numpy().T


def test_n1_closed_form(orc):
    rng = np.random.default_rng(0)
    a = rng.standard_normal((512, 1))
    out = orc.factor(a, 3, 1)
    nrm = np.linalg.norm(a)
    assert out["rc"] == 0
    assert abs(out["R"][0, 0] - nrm) <= 4 * U * nrm
    assert np.max(np.abs(out["Q"] - a / nrm)) <= 4 * U


def test_planted_factors_recovered(orc):
    m, n = 2048, 12
    rng = np.random.default_rng(3)
    Q0, _ = np.linalg.qr(rng.standard_normal((m, n)))
    R0 = np.triu(rng.standard_normal((n, n)))
    R0[np.diag_indices(n)] = np.abs(np.diag(R0)) + 0.5
    A = Q0 @ R0
    out = orc.factor(A, 3 * n, 5)
    kappa = np.linalg.cond(R0)
    assert out["rc"] == 0
    assert np.linalg.norm(out["Q"] - Q0) <= 10 * kappa * n * U
    assert np.linalg.norm(out["R"] - R0) <= 10 * kappa * n * U * np.linalg.norm(R0)


@pytest.mark.parametrize("name", ["C0"])
def test_config_invariants(orc, name):
    cfg = inputs.CONFIGS[name]
    A = as_np(inputs.make_config(cfg))
    out = orc.factor(A, cfg["s"], cfg["seed_draw"], want_intermediates=True)
    assert out["rc"] == 0
    Q, R = out["Q"], out["R"]
    assert orc.orth_error_fro(Q) <= 1e-13
    assert orc.residual_fro(A, Q, R) <= 1e-13
    assert np.all(np.diag(R) > 0) and np.array_equal(np.tril(R, -1), np.zeros_like(R))
    # kappa(A Rs^-1) = O(1) w.h.p.; SURVEY probe: 5-10 at s = 2n
    Y = orc.row_solve(A, out["Rs"])
    assert np.linalg.cond(Y) < 50
    # uniqueness: numpy's Householder QR with the same sign convention
    Qn, Rn = np.linalg.qr(A)
    sg = np.sign(np.diag(Rn))
    kappa = np.linalg.cond(Rn)
    assert np.linalg.norm(Q - Qn * sg) <= 10 * kappa * cfg["n"] * U


@pytest.mark.parametrize("exponent", [2, 8, 12, 15])
def test_reduced_size_high_kappa_invariants(orc, exponent):
    # same recipe as C1..C3 at reduced m (the full sizes run in the gpu-marked parity tests)
    m, n = 1 << 13, 48
    A = as_np(inputs.make_A(m, n, exponent, 100 + exponent, 200 + exponent))
    out = orc.factor(A, 2 * n, 7, want_intermediates=True)
    assert out["rc"] == 0
    assert orc.orth_error_fro(out["Q"]) <= 2e-14
    assert orc.residual_fro(A, out["Q"], out["R"]) <= 1e-14
    assert np.linalg.cond(orc.row_solve(A, out["Rs"])) < 50


def test_paper_eq3_levels(orc):
    # eq.(3) matrices, n = 50, kappa up to 1e16; FP64 sketch gives ~5e-15 (2-norm)
    m, n = 1 << 13, 50
    for kappa in (1e2, 1e8, 1e15):
        A = as_np(inputs.make_paper_eq3(m, n, kappa, 1, 2))
        assert abs(np.log10(np.linalg.cond(A)) - np.log10(kappa)) < 0.5
        out = orc.factor(A, 3 * n, 9)                     # paper default c = 3n
        assert out["rc"] == 0
        Q = out["Q"]
        orth2 = np.linalg.norm(np.eye(n) - Q.T @ Q, 2)
        assert orth2 <= 2e-14                             # paper prints ~5e-15
        assert orc.residual_fro(A, Q, out["R"]) <= 1e-14


def test_plain_cholqr_breaks_down_where_paper_says(orc):
    # CholQR (no preconditioner) loses positive definiteness for kappa >~ 1e8.
    m, n = 1 << 12, 32
    A = as_np(inputs.make_A(m, n, 12, 1, 2))
    _, info = orc.cholesky_upper(orc.gram(A))
    Qbad = None
    if info == 0:
        Rc, _ = orc.cholesky_upper(orc.gram(A))
        Qbad = orc.row_solve(A, Rc)
    assert info != 0 or orc.orth_error_fro(Qbad) > 1e-6
    # ...while Algorithm 2 on the same matrix is fine
    out = orc.factor(A, 2 * n, 4)
    assert out["rc"] == 0 and orc.orth_error_fro(out["Q"]) <= 1e-14


def test_metamorphic_seed_s_and_scaling(orc):
    m, n = 4096, 20
    A = as_np(inputs.make_A(m, n, 5, 11, 12))
    base = orc.factor(A, 2 * n, 1)
    kappa = np.linalg.cond(base["R"])
    for s, seed in [(2 * n, 2), (3 * n, 1), (n, 3)]:
        o = orc.factor(A, s, seed)
        assert o["rc"] == 0
        assert np.linalg.norm(o["Q"] - base["Q"]) <= 10 * kappa * n * U
        assert np.linalg.norm(o["R"] - base["R"]) <= 10 * kappa * n * U * np.linalg.norm(base["R"])
    # power-of-two scaling is exact in binary floating point: R scales, Q unchanged bit for bit
    o = orc.factor(np.asfortranarray(A * 8.0), 2 * n, 1)
    assert np.array_equal(o["Q"], base["Q"]) and np.array_equal(o["R"], base["R"] * 8.0)


def test_rank_deficient_is_reported(orc):
    A = np.zeros((256, 3), order="F")
    A[:, 0] = 1.0; A[:, 1] = 2.0; A[::2, 2] = 1.0           # column 1 = 2 * column 0
    out = orc.factor(A, 6, 1)
    assert out["rc"] in (2, 3)                               # singular R_s or Cholesky breakdown, never "ok"


def test_theorem1_bound(orc):
    # kappa(A (Rs+E)^-1) <= kappa(A Rs^-1) (1 + eps k(Rs)) / (1 - eps k(Rs))
    m, n = 2048, 10
    A = as_np(inputs.make_A(m, n, 3, 21, 22))
    signs, idx = orc.draw(m, 2 * n, 6)
    Rs, _ = orc.householder_r(orc.sketch(A, signs, idx))
    Rs32, _ = orc.householder_r(orc.sketch(A, signs, idx).astype(np.float32).astype(np.float64))
    E = Rs32 - Rs
    eps = np.linalg.norm(E, 2) / np.linalg.norm(Rs, 2)
    kR = np.linalg.cond(Rs)
    assert eps * kR < 1
    k1 = np.linalg.cond(orc.row_solve(A, Rs))
    k1hat = np.linalg.cond(orc.row_solve(A, Rs32))
    assert k1hat <= k1 * (1 + eps * kR) / (1 - eps * kR) * (1 + 1e-8)


def test_inputs_generator_is_seeded_and_shaped():
    a = inputs.make_A(1024, 8, 4, 1, 2)
    b = inputs.make_A(1024, 8, 4, 1, 2)
    assert a.shape == (8, 1024) and a.dtype == torch.float64 and torch.equal(a, b)
    sv = np.linalg.svd(a.numpy(), compute_uv=False)
    assert 1e3 < sv[0] / sv[-1] < 1e5
    g = inputs.gaussian_colmajor(1 << 16, 2, 3)
    assert abs(float(g.mean())) < 0.02 and abs(float(g.std()) - 1.0) < 0.02
