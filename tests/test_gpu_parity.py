"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs,
element by element, at sizes the oracle finishes in seconds.  Tolerances are north_star's:
sketch rel. Frobenius error <= 1e-2 / 1e-5 / 1e-12 (fp16 / fp32 / fp64); ||I-Q^TQ||_F <= 1e-13;
||A-QR||_F/||A||_F <= 1e-13; ||Q-Q_oracle||_F <= 10 kappa(A) n 1.1e-16."""
import numpy as np
import pytest
import torch

from helpers import U, colmajor_to_dev, draw_to_dev, to_np
from paper_2606_18411_b200 import binding as B
from paper_2606_18411_b200 import inputs

pytestmark = pytest.mark.gpu

SKETCH_TOL = {16: 1e-2, 32: 1e-5, 64: 1e-12}


def relf(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def stage_parity(orc, AT, s, seed, prec):
    """Runs every stage of the C ABI against the matching oracle step.  Returns the oracle dict."""
    A = to_np(AT)
    m, n = A.shape
    signs, idx = orc.draw(m, s, seed)
    o = orc.factor_from_draw(A, signs, idx, want_intermediates=True)
    assert o["rc"] == 0
    dsigns, didx = draw_to_dev(signs, idx)
    # stage 1: sketch (o2-o4) and R_s (o5)
    Rs, As = B.mrcqr_sketch(AT, prec, dsigns, didx, want_As=True)
    assert relf(to_np(As), o["As"]) <= SKETCH_TOL[prec]
    Rs_np = to_np(Rs)
    assert np.all(np.diag(Rs_np) > 0) and np.array_equal(np.tril(Rs_np, -1), np.zeros((n, n)))
    # R_s is the R-factor of the GPU's own precision-p sketch: R_s^T R_s = As^T As
    Asg = to_np(As)
    assert np.linalg.norm(Rs_np.T @ Rs_np - Asg.T @ Asg) <= 100 * n * U * np.linalg.norm(Asg) ** 2
    # stage 2a from the ORACLE's R_s, so that G and R_c are comparable element by element
    RsO = colmajor_to_dev(o["Rs"])
    Rc, G = B.mrcqr_precondition_gram(AT, RsO, want_G=True)
    kY = np.linalg.cond(o["Rs"])
    assert relf(to_np(G), o["G"]) <= 1e-15 * max(1.0, kY) * n
    assert np.array_equal(to_np(G), to_np(G).T)
    Rc_np = to_np(Rc)
    assert np.all(np.diag(Rc_np) > 0) and np.array_equal(np.tril(Rc_np, -1), np.zeros((n, n)))
    assert relf(Rc_np, o["Rc"]) <= 1e-15 * max(1.0, kY) * n * 10
    # stage 2b + 3 from the oracle's R_s, R_c
    RcO = colmajor_to_dev(o["Rc"])
    QT, R = B.mrcqr_form_q(AT, RsO, RcO)
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(to_np(QT) - o["Q"]) <= 10 * kappa * n * U
    assert relf(to_np(R), o["R"]) <= 10 * n * U
    assert np.array_equal(np.tril(to_np(R), -1), np.zeros((n, n)))
    return o


def factor_parity(orc, AT, s, seed, prec, o=None, q_compare=True):
    A = to_np(AT)
    m, n = A.shape
    if o is None:
        o = orc.factor(A, s, seed)
        assert o["rc"] == 0
    QT, R = B.mrcqr_factor(AT, prec, s, seed)
    Q, Rn = to_np(QT), to_np(R)
    assert orc.orth_error_fro(Q) <= 1e-13
    assert orc.residual_fro(A, Q, Rn) <= 1e-13
    assert np.all(np.diag(Rn) > 0) and np.array_equal(np.tril(Rn, -1), np.zeros((n, n)))
    kappa = np.linalg.cond(o["R"])
    if q_compare:
        assert np.linalg.norm(Q - o["Q"]) <= 10 * kappa * n * U
        assert np.linalg.norm(Rn - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
    return QT, R


def test_config0_all_stages(orc):
    cfg = inputs.CONFIGS["C0"]
    AT = inputs.make_config(cfg, "cuda")
    o = stage_parity(orc, AT, cfg["s"], cfg["seed_draw"], cfg["prec"])
    factor_parity(orc, AT, cfg["s"], cfg["seed_draw"], cfg["prec"], o)


@pytest.mark.parametrize("m,n,s,prec,expo", [
    (1 << 12, 1, 3, 64, 0),        # n = 1 closed form below
    (1 << 12, 5, 15, 32, 2),       # n < 8: padding columns
    (1 << 13, 20, 60, 64, 6),      # paper's n = 20, default c = 3n
    (1 << 13, 50, 150, 32, 5),     # paper's n = 50, not a multiple of 16
    (1 << 14, 72, 144, 16, 3),     # second tile geometry (n16 = 80), odd column pair count no
    (1 << 13, 129, 258, 64, 10),   # third tile geometry, ragged n, odd n (last FFT pair half empty)
    (1 << 12, 272, 544, 32, 4),    # fourth tile geometry (n16 > 256)
    (64, 16, 32, 64, 1),           # smallest m: single FFT tile, m1 = 2
    (32, 4, 17, 32, 1),            # m = 32, s = m/2 + 1 (every bin)
])
def test_small_shapes_all_stages(orc, m, n, s, prec, expo):
    AT = inputs.make_A(m, n, expo, 7 * n + 1, 7 * n + 2, "cuda")
    o = stage_parity(orc, AT, s, 1000 + n, prec)
    factor_parity(orc, AT, s, 1000 + n, prec, o)
    if n == 1:
        a = to_np(AT)
        QT, R = B.mrcqr_factor(AT, prec, s, 5)
        assert abs(float(R[0, 0]) - np.linalg.norm(a)) <= 8 * U * np.linalg.norm(a)
        assert np.max(np.abs(to_np(QT) - a / np.linalg.norm(a))) <= 8 * U


@pytest.mark.parametrize("prec", [16, 32, 64])
def test_three_precisions_same_factorization(orc, prec):
    # kappa ~ 1e3 is inside every precision's range: same (Q, R) to kappa*u
    m, n = 1 << 14, 32
    AT = inputs.make_A(m, n, 3, 51, 52, "cuda")
    factor_parity(orc, AT, 2 * n, 9, prec)


@pytest.mark.parametrize("m", [1000, 4097, 129, 128])
def test_stage2_ragged_rows(orc, m):
    # stages 2a/2b accept any m >= n: ragged last tile, rows not a multiple of anything
    n = 24
    rng = np.random.default_rng(m)
    A = np.asfortranarray(rng.standard_normal((m, n)))
    Rs = np.triu(rng.standard_normal((n, n))) + 5 * np.eye(n)
    AT, RsT = colmajor_to_dev(A), colmajor_to_dev(Rs)
    Rc, G = B.mrcqr_precondition_gram(AT, RsT, want_G=True)
    Y = orc.row_solve(A, Rs)
    Go = orc.gram(Y)
    assert relf(to_np(G), Go) <= 1e-13
    Rco, info = orc.cholesky_upper(Go)
    assert info == 0 and relf(to_np(Rc), Rco) <= 1e-12
    QT, R = B.mrcqr_form_q(AT, RsT, colmajor_to_dev(Rco))
    Qo = orc.row_solve(Y, Rco)
    assert np.linalg.norm(to_np(QT) - Qo) <= 1e-12
    assert relf(to_np(R), orc.triu_mul(Rco, Rs)) <= 1e-14


@pytest.mark.parametrize("m,n", [((1 << 22) + 100, 16), ((1 << 22) + 100, 24), ((1 << 21) + 100, 40), (5000, 40)])
def test_warp_private_gram_flushes_mid_run(orc, m, n):
    # K3 at n16 <= 48 keeps one Gram accumulator set per warp and sums the four sets of a CTA (fixed order) every
    # 32 tiles and at the end.  The large m values give every CTA more than 32 tiles, so that the first flush
    # (plain store) AND the later ones (ordered adds) run; 5000 rows: a single flush, ragged last tile, n16 = 48.
    AT = inputs.gaussian_colmajor(m, n, 900 + n, "cuda")
    A = to_np(AT)
    rng = np.random.default_rng(n)
    Rs = np.triu(rng.standard_normal((n, n))) + 6 * np.eye(n)
    Rc, G = B.mrcqr_precondition_gram(AT, colmajor_to_dev(Rs), want_G=True)
    Go = orc.gram(orc.row_solve(A, Rs))
    assert relf(to_np(G), Go) <= 1e-13
    Rc2, G2 = B.mrcqr_precondition_gram(AT, colmajor_to_dev(Rs), want_G=True)
    assert torch.equal(G, G2) and torch.equal(Rc, Rc2)          # deterministic split-m reduction
    Rco, info = orc.cholesky_upper(Go)
    assert info == 0 and relf(to_np(Rc), Rco) <= 1e-12


def test_lda_padding_and_unaligned_base(orc):
    # lda > m and a base pointer that is only 8-byte aligned (scalar load path)
    m, n, lda = 2048, 16, 2048 + 6
    rng = np.random.default_rng(3)
    buf = torch.zeros(n * lda + 1, dtype=torch.float64, device="cuda")
    A = rng.standard_normal((m, n))
    for off in (0, 1):
        view = buf[off:off + n * lda].view(n, lda)[:, :m]
        view.copy_(torch.from_numpy(np.ascontiguousarray(A.T)))
        QT, R = B.mrcqr_factor(view, 64, 2 * n, 3)
        Q, Rn = to_np(QT)[:m], to_np(R)
        assert QT.stride(0) == lda
        assert orc.orth_error_fro(Q) <= 1e-13 and orc.residual_fro(np.asfortranarray(A), Q, Rn) <= 1e-13


def test_bit_identical_y_and_determinism(orc):
    # the Y recomputed in stage 2b equals the Y stage 2a fed to the Gram
    for (m, n) in [(1 << 13, 64), (1 << 12, 144), (3000, 40), (1 << 11, 300)]:
        AT = inputs.make_A(1 << int(np.ceil(np.log2(m))), n, 1, 5, 6, "cuda")[:, :m].contiguous()
        A = to_np(AT)
        rng = np.random.default_rng(n)
        Rs = np.triu(rng.standard_normal((n, n))) / np.sqrt(n) + 3 * np.eye(n)
        RsT = colmajor_to_dev(Rs)
        Y3, Y5 = B.mrcqr_debug_dump_y(AT, RsT)
        assert torch.equal(Y3, Y5)
        Yo = orc.row_solve(A, Rs)
        assert np.linalg.norm(to_np(Y3) - Yo) <= 1e-13 * np.linalg.cond(Rs) * np.linalg.norm(Yo)
    # ill-conditioned A with a real preconditioner: kappa(R_s) ~ 1e12 is where a re-rounded Y would
    # differ by kappa*u; it must still be identical bit for bit
    AT = inputs.make_A(1 << 14, 96, 12, 15, 16, "cuda")
    sg, ix = B.mrcqr_draw(1 << 14, 192, 3)
    Rs, _ = B.mrcqr_sketch(AT, 64, sg.cuda(), ix.cuda())
    Y3, Y5 = B.mrcqr_debug_dump_y(AT, Rs)
    assert torch.equal(Y3, Y5)
    AT = inputs.make_A(1 << 14, 48, 6, 1, 2, "cuda")
    Q1, R1 = B.mrcqr_factor(AT, 32, 96, 4)
    Q2, R2 = B.mrcqr_factor(AT, 32, 96, 4)
    assert torch.equal(Q1, Q2) and torch.equal(R1, R2)


def test_power_of_two_scaling_is_exact(orc):
    AT = inputs.make_A(1 << 13, 24, 5, 8, 9, "cuda")
    Q1, R1 = B.mrcqr_factor(AT, 64, 48, 2)
    Q2, R2 = B.mrcqr_factor(AT * 16.0, 64, 48, 2)
    assert torch.equal(Q1, Q2) and torch.equal(R1 * 16.0, R2)


def test_breakdown_and_errors_are_reported(orc):
    m, n = 4096, 8
    rng = np.random.default_rng(0)
    # rank deficient by an exact zero column.  It is the unpaired last column (n odd) so that no
    # rounding noise of a neighbouring column leaks into it through the two-columns-per-complex-FFT
    # packing: its sketch is exactly zero and R_s[6,6] = 0.
    A7 = np.asfortranarray(rng.standard_normal((m, 7)))
    A7[:, 6] = 0.0
    rc = B.mrcqr_factor(colmajor_to_dev(A7), 64, 14, 1, check=False)
    assert rc == 2 and B.mrcqr_last_info() == 6               # PAPER.md:31 assumes rank n
    A = np.zeros((m, n), order="F")
    A[:, :] = rng.standard_normal((m, n))
    A[:, 5] = 2.0 * A[:, 2]                                   # numerically dependent column
    QT = torch.empty((n, m), dtype=torch.float64, device="cuda")
    R = torch.empty((n, n), dtype=torch.float64, device="cuda")
    rc = B.mrcqr_factor(colmajor_to_dev(A), 64, 16, 1, QT, R, check=False)
    # rounding makes R_s[5,5] tiny but non-zero: either a reported failure or a valid QR of A
    assert rc in (2, 3) or (orc.orth_error_fro(to_np(QT)) <= 1e-13 and
                            orc.residual_fro(A, to_np(QT), to_np(R)) <= 1e-13)
    # FP16 overflow of fl_p(D A): inputs beyond 65504 -> non-finite sketch, code 1
    big = colmajor_to_dev(rng.standard_normal((m, n)) * 1e6)
    assert B.mrcqr_factor(big, 16, 16, 1, check=False) == 1
    assert B.mrcqr_factor(big, 32, 16, 1, check=False) == 0
    # Cholesky breakdown through the stage call: a zero column with R_s = I gives
    # G[5,5] = 0 exactly, i.e. pivot 5 is not positive
    A[:, 5] = 0.0
    Rs = np.eye(n)
    with pytest.raises(B.MrcqrError) as e:
        B.mrcqr_precondition_gram(colmajor_to_dev(A), colmajor_to_dev(Rs))
    assert e.value.code == 3 and e.value.info == 5
    Rs[3, 3] = 0.0
    with pytest.raises(B.MrcqrError) as e:
        B.mrcqr_precondition_gram(colmajor_to_dev(A), colmajor_to_dev(Rs))
    assert e.value.code == 2 and e.value.info == 3


def test_fp16_degrades_beyond_its_range_never_silently(orc):
    # past kappa ~ 1e4..1e10 the FP16 sketch degrades orthogonality or breaks down;
    # it must never return "ok" with O(u) claimed falsely -- here we only require the honest outcome:
    # either a positive code, or a Q whose measured error is what it is while FP64 stays at O(u).
    m, n = 1 << 14, 32
    AT = inputs.make_A(m, n, 13, 61, 62, "cuda")
    A = to_np(AT)
    QT64, R64 = B.mrcqr_factor(AT, 64, 2 * n, 3)
    assert orc.orth_error_fro(to_np(QT64)) <= 1e-13
    QT16 = torch.empty_like(AT); R16 = torch.empty((n, n), dtype=torch.float64, device="cuda")
    rc = B.mrcqr_factor(AT, 16, 2 * n, 3, QT16, R16, check=False)
    if rc == 0:
        assert orc.orth_error_fro(to_np(QT16)) > 1e-13          # degraded, detectably
    else:
        assert rc in (2, 3)
