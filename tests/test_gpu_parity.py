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
    # rank deficient by an exact zero column: the transform is column-wise, so the sketch of a zero
    # column is exactly zero whatever its neighbours hold, and R_s[5,5] = 0 (PAPER.md:31 assumes rank n).  All three
    # sketch precisions, an interior column of an even n (the round-1 kernel packed column pairs and failed this)
    A8 = np.asfortranarray(rng.standard_normal((m, n)))
    A8[:, 5] = 0.0
    for prec in (64, 32, 16):
        rc = B.mrcqr_factor(colmajor_to_dev(A8), prec, 16, 1, check=False)
        assert rc == 2 and B.mrcqr_last_info() == 5
    # ... and the last column of an odd n
    A7 = np.asfortranarray(rng.standard_normal((m, 7)))
    A7[:, 6] = 0.0
    rc = B.mrcqr_factor(colmajor_to_dev(A7), 64, 14, 1, check=False)
    assert rc == 2 and B.mrcqr_last_info() == 6
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


@pytest.mark.parametrize("prec,m,n,s", [(64, 1 << 13, 6, 24), (32, 1 << 14, 7, 40), (64, 1 << 15, 4, 520), (32, 1 << 15, 5, 1030),
                                        (32, 64, 4, 16), (64, 32, 3, 9), (16, 1 << 14, 6, 200)])
def test_sketch_is_column_wise(orc, prec, m, n, s):
    """the transform runs down each column on its own.  Scaling column j of A by 2^-30 scales column j of
    the sketch by 2^-30 BIT FOR BIT and leaves every other column untouched, for even and odd j, in every tile width
    of the FFT form of K1 (the FP16 sketch would underflow: checked with 2^-3)."""
    AT = inputs.make_A(m, n, 2, 700 + n, 701 + n, "cuda")
    signs, idx = orc.draw(m, s, 31 + n)
    dsigns, didx = draw_to_dev(signs, idx)
    _, As0 = B.mrcqr_sketch(AT, prec, dsigns, didx, want_As=True) if s >= n else (None, None)
    f = 2.0 ** (-3 if prec == 16 else -30)
    for j in (0, 1, n - 1, n - 2):
        AT2 = AT.clone()
        AT2[j] *= f
        _, As1 = B.mrcqr_sketch(AT2, prec, dsigns, didx, want_As=True)
        want = As0.clone()
        want[j] *= f
        if prec == 16:                                   # FP16 rounding of the scaled input is not an exact scaling near the subnormals
            assert torch.equal(As1[torch.arange(n) != j], want[torch.arange(n) != j])
            assert relf(to_np(As1[j]), to_np(want[j])) <= 2e-3
        else:
            assert torch.equal(As1, want)
    # the sketch of one column alone equals that column of the whole sketch
    _, As_one = B.mrcqr_sketch(AT[1:2].contiguous(), prec, dsigns, didx, want_As=True) if s >= 1 else (None, None)
    assert torch.equal(As_one[0], As0[1])


@pytest.mark.parametrize("m,s,seed", [(32, 4, 5), (64, 33, 6), (1 << 15, 100, 7), (1 << 20, 128, 12), (1 << 21, 512, 32)])
def test_device_draw_is_bit_exact(orc, m, s, seed):
    """a0 (north_star: bit-exact for integer work): the sign words mrcqr_factor draws with its DEVICE
    kernel and the bins it copies are the oracle's, word for word (m = 2^15: 512 words, two CTAs of the draw kernel)."""
    osigns, oidx = orc.draw(m, s, seed)
    dsigns, didx = B.mrcqr_draw_device(m, s, seed)
    assert np.array_equal(dsigns.cpu().numpy().view(np.uint64), osigns)
    assert np.array_equal(didx.cpu().numpy(), oidx)


@pytest.mark.parametrize("m,n,s,prec", [(32, 4, 8, 64), (1 << 15, 24, 48, 32), (1 << 15, 64, 128, 16), (1 << 14, 100, 200, 64)])
def test_factor_equals_its_stages_on_the_oracle_draw(orc, m, n, s, prec):
    """mrcqr_factor(seed) is bit for bit the composition sketch(oracle.draw) -> precondition_gram -> form_q: every
    kernel is deterministic, so equality holds iff the device-drawn sign words and bins equal the oracle's."""
    AT = inputs.make_A(m, n, 3, 800 + n, 801 + n, "cuda")
    B.mrcqr_set_store_y(False)        # the stage calls are the fused form of stage 2; at n16 = 128 mrcqr_factor's default is the SYRK form
    try:
        QT, R = B.mrcqr_factor(AT, prec, s, 77)
    finally:
        B.mrcqr_set_store_y(None)
    signs, idx = orc.draw(m, s, 77)
    dsigns, didx = draw_to_dev(signs, idx)
    Rs, _ = B.mrcqr_sketch(AT, prec, dsigns, didx)
    Rc, _ = B.mrcqr_precondition_gram(AT, Rs)
    Q2, R2 = B.mrcqr_form_q(AT, Rs, Rc)
    assert torch.equal(QT, Q2) and torch.equal(R, R2)


def test_default_s_is_3n(orc):
    """c = 3n by default.  s <= 0 in mrcqr_factor is exactly s = 3n."""
    m, n = 1 << 13, 20
    AT = inputs.make_A(m, n, 4, 5, 6, "cuda")
    Q0, R0 = B.mrcqr_factor(AT, 32, 0, 9)
    Q1, R1 = B.mrcqr_factor(AT, 32, 3 * n, 9)
    assert torch.equal(Q0, Q1) and torch.equal(R0, R1)
    Q2, R2 = B.mrcqr_factor(AT, 32, 2 * n, 9)
    assert not torch.equal(R0, R2)                        # a different sketch: same QR only to rounding
    factor_parity(orc, AT, 3 * n, 9, 32)
    Qa, Ra, used, orth = B.mrcqr_factor_auto(AT, 32, -1, 9)
    assert torch.equal(Qa, Q1) and used == 32


@pytest.mark.parametrize("name,m,n,s,prec,expo,pad", [("C0", 4096, 16, 32, 32, 6, 0), ("wide", 1 << 12, 136, 272, 64, 5, 0),
                                                      ("lda", 1 << 12, 24, 48, 64, 3, 10)])
def test_factor_host_matches_oracle(orc, name, m, n, s, prec, expo, pad):
    """mrcqr_factor_host (the path bench.py times as e2e) against the oracle, element by element; with lda > m the
    padding rows of A_host are not read (NaN there) and those of Q_host are not written (sentinels survive)."""
    if name == "C0":
        cfg = inputs.CONFIGS["C0"]
        AT = inputs.make_config(cfg, "cpu")
        seed = cfg["seed_draw"]
    else:
        AT = inputs.make_A(m, n, expo, 900 + n, 901 + n, "cpu")
        seed = 5
    lda = m + pad
    A_host = torch.full((n, lda), float("nan"), dtype=torch.float64).pin_memory()
    A_host[:, :m] = AT
    Q_host = torch.full((n, lda), -7.0, dtype=torch.float64).pin_memory()
    R_host = torch.empty((n, n), dtype=torch.float64).pin_memory()
    B.mrcqr_factor_host(A_host[:, :m], prec, s, seed, Q_host[:, :m], R_host)
    A = to_np(AT)
    Q, Rn = Q_host[:, :m].numpy().T, R_host.numpy().T
    assert np.all(Q_host[:, m:].numpy() == -7.0)
    o = orc.factor(A, s, seed)
    assert o["rc"] == 0
    assert orc.orth_error_fro(Q) <= 1e-13 and orc.residual_fro(A, Q, Rn) <= 1e-13
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(Q - o["Q"]) <= 10 * kappa * n * U
    assert np.linalg.norm(Rn - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
    # same bits as the device-buffer call
    QT, R = B.mrcqr_factor(AT.cuda(), prec, s, seed)
    assert torch.equal(QT.cpu(), Q_host[:, :m]) and torch.equal(R.cpu(), R_host)
