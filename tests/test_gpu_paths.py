"""GPU parity of the kernel variants mrcqr_factor dispatches to beyond the basic shapes of
test_gpu_parity.py: the register radix-16 form of K1 for the FP16 sketch (odd bin counts, one and several tiles), the
store-Y form of stage 2 for n16 > 128 (panel passes + SYRK Gram, every panel width, ragged n),
and the fall-backs taken for unaligned operands.  Same tolerances as test_gpu_parity.py."""
import numpy as np
import pytest
import torch

from helpers import U, draw_to_dev, gpu_residual_fro, to_np
from paper_2606_18411_b200 import binding as B
from paper_2606_18411_b200 import inputs
from test_gpu_parity import factor_parity, relf

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("m,n,s", [
    (1 << 13, 8, 24),        # one tile per column (m2 = 32)
    (1 << 14, 25, 50),       # two tiles per column, odd n
    (1 << 15, 33, 100),      # four tiles, s not a multiple of 32
    (1 << 14, 64, 128),      # the C1 geometry at small m
    (1 << 13, 150, 128),     # n > s is illegal for QR: the stage call rejects it
])
def test_half_sketch_matches_oracle(orc, m, n, s):
    AT = inputs.make_A(m, n, 2, 300 + n, 301 + n, "cuda")
    A = to_np(AT)
    signs, idx = orc.draw(m, s, 77 + n)
    As_o = orc.sketch(np.asfortranarray(A), signs, idx)
    dsigns, didx = draw_to_dev(signs, idx)
    if s >= n:
        _, As = B.mrcqr_sketch(AT, B.FP16, dsigns, didx, want_As=True)
        Asg = to_np(As)
        assert relf(Asg, As_o) <= 1e-2
        # every stored value is an FP16 number (the sketch lives in precision p)
        assert np.array_equal(Asg, Asg.astype(np.float16).astype(np.float64))
        factor_parity(orc, AT, s, 77 + n, B.FP16)
    else:
        with pytest.raises(B.MrcqrError):
            B.mrcqr_sketch(AT, B.FP16, dsigns, didx, want_As=True)


def test_half_sketch_closed_form(orc):
    """Column j = d * cos(2 pi k_j t / m) (signs undone): the transform has one line, at bin k_j, of height
    m/2 (m at DC / Nyquist); after the sqrt(s/m) scale the sketch is that value at (j, j) and zero elsewhere."""
    m, n, s = 1 << 13, 16, 32
    signs, idx = orc.draw(m, s, 5)
    bits = np.unpackbits(np.ascontiguousarray(signs).view(np.uint8), bitorder="little")[:m]
    d = 1.0 - 2.0 * bits
    t = np.arange(m)
    A = np.stack([d * np.cos(2 * np.pi * int(idx[j]) * t / m) for j in range(n)], axis=1)
    AT = torch.from_numpy(np.ascontiguousarray(A.T)).cuda()
    dsigns, didx = draw_to_dev(signs, idx)
    _, As = B.mrcqr_sketch(AT, B.FP16, dsigns, didx, want_As=True)
    Asg = to_np(As)
    scale = np.sqrt(s / m)
    want = np.zeros((s, n))
    for j in range(n):
        k0 = int(idx[j])
        want[j, j] = (m if k0 in (0, m // 2) else 0.5 * m) * scale
    assert np.linalg.norm(Asg - want) <= 1e-2 * np.linalg.norm(want)


@pytest.mark.parametrize("m,n,s,prec,tol", [
    (1 << 13, 5, 40, 64, 1e-12),       # radix-16 form, FP64: one tile per column (m2 = 32)
    (1 << 15, 6, 96, 64, 1e-12),       # radix-16 form, FP64: four tiles per column, even n
    (1 << 14, 4, 520, 64, 1e-12),      # radix-16 form, s > 256: three bins per thread in stage 2
    (1 << 14, 3, 1024, 32, 5e-5),      # radix-16 form, FP32, s = 1024, odd n
    (1 << 15, 4, 1030, 16, 1e-2),      # radix-16 form, FP16 tile storage, ragged s
    (1 << 17, 3, 48, 32, 5e-5),        # radix-16 form, several tiles per chunk
    (1 << 12, 5, 40, 64, 1e-12),       # radix-4 form (m < 8192): 32-wide tiles, m1 = 64
    (1 << 12, 6, 200, 32, 5e-5),       # radix-4 form, FP32
    (1 << 10, 4, 100, 16, 1e-2),       # radix-4 form, FP16 rounding, m1 = 16
    (256, 3, 129, 64, 1e-12),          # radix-4 form, every bin (s = m/2 + 1), m1 = 4
])
def test_fft_sketch_tile_widths_match_oracle(orc, m, n, s, prec, tol):
    """K1 (k1_srtt.cu) takes the register radix-16 form for m >= 8192 and the shared-memory radix-4 form, whose tile
    width depends on (m, prec, s), below; every choice is the same transform."""
    AT = inputs.make_A(m, n, 3, 500 + n, 501 + n, "cuda")
    A = to_np(AT)
    signs, idx = orc.draw(m, s, 900 + n)
    As_o = orc.sketch(np.asfortranarray(A), signs, idx)        # the oracle's sketch is the double one
    dsigns, didx = draw_to_dev(signs, idx)
    _, As = B.mrcqr_sketch(AT, {16: B.FP16, 32: B.FP32, 64: B.FP64}[prec], dsigns, didx, want_As=True)
    assert relf(to_np(As), As_o) <= tol


@pytest.mark.parametrize("m,n,expo,prec", [
    (1 << 12, 136, 3, 32),     # n16 = 144: panels of 8, 8, 2 blocks; SYRK with P = 2 and a ragged second panel
    (1 << 12, 160, 6, 64),     # n16 = 160: panels 8, 8, 4
    (1 << 12, 240, 8, 64),     # n16 = 240: panels 8, 8, 8, 6
    (1 << 11, 400, 4, 32),     # P = 4 SYRK blocks, 7 panels
    (1 << 11, 512, 5, 64),     # the largest n
    (1 << 12, 256, 7, 64),     # n16 % 64 == 0: all panels of a solve in one launch (mrcqr_panel_fused), 4 panels
    (1 << 12, 250, 5, 32),     # the same with a ragged last panel (58 columns)
    (1 << 12, 180, 4, 32),     # 3 panels (n16 = 192), last one ragged
    (1 << 11, 500, 3, 64),     # 8 panels, last one ragged
    (1 << 12, 200, 4, 32),     # n16 = 208: a ragged first panel of 2 blocks + 3 full ones; SYRK with 10 live blocks in the last panel
    (1 << 11, 330, 3, 64),     # n16 = 336: P = 3 SYRK blocks, 10 live blocks, ragged first panel of 2 blocks + 5 full ones
    (1 << 11, 304, 6, 32),     # n16 = 304: P = 3, 6 live blocks, ragged first panel of 6 blocks
])
def test_store_y_path_factorization(orc, m, n, expo, prec):
    AT = inputs.make_A(m, n, expo, 500 + n, 501 + n, "cuda")
    factor_parity(orc, AT, 2 * n, 600 + n, prec)


def test_store_y_path_is_deterministic_and_handles_strides(orc):
    m, n = 1 << 12, 272
    AT = inputs.make_A(m, n, 5, 11, 12, "cuda")
    Q1, R1 = B.mrcqr_factor(AT, B.FP64, 2 * n, 3)
    Q2, R2 = B.mrcqr_factor(AT, B.FP64, 2 * n, 3)
    assert torch.equal(Q1, Q2) and torch.equal(R1, R2)
    # lda = m + 6 (16-byte aligned columns): same arithmetic, same bits
    big = torch.zeros((n, m + 6), dtype=torch.float64, device="cuda")
    big[:, :m] = AT
    Q3, R3 = B.mrcqr_factor(big[:, :m], B.FP64, 2 * n, 3)
    assert Q3.shape == (n, m) and Q3.stride(0) == m + 6                # Q takes A's leading dimension
    assert torch.equal(Q3, Q1) and torch.equal(R3, R1)
    # columns that start on an odd element (8-byte aligned only): the fall-back kernels run; same Q to rounding
    odd = torch.zeros((n, m + 7), dtype=torch.float64, device="cuda")
    odd[:, 1:m + 1] = AT
    Q4, R4 = B.mrcqr_factor(odd[:, 1:m + 1], B.FP64, 2 * n, 3)
    A = to_np(AT)
    Q4n, R4n = to_np(Q4), to_np(R4)
    assert orc.orth_error_fro(Q4n) <= 1e-13 and orc.residual_fro(A, Q4n, R4n) <= 1e-13
    kappa = np.linalg.cond(to_np(R1))
    assert np.linalg.norm(Q4n - to_np(Q1)) <= 10 * kappa * n * U


@pytest.mark.parametrize("m,n,prec,aligned", [(1 << 14, 64, 16, True), (1 << 13, 100, 32, True), (1 << 13, 20, 64, True),
                                              (1 << 14, 128, 32, True), (1 << 13, 40, 32, True), (1 << 13, 128, 32, False),
                                              (1 << 13, 100, 32, False), (1 << 13, 20, 64, False)])
def test_three_forms_of_stage2_up_to_128_columns(orc, m, n, prec, aligned):
    """mrcqr_set_store_y (include/mrcqr.h): 0 = fused form (north_star's: Y stays on chip, K5 recomputes
    it), 1 = Y stored in Q's buffer, default = the fastest measured form (fused for n16 <= 32, stored from 48 on).
    A stored Y below n16 = 128, or with operands the panel kernels cannot take (A starting on an odd element), is K3 with
    a Y dump + K5 in place: the stored Y is the Y the Gram matrix saw, so Q is bit-identical to the fused form's.
    n16 = 128 with aligned operands takes the kernels of the n16 > 128 path (panel solves + SYRK): the same factorization
    up to the rounding of a differently ordered Gram sum.  Every form against the oracle."""
    A0 = inputs.make_A(m, n, 4, 900 + n, 901 + n, "cuda")
    if aligned:
        AT = A0
    else:
        buf = torch.empty((n, m + 2), dtype=torch.float64, device="cuda")
        AT = buf[:, 1:m + 1]
        AT.copy_(A0)
    n16 = (n + 15) // 16 * 16
    try:
        B.mrcqr_set_store_y(False)
        Q0, R0 = factor_parity(orc, AT, 2 * n, 31, prec)
        assert not B.mrcqr_last_used_store_y()
        B.mrcqr_set_store_y(True)
        Q1, R1 = factor_parity(orc, AT, 2 * n, 31, prec)
        assert B.mrcqr_last_used_store_y()
        B.mrcqr_set_store_y(None)
        Q2, R2 = B.mrcqr_factor(AT, prec, 2 * n, 31)
        assert B.mrcqr_last_used_store_y() == (n16 >= 48)                   # the measured threshold (include/mrcqr.h)
    finally:
        B.mrcqr_set_store_y(None)
    assert torch.equal(Q2, Q1 if n16 >= 48 else Q0)
    if aligned and n16 >= 128:
        kappa = np.linalg.cond(to_np(R0))
        assert not torch.equal(Q0, Q1)                                       # really the other kernels
        assert np.linalg.norm(to_np(Q1) - to_np(Q0)) <= 10 * kappa * n * U
        assert np.linalg.norm(to_np(R1) - to_np(R0)) <= 10 * kappa * n * U * np.linalg.norm(to_np(R0))
    else:
        assert torch.equal(Q0, Q1) and torch.equal(R0, R1)


def test_large_n_kernels_report_breakdown(orc):
    """The cooperative-grid Cholesky (n16 > 160) and the blocked sketch QR (n > 64) report what the small
    kernels report: a non-positive pivot -> code 3 with its index; a zero R_s diagonal -> code 2 with its index."""
    from helpers import colmajor_to_dev
    m, n = 2048, 200
    rng = np.random.default_rng(3)
    A = np.asfortranarray(rng.standard_normal((m, n)))
    A[:, 150] = 0.0                                            # with R_s = I: G[150,150] = 0 exactly
    with pytest.raises(B.MrcqrError) as e:
        B.mrcqr_precondition_gram(colmajor_to_dev(A), colmajor_to_dev(np.eye(n)))
    assert e.value.code == 3 and e.value.info == 150
    # the stage call returns G and R_c of a healthy matrix through the same kernel
    A[:, 150] = rng.standard_normal(m)
    Rc, G = B.mrcqr_precondition_gram(colmajor_to_dev(A), colmajor_to_dev(np.eye(n)), want_G=True)
    Gn, Rcn = to_np(G), to_np(Rc)
    assert np.linalg.norm(Gn - A.T @ A) <= 1e-13 * np.linalg.norm(Gn)
    assert np.linalg.norm(Rcn.T @ Rcn - Gn) <= 1e-13 * np.linalg.norm(Gn)
    assert np.all(np.diag(Rcn) > 0) and np.array_equal(np.tril(Rcn, -1), np.zeros((n, n)))
    # blocked sketch QR: the last column of an odd-n matrix is exactly zero -> its sketch is exactly zero
    m2, n2 = 1 << 13, 131
    A2 = np.asfortranarray(rng.standard_normal((m2, n2)))
    A2[:, 130] = 0.0
    rc = B.mrcqr_factor(colmajor_to_dev(A2), B.FP64, 2 * n2, 1, check=False)
    assert rc == 2 and B.mrcqr_last_info() == 130


def test_blocked_sketch_qr_is_a_qr_of_the_sketch(orc):
    """R_s^T R_s = A_s^T A_s to n u ||A_s||^2, upper triangular, diag > 0, for the blocked kernel's shapes
    (panel remainders: n = 100 -> last panel of 4; s not a multiple of 256; s = 3n)."""
    for m, n, s in [(1 << 13, 100, 200), (1 << 13, 72, 216), (1 << 12, 300, 600)]:
        AT = inputs.make_A(m, n, 6, 40 + n, 41 + n, "cuda")
        signs, idx = orc.draw(m, s, 9)
        dsigns, didx = draw_to_dev(signs, idx)
        Rs, As = B.mrcqr_sketch(AT, B.FP64, dsigns, didx, want_As=True)
        Rsn, Asn = to_np(Rs), to_np(As)
        assert np.all(np.diag(Rsn) > 0) and np.array_equal(np.tril(Rsn, -1), np.zeros((n, n)))
        assert np.linalg.norm(Rsn.T @ Rsn - Asn.T @ Asn) <= 100 * n * U * np.linalg.norm(Asn) ** 2
        # same R as the oracle's Householder QR of the oracle's sketch, to kappa(A_s) u
        o = orc.factor_from_draw(to_np(AT), signs, idx, want_intermediates=True)
        kap = np.linalg.cond(o["Rs"])
        assert np.linalg.norm(Rsn - o["Rs"]) <= 100 * n * U * kap * np.linalg.norm(o["Rs"])


def test_orth_error_matches_the_oracle_checker(orc):
    """mrcqr_orth_error against the oracle's blocked-pairwise ||I - Q^T Q||_F: on an orthonormal Q (rounding level:
    same order of magnitude) and on a Q with a planted defect (closed form: Q (I + E) with small E gives
    ||E + E^T + E^T E||_F)."""
    m, n = 1 << 14, 48
    AT = inputs.make_A(m, n, 2, 5, 6, "cuda")
    QT, _ = B.mrcqr_factor(AT, B.FP64, 2 * n, 1)
    e_gpu, e_orc = B.mrcqr_orth_error(QT), orc.orth_error_fro(to_np(QT))
    assert e_gpu <= 1e-13 and e_orc <= 1e-13 and 0.2 * e_orc <= e_gpu <= 5 * e_orc
    rng = np.random.default_rng(1)
    E = 1e-6 * rng.standard_normal((n, n))
    Qd = to_np(QT) @ (np.eye(n) + E)
    want = np.linalg.norm(E + E.T + E.T @ E)
    QdT = torch.from_numpy(np.ascontiguousarray(Qd.T)).cuda()
    assert abs(B.mrcqr_orth_error(QdT) - want) <= 1e-6 * want
    assert abs(orc.orth_error_fro(Qd) - want) <= 1e-6 * want
    # n > 128 goes through several 128 x 128 blocks
    AT2 = inputs.make_A(1 << 12, 200, 2, 7, 8, "cuda")
    QT2, _ = B.mrcqr_factor(AT2, B.FP64, 400, 1)
    assert 0.2 * orc.orth_error_fro(to_np(QT2)) <= B.mrcqr_orth_error(QT2) <= 5 * orc.orth_error_fro(to_np(QT2))


def test_factor_auto_escalates_only_when_needed(orc):
    """an underestimated precision is detected by ||I - Q^T Q|| and cured by the next level."""
    m, n = 1 << 14, 32
    # kappa ~ 1e3: the FP16 sketch is enough -> no escalation, same factorization as the oracle
    AT = inputs.make_A(m, n, 3, 21, 22, "cuda")
    QT, R, used, orth = B.mrcqr_factor_auto(AT, B.FP16, 2 * n, 4)
    assert used == 16 and 0 <= orth <= 1e-13
    A = to_np(AT)
    o = orc.factor(A, 2 * n, 4)
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(to_np(QT) - o["Q"]) <= 10 * kappa * n * U
    # kappa ~ 1e13: FP16 (and possibly FP32) must be given up; the returned factorization meets the bar
    AT = inputs.make_A(m, n, 13, 61, 62, "cuda")
    rc16 = B.mrcqr_factor(AT, B.FP16, 2 * n, 3, check=False)
    QT, R, used, orth = B.mrcqr_factor_auto(AT, B.FP16, 2 * n, 3)
    assert used in (32, 64) and 0 <= orth <= 1e-13
    if rc16 == 0:                                             # FP16 "worked" but degraded: that is what was detected
        Q16, _ = B.mrcqr_factor(AT, B.FP16, 2 * n, 3)
        assert B.mrcqr_orth_error(Q16) > 1e-13
    A = to_np(AT)
    assert orc.orth_error_fro(to_np(QT)) <= 1e-13 and orc.residual_fro(A, to_np(QT), to_np(R)) <= 1e-13
    # an impossible tolerance: the FP64 result comes back with code 5 and its measured error
    rc, used, orth = B.mrcqr_factor_auto(AT, B.FP32, 2 * n, 3, tol=1e-18, check=False)
    assert rc == 5 and used == 64 and orth > 1e-18
    # a rank-deficient matrix is reported, not hidden, after the last level
    Az = A.copy(); Az[:, 31] = 0.0; Az = Az[:, :31]
    rc, used, orth = B.mrcqr_factor_auto(torch.from_numpy(np.ascontiguousarray(Az.T)).cuda(), B.FP32, 62, 3, check=False)
    assert rc == 0 or rc in (2, 3)


@pytest.mark.parametrize("m,n", [(32 * 1301, 192), (32 * 1301, 136), (32 * 2500, 128), (32 * 1301 + 8, 200)])
def test_panel_kernels_over_several_rounds(orc, m, n):
    """The panel kernels give every warp slab after slab (296 CTAs x 4 warps of 32 rows): m = 32 x 1301 is a second round
    that only some warps take part in, with the landing zone re-requested across rounds; n = 192: three full panels in the
    fused launch; n = 136: two full panels + a ragged one in its own launch; n = 128: the SYRK form below 128 < n;
    m not a multiple of 32: the slab-kernel fallback.  CholQR2 (mrcqr_cholqr, any m) on a well-conditioned A against
    numpy's QR: two passes through solve -> Gram -> Cholesky -> solve, the second one in place."""
    gen = torch.Generator(device="cuda").manual_seed(n + m)
    AT = torch.randn((n, m), dtype=torch.float64, device="cuda", generator=gen)
    AT[: n // 2] *= 1e-2                                                  # kappa ~ 1e2: CholQR2 territory
    QT, R = B.mrcqr_cholqr(AT, 2)
    assert B.mrcqr_orth_error(QT) <= 1e-13
    assert gpu_residual_fro(AT, QT, R) <= 1e-13
    Rn = to_np(R)
    assert np.all(np.diag(Rn) > 0) and np.array_equal(np.tril(Rn, -1), np.zeros((n, n)))
    Rref = torch.linalg.qr(AT.T.contiguous(), mode="r").R
    Rref = Rref * torch.sign(torch.diagonal(Rref)).unsqueeze(1)          # positive diagonal: the unique R
    kappa = float(torch.linalg.cond(Rref))
    assert float((R.T - Rref).norm()) <= 10 * kappa * n * U * float(Rref.norm())
    Q2, R2 = B.mrcqr_cholqr(AT, 2)
    assert torch.equal(QT, Q2) and torch.equal(R, R2)                     # deterministic across launches


def test_cholqr_cholqr2_and_the_kappa_probe(orc):
    """Algorithm 1 on A against the oracle's Gram / Cholesky / row solves; its kappa^2 u loss
    of orthogonality and its breakdown near kappa ~ 1e8; CholQR2; eq. (2) as a lower bound."""
    m, n = 1 << 13, 40
    AT = inputs.make_A(m, n, 3, 71, 72, "cuda")                 # kappa ~ 1e3
    A = to_np(AT)
    Go = orc.gram(np.asfortranarray(A))
    Ro, info = orc.cholesky_upper(Go)
    assert info == 0
    Qo = orc.row_solve(np.asfortranarray(A), Ro)
    QT, R = B.mrcqr_cholqr(AT, 1)
    kappa = np.linalg.cond(Ro)
    assert np.linalg.norm(to_np(R) - Ro) <= 10 * kappa * n * U * np.linalg.norm(Ro)
    assert np.linalg.norm(to_np(QT) - Qo) <= 10 * kappa ** 2 * n * U
    e1 = B.mrcqr_orth_error(QT)
    assert e1 <= 10 * n * kappa ** 2 * U                          # O(kappa^2 u)
    assert orc.residual_fro(A, to_np(QT), to_np(R)) <= 1e-13
    Q2, R2 = B.mrcqr_cholqr(AT, 2)
    assert B.mrcqr_orth_error(Q2) <= 1e-13 and orc.residual_fro(A, to_np(Q2), to_np(R2)) <= 1e-13
    assert np.all(np.diag(to_np(R2)) > 0) and np.array_equal(np.tril(to_np(R2), -1), np.zeros((n, n)))
    # eq. (2): a lower bound of kappa_2(A), within two orders of magnitude here
    lb, prec = B.mrcqr_kappa_probe(AT)
    ktrue = np.linalg.cond(A)
    assert ktrue / 100 <= lb <= ktrue * 1.001 and prec == 16
    # kappa ~ 1e10: Cholesky of A^T A breaks down (or, if rounding lets it through, Q is far from orthonormal)
    ATb = inputs.make_A(m, n, 10, 73, 74, "cuda")
    rc = B.mrcqr_cholqr(ATb, 1, check=False)
    assert rc == 3 or (rc == 0 and B.mrcqr_orth_error(B.mrcqr_cholqr(ATb, 1)[0]) > 1e-8)
    lb, prec = B.mrcqr_kappa_probe(ATb)
    assert lb >= 1e6 and prec in (32, 64)
    # m not a power of two is fine here (no transform involved)
    AT3 = inputs.make_A(5000, 24, 2, 75, 76, "cuda")
    Q3, R3 = B.mrcqr_cholqr(AT3, 2)
    assert B.mrcqr_orth_error(Q3) <= 1e-13 and orc.residual_fro(to_np(AT3), to_np(Q3), to_np(R3)) <= 1e-13


@pytest.mark.parametrize("m,n,prec", [(4096, 16, 32), (1 << 14, 64, 16), (1 << 12, 200, 64), (1 << 12, 131, 64)])
def test_graph_replay_gives_the_same_bits(orc, m, n, prec):
    """mrcqr_set_graph(1): the captured pipeline replays with new seeds (seed and bins are graph data) and returns
    exactly what the ordinary path returns, positive codes included.  Capture is illegal on the legacy default stream,
    so the replays run on a stream of their own and mrcqr_last_used_graph() must say that a graph ran (n = 16: the
    register QR, n = 64: the half-storage sketch, n > 128: the cooperative K2 / K4 launches
    and the panel passes)."""
    AT = inputs.make_A(m, n, 3, 300 + n, 301 + n, "cuda")
    QT = torch.empty_like(AT); R = torch.empty((n, n), dtype=torch.float64, device="cuda")
    ref = {}
    for seed in (1, 2, 3):
        B.mrcqr_factor(AT, prec, 2 * n, seed, QT, R)
        ref[seed] = (QT.clone(), R.clone())
    assert not B.mrcqr_last_used_graph()
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    B.mrcqr_set_graph(True)
    try:
        # the legacy default stream cannot be captured: the ordinary path runs, same bits
        B.mrcqr_factor(AT, prec, 2 * n, 2, QT, R, stream=torch.cuda.default_stream())
        assert not B.mrcqr_last_used_graph() and torch.equal(QT, ref[2][0])
        with torch.cuda.stream(side):
            for seed in (1, 2, 3, 1):
                B.mrcqr_factor(AT, prec, 2 * n, seed, QT, R, stream=side)
                assert B.mrcqr_last_used_graph()
                assert torch.equal(QT, ref[seed][0]) and torch.equal(R, ref[seed][1])
            assert B.mrcqr_last_launch_count() > 0
            bad = AT.clone(); bad[n - 1, :] = 0.0                # exact zero last column -> code 2 from a replayed graph too
            Qb = torch.empty_like(bad)
            for _ in range(2):
                rc = B.mrcqr_factor(bad, prec, 2 * n, 1, Qb, R, stream=side, check=False)
                assert rc == 2 and B.mrcqr_last_info() == n - 1 and B.mrcqr_last_used_graph()
    finally:
        B.mrcqr_set_graph(False)


@pytest.mark.parametrize("m,n,s,prec,tol", [
    (1 << 13, 6, 20, 64, 1e-12),       # FP64, single chunk
    (1 << 14, 33, 100, 32, 5e-5),      # FP32, odd n (last column pair half empty), 2s = 200 sketch rows
    (1 << 15, 64, 128, 16, 1e-2),      # the C1 geometry at small m: FP16, 2s = 256 rows (the FFT form, not the tensor-core one)
    (1 << 12, 150, 300, 32, 5e-5),     # n > 64: blocked sketch QR on 600 rows, store-Y stage 2
])
def test_reim_sketch_variant(orc, m, n, s, prec, tol):
    """mrcqr_set_sketch_reim: the 2s x n sketch [Re X[S]; Im X[S]] against the oracle's, then the
    whole factorization with that sketch: same invariants, and R equal to the oracle's stages run on the oracle's
    Re+Im sketch (Q, R are unique given diag(R) > 0, so the sketch only enters through rounding)."""
    AT = inputs.make_A(m, n, 4, 600 + n, 601 + n, "cuda")
    A = np.asfortranarray(to_np(AT))
    seed = 1200 + n
    signs, idx = orc.draw(m, s, seed)
    As_o = orc.sketch_reim(A, signs, idx)
    dsigns, didx = draw_to_dev(signs, idx)
    p = {16: B.FP16, 32: B.FP32, 64: B.FP64}[prec]
    B.mrcqr_set_sketch_reim(True)
    try:
        Rs, As = B.mrcqr_sketch(AT, p, dsigns, didx, want_As=True)
        Asg = to_np(As)
        assert Asg.shape == (2 * s, n)
        assert relf(Asg, As_o) <= tol
        assert relf(Asg[s:], As_o[s:]) <= 2 * tol          # the imaginary rows on their own
        if prec == 16:
            assert np.array_equal(Asg, Asg.astype(np.float16).astype(np.float64))
        # R_s is the R factor of the GPU's own sketch: R_s^T R_s = A_s^T A_s, upper triangular, diag > 0
        Rsn = to_np(Rs)
        assert np.all(np.diag(Rsn) > 0) and np.array_equal(np.tril(Rsn, -1), np.zeros((n, n)))
        assert relf(Rsn.T @ Rsn, Asg.T @ Asg) <= 1e-12
        QT, R = B.mrcqr_factor(AT, p, s, seed)
    finally:
        B.mrcqr_set_sketch_reim(False)
    Q, Rn = to_np(QT), to_np(R)
    assert orc.orth_error_fro(Q) <= 1e-13
    assert orc.residual_fro(A, Q, Rn) <= 1e-13
    assert np.all(np.diag(Rn) > 0)
    o = orc.factor(A, s, seed)                              # Re-only oracle factorization: same unique (Q, R)
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(Rn - o["R"]) <= 10 * kappa * n * U * np.linalg.norm(o["R"])
    assert np.linalg.norm(Q - o["Q"]) <= 10 * kappa * n * U
    # and the switch is off again: the default sketch has s rows
    _, As1 = B.mrcqr_sketch(AT, p, dsigns, didx, want_As=True)
    assert to_np(As1).shape == (s, n)


def _guarded(shape_elems, margin=4096, fill=-1234.5):
    """A float64 CUDA buffer of `shape_elems` elements with `margin` sentinel elements on both sides (16-byte aligned)."""
    buf = torch.full((shape_elems + 2 * margin,), fill, dtype=torch.float64, device="cuda")
    return buf, buf[margin:margin + shape_elems]


def _margins_intact(buf, inner_elems, margin=4096, fill=-1234.5):
    return bool((buf[:margin] == fill).all()) and bool((buf[margin + inner_elems:] == fill).all())


@pytest.mark.parametrize("m,n,s,prec,pad", [
    (4096, 16, 32, 32, 0),       # register K2, K3 / K5 at n16 = 16, single-CTA Cholesky
    (1 << 14, 64, 128, 16, 0),   # FP16 tile storage in K1, n16 = 64
    (1 << 13, 50, 150, 64, 6),   # ragged n, lda > m: the padding rows of Q must stay untouched
    (1 << 13, 100, 200, 32, 0),  # blocked (cooperative) K2, n16 = 112
    (1 << 12, 136, 272, 64, 2),  # panel passes + SYRK, cooperative K4... n16 = 144, lda > m
    (1 << 11, 300, 600, 32, 0),  # n16 > 256
    (64, 8, 16, 64, 0),          # tiny m
])
def test_no_writes_outside_the_outputs(orc, m, n, s, prec, pad):
    """Stand-in for compute-sanitizer memcheck (closed on this pool, profiles/r02_sanitizer.md): every output lives inside a
    larger buffer of sentinels; after mrcqr_factor and the three stage calls the sentinels (margins, and the padding rows
    m..lda-1 of every column of Q) are unchanged and A is bit-identical to its copy."""
    lda = m + pad
    A0 = inputs.make_A(m, n, 3, 50 + n, 51 + n, "cuda")
    abuf, aflat = _guarded(n * lda)
    AT = aflat.view(n, lda)[:, :m]
    AT.copy_(A0)
    a_before = abuf.clone()
    qbuf, qflat = _guarded(n * lda)
    QT = qflat.view(n, lda)[:, :m]
    rbuf, rflat = _guarded(n * n)
    R = rflat.view(n, n)
    B.mrcqr_factor(AT, prec, s, 5, QT, R)
    assert _margins_intact(qbuf, n * lda) and _margins_intact(rbuf, n * n)
    if pad:
        assert bool((qflat.view(n, lda)[:, m:] == -1234.5).all())
    assert torch.equal(abuf, a_before)
    Qn, Rn = to_np(QT.contiguous()), to_np(R)
    assert orc.orth_error_fro(Qn) <= 1e-13 and orc.residual_fro(to_np(A0), Qn, Rn) <= 1e-13
    # stage calls: As, Rs, G, Rc, Q, R inside guards
    signs, idx = orc.draw(m, s, 5)
    dsigns, didx = draw_to_dev(signs, idx)
    L = B.lib()
    asbuf, asflat = _guarded(s * n)
    rsbuf, rsflat = _guarded(n * n)
    st = torch.cuda.current_stream().cuda_stream
    assert L.mrcqr_sketch(m, n, lda, AT.data_ptr(), prec, s, dsigns.data_ptr(), didx.data_ptr(), asflat.data_ptr(), rsflat.data_ptr(), st) == 0
    assert _margins_intact(asbuf, s * n) and _margins_intact(rsbuf, n * n)
    gbuf, gflat = _guarded(n * n)
    rcbuf, rcflat = _guarded(n * n)
    assert L.mrcqr_precondition_gram(m, n, lda, AT.data_ptr(), rsflat.data_ptr(), gflat.data_ptr(), rcflat.data_ptr(), st) == 0
    assert _margins_intact(gbuf, n * n) and _margins_intact(rcbuf, n * n)
    qbuf.fill_(-1234.5); rbuf.fill_(-1234.5)
    assert L.mrcqr_form_q(m, n, lda, AT.data_ptr(), rsflat.data_ptr(), rcflat.data_ptr(), lda, QT.data_ptr(), R.data_ptr(), st) == 0
    assert _margins_intact(qbuf, n * lda) and _margins_intact(rbuf, n * n)
    if pad:
        assert bool((qflat.view(n, lda)[:, m:] == -1234.5).all())
    assert torch.equal(abuf, a_before)
    # the signs / bins the caller passed are not modified either
    assert np.array_equal(dsigns.cpu().numpy().view(np.uint64), signs) and np.array_equal(didx.cpu().numpy(), idx)


def test_batched_writes_stay_inside(orc):
    batch, m, n, s = 7, 1024, 12, 30
    abuf, aflat = _guarded(batch * n * m)
    AB = aflat.view(batch, n, m)
    for b in range(batch):
        AB[b] = inputs.make_A(m, n, 2, 60 + b, 61 + b, "cuda")
    a_before = abuf.clone()
    qbuf, qflat = _guarded(batch * n * m)
    rbuf, rflat = _guarded(batch * n * n)
    QB, RB, codes = B.mrcqr_factor_batched(AB, 64, s, 1, qflat.view(batch, n, m), rflat.view(batch, n, n))
    assert codes == [0] * batch
    assert _margins_intact(qbuf, batch * n * m) and _margins_intact(rbuf, batch * n * n) and torch.equal(abuf, a_before)


def test_two_contexts_factor_concurrently(orc):
    """mrcqr_create / mrcqr_set_current: two host threads, each with a context and a stream of its own, factor different
    matrices at the same time (ctypes drops the GIL during the calls), interleaving the small-n kernels, the panel passes
    and batched calls.  Every result is bit for bit the one a lone call gives: the contexts share nothing but the
    constant-bank gate, which orders their coefficient uploads on the device."""
    import threading
    jobs = [(1 << 14, 64, 16), (1 << 12, 200, 64), (1 << 13, 24, 32), (1 << 12, 136, 32)]
    mats = [inputs.make_A(m, n, 3, 70 + n, 71 + n, "cuda") for (m, n, _) in jobs]
    ref = [B.mrcqr_factor(A, p, 2 * n, 5) for A, (m, n, p) in zip(mats, jobs)]
    AB = torch.stack([inputs.make_A(1024, 12, 2, 90 + b, 91 + b, "cuda") for b in range(6)])
    QBr, RBr, _ = B.mrcqr_factor_batched(AB, 64, 30, 1)
    torch.cuda.synchronize()
    errors = []

    def worker(tix):
        try:
            h = B.mrcqr_create()
            B.mrcqr_set_current(h)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for it in range(12):
                    j = (2 * it + tix) % len(jobs)
                    m, n, p = jobs[j]
                    Q, R = B.mrcqr_factor(mats[j], p, 2 * n, 5, stream=st)
                    if not (torch.equal(Q, ref[j][0]) and torch.equal(R, ref[j][1])):
                        errors.append(("factor", tix, it, j))
                    if it % 4 == tix:
                        QB, RB, codes = B.mrcqr_factor_batched(AB, 64, 30, 1, stream=st)
                        if not (torch.equal(QB, QBr) and torch.equal(RB, RBr)):
                            errors.append(("batched", tix, it))
                st.synchronize()
            B.mrcqr_set_current(None)
            B.mrcqr_destroy(h)
        except Exception as e:                                   # noqa: BLE001
            errors.append(("exception", tix, repr(e)))

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert errors == []
    # the default context is untouched and still works
    Q, R = B.mrcqr_factor(mats[0], jobs[0][2], 2 * jobs[0][1], 5)
    assert torch.equal(Q, ref[0][0])


@pytest.mark.parametrize("prec,tol", [(64, 1e-12), (32, 5e-5), (16, 1e-2)])
def test_radix16_sketch_unaligned_operands(orc, prec, tol):
    """The register radix-16 form of K1 (m >= 8192) on an A whose columns start on an odd element and whose leading
    dimension is odd: the 8-byte load path.  Same sketch as the aligned matrix, bit for bit, and within tolerance of the oracle."""
    m, n, s = 1 << 14, 5, 40
    A0 = inputs.make_A(m, n, 2, 11, 12, "cuda")
    signs, idx = orc.draw(m, s, 4)
    dsigns, didx = draw_to_dev(signs, idx)
    _, As0 = B.mrcqr_sketch(A0, prec, dsigns, didx, want_As=True)
    buf = torch.zeros(n * (m + 3) + 1, dtype=torch.float64, device="cuda")
    view = buf[1:1 + n * (m + 3)].view(n, m + 3)[:, :m]
    view.copy_(A0)
    assert view.data_ptr() % 16 == 8 and view.stride(0) % 2 == 1
    _, As1 = B.mrcqr_sketch(view, prec, dsigns, didx, want_As=True)
    assert torch.equal(As0, As1)
    As_o = orc.sketch(np.asfortranarray(to_np(A0)), signs, idx)
    assert relf(to_np(As1), As_o) <= tol
