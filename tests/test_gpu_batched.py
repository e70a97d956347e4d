"""GPU parity of mrcqr_factor_batched (repeated small factorizations): every problem
of a batch against the oracle's factorization of that problem with seed + b, element by element, plus the invariants;
per-problem status codes; the one-after-the-other path for shapes beyond one CTA; determinism."""
import numpy as np
import pytest
import torch

from helpers import U, to_np
from paper_2606_18411_b200 import binding as B
from paper_2606_18411_b200 import inputs

pytestmark = pytest.mark.gpu


def make_batch(batch, m, n, expo, seed0, pad=0, gap=0):
    """(batch, n, m) view into a buffer with leading dimension m + pad and `gap` extra doubles between problems."""
    lda = m + pad
    stride = n * lda + gap
    buf = torch.full((batch * stride + 2,), float("nan"), dtype=torch.float64, device="cuda")
    AB = torch.as_strided(buf, (batch, n, m), (stride, lda, 1))
    for b in range(batch):
        AB[b] = inputs.make_A(m, n, expo, seed0 + 2 * b, seed0 + 2 * b + 1, "cuda")
    return AB


def check_problem(orc, A_T, Q_T, R_T, s, seed, n, q_tol_scale=10.0):
    A, Q, Rn = to_np(A_T), to_np(Q_T), to_np(R_T)
    o = orc.factor(A, s, seed)
    assert o["rc"] == 0
    assert orc.orth_error_fro(Q) <= 1e-13
    assert orc.residual_fro(A, Q, Rn) <= 1e-13
    assert np.all(np.diag(Rn) > 0) and np.array_equal(np.tril(Rn, -1), np.zeros((n, n)))
    kappa = np.linalg.cond(o["R"])
    assert np.linalg.norm(Q - o["Q"]) <= q_tol_scale * kappa * n * U
    assert np.linalg.norm(Rn - o["R"]) <= q_tol_scale * kappa * n * U * np.linalg.norm(o["R"])


@pytest.mark.parametrize("batch,m,n,s,prec,expo,pad,gap", [
    (5, 4096, 16, 32, 32, 6, 0, 0),        # the C0 shape (BASELINE.json configs[0]) five times over
    (3, 32, 4, 9, 64, 1, 0, 0),            # smallest m: one 32-row tile, four rows per row group
    (4, 64, 3, 33, 64, 2, 0, 0),           # every bin (s = m/2 + 1), two warps of bins
    (3, 8192, 20, 60, 16, 3, 0, 0),        # FP16 sketch, n16 = 32, default c = 3n
    (2, 2048, 32, 128, 64, 8, 0, 0),       # widest fused shape: n = 32, s = 128, FP64
    (3, 1024, 7, 21, 32, 4, 6, 10),        # lda > m and a gap between the problems (still 16-byte aligned)
    (3, 1024, 9, 20, 64, 4, 3, 1),         # odd lda and stride: the 8-byte load path
    (2, 1 << 16, 8, 16, 32, 2, 0, 0),      # the longest fused m
])
def test_batched_matches_oracle_per_problem(orc, batch, m, n, s, prec, expo, pad, gap):
    AB = make_batch(batch, m, n, expo, 1000 + n, pad, gap)
    QB, RB, codes = B.mrcqr_factor_batched(AB, prec, s, 40)
    assert codes == [0] * batch and B.mrcqr_last_launch_count() == 1
    for b in range(batch):
        check_problem(orc, AB[b].contiguous(), QB[b].contiguous(), RB[b], s, 40 + b, n)
    # the same problems through mrcqr_factor with seed + b: the same unique (Q, R) to rounding
    Q1, R1 = B.mrcqr_factor(AB[1].contiguous(), prec, s, 41)
    kappa = np.linalg.cond(to_np(R1))
    assert np.linalg.norm(to_np(QB[1].contiguous()) - to_np(Q1)) <= 10 * kappa * n * U
    # deterministic
    Q2, R2, _ = B.mrcqr_factor_batched(AB, prec, s, 40)
    assert torch.equal(RB, R2) and torch.equal(torch.nan_to_num(QB.contiguous()), torch.nan_to_num(Q2.contiguous()))


def test_batched_more_problems_than_ctas(orc):
    """1024 C0-sized problems (the VERDICT's measure of the repeated-call mode): the persistent grid walks them; a sample
    is compared with the oracle, all of them with the invariants computed on the device."""
    batch, m, n, s = 1024, 4096, 16, 32
    G = inputs.gaussian_colmajor(m, n * batch, 77, "cuda").view(batch, n, m)
    sig = inputs.sigma_logspaced(n, 6, "cuda")
    V = inputs.orthogonal_factor(n, 78, "cuda")
    AB = torch.matmul((V * sig.unsqueeze(0)).unsqueeze(0), G).contiguous()
    QB, RB, codes = B.mrcqr_factor_batched(AB, 32, s, 7)
    assert codes == [0] * batch
    for b in (0, 1, 147, 148, 500, 1023):
        check_problem(orc, AB[b], QB[b], RB[b], s, 7 + b, n)
    E = torch.bmm(QB, QB.transpose(1, 2)) - torch.eye(n, dtype=torch.float64, device="cuda")
    assert float(E.flatten(1).norm(dim=1).max()) <= 1e-13
    Res = AB - torch.bmm(RB, QB)                                  # A^T - R^T Q^T per problem
    assert float((Res.flatten(1).norm(dim=1) / AB.flatten(1).norm(dim=1)).max()) <= 1e-13


def test_batched_reports_codes_per_problem(orc):
    batch, m, n, s = 6, 2048, 8, 16
    AB = make_batch(batch, m, n, 2, 300)
    AB[2, 5] = 0.0                                                # exact zero column: R_s[5,5] = 0 -> code 2, info 5
    AB[4] *= 1e6                                                  # beyond FP16 range -> code 1 with the FP16 sketch
    QB, RB, codes = B.mrcqr_factor_batched(AB, 16, s, 3, check=False)
    assert codes == [0, 0, 2, 0, 1, 0]
    rc = B.lib().mrcqr_factor_batched(batch, m, n, m, n * m, AB.data_ptr(), n * m, QB.data_ptr(), RB.data_ptr(), 16, s, 3, None, None)
    assert rc == 2 and B.mrcqr_last_info() == 5                   # the first failing problem
    for b in (0, 1, 3, 5):
        check_problem(orc, AB[b], QB[b], RB[b], s, 3 + b, n)
    QB, RB, codes = B.mrcqr_factor_batched(AB, 32, s, 3, check=False)
    assert codes == [0, 0, 2, 0, 0, 0]


def test_batched_large_shapes_take_the_ordinary_path(orc):
    batch, m, n, s = 2, 1 << 13, 40, 80                           # n > 32: one mrcqr_factor after the other
    AB = make_batch(batch, m, n, 3, 500)
    QB, RB, codes = B.mrcqr_factor_batched(AB, 32, s, 11)
    assert codes == [0, 0] and B.mrcqr_last_launch_count() > 2
    for b in range(batch):
        check_problem(orc, AB[b], QB[b], RB[b], s, 11 + b, n)
        Q1, R1 = B.mrcqr_factor(AB[b], 32, s, 11 + b)
        assert torch.equal(Q1, QB[b]) and torch.equal(R1, RB[b])
