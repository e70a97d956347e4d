"""Pins for the oracle's Householder R (o5), row solves (o6/o9), Gram (o7), Cholesky (o8), R_c R_s
(o10) and the invariant checkers.  CPU only.  numpy/scipy appear as test-only cross-checks."""
import numpy as np
import pytest
import scipy.linalg as sla


def test_householder_n1_closed_form(orc):
    x = np.array([[3.0], [-4.0], [12.0]])
    R, info = orc.householder_r(x)
    assert info == 0 and abs(R[0, 0] - 13.0) < 1e-15


def test_householder_hand_worked_2x2(orc):
    # A = [[3, 1], [4, 2]]: ||a1|| = 5, q1 = (3,4)/5, r12 = q1.a2 = 11/5, r22 = ||a2 - r12 q1|| = 2/5
    R, info = orc.householder_r(np.array([[3.0, 1.0], [4.0, 2.0]]))
    assert info == 0
    assert np.allclose(R, [[5.0, 2.2], [0.0, 0.4]], atol=1e-15)


@pytest.mark.parametrize("s,n,cond", [(32, 16, 1e2), (128, 64, 1e6), (97, 31, 1e12), (16, 16, 1e3)])
def test_householder_properties_and_numpy(orc, s, n, cond):
    rng = np.random.default_rng(s * n)
    U, _ = np.linalg.qr(rng.standard_normal((s, n)))
    V, _ = np.linalg.qr(rng.standard_normal((n, n)))
    As = (U * np.logspace(0, -np.log10(cond), n)) @ V.T
    R, info = orc.householder_r(As)
    assert info == 0
    assert np.all(np.diag(R) > 0) and np.allclose(np.tril(R, -1), 0.0)
    # R^T R = As^T As to n u ||As||^2
    assert np.linalg.norm(R.T @ R - As.T @ As) <= 50 * n * 1.1e-16 * np.linalg.norm(As) ** 2
    # As R^-1 has orthonormal columns (up to kappa u)
    Qs = sla.solve_triangular(R, As.T, trans="T", lower=False).T
    assert np.linalg.norm(Qs.T @ Qs - np.eye(n)) <= 100 * n * 1.1e-16 * cond
    # numpy (LAPACK) R with the same sign normalisation, column-scaled comparison
    Rn = np.linalg.qr(As, mode="r")
    Rn = Rn * np.sign(np.diag(Rn))[:, None]
    err = np.linalg.norm((R - Rn) / np.linalg.norm(As, axis=0)[None, :])
    assert err <= 1e-13 * cond ** 0 * n * 10 or err <= 1e-15 * cond


def test_householder_gram_schmidt_tiny(orc):
    rng = np.random.default_rng(1)
    As = rng.standard_normal((7, 3))
    # classical Gram-Schmidt in extended precision
    A = As.astype(np.longdouble)
    Q = np.zeros_like(A); Rg = np.zeros((3, 3), dtype=np.longdouble)
    for j in range(3):
        v = A[:, j].copy()
        for i in range(j):
            Rg[i, j] = Q[:, i] @ A[:, j]
            v -= Rg[i, j] * Q[:, i]
        Rg[j, j] = np.sqrt(v @ v); Q[:, j] = v / Rg[j, j]
    R, _ = orc.householder_r(As)
    assert np.max(np.abs(R - Rg.astype(float))) < 1e-14


def test_householder_rank_deficient_reported(orc):
    As = np.zeros((6, 3)); As[:, 0] = 1.0; As[:, 2] = np.arange(6)
    R, info = orc.householder_r(As)
    assert info == 2


def test_row_solve_identity_diagonal_and_hand(orc):
    rng = np.random.default_rng(2)
    A = rng.standard_normal((50, 4))
    assert np.array_equal(orc.row_solve(A, np.eye(4)), A)
    d = np.array([2.0, 4.0, 0.5, 8.0])
    assert np.array_equal(orc.row_solve(A, np.diag(d)), A / d)
    # hand: [y0 y1] [[2,1],[0,4]] = [6, 11] -> y0 = 3, y1 = (11 - 3)/4 = 2
    Y = orc.row_solve(np.array([[6.0, 11.0]]), np.array([[2.0, 1.0], [0.0, 4.0]]))
    assert np.array_equal(Y, [[3.0, 2.0]])


@pytest.mark.parametrize("m,n", [(300, 17), (1000, 64)])
def test_row_solve_residual_and_scipy(orc, m, n):
    rng = np.random.default_rng(m)
    A = rng.standard_normal((m, n))
    R = np.triu(rng.standard_normal((n, n))) + 4 * np.eye(n)
    Y = orc.row_solve(A, R)
    res = np.linalg.norm(Y @ R - A, axis=1)
    bound = 4 * n * 1.1e-16 * np.linalg.norm(Y, axis=1) * np.linalg.norm(R)
    assert np.all(res <= bound)
    Ys = sla.solve_triangular(R, A.T, trans="T", lower=False).T
    assert np.linalg.norm(Y - Ys) <= 1e-13 * np.linalg.norm(Ys) * np.linalg.cond(R)
    # a transposed / lower-triangular mistake would fail this: strictly lower part must be ignored
    R2 = R + np.tril(rng.standard_normal((n, n)), -1)
    assert np.array_equal(orc.row_solve(A, R2), Y)


@pytest.mark.parametrize("m,n", [(1, 3), (255, 4), (256, 4), (257, 4), (5000, 9), (70000, 3)])
def test_gram_exact_on_integers(orc, m, n):
    rng = np.random.default_rng(m + n)
    Y = rng.integers(-8, 9, size=(m, n)).astype(float)
    G = orc.gram(Y)
    want = (Y.astype(np.int64).T @ Y.astype(np.int64)).astype(float)
    assert np.array_equal(G, want)          # integers: any correct summation order is exact


def test_gram_vs_longdouble(orc):
    rng = np.random.default_rng(5)
    Y = rng.standard_normal((3000, 6))
    want = (Y.astype(np.longdouble).T @ Y.astype(np.longdouble)).astype(float)
    G = orc.gram(Y)
    assert np.max(np.abs(G - want)) <= 20 * 1.1e-16 * np.max(np.abs(want))
    assert np.array_equal(G, G.T)


def test_cholesky_hand_worked_3x3(orc):
    # G = R^T R with R = [[2,1,3],[0,3,1],[0,0,4]]
    R0 = np.array([[2.0, 1.0, 3.0], [0.0, 3.0, 1.0], [0.0, 0.0, 4.0]])
    Rc, info = orc.cholesky_upper(R0.T @ R0)
    assert info == 0 and np.array_equal(Rc, R0)


def test_cholesky_vs_numpy_and_reconstruction(orc):
    rng = np.random.default_rng(6)
    B = rng.standard_normal((200, 40))
    G = B.T @ B
    Rc, info = orc.cholesky_upper(G)
    assert info == 0 and np.all(np.diag(Rc) > 0) and np.allclose(np.tril(Rc, -1), 0)
    assert np.linalg.norm(Rc.T @ Rc - G) <= 40 * 1.1e-16 * np.linalg.norm(G)
    assert np.linalg.norm(Rc - np.linalg.cholesky(G).T) <= 1e-12 * np.linalg.norm(Rc)
    # only the upper triangle is read
    G2 = np.triu(G) + np.tril(rng.standard_normal((40, 40)), -1)
    assert np.array_equal(orc.cholesky_upper(G2)[0], Rc)


def test_cholesky_breakdown_reported(orc):
    G = np.diag([4.0, 1.0, -1e-3, 2.0])
    _, info = orc.cholesky_upper(G)
    assert info == 3                              # pivot index 2, reported as j+1
    G = np.array([[1.0, 2.0], [2.0, 1.0]])        # indefinite
    assert orc.cholesky_upper(G)[1] == 2
    assert orc.cholesky_upper(np.array([[np.nan]]))[1] == 1


def test_triu_mul(orc):
    rng = np.random.default_rng(7)
    Rc = np.triu(rng.standard_normal((9, 9))); Rs = np.triu(rng.standard_normal((9, 9)))
    R = orc.triu_mul(Rc, Rs)
    assert np.allclose(R, Rc @ Rs, atol=1e-14) and np.array_equal(np.tril(R, -1), np.zeros((9, 9)))
    assert np.allclose(np.diag(R), np.diag(Rc) * np.diag(Rs), rtol=1e-15)
    # garbage below the diagonals must be ignored
    R2 = orc.triu_mul(Rc + np.tril(np.ones((9, 9)), -1), Rs + np.tril(np.ones((9, 9)), -1))
    assert np.array_equal(R, R2)


def test_checkers(orc):
    m, n = 1024, 4
    Q = np.zeros((m, n))
    for j in range(n):
        Q[j * 256:(j + 1) * 256, j] = 1.0 / 16.0          # exactly orthonormal (256 * 2^-8 = 1)
    assert orc.orth_error_fro(Q) == 0.0
    Q2 = Q.copy(); Q2[:, 1] += 1e-6 * Q[:, 0]
    # I - Q^T Q = -[[0,e],[e,e^2]] block -> Frobenius ~ sqrt(2) e
    assert abs(orc.orth_error_fro(Q2) - np.sqrt(2) * 1e-6) < 1e-11
    R = np.triu(np.arange(1.0, 17.0).reshape(4, 4))
    A = Q @ R
    assert orc.residual_fro(A, Q, R) < 1e-16
    A2 = A.copy(); A2[0, 0] += 1e-3
    assert abs(orc.residual_fro(A2, Q, R) - 1e-3 / np.linalg.norm(A2)) < 1e-12
