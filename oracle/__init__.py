"""CPU oracle for MRCQR (arxiv/paper_2606_18411) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper over oracle/mrcqr_oracle.c (plain C, IEEE double).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from paper_2606_18411_b200 and shares no code with the CUDA path.

All matrices cross this boundary as numpy float64 arrays in Fortran (column-major) order; a
2-D array M[r, j] with M.flags.f_contiguous is the paper's m x n matrix with ld = m.
"""
import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        i64, u64, dp, vp = C.c_int64, C.c_uint64, C.POINTER(C.c_double), C.c_void_p
        L.orc_splitmix64_at.restype = u64
        L.orc_splitmix64_at.argtypes = [u64, u64]
        L.orc_draw.argtypes = [i64, C.c_int, u64, vp, vp]
        L.orc_fft_radix2.restype = None
        L.orc_fft_radix2.argtypes = [i64, vp, vp]
        L.orc_sketch.argtypes = [i64, C.c_int, i64, vp, vp, C.c_int, vp, vp]
        L.orc_sketch_reim.argtypes = [i64, C.c_int, i64, vp, vp, C.c_int, vp, vp]
        L.orc_householder_r.argtypes = [C.c_int, C.c_int, vp, vp]
        L.orc_row_solve.restype = None
        L.orc_row_solve.argtypes = [i64, C.c_int, i64, vp, vp, i64, vp]
        L.orc_gram.restype = None
        L.orc_gram.argtypes = [i64, C.c_int, i64, vp, vp]
        L.orc_cholesky_upper.argtypes = [C.c_int, vp, vp]
        L.orc_triu_mul.restype = None
        L.orc_triu_mul.argtypes = [C.c_int, vp, vp, vp]
        L.orc_factor_from_draw.argtypes = [i64, C.c_int, i64, vp, vp, C.c_int, vp, i64, vp, vp,
                                           vp, vp, vp, vp, C.POINTER(C.c_int)]
        L.orc_orth_error_fro.restype = C.c_double
        L.orc_orth_error_fro.argtypes = [i64, C.c_int, i64, vp]
        L.orc_residual_fro.restype = C.c_double
        L.orc_residual_fro.argtypes = [i64, C.c_int, i64, vp, i64, vp, vp]
        L.orc_num_threads.restype = C.c_int
        del dp
        _lib = L
    return _lib


def _f(a):
    """float64, column-major; copies only if needed."""
    return np.asfortranarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _new(shape):
    return np.zeros(shape, dtype=np.float64, order="F")


def num_threads():
    return int(lib().orc_num_threads())


def splitmix64_at(seed, k):
    return int(lib().orc_splitmix64_at(C.c_uint64(seed), C.c_uint64(k)))


def draw(m, s, seed):
    """(signs, idx): signs = ceil(m/64) uint64 words (bit t%64 of word t//64 set -> d_t = -1),
    idx = s sorted distinct bins in [0, m//2].  Algorithm 2 step 1."""
    signs = np.zeros((m + 63) // 64, dtype=np.uint64)
    idx = np.zeros(max(s, 1), dtype=np.int64)
    rc = lib().orc_draw(m, s, C.c_uint64(seed), _p(signs), _p(idx))
    if rc != 0:
        raise ValueError("orc_draw: s out of range")
    return signs, idx[:s].copy()


def fft(x):
    """Unnormalised complex DFT (exp(-2 pi i k t/m)) of a length-2^k vector."""
    x = np.asarray(x)
    re = np.ascontiguousarray(x.real, dtype=np.float64).copy()
    im = np.ascontiguousarray(x.imag, dtype=np.float64).copy() if np.iscomplexobj(x) else np.zeros_like(re)
    lib().orc_fft_radix2(re.shape[0], _p(re), _p(im))
    return re + 1j * im


def sketch(A, signs, idx):
    """A_s = sqrt(s/m) Re(FFT(D A))[S,:]  (Algorithm 2 steps 2-4), in double."""
    A = _f(A)
    m, n = A.shape
    s = int(len(idx))
    signs = np.ascontiguousarray(signs, dtype=np.uint64)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    As = _new((s, n))
    lib().orc_sketch(m, n, m, _p(A), _p(signs), s, _p(idx), _p(As))
    return As


def sketch_reim(A, signs, idx):
    """Re+Im variant: (2s, n) sketch, rows [0, s) = sqrt(s/m) Re X[S], rows [s, 2s) = sqrt(s/m) Im X[S]."""
    A = _f(A)
    m, n = A.shape
    s = int(len(idx))
    signs = np.ascontiguousarray(signs, dtype=np.uint64)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    As = _new((2 * s, n))
    lib().orc_sketch_reim(m, n, m, _p(A), _p(signs), s, _p(idx), _p(As))
    return As


def householder_r(As):
    """(R_s, info): R-factor of Householder QR of the sketch, diag > 0 (step 5)."""
    As = _f(As)
    s, n = As.shape
    Rs = _new((n, n))
    info = lib().orc_householder_r(s, n, _p(As), _p(Rs))
    return Rs, int(info)


def row_solve(A, R):
    """Y = A R^{-1} row by row, R upper (step 7 PAPER.md:103 / Alg.1 step 3 PAPER.md:53)."""
    A, R = _f(A), _f(R)
    m, n = A.shape
    Y = _new((m, n))
    lib().orc_row_solve(m, n, m, _p(A), _p(R), m, _p(Y))
    return Y


def gram(Y):
    """G = Y^T Y (Alg.1 step 1), leaf-256 + binary-tree summation."""
    Y = _f(Y)
    m, n = Y.shape
    G = _new((n, n))
    lib().orc_gram(m, n, m, _p(Y), _p(G))
    return G


def cholesky_upper(G):
    """(R_c, info): G = R_c^T R_c; info = j+1 for the first non-positive pivot (breakdown)."""
    G = _f(G)
    n = G.shape[0]
    Rc = _new((n, n))
    info = lib().orc_cholesky_upper(n, _p(G), _p(Rc))
    return Rc, int(info)


def triu_mul(Rc, Rs):
    """R = R_c R_s (step 9)."""
    Rc, Rs = _f(Rc), _f(Rs)
    n = Rc.shape[0]
    R = _new((n, n))
    lib().orc_triu_mul(n, _p(Rc), _p(Rs), _p(R))
    return R


def factor_from_draw(A, signs, idx, want_intermediates=False):
    """Whole Algorithm 2 from a given draw.  Returns dict(rc, info, Q, R[, As, Rs, G, Rc])."""
    A = _f(A)
    m, n = A.shape
    s = int(len(idx))
    signs = np.ascontiguousarray(signs, dtype=np.uint64)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    Q, R = _new((m, n)), _new((n, n))
    As, Rs, G, Rc = _new((s, n)), _new((n, n)), _new((n, n)), _new((n, n))
    info = C.c_int(0)
    rc = lib().orc_factor_from_draw(m, n, m, _p(A), _p(signs), s, _p(idx), m, _p(Q), _p(R),
                                    _p(As), _p(Rs), _p(G), _p(Rc), C.byref(info))
    out = dict(rc=int(rc), info=int(info.value), Q=Q, R=R)
    if want_intermediates:
        out.update(As=As, Rs=Rs, G=G, Rc=Rc)
    return out


def factor(A, s, seed, want_intermediates=False):
    A = _f(A)
    signs, idx = draw(A.shape[0], s, seed)
    return factor_from_draw(A, signs, idx, want_intermediates)


def orth_error_fro(Q):
    """||I - Q^T Q||_F with tree summation over rows (eq.(1); Frobenius per BASELINE)."""
    Q = _f(Q)
    m, n = Q.shape
    return float(lib().orc_orth_error_fro(m, n, m, _p(Q)))


def residual_fro(A, Q, R):
    """||A - Q R||_F / ||A||_F, long-double accumulation."""
    A, Q, R = _f(A), _f(Q), _f(R)
    m, n = A.shape
    return float(lib().orc_residual_fro(m, n, m, _p(A), m, _p(Q), _p(R)))
