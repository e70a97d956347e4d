"""Thin ctypes binding of the C ABI in include/mrcqr.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libmrcqr.so; there is no Python or CPU
fallback: a missing library or a missing device raises.  PyTorch is used for device memory and
streams only.

Matrices are torch float64 CUDA tensors of shape (n, m), C-contiguous = the m x n column-major
matrix with leading dimension m (see inputs.py).  n x n factors are (n, n) tensors holding the
column-major matrix, i.e. tensor[j, i] = R[i, j]; use `.t()` to read them as R[i, j].
"""
import ctypes as C
import os

import torch

from . import build as _build

FP16, FP32, FP64 = 16, 32, 64
ERRORS = {1: "non-finite value in the sketch", 2: "R_s singular (A rank deficient)",
          3: "Cholesky breakdown", 4: "CUDA error / no device", 5: "not orthogonal to tolerance at FP64",
          6: "problem exceeds the static scratch of a no-alloc entry point (n > 128)"}

_lib = None


class MrcqrError(RuntimeError):
    def __init__(self, code, info=0):
        self.code, self.info = code, info
        what = ERRORS.get(code, "illegal argument %d" % (-code) if code < 0 else "unknown")
        super().__init__("mrcqr: code %d (%s), info %d" % (code, what, info))


def lib():
    """Loads (building if needed) libmrcqr.so.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if not os.path.exists(path) or os.environ.get("MRCQR_REBUILD"):
            path = _build.build()
        L = C.CDLL(path)
        i64, u64, vp, ci = C.c_int64, C.c_uint64, C.c_void_p, C.c_int
        L.mrcqr_draw.argtypes = [i64, ci, u64, vp, vp]
        L.mrcqr_create.argtypes = [vp]
        L.mrcqr_set_current.argtypes = [vp]
        L.mrcqr_destroy.argtypes = [vp]
        L.mrcqr_draw_device.argtypes = [i64, ci, u64, vp, vp, vp]
        L.mrcqr_sketch.argtypes = [i64, ci, i64, vp, ci, ci, vp, vp, vp, vp, vp]
        L.mrcqr_precondition_gram.argtypes = [i64, ci, i64, vp, vp, vp, vp, vp]
        L.mrcqr_form_q.argtypes = [i64, ci, i64, vp, vp, vp, i64, vp, vp, vp]
        L.mrcqr_factor.argtypes = [i64, ci, i64, vp, vp, vp, ci, ci, u64, vp]
        L.mrcqr_factor_async.argtypes = [i64, ci, i64, vp, vp, vp, ci, ci, u64, vp]
        L.mrcqr_wait.argtypes = [vp]
        L.mrcqr_factor_batched.argtypes = [ci, i64, ci, i64, i64, vp, i64, vp, vp, ci, ci, u64, vp, vp]
        L.mrcqr_factor_host.argtypes = [i64, ci, i64, vp, vp, vp, ci, ci, u64]
        L.mrcqr_workspace_bytes.restype = C.c_size_t
        L.mrcqr_workspace_bytes.argtypes = [i64, ci, ci, ci]
        L.mrcqr_debug_dump_y.argtypes = [i64, ci, i64, vp, vp, vp, vp, vp]
        L.mrcqr_shutdown.restype = None
        L.mrcqr_set_timing.argtypes = [ci]
        L.mrcqr_cholqr.argtypes = [i64, ci, i64, vp, vp, vp, ci, vp]
        L.mrcqr_kappa_probe.argtypes = [i64, ci, i64, vp, vp, vp, vp, vp, vp]
        L.mrcqr_orth_error.argtypes = [i64, ci, i64, vp, vp, vp]
        L.mrcqr_orth_error_noalloc.argtypes = [i64, ci, i64, vp, vp, vp, vp]
        L.mrcqr_factor_auto.argtypes = [i64, ci, i64, vp, vp, vp, ci, ci, u64, C.c_double, vp, vp, vp]
        L.mrcqr_set_store_y.argtypes = [ci]
        L.mrcqr_set_sketch_reim.argtypes = [ci]
        L.mrcqr_set_graph.argtypes = [ci]
        L.mrcqr_last_timing.argtypes = [vp]
        for f in ("mrcqr_create", "mrcqr_set_current", "mrcqr_destroy", "mrcqr_draw", "mrcqr_draw_device", "mrcqr_last_used_graph", "mrcqr_factor_batched", "mrcqr_sketch", "mrcqr_precondition_gram", "mrcqr_form_q", "mrcqr_factor",
                  "mrcqr_factor_host", "mrcqr_last_info", "mrcqr_last_launch_count", "mrcqr_debug_dump_y",
                  "mrcqr_set_timing", "mrcqr_last_timing", "mrcqr_set_store_y", "mrcqr_orth_error", "mrcqr_factor_auto", "mrcqr_cholqr", "mrcqr_kappa_probe", "mrcqr_set_graph", "mrcqr_set_sketch_reim", "mrcqr_factor_async", "mrcqr_wait"):
            getattr(L, f).restype = ci
        _lib = L
    return _lib


EXPORTS = ["mrcqr_create", "mrcqr_set_current", "mrcqr_destroy", "mrcqr_draw", "mrcqr_draw_device", "mrcqr_last_used_graph", "mrcqr_factor_batched", "mrcqr_sketch", "mrcqr_precondition_gram", "mrcqr_form_q", "mrcqr_factor",
           "mrcqr_factor_host", "mrcqr_workspace_bytes", "mrcqr_last_info", "mrcqr_last_launch_count",
           "mrcqr_debug_dump_y", "mrcqr_shutdown", "mrcqr_set_timing", "mrcqr_last_timing", "mrcqr_set_store_y", "mrcqr_orth_error", "mrcqr_factor_auto", "mrcqr_cholqr", "mrcqr_kappa_probe", "mrcqr_set_graph", "mrcqr_set_sketch_reim",
           "mrcqr_orth_error_noalloc", "mrcqr_last_used_store_y", "mrcqr_factor_async", "mrcqr_wait"]

STAGES = ["k1_srtt", "k2_sketch_qr", "prep_rs", "k3_gram", "gram_reduce", "k4_chol", "k5_form_q"]


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _chk(rc):
    if rc != 0:
        raise MrcqrError(rc, lib().mrcqr_last_info())


def _mat(AT):
    assert AT.is_cuda and AT.dtype == torch.float64 and AT.dim() == 2 and AT.stride(1) == 1
    n, m = AT.shape
    return m, n, AT.stride(0), AT.data_ptr()


def mrcqr_create():
    """A new context (own workspace, switches, status); make it the calling thread's with mrcqr_set_current."""
    h = C.c_void_p(None)
    rc = lib().mrcqr_create(C.byref(h))
    if rc != 0:
        raise MrcqrError(rc)
    return h


def mrcqr_set_current(handle):
    """handle from mrcqr_create, or None for the process default context."""
    lib().mrcqr_set_current(handle)


def mrcqr_destroy(handle):
    lib().mrcqr_destroy(handle)


def mrcqr_draw(m, s, seed):
    """Host draw (Algorithm 2 step 1): returns (signs uint64-as-int64 tensor, idx int64 tensor) on CPU."""
    signs = torch.zeros((m + 63) // 64, dtype=torch.int64)
    idx = torch.zeros(max(s, 1), dtype=torch.int64)
    rc = lib().mrcqr_draw(m, s, seed, signs.data_ptr(), idx.data_ptr())
    if rc != 0:
        raise MrcqrError(rc)
    return signs, idx[:s].clone()


def mrcqr_draw_device(m, s, seed, stream=None):
    """The draw as mrcqr_factor performs it (device kernel for the sign words): (signs int64 tensor, idx int64 tensor) on the GPU."""
    signs = torch.zeros((m + 63) // 64, dtype=torch.int64, device="cuda")
    idx = torch.zeros(max(s, 1), dtype=torch.int64, device="cuda")
    _chk(lib().mrcqr_draw_device(m, s, seed, signs.data_ptr(), idx.data_ptr(), _stream(stream)))
    return signs, idx[:s].clone()


def _out(QT, AT):
    """A caller-supplied Q must have A's shape and leading dimension (the C ABI gives mrcqr_factor one lda)."""
    assert QT.is_cuda and QT.dtype == torch.float64 and QT.device == AT.device
    assert QT.shape == AT.shape and QT.stride(1) == 1 and QT.stride(0) == AT.stride(0), "Q must share A's shape and lda"
    return QT


def mrcqr_sketch(AT, prec, signs, idx, want_As=False, stream=None):
    """Stage 1.  signs/idx: device tensors.  Returns (Rs (n,n) col-major, As (n,s) col-major or None)."""
    m, n, lda, pA = _mat(AT)
    s = idx.numel()
    Rs = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    As = torch.empty((n, 2 * s if _reim else s), dtype=torch.float64, device=AT.device) if want_As else None
    rc = lib().mrcqr_sketch(m, n, lda, pA, prec, s, signs.data_ptr(), idx.data_ptr(),
                            As.data_ptr() if want_As else None, Rs.data_ptr(), _stream(stream))
    _chk(rc)
    return Rs, As


def mrcqr_precondition_gram(AT, Rs, want_G=False, stream=None):
    """Stage 2a.  Returns (Rc, G or None), both (n,n) col-major."""
    m, n, lda, pA = _mat(AT)
    Rc = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    G = torch.empty((n, n), dtype=torch.float64, device=AT.device) if want_G else None
    rc = lib().mrcqr_precondition_gram(m, n, lda, pA, Rs.data_ptr(), G.data_ptr() if want_G else None,
                                       Rc.data_ptr(), _stream(stream))
    _chk(rc)
    return Rc, G


def mrcqr_form_q(AT, Rs, Rc, QT=None, stream=None):
    """Stage 2b + 3.  Returns (QT (n,m) col-major Q, R (n,n) col-major)."""
    m, n, lda, pA = _mat(AT)
    if QT is None:
        QT = torch.empty((n, m), dtype=torch.float64, device=AT.device)
    assert QT.is_cuda and QT.dtype == torch.float64 and QT.shape == AT.shape and QT.stride(1) == 1 and QT.stride(0) >= m
    R = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    rc = lib().mrcqr_form_q(m, n, lda, pA, Rs.data_ptr(), Rc.data_ptr(), QT.stride(0), QT.data_ptr(),
                            R.data_ptr(), _stream(stream))
    _chk(rc)
    return QT, R


def mrcqr_factor(AT, prec, s, seed, QT=None, R=None, stream=None, check=True):
    """Whole Algorithm 2 on device buffers.  Returns (QT, R) (or the return code if check=False)."""
    m, n, lda, pA = _mat(AT)
    if QT is None:
        QT = torch.empty_strided((n, m), (lda, 1), dtype=torch.float64, device=AT.device)
    if R is None:
        R = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    _out(QT, AT)
    rc = lib().mrcqr_factor(m, n, lda, pA, QT.data_ptr(), R.data_ptr(), prec, s, seed, _stream(stream))
    if not check:
        return rc
    _chk(rc)
    return QT, R


def mrcqr_factor_async(AT, prec, s, seed, QT, R, stream=None):
    """mrcqr_factor without the synchronisation: enqueues and returns; the status comes from mrcqr_wait()."""
    m, n, lda, pA = _mat(AT)
    _out(QT, AT)
    _chk(lib().mrcqr_factor_async(m, n, lda, pA, QT.data_ptr(), R.data_ptr(), prec, s, seed, _stream(stream)))


def mrcqr_wait(check=True):
    """Synchronises the pending mrcqr_factor_async calls; returns (code, info) of the first error among them (0, 0 if
    none) or raises it when check=True."""
    info = C.c_int(0)
    rc = lib().mrcqr_wait(C.byref(info))
    if check:
        _chk(rc)
    return rc, info.value


def mrcqr_factor_batched(AB, prec, s, seed, QB=None, RB=None, stream=None, check=True):
    """Batch of problems: AB is a (batch, n, m) float64 CUDA tensor (problem b = AB[b], column-major m x n).  Problem b is
    drawn with seed + b.  Returns (QB (batch, n, m), RB (batch, n, n), codes list) -- raises on the first failing problem
    unless check=False."""
    assert AB.is_cuda and AB.dtype == torch.float64 and AB.dim() == 3 and AB.stride(2) == 1
    batch, n, m = AB.shape
    if QB is None:
        QB = torch.empty_strided((batch, n, m), AB.stride(), dtype=torch.float64, device=AB.device)
    if RB is None:
        RB = torch.empty((batch, n, n), dtype=torch.float64, device=AB.device)
    assert QB.shape == AB.shape and QB.stride(2) == 1 and QB.stride(1) == AB.stride(1) and RB.is_contiguous()
    codes = (C.c_int * batch)()
    rc = lib().mrcqr_factor_batched(batch, m, n, AB.stride(1), AB.stride(0), AB.data_ptr(), QB.stride(0), QB.data_ptr(),
                                    RB.data_ptr(), prec, s, seed, codes, _stream(stream))
    if check:
        _chk(rc)
    return QB, RB, list(codes)


def mrcqr_factor_host(AT_host, prec, s, seed, QT_host=None, R_host=None):
    """Whole Algorithm 2 on HOST buffers (copies inside the call): the end-to-end path."""
    assert (not AT_host.is_cuda) and AT_host.dtype == torch.float64 and AT_host.stride(1) == 1
    n, m = AT_host.shape
    if QT_host is None:
        QT_host = torch.empty((n, AT_host.stride(0)), dtype=torch.float64, pin_memory=True)[:, :m]
    assert (not QT_host.is_cuda) and QT_host.shape == AT_host.shape and QT_host.stride(1) == 1 \
        and QT_host.stride(0) == AT_host.stride(0), "Q_host must share A_host's shape and lda"
    if R_host is None:
        R_host = torch.empty((n, n), dtype=torch.float64, pin_memory=True)
    rc = lib().mrcqr_factor_host(m, n, AT_host.stride(0), AT_host.data_ptr(), QT_host.data_ptr(),
                                 R_host.data_ptr(), prec, s, seed)
    _chk(rc)
    return QT_host, R_host


def mrcqr_debug_dump_y(AT, Rs, stream=None):
    m, n, lda, pA = _mat(AT)
    Y3 = torch.empty((n, m), dtype=torch.float64, device=AT.device)
    Y5 = torch.empty((n, m), dtype=torch.float64, device=AT.device)
    rc = lib().mrcqr_debug_dump_y(m, n, lda, pA, Rs.data_ptr(), Y3.data_ptr(), Y5.data_ptr(), _stream(stream))
    _chk(rc)
    return Y3, Y5


def mrcqr_workspace_bytes(m, n, s, prec):
    return int(lib().mrcqr_workspace_bytes(m, n, s, prec))


def mrcqr_last_info():
    return int(lib().mrcqr_last_info())


def mrcqr_last_launch_count():
    return int(lib().mrcqr_last_launch_count())


def mrcqr_shutdown():
    lib().mrcqr_shutdown()


def mrcqr_orth_error(QT, stream=None):
    """||I - Q^T Q||_F of the column-major Q held in QT (n, m), computed on the device."""
    m, n, ldq, pQ = _mat(QT)
    err = C.c_double(0.0)
    _chk(lib().mrcqr_orth_error(m, n, ldq, pQ, C.byref(err), _stream(stream)))
    return float(err.value)


NOALLOC_N_MAX = 128


def mrcqr_orth_error_noalloc(QT, err, G=None, stream=None):
    """||I - Q^T Q||_F into the DEVICE double err[0] (and Q^T Q into the (n, n) device tensor G) with no allocation:
    the scratch is a static 19.1 MiB device array, n <= NOALLOC_N_MAX (code 6 beyond); enqueues only, no sync;
    overlapping calls race on the array (include/mrcqr.h)."""
    m, n, ldq, pQ = _mat(QT)
    assert err.is_cuda and err.dtype == torch.float64 and err.numel() >= 1
    pG = None
    if G is not None:
        assert G.is_cuda and G.dtype == torch.float64 and G.shape == (n, n) and G.is_contiguous()
        pG = G.data_ptr()
    _chk(lib().mrcqr_orth_error_noalloc(m, n, ldq, pQ, err.data_ptr(), pG, _stream(stream)))


def mrcqr_factor_auto(AT, first_prec, s, seed, tol=0.0, QT=None, R=None, stream=None, check=True):
    """Self-correcting MRCQR.  Returns (QT, R, prec_used, orth) (or (rc, prec_used, orth) if check=False)."""
    m, n, lda, pA = _mat(AT)
    if QT is None:
        QT = torch.empty_strided((n, m), (lda, 1), dtype=torch.float64, device=AT.device)
    if R is None:
        R = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    used, orth = C.c_int(0), C.c_double(0.0)
    _out(QT, AT)
    rc = lib().mrcqr_factor_auto(m, n, lda, pA, QT.data_ptr(), R.data_ptr(), first_prec, s, seed, float(tol),
                                 C.byref(used), C.byref(orth), _stream(stream))
    if not check:
        return rc, int(used.value), float(orth.value)
    _chk(rc)
    return QT, R, int(used.value), float(orth.value)


def mrcqr_cholqr(AT, passes=1, QT=None, R=None, stream=None, check=True):
    """Algorithm 1 (CholQR) on A; passes = 2: CholQR2.  Returns (QT, R) (or the code if check=False)."""
    m, n, lda, pA = _mat(AT)
    if QT is None:
        QT = torch.empty_strided((n, m), (lda, 1), dtype=torch.float64, device=AT.device)
    if R is None:
        R = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    _out(QT, AT)
    rc = lib().mrcqr_cholqr(m, n, lda, pA, QT.data_ptr(), R.data_ptr(), passes, _stream(stream))
    if not check:
        return rc
    _chk(rc)
    return QT, R


def mrcqr_kappa_probe(AT, stream=None):
    """CholQR probe (eq. (2)): returns (kappa lower bound, suggested sketch precision)."""
    m, n, lda, pA = _mat(AT)
    QT = torch.empty_strided((n, m), (lda, 1), dtype=torch.float64, device=AT.device)
    R = torch.empty((n, n), dtype=torch.float64, device=AT.device)
    lb, prec = C.c_double(0.0), C.c_int(0)
    _chk(lib().mrcqr_kappa_probe(m, n, lda, pA, QT.data_ptr(), R.data_ptr(), C.byref(lb), C.byref(prec), _stream(stream)))
    return float(lb.value), int(prec.value)


def mrcqr_set_graph(on):
    """Repeated-call mode: mrcqr_factor replays a CUDA graph captured per (shape, buffers)."""
    lib().mrcqr_set_graph(1 if on else 0)


def mrcqr_last_used_graph():
    return bool(lib().mrcqr_last_used_graph())


_reim = False


def mrcqr_set_sketch_reim(on):
    """Re+Im sketch variant: 2s sketch rows; mrcqr_sketch(want_As=True) then returns (n, 2s)."""
    global _reim
    lib().mrcqr_set_sketch_reim(1 if on else 0)
    _reim = bool(on)


def mrcqr_set_store_y(mode):
    """Form of stage 2 for n16 <= 128: None = the faster one as measured (default: Y stored from n16 = 48 on), False = always
    fused (Y stays on chip and is recomputed: north_star's form), True = always stored."""
    lib().mrcqr_set_store_y(-1 if mode is None else (1 if mode else 0))


def mrcqr_last_used_store_y():
    return bool(lib().mrcqr_last_used_store_y())


def mrcqr_set_timing(on):
    lib().mrcqr_set_timing(1 if on else 0)


def mrcqr_last_timing():
    """dict stage name -> ms of the last mrcqr_factor call (needs mrcqr_set_timing(True))."""
    buf = (C.c_float * 7)()
    lib().mrcqr_last_timing(buf)
    return {k: float(buf[i]) for i, k in enumerate(STAGES)}
