/*
 * mrcqr.h -- C ABI of the B200-native (sm_100a) MRCQR library: FP64 thin QR  A = Q R  of a
 * tall-skinny m x n matrix by mixed-precision randomized-preconditioned Cholesky-QR
 * (arxiv/paper_2606_18411, Algorithm 2; Algorithm 1).
 *
 * Conventions (all entry points)
 *   Layout     column-major; A is m x n with leading dimension lda >= m (the paper's libraries
 *              and its "column-wise" FFT are column-major).  R, Rs, Rc, G are
 *              n x n, ld = n, upper triangle meaningful, strictly-lower part written as zero
 *              (G is written full symmetric).
 *   Pointers   DEVICE pointers unless the argument name ends in _host.  The caller owns every
 *              buffer it passes; A is never modified; Q must not overlap A.
 *   Workspace  every CONTEXT owns one grow-only device workspace (sketch partials, A_s, R_s, Gram
 *              partials, status word), its staging buffers, its switches (mrcqr_set_*), its status
 *              (mrcqr_last_*) and its graph cache, allocated on first use, freed by mrcqr_shutdown().
 *              All entry points act on the calling thread's CURRENT context: the process default
 *              one, or a handle made current by mrcqr_set_current (mrcqr_create / mrcqr_destroy).
 *              One call at a time per context; host threads with a context and a stream each may
 *              call concurrently (the library orders, on the device, the one stretch of a
 *              factorization that uses a device-wide resource, the constant-bank coefficients of
 *              the row kernels; sketches and batched calls overlap freely).
 *   stream     a cudaStream_t passed as void* (NULL = default stream).  Kernels are enqueued on
 *              it; the call then reads back an 8-byte status word and synchronises the stream, so
 *              the return value is final when the call returns.
 *   Returns    0 ok.  -k: the k-th argument is illegal (LAPACK style).  Positive codes below.
 *              On a positive code Q and R are unspecified.  Nothing is retried, shifted or
 *              hidden (breakdown is a reported event).
 *   No CPU fallback exists: without a CUDA device every compute entry point returns MRCQR_ERR_CUDA.
 */
#ifndef MRCQR_H
#define MRCQR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Contexts.  mrcqr_create makes a new context (nothing is allocated until its first use), mrcqr_set_current makes it the
 * calling thread's current one (NULL: back to the process default context), mrcqr_destroy frees everything it owns (it
 * must not be current in another thread, nor in use).  Return 0, or -1 for a null argument.
 */
typedef struct mrcqr_handle_s* mrcqr_handle_t;
int mrcqr_create(mrcqr_handle_t* handle);
int mrcqr_set_current(mrcqr_handle_t handle);
int mrcqr_destroy(mrcqr_handle_t handle);

/* sketch precision p of Algorithm 2: half, single, double */
typedef enum { MRCQR_FP16 = 16, MRCQR_FP32 = 32, MRCQR_FP64 = 64 } mrcqr_prec_t;

enum {
    MRCQR_OK            = 0,
    MRCQR_ERR_NONFINITE = 1,  /* non-finite value in the sketch (e.g. FP16 overflow of fl_p(D A))        */
    MRCQR_ERR_SINGULAR  = 2,  /* R_s has a zero / non-finite diagonal: A rank deficient   */
    MRCQR_ERR_BREAKDOWN = 3,  /* Cholesky pivot <= 0 or NaN; index: mrcqr_last_info() */
    MRCQR_ERR_CUDA      = 4,  /* CUDA runtime error, or no device                                        */
    MRCQR_ERR_NOT_ORTHOGONAL = 5, /* mrcqr_factor_auto: ||I - Q^T Q||_F > tol even with the FP64 sketch       */
    MRCQR_ERR_TOO_LARGE = 6   /* mrcqr_orth_error_noalloc: the problem exceeds its fixed static scratch       */
};

/*
 * Algorithm 2 step 1: draw the Rademacher diagonal D and the sampled bins S from a
 * splitmix64 stream (BASELINE.json configs).  HOST function, integer arithmetic only.
 *   X(k) = k-th output of splitmix64 seeded with `seed`.
 *   signs_host: ceil(m/64) words; d_t = -1 iff bit (t mod 64) of word floor(t/64) = X(floor(t/64)) is 1.
 *   idx_host:   s distinct 0-based bins in [0, floor(m/2)], ascending.  Candidates
 *               floor(X(k) * (floor(m/2)+1) / 2^64) for k = ceil(m/64), ceil(m/64)+1, ...;
 *               a candidate is kept if new, until s are kept.
 * Returns 0, -1 (m < 1), -2 (s < 0 or s > floor(m/2)+1), -4/-5 (null pointer).
 */
int mrcqr_draw(int64_t m, int s, uint64_t seed, uint64_t* signs_host, int64_t* idx_host);

/*
 * The same draw (Algorithm 2 step 1) into DEVICE buffers: the ceil(m/64) sign words by the device kernel
 * of the library, the s bins drawn on the host and copied.  The words and bins are bit-identical to mrcqr_draw's (and
 * the oracle's); the GPU tests pin that.  mrcqr_factor draws the same words: with this kernel when m < 8192, in the
 * Re+Im variant and under graph replay, otherwise inside its transform kernel, which evaluates X(word) where it uses
 * it (the tests require mrcqr_factor to equal, bit for bit, its stage calls run on these buffers).  signs / idx:
 * device.  Synchronises the stream.  Returns as mrcqr_draw, or 4.
 */
int mrcqr_draw_device(int64_t m, int s, uint64_t seed, uint64_t* signs, int64_t* idx, void* stream);

/*
 * Stage 1, Algorithm 2 steps 2-6: the subsampled randomized trigonometric
 * transform and the sketch QR.
 *   x~ = fl_p(D a_j) (sign-bit flip + round to p), X = DFT_m(x~) down each column,
 *   A_s[i,j] = sqrt(s/m) Re X[idx[i]], A_s stored in precision p;
 *   R_s = R-factor of the Householder QR of A_s with rows sign-normalised to diag > 0, in FP64.
 * Arithmetic is at least precision p (FP16: FP16 input/output rounding, FP32 arithmetic).
 *   m       power of two, m >= n            signs  ceil(m/64) uint64 words (device)
 *   s       n <= s <= m/2+1                 idx    s ascending bins, int64 (device)
 *   As_out  nullable; s x n, ld = s, FP64 container holding the precision-p values exactly
 *   Rs      n x n, ld = n (out)
 * Positive returns: 1 (non-finite sketch), 2 (singular R_s; index via mrcqr_last_info()).
 */
int mrcqr_sketch(int64_t m, int n, int64_t lda, const double* A, mrcqr_prec_t prec, int s,
                 const uint64_t* signs, const int64_t* idx, double* As_out, double* Rs,
                 void* stream);

/*
 * Stage 2a, Algorithm 2 step 7 fused with Algorithm 1 steps 1-2.
 * For every row a of A: y R_s = a by forward substitution in FP64 (R_s^-1 is never formed,
 * PAPER.md:121); G = sum_rows y^T y on FP64 tensor cores (DMMA) with a deterministic split-m
 * reduction; Y = A R_s^-1 is never written to memory.  Then G = Rc^T Rc (Cholesky, Rc upper,
 * diag > 0).  Any m >= n.  G_out nullable (n x n full symmetric).  Rc: n x n (out).
 * Positive returns: 2 (Rs diagonal zero/non-finite), 3 (Cholesky breakdown, pivot index via
 * mrcqr_last_info()).
 */
int mrcqr_precondition_gram(int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                            double* G_out, double* Rc, void* stream);

/*
 * Stage 2b + 3, Algorithm 1 step 3 and Algorithm 2 step 9.
 * For every row: y = a R_s^-1 recomputed bit-identically to stage 2a, then q R_c = y; Q written
 * (m x n, ldq >= m).  R = R_c R_s (n x n, nullable).
 */
int mrcqr_form_q(int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                 const double* Rc, int64_t ldq, double* Q, double* R, void* stream);

/*
 * Whole Algorithm 2 = draw(seed) -> mrcqr_sketch -> mrcqr_precondition_gram ->
 * mrcqr_form_q on one stream with a single status read-back at the end.
 *   Q uses the same leading dimension lda as A.   s <= 0 selects the paper default 3n.
 *   sketch_prec: the caller's choice by the rule of PAPER.md:163 (half if kappa < 1e4, single if
 *   kappa < 1e8, double otherwise).
 * Argument errors: -1 m (not a power of two or < n), -2 n, -3 lda, -4 A, -5 Q, -6 R, -7 prec, -8 s.
 */
int mrcqr_factor(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R,
                 mrcqr_prec_t sketch_prec, int s, uint64_t seed, void* stream);

/*
 * Algorithm 2 for a BATCH of independent problems of one shape: the repeated-call regime the paper motivates (block
 * Arnoldi, randomized-SVD power iterations, time stepping), where one small factorization is a chain of
 * dependent kernels whose latency no loop or graph can hide.  Problem b (0 <= b < batch) is
 *     A_b = A + b * strideA  (m x n, column-major, leading dimension lda),   Q_b = Q + b * strideQ (same lda),
 *     R_b = R + b * n * n,   drawn with seed + b: its result is that of mrcqr_factor(..., seed + b, ...).
 * Shapes with n <= 32, s <= 128, m <= 2^16 run as ONE kernel, one CTA per problem, out of shared memory and L2 (the sketch
 * is the defining cosine sum evaluated directly in the arithmetic of p; everything else as in mrcqr_factor); other shapes
 * are factored one after the other by the ordinary path.  Strides count doubles; strideA, strideQ >= (n-1) lda + m.
 * codes_host (nullable, HOST, batch ints): the code of every problem (0, 1, 2, 3).  Returns 0 if every problem succeeded,
 * else the code of the first failing problem (its index detail via mrcqr_last_info()); a negative argument index:
 * -1 batch, -2 m, -3 n, -4 lda, -5 strideA, -6 A, -7 strideQ, -8 Q, -9 R, -10 prec, -11 s; or 4.
 */
int mrcqr_factor_batched(int batch, int64_t m, int n, int64_t lda, int64_t strideA, const double* A,
                         int64_t strideQ, double* Q, double* R, mrcqr_prec_t sketch_prec, int s,
                         uint64_t seed, int* codes_host, void* stream);

/*
 * mrcqr_factor with HOST buffers: copies the m x n part of A (lda >= m; the padding rows m..lda-1 of a column are
 * neither read nor written) to library-owned device buffers on a stream of the library's own, factors, copies Q
 * (same lda) and R back; synchronous.  This is the end-to-end path bench.py times as `e2e`.
 */
int mrcqr_factor_host(int64_t m, int n, int64_t lda, const double* A_host, double* Q_host,
                      double* R_host, mrcqr_prec_t sketch_prec, int s, uint64_t seed);

/* Bytes of library-owned device workspace a factorization of this shape uses. */
size_t mrcqr_workspace_bytes(int64_t m, int n, int s, mrcqr_prec_t prec);

/* Detail of the last positive return code: 0-based pivot / diagonal index (codes 2, 3), else 0. */
int mrcqr_last_info(void);

/* Number of kernel launches enqueued by the last compute call (bench.py's gpu_launches). */
int mrcqr_last_launch_count(void);

/*
 * Per-kernel device timing of mrcqr_factor (CUDA events recorded on the call's stream between the
 * kernels; off by default).  mrcqr_last_timing fills 7 floats, milliseconds of the last
 * mrcqr_factor / mrcqr_factor_host call:  [0] K1 sampled transform (Alg.2 steps 2-4),  [1] K2 sketch QR
 * (steps 5-6),  [2] upload of the prepared R_s,  [3] K3 precondition + Gram (step 7, Alg.1 step 1; n > 128: the
 * first triangular solve, Y = A R_s^-1 into Q's buffer),  [4] reduction of the Gram partials (n > 128: the SYRK
 * G = Y^T Y and its reduction),  [5] K4 Cholesky + R = Rc Rs (Alg.1 step 2, Alg.2 step 9),  [6] K5 form Q
 * (Alg.1 step 3; n > 128: the second triangular solve, in place).
 */
int mrcqr_set_timing(int on);
int mrcqr_last_timing(float* ms_out_host);

/*
 * ||I - Q^T Q||_F of a column-major m x n Q (device), the quantity the paper monitors (Frobenius
 * instead of the 2-norm, R13).  Q^T Q is accumulated on the FP64 tensor cores in chains of 1024 rows with a
 * fixed-order reduction (a plain long accumulation adds ~1e-14 of its own at m = 2^20).  err_host: one double (host).
 * Returns 0 or -1 m, -2 n, -3 ldq, -4 Q, -5 err_host, 4.
 */
int mrcqr_orth_error(int64_t m, int n, int64_t ldq, const double* Q, double* err_host, void* stream);

/*
 * The same quantity for callers that must not allocate (stream capture, serving loops, harnesses that forbid
 * cudaMalloc): the kernels of mrcqr_orth_error in the same order (bit-identical result), their scratch (one Gram
 * partial per SYRK CTA, the 128 x 128 Gram matrix) in a static device array of 20 054 016 bytes (19.1 MiB) that every
 * GPU which loads the library holds until the process exits.  Limit: n <= MRCQR_NOALLOC_N_MAX, any m >= n; a larger n
 * (or a device with more than 151 SMs) returns MRCQR_ERR_TOO_LARGE before anything is launched.
 * err: ONE double, DEVICE (written by the last kernel).  G: nullable, DEVICE, n x n, ld n, receives Q^T Q (full
 * symmetric).  The call uses no context and no workspace, calls no cudaMalloc / cudaFree / allocating routine, copies
 * nothing to the host and does not synchronise: it enqueues 3 (4 with G) kernels on `stream` and returns; a failure of
 * a kernel on the device surfaces at the caller's next synchronisation.  Every call shares the array (it needs no
 * clearing: each call overwrites what it reads): calls that OVERLAP on the GPU race on it, serialise them.  The first
 * call on a device resolves the array's device address (cudaGetSymbolAddress, that device current).
 * Returns 0 or -1 m, -2 n < 1, -3 ldq, -4 Q, -5 err, MRCQR_ERR_CUDA, MRCQR_ERR_TOO_LARGE.
 */
#define MRCQR_NOALLOC_N_MAX 128
int mrcqr_orth_error_noalloc(int64_t m, int n, int64_t ldq, const double* Q, double* err, double* G, void* stream);

/*
 * Self-correcting MRCQR ("the remedy is to rerun MRCQR at the next higher precision level"):
 * factor with the sketch precision first_prec; if the factorization reports a positive code or
 * ||I - Q^T Q||_F > tol, rerun at the next precision (half -> single -> double).  tol <= 0 means 1e-13.
 * prec_used_host / orth_host (nullable, host): the precision of the returned (Q, R) and its measured
 * ||I - Q^T Q||_F (-1 if that run reported a positive code).  Returns 0; a negative argument index as
 * mrcqr_factor; or the outcome at FP64: codes 1-3, or MRCQR_ERR_NOT_ORTHOGONAL with the FP64 result in (Q, R).
 * Nothing is hidden: every escalation is visible through prec_used_host.
 */
int mrcqr_factor_auto(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R,
                      mrcqr_prec_t first_prec, int s, uint64_t seed, double tol,
                      int* prec_used_host, double* orth_host, void* stream);

/*
 * Algorithm 1, CholQR, on A itself: G = A^T A, G = R^T R, Q = A R^-1, with the stage-2/3 kernels
 * of MRCQR (R_s = I).  passes = 2: CholQR2: Algorithm 1 again on Q, R = R2 R1.  Breaks down
 * (MRCQR_ERR_BREAKDOWN) once kappa(A)^2 u >~ 1, i.e. kappa >~ 1e8; loses orthogonality as kappa^2 u
 * before that (one pass).  m need not be a power of two.  Returns 0, -1 m, -2 n, -3 lda, -4 A, -5 Q, -6 R, -7 passes, 3, 4.
 */
int mrcqr_cholqr(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R, int passes, void* stream);

/*
 * CholQR probe for the conditioning regime (eq. (2)): one CholQR of A into the caller's work
 * buffers Qwork (m x n, ld = lda) and Rwork (n x n), q = ||I - Q^T Q||_F / sqrt(n) (a lower bound of the 2-norm the
 * paper uses), kappa_lb = sqrt(q / (u (1 + q))) <= kappa_2(A), u = 2^-53.  A CholQR breakdown means kappa >~ u^-1/2:
 * kappa_lb = 2^26.5.  prec_host (nullable): the paper's rule applied to the bound: 16 if
 * kappa_lb < 1e4, 32 if < 1e8, else 64 -- a LOWER bound, so the suggestion may be too low; mrcqr_factor_auto
 * corrects that.  Returns 0, a negative argument index (as mrcqr_cholqr; -7 kappa_lb_host) or 4.
 */
int mrcqr_kappa_probe(int64_t m, int n, int64_t lda, const double* A, double* Qwork, double* Rwork,
                      double* kappa_lb_host, int* prec_host, void* stream);

/*
 * Form of stage 2 for n16 <= 128 (n16 = n rounded up to 16) in mrcqr_factor / mrcqr_factor_host:
 *   fused    stage 2a keeps Y = A R_s^-1 on chip and stage 2b recomputes it bit-identically (north_star's form:
 *            4 passes over m x n, 4 m n^2 flops, Y never written);
 *   stored   stage 2a writes Y into Q's buffer and stage 2b solves it in place against R_c (5 passes, 3 m n^2 flops:
 *            the paper's own TrsmPre / TrsmFin order).  Below n16 = 128 (and for operands that are
 *            not 16-byte aligned or m not a multiple of 32) the Gram matrix is still accumulated on chip beside the
 *            write, and Q, R are bit-identical to the fused form's; at n16 = 128 the kernels of the n > 128 path run
 *            (panel solve, Gram of the stored Y, panel solve), same tolerances, a differently ordered Gram sum.
 * mode < 0 (default): the faster one as measured on B200: fused for n16 <= 32, where HBM binds;
 * stored from n16 = 48 on, where the FP64 pipe binds (m = 2^21: n = 64 1.79 vs 1.69 ms, n = 128 6.69 vs 5.09 ms).
 * mode 0: always fused; mode > 0: always stored.  For n16 > 128 Y is always stored (the Gram matrix no longer fits one
 * SM).  Returns 0.  mrcqr_last_used_store_y: 1 if the last mrcqr_factor of this context stored Y, else 0.
 */
int mrcqr_set_store_y(int mode);
int mrcqr_last_used_store_y(void);

/*
 * Variant switch of the sketch (SURVEY.md 8(f)3 iii; "retain both real and imaginary parts,
 * yielding a 2c x n sketch at no extra FFT cost but doubling the sketch QR cost" -- measured by the authors,
 * who kept Re-only).  On, every call that sketches (mrcqr_sketch, mrcqr_factor, mrcqr_factor_host,
 * mrcqr_factor_auto) forms the 2s x n matrix  [ sqrt(s/m) Re X[S] ; sqrt(s/m) Im X[S] ]  (reading R11: Re rows
 * first, same scale) in the FFT form of K1 and QR-factors that; the As argument of mrcqr_sketch then receives
 * 2s x n values (column-major, ld = 2s).  Requires 2s <= 4096 (else the s argument is reported invalid).
 * Off (default): Algorithm 2 as printed.  Returns 0.
 */
int mrcqr_set_sketch_reim(int on);

/*
 * Repeated-call mode (block Arnoldi, randomized-SVD power iteration, time stepping): on, the
 * kernels, copies and the status read-back of mrcqr_factor are captured ONCE into a CUDA graph per (m, n, lda, A, Q, R,
 * precision, s) and replayed by later calls with the same arguments; the seed and the drawn bins are data of the graph
 * (read from pinned host memory at replay), so they may change from call to call.  Same results bit for bit.  Per-kernel
 * timing (mrcqr_set_timing) takes the ordinary path.  Stream capture is not permitted on the legacy default stream
 * (stream = NULL): such calls take the ordinary path; mrcqr_last_used_graph() tells which one ran.  Returns 0.
 */
int mrcqr_set_graph(int on);

/*
 * Calls in flight (repeated-call mode: the QR inside a block-Arnoldi or power-iteration loop, whose
 * caller does not need the status of one factorization before it enqueues the next).  mrcqr_factor_async takes the
 * arguments of mrcqr_factor (device pointers, same layouts, same checks), enqueues Algorithm 2 on `stream` and returns
 * WITHOUT synchronising: 0 = enqueued, < 0 = argument -rc invalid, MRCQR_ERR_CUDA.  Nothing is allocated once the
 * context's workspace fits the shape and its ring of 8 pinned bin buffers fits s.  Q and R are ready when the work
 * enqueued on `stream` has run.  Same kernels, same results bit for bit as mrcqr_factor.
 * The run-time status (MRCQR_ERR_OVERFLOW / _SINGULAR / _BREAKDOWN and its column) is NOT returned per call: the
 * device status block keeps the FIRST error of the calls in flight, and the later calls still run in full.
 * mrcqr_wait synchronises the stream of the pending calls, returns that status (0 if every call was clean), writes its
 * column to *info_host (may be NULL; also mrcqr_last_info) and clears it; with nothing pending it returns 0 at once.
 * All calls between two waits share the context's workspace and must use ONE stream (a call on another stream, or one
 * whose workspace must grow, first waits for the pending ones and carries their status over).  Call mrcqr_wait before
 * any other entry point of the same context: a synchronous entry point drains the pending calls and DROPS their status.
 * mrcqr_set_timing / mrcqr_set_graph do not apply to these calls.
 */
int mrcqr_factor_async(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R,
                       mrcqr_prec_t sketch_prec, int s, uint64_t seed, void* stream);
int mrcqr_wait(int* info_host);

/* 1 if the last mrcqr_factor / mrcqr_factor_host call replayed (or captured and replayed) a CUDA graph, else 0. */
int mrcqr_last_used_graph(void);

/*
 * Test hook for the "bit-identical Y" requirement: runs the stage-2a and the stage-2b
 * tile solves and dumps the Y = A R_s^-1 each of them computed (m x n, ld = m).  The two dumps
 * must be equal bit for bit.
 */
int mrcqr_debug_dump_y(int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                       double* Y_stage2a, double* Y_stage2b, void* stream);

/* Frees everything the current context owns (workspace, staging buffers, graph); the context stays usable. */
void mrcqr_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* MRCQR_H */
