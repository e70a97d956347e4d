/*
 * mrcqr_oracle.c -- CPU ORACLE for MRCQR (arxiv/paper_2606_18411), IEEE double throughout.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant with paper_2606_18411_b200/csrc (the CUDA path) and neither
 * imports the other.
 *
 * It is a plain, slow, step-by-step restatement of the paper's Algorithm 2 and
 * Algorithm 1 in the paper's order.  No blocking, fusion or reordering beyond
 * what DESIGN.md "Readings of the paper" lists (the one deliberate choice is the summation tree
 * of the Gram matrix, reading R7).  OpenMP is used only over independent columns / rows /
 * fixed-shape tree leaves, so results do not depend on the thread count.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): every function below is pinned to something
 * other than itself -- see the "pin:" line in each header comment.  Nothing here is
 * "parity unpinned".
 *
 * All matrices are column-major.  Build: see oracle/build.py (gcc -O2 -fopenmp, no fast-math).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------------
 * o1. Random draw (Algorithm 2 step 1).  The paper does not name a generator;
 * BASELINE.json's configs fix "a splitmix64 stream".  Reading R1: X(k) is the k-th
 * output (k = 0,1,...) of splitmix64 seeded with `seed`; counter-based: state_k = seed+(k+1)*gamma.
 * pin: published splitmix64 test vector (seed 1234567) + a pure-Python big-int re-implementation.
 * ------------------------------------------------------------------------------------------ */
uint64_t orc_splitmix64_at(uint64_t seed, uint64_t k)
{
    uint64_t z = seed + (k + 1u) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static int cmp_i64(const void *a, const void *b)
{
    int64_t x = *(const int64_t *)a, y = *(const int64_t *)b;
    return (x > y) - (x < y);
}

/* Signs: d_t = -1 iff bit (t mod 64) of X(floor(t/64)) is 1; signs[] holds ceil(m/64) words.
 * Bins: S is a set of s DISTINCT 0-based bins in [0, floor(m/2)] (PAPER.md:94 prints the 1-based
 * range {1..floor(m/2)+1}).  Candidates floor(X(k)*B / 2^64), B = floor(m/2)+1, for
 * k = ceil(m/64), ceil(m/64)+1, ...; a candidate is kept if new; stop at s kept; sort ascending.
 * Returns 0, or -1 if s is out of range. */
int orc_draw(int64_t m, int s, uint64_t seed, uint64_t *signs, int64_t *idx)
{
    int64_t nw = (m + 63) / 64, B = m / 2 + 1;
    if (s < 0 || (int64_t)s > B) return -1;
    for (int64_t w = 0; w < nw; ++w) signs[w] = orc_splitmix64_at(seed, (uint64_t)w);
    int kept = 0;
    for (uint64_t k = (uint64_t)nw; kept < s; ++k) {
        unsigned __int128 p = (unsigned __int128)orc_splitmix64_at(seed, k) * (unsigned __int128)(uint64_t)B;
        int64_t cand = (int64_t)(uint64_t)(p >> 64);
        int dup = 0;
        for (int i = 0; i < kept; ++i) if (idx[i] == cand) { dup = 1; break; }
        if (!dup) idx[kept++] = cand;
    }
    qsort(idx, (size_t)s, sizeof(int64_t), cmp_i64);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * o3. Unnormalised complex DFT of length m = 2^k, X_k = sum_t x_t exp(-2 pi i k t / m)
 * (Algorithm 2 step 3 "column-wise real-to-complex FFT").  Textbook iterative
 * radix-2 decimation-in-time: bit-reversal permutation, then log2(m) butterfly passes.  Every
 * twiddle is evaluated directly as cos/sin(-2 pi j / len) (no recurrence).
 * pin: O(m^2) direct sum written in the tests, numpy.fft (test-only), closed forms, Parseval.
 * ------------------------------------------------------------------------------------------ */
void orc_fft_radix2(int64_t m, double *re, double *im)
{
    for (int64_t i = 1, j = 0; i < m; ++i) {           /* bit reversal */
        int64_t bit = m >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double t = re[i]; re[i] = re[j]; re[j] = t;
            t = im[i]; im[i] = im[j]; im[j] = t;
        }
    }
    for (int64_t len = 2; len <= m; len <<= 1) {
        int64_t half = len >> 1;
        for (int64_t j = 0; j < half; ++j) {
            double ang = -2.0 * ORC_PI * (double)j / (double)len;
            double wr = cos(ang), wi = sin(ang);
            for (int64_t b = 0; b < m; b += len) {
                int64_t u = b + j, v = u + half;
                double tr = re[v] * wr - im[v] * wi;
                double ti = re[v] * wi + im[v] * wr;
                re[v] = re[u] - tr; im[v] = im[u] - ti;
                re[u] = re[u] + tr; im[u] = im[u] + ti;
            }
        }
    }
}

static int is_pow2(int64_t m) { return m > 0 && (m & (m - 1)) == 0; }

static inline double sign_of(const uint64_t *signs, int64_t t)
{
    return ((signs[t >> 6] >> (t & 63)) & 1u) ? -1.0 : 1.0;
}

/* ------------------------------------------------------------------------------------------
 * o2-o4. Sketch A_s = sqrt(s/m) * Re(FFT(D A))[S,:]  (Algorithm 2 steps 2-4).
 * x~ = d .* a_j exactly in double: the oracle does NOT round to the sketch precision p; the
 * precision-p GPU sketch is compared with this within north_star's tolerances (reading R5).
 * m = 2^k: FFT of each column then gather.  Other m: the defining sum
 * Re X_k = sum_t x~_t cos(2 pi k t / m), with the angle reduced as (k t mod m) in integers.
 * As is s x n column-major, ld = s.  Returns 0.
 * pin: brute-force cosine sum in tests, impulse / pure-cosine / constant closed forms.
 * ------------------------------------------------------------------------------------------ */
int orc_sketch(int64_t m, int n, int64_t lda, const double *A, const uint64_t *signs,
               int s, const int64_t *idx, double *As)
{
    const double scale = sqrt((double)s / (double)m);
    if (is_pow2(m)) {
        #pragma omp parallel
        {
            double *re = (double *)malloc(sizeof(double) * (size_t)m);
            double *im = (double *)malloc(sizeof(double) * (size_t)m);
            #pragma omp for schedule(dynamic, 1)
            for (int j = 0; j < n; ++j) {
                const double *a = A + (size_t)j * (size_t)lda;
                for (int64_t t = 0; t < m; ++t) { re[t] = sign_of(signs, t) * a[t]; im[t] = 0.0; }
                orc_fft_radix2(m, re, im);
                for (int i = 0; i < s; ++i) As[(size_t)j * s + i] = scale * re[idx[i]];
            }
            free(re); free(im);
        }
    } else {
        #pragma omp parallel for collapse(2) schedule(static)
        for (int j = 0; j < n; ++j)
            for (int i = 0; i < s; ++i) {
                const double *a = A + (size_t)j * (size_t)lda;
                double acc = 0.0;
                for (int64_t t = 0; t < m; ++t) {
                    int64_t r = (int64_t)(((unsigned __int128)idx[i] * (unsigned __int128)t) % (unsigned __int128)m);
                    acc += sign_of(signs, t) * a[t] * cos(2.0 * ORC_PI * (double)r / (double)m);
                }
                As[(size_t)j * s + i] = scale * acc;
            }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * o4'. Re+Im variant of the sketch ("retain both real and imaginary parts, yielding a
 * 2c x n sketch at no extra FFT cost but doubling the sketch QR cost"; the authors measured it and
 * kept Re-only).  With X = FFT(D a_j), X_k = sum_t x~_t exp(-2 pi i k t / m):
 *   As[i, j]     = sqrt(s/m) * Re X[k_i],   As[s + i, j] = sqrt(s/m) * Im X[k_i],   i < s.
 * Reading R11: the paper gives neither the row order nor a scale for this variant; the
 * Re rows keep their place and scale, the Im rows follow (a common factor only scales R_s).
 * As is 2s x n column-major, ld = 2s.  Returns 0.
 * pin: brute-force sine sum, pure-sine closed form, Im = 0 at DC / Nyquist, Re rows equal o2-o4.
 * ------------------------------------------------------------------------------------------ */
int orc_sketch_reim(int64_t m, int n, int64_t lda, const double *A, const uint64_t *signs,
                    int s, const int64_t *idx, double *As)
{
    const double scale = sqrt((double)s / (double)m);
    const size_t ld = 2 * (size_t)s;
    if (is_pow2(m)) {
        #pragma omp parallel
        {
            double *re = (double *)malloc(sizeof(double) * (size_t)m);
            double *im = (double *)malloc(sizeof(double) * (size_t)m);
            #pragma omp for schedule(dynamic, 1)
            for (int j = 0; j < n; ++j) {
                const double *a = A + (size_t)j * (size_t)lda;
                for (int64_t t = 0; t < m; ++t) { re[t] = sign_of(signs, t) * a[t]; im[t] = 0.0; }
                orc_fft_radix2(m, re, im);
                for (int i = 0; i < s; ++i) {
                    As[(size_t)j * ld + i] = scale * re[idx[i]];
                    As[(size_t)j * ld + s + i] = scale * im[idx[i]];
                }
            }
            free(re); free(im);
        }
    } else {
        #pragma omp parallel for collapse(2) schedule(static)
        for (int j = 0; j < n; ++j)
            for (int i = 0; i < s; ++i) {
                const double *a = A + (size_t)j * (size_t)lda;
                double accr = 0.0, acci = 0.0;
                for (int64_t t = 0; t < m; ++t) {
                    int64_t r = (int64_t)(((unsigned __int128)idx[i] * (unsigned __int128)t) % (unsigned __int128)m);
                    const double x = sign_of(signs, t) * a[t], th = 2.0 * ORC_PI * (double)r / (double)m;
                    accr += x * cos(th);
                    acci -= x * sin(th);
                }
                As[(size_t)j * ld + i] = scale * accr;
                As[(size_t)j * ld + s + i] = scale * acci;
            }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * o5. R-factor of the Householder QR of the s x n sketch (Algorithm 2 step 5), then
 * rows negated so that diag(R_s) > 0 (reading R6: the paper is silent; positive diagonals make
 * (Q,R) unique as north_star requires).  Unblocked textbook Householder (Golub & Van Loan
 * Alg. 5.2.1 / LAPACK dgeqr2 convention): for column j, x = W[j:s, j],
 *   beta = -sign(x_0) ||x||_2,  v = x - beta e_1 (normalised v_0 = 1),  tau = (beta - x_0)/beta,
 *   W[j:s, j+1:n] -= tau v (v^T W[j:s, j+1:n]).
 * ||x|| uses a scaled sum of squares (no overflow/underflow).  Rs: n x n col-major, ld = n,
 * strictly-lower part zero.  Returns 0, or j+1 if R_s[j,j] is zero or non-finite.
 * pin: R^T R = As^T As, numpy.linalg.qr (test-only), n = 1 closed form, Gram-Schmidt on tiny input.
 * ------------------------------------------------------------------------------------------ */
static double scaled_norm2(int64_t len, const double *x)
{
    double scale = 0.0, ssq = 1.0;
    for (int64_t i = 0; i < len; ++i) {
        double ax = fabs(x[i]);
        if (ax > 0.0) {
            if (scale < ax) { ssq = 1.0 + ssq * (scale / ax) * (scale / ax); scale = ax; }
            else            { ssq += (ax / scale) * (ax / scale); }
        }
    }
    return scale * sqrt(ssq);
}

int orc_householder_r(int s, int n, const double *As, double *Rs)
{
    double *W = (double *)malloc(sizeof(double) * (size_t)s * (size_t)n);
    memcpy(W, As, sizeof(double) * (size_t)s * (size_t)n);
    int info = 0;
    for (int j = 0; j < n && j < s; ++j) {
        double *x = W + (size_t)j * s + j;
        int64_t len = s - j;
        double alpha = x[0];
        double xnorm = scaled_norm2(len - 1, x + 1);
        if (xnorm == 0.0) continue;                      /* H = I, R[j,j] = alpha */
        double nrm = scaled_norm2(len, x);
        double beta = (alpha >= 0.0) ? -nrm : nrm;
        double tau = (beta - alpha) / beta;
        double inv = 1.0 / (alpha - beta);
        for (int64_t i = 1; i < len; ++i) x[i] *= inv;   /* v, with v_0 = 1 implied */
        x[0] = beta;
        #pragma omp parallel for schedule(static) if ((int64_t)(n - j) * len > 65536)
        for (int c = j + 1; c < n; ++c) {
            double *y = W + (size_t)c * s + j;
            double w = y[0];
            for (int64_t i = 1; i < len; ++i) w += x[i] * y[i];
            w *= tau;
            y[0] -= w;
            for (int64_t i = 1; i < len; ++i) y[i] -= w * x[i];
        }
    }
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i)
            Rs[(size_t)j * n + i] = (i <= j && i < s) ? W[(size_t)j * s + i] : 0.0;
    for (int i = 0; i < n; ++i) {
        double d = Rs[(size_t)i * n + i];
        if (!(fabs(d) > 0.0) || !isfinite(d)) { if (!info) info = i + 1; continue; }
        if (d < 0.0) for (int j = i; j < n; ++j) Rs[(size_t)j * n + i] = -Rs[(size_t)j * n + i];
    }
    free(W);
    return info;
}

/* ------------------------------------------------------------------------------------------
 * o6 / o9. Row-wise triangular solve Y = A R^{-1}, R upper (Algorithm 2 step 7 "A_1 <- A R_s^-1",
 * PAPER.md:103, and Algorithm 1 step 3 "Q <- A R^-1").  For each row a (1 x n):
 *   y_j = (a_j - sum_{k<j} y_k R[k,j]) / R[j,j],  j ascending, true division.
 * R^{-1} is never formed.  Y may alias A (in place).  R: n x n col-major ld = n.
 * pin: residual ||Y R - A||, R = I, diagonal R, 2x2 worked by hand, scipy solve_triangular.
 * ------------------------------------------------------------------------------------------ */
void orc_row_solve(int64_t m, int n, int64_t lda, const double *A, const double *R,
                   int64_t ldy, double *Y)
{
    #pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < m; ++r) {
        for (int j = 0; j < n; ++j) {
            double t = A[(size_t)j * (size_t)lda + r];
            for (int k = 0; k < j; ++k) t -= Y[(size_t)k * (size_t)ldy + r] * R[(size_t)j * n + k];
            Y[(size_t)j * (size_t)ldy + r] = t / R[(size_t)j * n + j];
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * o7. Gram matrix G = Y^T Y (Algorithm 1 step 1).  The definition is a sum over the
 * m rows; reading R7 fixes the summation tree: leaves of 256 consecutive rows summed in row
 * order, leaves combined by a balanced binary tree over the leaf index (split at the midpoint).
 * A single chain of m additions loses the 1e-13 orthogonality bar at m = 2^18..2^21 (SURVEY.md
 * appendix), a tree does not.  Full symmetric n x n is returned (ld = n).
 * pin: exact on integer-valued Y (any order gives the same integers), long-double reference,
 *      numpy Y.T@Y (test-only).
 * ------------------------------------------------------------------------------------------ */
#define ORC_GRAM_LEAF 256

static void gram_leaf(int64_t r0, int64_t r1, int n, int64_t ldy, const double *Y, double *G)
{
    for (int j = 0; j < n; ++j)
        for (int i = 0; i <= j; ++i) {
            const double *yi = Y + (size_t)i * (size_t)ldy, *yj = Y + (size_t)j * (size_t)ldy;
            double acc = 0.0;
            for (int64_t r = r0; r < r1; ++r) acc += yi[r] * yj[r];
            G[(size_t)j * n + i] = acc;
        }
}

/* sums leaves [l0, l1) into G (upper triangle); tmp is scratch of n*n doubles per level */
static void gram_tree(int64_t l0, int64_t l1, int64_t m, int n, int64_t ldy, const double *Y, double *G)
{
    if (l1 - l0 == 1) {
        int64_t r0 = l0 * ORC_GRAM_LEAF, r1 = r0 + ORC_GRAM_LEAF;
        if (r1 > m) r1 = m;
        gram_leaf(r0, r1, n, ldy, Y, G);
        return;
    }
    int64_t mid = l0 + (l1 - l0) / 2;
    double *T = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    int par = (l1 - l0) >= 64;                 /* independent subtrees: safe to run as tasks */
    #pragma omp task if (par)
    gram_tree(l0, mid, m, n, ldy, Y, G);
    #pragma omp task if (par)
    gram_tree(mid, l1, m, n, ldy, Y, T);
    #pragma omp taskwait
    for (int j = 0; j < n; ++j)
        for (int i = 0; i <= j; ++i) G[(size_t)j * n + i] += T[(size_t)j * n + i];
    free(T);
}

void orc_gram(int64_t m, int n, int64_t ldy, const double *Y, double *G)
{
    int64_t leaves = (m + ORC_GRAM_LEAF - 1) / ORC_GRAM_LEAF;
    if (leaves < 1) leaves = 1;
    #pragma omp parallel
    #pragma omp single
    gram_tree(0, leaves, m, n, ldy, Y, G);
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < j; ++i) G[(size_t)i * n + j] = G[(size_t)j * n + i];
}

/* ------------------------------------------------------------------------------------------
 * o8. Cholesky G = Rc^T Rc, Rc upper with positive diagonal (Algorithm 1 step 2).
 * Textbook Cholesky-Crout by columns.  "Breakdown": a pivot that is <= 0 or
 * not finite is reported, never hidden: returns j+1 for the first such pivot j (Rc then
 * unspecified), 0 on success.  Only the upper triangle of G is read.
 * pin: Rc^T Rc = G, a 3x3 worked by hand, non-PD input -> reported index, numpy cholesky.
 * ------------------------------------------------------------------------------------------ */
int orc_cholesky_upper(int n, const double *G, double *Rc)
{
    memset(Rc, 0, sizeof(double) * (size_t)n * (size_t)n);
    for (int j = 0; j < n; ++j) {
        for (int i = 0; i <= j; ++i) {
            double t = G[(size_t)j * n + i];
            for (int k = 0; k < i; ++k) t -= Rc[(size_t)i * n + k] * Rc[(size_t)j * n + k];
            if (i < j) Rc[(size_t)j * n + i] = t / Rc[(size_t)i * n + i];
            else {
                if (!(t > 0.0) || !isfinite(t)) return j + 1;
                Rc[(size_t)j * n + j] = sqrt(t);
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * o10. R = Rc * Rs, both upper triangular (Algorithm 2 step 9 "R <- R_2 R_s"):
 * R[i,j] = sum_{k=i..j} Rc[i,k] Rs[k,j]; strictly-lower part zero.
 * pin: numpy matmul of the two triangles (test-only), diag(R) = diag(Rc) diag(Rs).
 * ------------------------------------------------------------------------------------------ */
void orc_triu_mul(int n, const double *Rc, const double *Rs, double *R)
{
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            double acc = 0.0;
            if (i <= j) for (int k = i; k <= j; ++k) acc += Rc[(size_t)k * n + i] * Rs[(size_t)j * n + k];
            R[(size_t)j * n + i] = acc;
        }
}

/* ------------------------------------------------------------------------------------------
 * Whole Algorithm 2 from a given draw: steps 2-9 in order.
 * Optional outputs (NULL to skip): As (s x n), Rs, G, Rc (n x n).  Q: m x n, ldq.  R: n x n.
 * Q is used as the store of A_1 = A Rs^-1 between steps 7 and 8 and solved in place (the paper's
 * own TrsmPre / TrsmFin structure).
 * Returns 0 ok, 2 = singular/non-finite R_s (+ index in *info), 3 = Cholesky breakdown (+ index).
 * pin: invariants Q^T Q = I, A = QR, R upper with diag > 0, kappa(A Rs^-1) = O(1); recovery of a
 *      planted (Q0, R0); n = 1 closed form.
 * ------------------------------------------------------------------------------------------ */
int orc_factor_from_draw(int64_t m, int n, int64_t lda, const double *A,
                         const uint64_t *signs, int s, const int64_t *idx,
                         int64_t ldq, double *Q, double *R,
                         double *As_out, double *Rs_out, double *G_out, double *Rc_out, int *info)
{
    size_t nn = (size_t)n * (size_t)n;
    double *As = (double *)malloc(sizeof(double) * (size_t)s * (size_t)n);
    double *Rs = (double *)malloc(sizeof(double) * nn);
    double *G  = (double *)malloc(sizeof(double) * nn);
    double *Rc = (double *)malloc(sizeof(double) * nn);
    int rc = 0, inf = 0;
    orc_sketch(m, n, lda, A, signs, s, idx, As);                 /* steps 2-4 */
    inf = orc_householder_r(s, n, As, Rs);                        /* steps 5-6 */
    if (As_out) memcpy(As_out, As, sizeof(double) * (size_t)s * (size_t)n);
    if (Rs_out) memcpy(Rs_out, Rs, sizeof(double) * nn);
    if (inf) { rc = 2; goto done; }
    orc_row_solve(m, n, lda, A, Rs, ldq, Q);                      /* step 7: A_1 (kept in Q) */
    orc_gram(m, n, ldq, Q, G);                                    /* Alg.1 step 1 */
    if (G_out) memcpy(G_out, G, sizeof(double) * nn);
    inf = orc_cholesky_upper(n, G, Rc);                           /* Alg.1 step 2 */
    if (inf) { rc = 3; goto done; }
    if (Rc_out) memcpy(Rc_out, Rc, sizeof(double) * nn);
    orc_row_solve(m, n, ldq, Q, Rc, ldq, Q);                      /* Alg.1 step 3 */
    orc_triu_mul(n, Rc, Rs, R);                                   /* step 9 */
done:
    if (info) *info = inf;
    free(As); free(Rs); free(G); free(Rc);
    return rc;
}

int orc_factor(int64_t m, int n, int64_t lda, const double *A, int64_t ldq, double *Q, double *R,
               int s, uint64_t seed, int *info)
{
    uint64_t *signs = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)((m + 63) / 64));
    int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * (size_t)(s > 0 ? s : 1));
    int rc = orc_draw(m, s, seed, signs, idx);
    if (rc == 0) rc = orc_factor_from_draw(m, n, lda, A, signs, s, idx, ldq, Q, R, 0, 0, 0, 0, info);
    free(signs); free(idx);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Checkers for the invariants of PAPER.md:31-35 / eq.(1) in the Frobenius norm
 * (BASELINE.json).  Sums over the m rows use the same leaf-256 + binary-tree shape as o7 so the
 * checker's own rounding (about 1e-14 for a plain chain at m = 2^20) stays
 * below what it measures.
 * pin: exactly orthonormal columns built from signed unit vectors -> 0; planted perturbation.
 * ------------------------------------------------------------------------------------------ */
double orc_orth_error_fro(int64_t m, int n, int64_t ldq, const double *Q)
{
    double *G = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    orc_gram(m, n, ldq, Q, G);
    double acc = 0.0;
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            double d = G[(size_t)j * n + i] - (i == j ? 1.0 : 0.0);
            acc += d * d;
        }
    free(G);
    return sqrt(acc);
}

/* ||A - Q R||_F / ||A||_F ; each entry of QR is a short (<= n terms) dot product; the squared
 * norms are accumulated per row block of 256 and then over a binary tree via long double. */
double orc_residual_fro(int64_t m, int n, int64_t lda, const double *A, int64_t ldq,
                        const double *Q, const double *R)
{
    int64_t leaves = (m + ORC_GRAM_LEAF - 1) / ORC_GRAM_LEAF;
    long double *num = (long double *)calloc((size_t)leaves, sizeof(long double));
    long double *den = (long double *)calloc((size_t)leaves, sizeof(long double));
    #pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < leaves; ++l) {
        int64_t r0 = l * ORC_GRAM_LEAF, r1 = r0 + ORC_GRAM_LEAF;
        if (r1 > m) r1 = m;
        long double sn = 0.0L, sd = 0.0L;
        for (int64_t r = r0; r < r1; ++r)
            for (int j = 0; j < n; ++j) {
                long double qr = 0.0L;
                for (int k = 0; k <= j; ++k)
                    qr += (long double)Q[(size_t)k * (size_t)ldq + r] * (long double)R[(size_t)j * n + k];
                long double a = (long double)A[(size_t)j * (size_t)lda + r];
                sn += (a - qr) * (a - qr);
                sd += a * a;
            }
        num[l] = sn; den[l] = sd;
    }
    for (int64_t w = 1; w < leaves; w <<= 1)
        for (int64_t l = 0; l + w < leaves; l += 2 * w) { num[l] += num[l + w]; den[l] += den[l + w]; }
    double out = (double)sqrtl(num[0] / den[0]);
    free(num); free(den);
    return out;
}

int orc_num_threads(void)
{
    int nt = 1;
#ifdef _OPENMP
    #pragma omp parallel
    {
        #pragma omp master
        nt = omp_get_num_threads();
    }
#endif
    return nt;
}
