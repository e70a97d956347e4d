// mrcqr_internal.cuh -- shared declarations of the CUDA path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstddef>

namespace mrcqr {

// device status block (8 ints): [0] = first error code, [1] = info (pivot index), rest scratch
struct Status { int code; int info; int pad[6]; };

__device__ __forceinline__ void report(Status* st, int code, int info)
{
    if (atomicCAS(&st->code, 0, code) == 0) st->info = info;
}

inline int round_up(int x, int q) { return (x + q - 1) / q * q; }

// splitmix64, counter form: X(k) = mix(seed + (k+1) * gamma), the stream of the draw (reading R1)
__host__ __device__ __forceinline__ uint64_t splitmix64_at(uint64_t seed, uint64_t k)
{
    uint64_t z = seed + (k + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// ---- slab geometry of the row-streaming kernels (K3 / K5), chosen from n only -----------------
// n16 = n padded to a multiple of 16 (8-wide DMMA blocks in pairs).  A warp owns a slab of 8*RG rows,
// a CTA NW slabs; slab = n16 x (8*RG + 4) doubles of shared memory.
struct RowCfg { int n16; int RG; int NW; int smem_bytes; };
RowCfg row_config(int n);

// "prepared" upper-triangular factor consumed by the slab solve (n16 x n16 doubles reserved), nB = n16/8:
//   [0, 64 * nB(nB-1)/2)   off-diagonal 8x8 blocks (K < J) in DMMA B-fragment order, pair index
//                          J(J-1)/2 + K, 32 lanes x (k = t, k = t + 4) of -R   (see rows.cuh)
//   [.., + 36 * nB)        diagonal blocks: 8 reciprocals 1/R[j,j], then 28 values -R[j,jj]/R[jj,jj], j < jj
// padding rows / columns (>= n) are the identity.  Built once per factor by prep_R (R_s) and by the
// Cholesky kernel (R_c); K3 and K5 read the same buffer (bit-identical Y).  The diagonal part is also
// copied to constant memory (upload_diag) before the row kernels run.
constexpr int PREP_DIAG = 36;
constexpr int PREP_MAX_NB = 64;
__host__ __device__ inline size_t prep_diag_offset(int nB) { return (size_t)32 * nB * (nB - 1); }
// value of prepared element o (0 <= o < prep_diag_offset + 36 nB) from R (n x n, element (i,j) = R[j*ldr+i]);
// *zero_diag is set when a diagonal entry is 0 / non-finite
__device__ __forceinline__ double prep_value(const double* R, int ldr, int n, int nB, size_t o, int* bad_col)
{
    const size_t doff = prep_diag_offset(nB);
    if (o < doff) {
        const int pair = (int)(o >> 6), w = (int)(o & 63), lane = w >> 1, h = w & 1;
        int J = 1;
        while ((J + 1) * J / 2 <= pair) ++J;
        const int K = pair - J * (J - 1) / 2;
        const int g = lane >> 2, t = lane & 3;
        const int row = 8 * K + t + 4 * h, col = 8 * J + (g >> 1) + 4 * (g & 1);
        return (row < n && col < n) ? -R[(size_t)col * ldr + row] : 0.0;
    }
    const int e = (int)(o - doff), J = e / PREP_DIAG, i = e % PREP_DIAG;
    if (i < 8) {
        const int j = 8 * J + i;
        if (j >= n) return 1.0;
        const double d = R[(size_t)j * ldr + j];
        if (!(fabs(d) > 0.0) || isinf(d)) *bad_col = j;
        return 1.0 / d;
    }
    int j = 0, rem = i - 8;
    while (rem >= 7 - j) { rem -= 7 - j; ++j; }
    const int row = 8 * J + j, col = 8 * J + j + 1 + rem;
    return (row < n && col < n) ? -R[(size_t)col * ldr + row] / R[(size_t)col * ldr + col] : 0.0;
}

// 1/sqrt(x) and 1/x for a positive, finite, normal double: hardware seed + two Newton steps (a few ulp).  They sit on
// the serial chain of every Cholesky pivot and every Householder reflector, where the correctly rounded sqrt / division
// routines cost 150-250 cycles each.
__device__ __forceinline__ double rsqrt_fast(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double h = 0.5 * x;
    y = y * fma(-h * y, y, 1.5);
    y = y * fma(-h * y, y, 1.5);
    return y;
}
__device__ __forceinline__ double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    y = fma(y, fma(-x, y, 1.0), y);
    y = fma(y, fma(-x, y, 1.0), y);
    return y;
}
// Householder coefficients of a column with pivot alpha and sigma = sum of squares below it (sigma > 0):
// beta = -sign(alpha) sqrt(alpha^2 + sigma), c = 1 / (beta (beta - alpha)).  Falls back to the exact routines outside the
// range where the approximations are safe.
__device__ __forceinline__ void householder_coeffs(double alpha, double sigma, double& beta, double& c)
{
    const double x = fma(alpha, alpha, sigma);
    double nrm;
    if (x > 1e-280 && x < 1e280) nrm = x * rsqrt_fast(x); else nrm = sqrt(x);
    beta = (alpha >= 0.0) ? -nrm : nrm;
    const double d = beta * (beta - alpha);
    c = (d > 1e-280 && d < 1e280) ? rcp_fast(d) : 1.0 / d;
}

// The whole prepared factor written by one CTA (same values as prep_value element by element): a warp takes an
// off-diagonal pair (K, J) at a time, so the pair index is decoded once per 64 elements, not once per element.
// *bad_col: a column with a zero / non-finite diagonal, or left untouched.
__device__ __forceinline__ void prep_cta(const double* R, int ldr, int n, int nB, double* out, int* bad_col)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int npair = nB * (nB - 1) / 2;
    int J = 1, base = 0;                                   // base = J (J - 1) / 2
    for (int pair = warp; pair < npair; pair += nwarp) {
        while (base + J <= pair) { base += J; ++J; }
        const int K = pair - base;
        const int col = 8 * J + (g >> 1) + 4 * (g & 1), r0 = 8 * K + t, r1 = r0 + 4;
        double2 v;
        v.x = (r0 < n && col < n) ? -R[(size_t)col * ldr + r0] : 0.0;
        v.y = (r1 < n && col < n) ? -R[(size_t)col * ldr + r1] : 0.0;
        *reinterpret_cast<double2*>(out + (size_t)pair * 64 + 2 * lane) = v;
    }
    const size_t doff = prep_diag_offset(nB);
    for (int e = threadIdx.x; e < PREP_DIAG * nB; e += blockDim.x) out[doff + e] = prep_value(R, ldr, n, nB, doff + e, bad_col);
}

// launchers (each returns the number of kernel launches it enqueued)
int launch_prep_R(const double* R, int n, double* Rprep, int n16, Status* st, int err_code, cudaStream_t s);
int upload_diag(const double* prep, int n16, int fac, cudaStream_t s);      // prepared diagonal blocks -> constant memory
// Ystore (nullable, n16 <= 128 only): also write Y = A Rs^-1 (store-Y variant)
int launch_k3_gram(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                   double* partials, int* n_partials_out, double* Ydump, double* Ystore, int64_t ldys, cudaStream_t s);
int launch_reduce_partials(const double* partials, int n_partials, int n, int n16, double* G16, cudaStream_t s);
int launch_k4_cholesky(const double* G16, int n, int n16, double* G_out, double* Rc, double* RcPrep,
                       const double* Rs, double* R, Status* st, cudaStream_t s);   // Rs, R nullable: R = Rc Rs
// mode 3: Q = (A Rs^-1) Rc^-1; mode 1: Q = A Rs^-1 (store-Y); mode 2: Q = A Rc^-1 (A = the stored Y, may alias Q)
int launch_k5_formq(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                    const double* RcPrep, int64_t ldq, double* Q, double* Ydump, int mode, cudaStream_t s);
// panel passes of the store-Y form (n16 > 128): dst <- src * R^-1 one 64-column panel per launch
bool panel_pass_usable(int64_t m, int n, const double* src, int64_t lds, const double* dst, int64_t ldd);
int launch_panel_solve(int64_t m, int n, int fac, const double* src, int64_t lds, const double* prep,
                       double* dst, int64_t ldd, cudaStream_t s);
// G = Y^T Y of a stored m x n Y (n16 > 128): DMMA SYRK over 128 x 128 blocks with a deterministic split of the rows
size_t syrk_partials_bytes(int n);
int launch_orth_norm(const double* G16, int n, int n16, double* err, cudaStream_t s);   // err[0] = ||I - G||_F
int launch_syrk(int64_t m, int n, int64_t ldy, const double* Y, double* partials, int n16, double* G16, cudaStream_t s);
int launch_triu_mul(const double* Rc, const double* Rs, int n, double* R, cudaStream_t s);
// RsPrep nullable: when given, the kernel also writes the prepared Rs and reports a singular diagonal.
// betas: n doubles of workspace (nullable: then the single-CTA kernels are used for every n).
// NOTE: for n > 64 the sketch `As` is overwritten (factored in place by the blocked kernel).
int launch_k2_sketch_qr(const double* As, int s_rows, int n, double* Rs, double* RsPrep, int n16,
                        double* betas, Status* st, cudaStream_t s);
int launch_k4_coop(double* G16, int n, int n16, double* G_out, double* Rc, double* RcPrep, const double* Rs,
                   double* R, Status* st, cudaStream_t stream);
bool k2_blocked_usable(int s_rows, int n);
int launch_k2_blocked(double* As, int s_rows, int n, double* betas, double* Rs, double* RsPrep, int n16,
                      Status* st, cudaStream_t stream);

// epilogue shared by the K2 kernels: Rs (just written by this CTA) -> prepared Rs, singular check
__device__ __forceinline__ void k2_prepare(const double* Rs, int n, double* RsPrep, int n16, Status* st)
{
    if (!RsPrep) return;
    __syncthreads();
    int bad = -1;
    prep_cta(Rs, n, n, n16 >> 3, RsPrep, &bad);
    if (bad >= 0) report(st, 2, bad);
}

// K1: sampled transform.  Returns launches.  As (s x n, ld = s) receives precision-p values in FP64.
size_t k1_workspace_bytes(int64_t m, int n, int s, int prec);
int launch_k1_srtt(int64_t m, int n, int64_t lda, const double* A, int prec, int s,
                   const uint64_t* signs, const int64_t* idx, void* k1_work, double* As,
                   Status* st, cudaStream_t stream, int reim = 0,       // reim: 2s rows, Im X[S] below Re X[S]
                   const uint64_t* gen_seed = nullptr, bool reset_status = false, const int64_t* h_bins = nullptr);
// h_bins != nullptr (HOST pointer, read during the call) and k1_takes_host_bins(m, s, reim): the bins travel as a launch
// parameter and `idx` is not read.
// gen_seed != nullptr and k1_generates_signs(m, reim): K1 evaluates the sign words from *gen_seed itself (`signs` is not
// read) and, with reset_status, clears the status block as the first kernel of the call.
bool k1_generates_signs(int64_t m, int reim);
bool k1_takes_host_bins(int64_t m, int s, int reim);

// batched small problems, one CTA per problem (k_batched.cu); codes_dev: batch x 2 ints (code, info)
bool batched_fused_usable(int64_t m, int n, int s);
int launch_factor_batched(int batch, int64_t m, int n, int64_t lda, int64_t strideA, const double* A, int64_t ldq,
                          int64_t strideQ, double* Q, double* R, int prec, int s, uint64_t seed, int* codes_dev,
                          cudaStream_t st);

size_t k3_partials_bytes(int n);
int num_sms();

} // namespace mrcqr
