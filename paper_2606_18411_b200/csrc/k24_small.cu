// k24_small.cu -- the latency-bound single-CTA steps and the tiny glue kernels:
//   K2  mrcqr_k2_sketch_qr  Algorithm 2 steps 5-6: Householder R-factor of the
//                           s x n sketch, rows sign-normalised to diag > 0, FP64 arithmetic on the
//                           precision-p sketch values (>= p; PAPER.md:119 promotes FP16 to FP32).
//   K4  mrcqr_k4_blocked   Algorithm 1 step 2: G = Rc^T Rc; a pivot <= 0 or NaN is
//                           reported, never shifted away.
//   prep_R                  builds the "prepared" factor the tile solve consumes.
//   triu_mul                Algorithm 2 step 9: R = Rc Rs.
#include "mrcqr_internal.cuh"

namespace mrcqr {

constexpr int SMALL_NT = 1024;
constexpr int SMALL_SMEM_MAX = 220 * 1024;

__global__ void mrcqr_prep_R(const double* __restrict__ R, int n, double* __restrict__ Rp, int n16,
                             Status* st, int err_code)
{
    const int nB = n16 >> 3;
    const size_t total = prep_diag_offset(nB) + (size_t)PREP_DIAG * nB;
    const size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= total) return;
    int bad = -1;
    Rp[o] = prep_value(R, n, n, nB, o, &bad);
    if (bad >= 0) report(st, err_code, bad);
}

__global__ void mrcqr_triu_mul(const double* __restrict__ Rc, const double* __restrict__ Rs, int n,
                               double* __restrict__ R)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n * n) return;
    const int i = e % n, j = e / n;
    double acc = 0.0;
    if (i <= j)
        for (int k = i; k <= j; ++k) acc = fma(Rc[(size_t)k * n + i], Rs[(size_t)j * n + k], acc);
    R[e] = acc;
}

// ---- K4 ---------------------------------------------------------------------------------------
// ---- K4, blocked form with the trailing update on DMMA (n16 <= 160) ---------------------------------------
// Eight pivots per step and three block barriers per step instead of one per pivot:
//   (1) warp 0 factors the 8x8 diagonal block in registers (lane j owns column j; shuffles; rsqrt_fast pivots),
//   (2) one thread per trailing column solves its 8 rows against the block, the block's 36 entries in registers first
//       (a first blocked kernel read them from shared memory inside the dependent chain and lost to the unblocked
//       one-barrier-per-pivot kernel of round 1: 71 vs 48 us at n = 64; this one: 38 us, and 131 vs 183 us at n = 128),
//   (3) the rank-8 update G22 -= R12^T R12 runs on the FP64 tensor cores: an 8x8 block of G22 is one accumulator
//       fragment, R12^T / R12 are the A / B fragments (k = 8: two DMMAs per block), the upper-triangular blocks dealt
//       round-robin to the 16 warps.
// W: working copy of G (upper triangle), col-major, ld = n16 + 2 (conflict-free accumulator fragments); Pn: the current
// 8-row panel, ld = n16 + 4 (conflict-free A / B fragments).  Epilogue: Rc, the prepared Rc and, if Rs is given,
// R = Rc Rs (Algorithm 2 step 9; Rs staged in the free strictly-lower triangle).
constexpr int K4B_NT = 512;

__global__ void __launch_bounds__(K4B_NT)
mrcqr_k4_blocked(const double* __restrict__ G16, int n, int n16, double* __restrict__ G_out,
                 double* __restrict__ Rc, double* __restrict__ RcPrep, const double* __restrict__ Rs,
                 double* __restrict__ R, Status* st)
{
    extern __shared__ __align__(16) double sm[];
    const int ldw = n16 + 2, pld = n16 + 4;
    double* W = sm;                              // n16 x ldw
    double* Pn = W + (size_t)n16 * ldw;          // 8 x pld
    double* D = Pn + 8 * pld;                    // 8 x 8: D[q * 8 + p] = Rc[k0 + p, k0 + q], p <= q
    double* dinv = D + 64;                       // 8
    double* rsd = dinv + 8;                      // n16
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    for (int j = warp; j < n16; j += K4B_NT / 32)             // column per warp, rows per lane: no index division
        for (int i = lane; i < ldw; i += 32) {
            double v = 0.0;
            if (i < n && j < n) { v = G16[(size_t)j * n16 + i]; if (G_out) G_out[(size_t)j * n + i] = v; }
            else if (i == j) v = 1.0;            // identity padding: its pivots are harmless
            W[j * ldw + i] = v;
        }
    for (int e = tid; e < 8 * pld; e += K4B_NT) Pn[e] = 0.0;
    __syncthreads();
    const int nB = n16 >> 3;
    for (int k0 = 0; k0 < n; k0 += 8) {
        const int kb = min(8, n - k0);
        if (warp == 0) {                         // (1) lane j < 8 owns column k0 + j of the diagonal block
            const int j = lane;
            double c[8];
#pragma unroll
            for (int p = 0; p < 8; ++p) c[p] = (j < 8 && p <= j) ? W[(k0 + j) * ldw + k0 + p] : 0.0;
#pragma unroll
            for (int p = 0; p < 8; ++p) {
                const double piv = __shfl_sync(0xffffffffu, c[p], p);
                if (p < kb && j == p && (!(piv > 0.0) || isinf(piv))) report(st, 3, k0 + p);
                const double ri = rsqrt_fast(piv);
                const double rp = (j == p) ? piv * ri : c[p] * ri;       // Rc[k0+p, k0+j] for j >= p
                c[p] = rp;
                if (j == p) dinv[p] = ri;
#pragma unroll
                for (int q = p + 1; q < 8; ++q) {                        // c[q] -= Rc[p, q] * Rc[p, j]  (q <= j)
                    const double rq = __shfl_sync(0xffffffffu, rp, q);
                    if (q <= j) c[q] = fma(-rq, rp, c[q]);
                }
            }
#pragma unroll
            for (int p = 0; p < 8; ++p)
                if (j < 8) { const double v = (p <= j) ? c[p] : 0.0; D[j * 8 + p] = v; if (p <= j) W[(k0 + j) * ldw + k0 + p] = v; }
        }
        __syncthreads();
        const int t0 = k0 + 8;
        if (t0 < n16) {
            if (tid < n16 - t0) {                // (2) row panel: column j = t0 + tid (padding columns give zeros)
                const int j = t0 + tid;
                double d[8][8], di[8], x[8];
#pragma unroll
                for (int p = 0; p < 8; ++p) {
                    di[p] = dinv[p];
#pragma unroll
                    for (int q = 0; q < p; ++q) d[p][q] = D[p * 8 + q];  // Rc[k0+q, k0+p]
                }
#pragma unroll
                for (int p = 0; p < 8; ++p) x[p] = W[j * ldw + k0 + p];
#pragma unroll
                for (int p = 0; p < 8; ++p) {
                    double acc = x[p];
#pragma unroll
                    for (int q = 0; q < p; ++q) acc = fma(-d[p][q], x[q], acc);
                    x[p] = acc * di[p];
                }
#pragma unroll
                for (int p = 0; p < 8; ++p) { W[j * ldw + k0 + p] = x[p]; Pn[p * pld + j] = x[p]; }
            }
            __syncthreads();
            // (3) trailing update on DMMA: blocks (I, J), t0/8 <= I <= J < nB
            const int b0 = t0 >> 3, T = nB - b0, nblk = T * (T + 1) / 2;
            int ii = warp, jj = 0;                   // block bi = warp, warp + 16, ...: (ii, jj) walks the upper triangle column by column
            while (ii > jj) { ii -= jj + 1; ++jj; }
            for (int bi = warp; bi < nblk; bi += K4B_NT / 32) {
                const int I = b0 + ii, J = b0 + jj;
                ii += K4B_NT / 32;
                while (ii > jj) { ii -= jj + 1; ++jj; }
                double* cp = W + (size_t)(8 * J + 2 * t) * ldw + 8 * I + g;
                double c2[2] = {cp[0], cp[ldw]};
                const double a0 = -Pn[t * pld + 8 * I + g], a1 = -Pn[(t + 4) * pld + 8 * I + g];
                const double bb0 = Pn[t * pld + 8 * J + g], bb1 = Pn[(t + 4) * pld + 8 * J + g];
                asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c2[0]), "+d"(c2[1]) : "d"(a0), "d"(bb0));
                asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c2[0]), "+d"(c2[1]) : "d"(a1), "d"(bb1));
                cp[0] = c2[0]; cp[ldw] = c2[1];
            }
            __syncthreads();
        }
    }
    __syncthreads();
    // stage Rs in the free strictly-lower triangle, transposed: Rs[k,j] (k < j) at W[k*ldw + j], diag(Rs) in rsd
    // (column per warp, rows per lane: coalesced reads, independent loads)
    if (R)
        for (int j = warp; j < n; j += K4B_NT / 32)
            for (int i = lane; i <= j; i += 32) {
                const double v = Rs[(size_t)j * n + i];
                if (i < j) W[i * ldw + j] = v; else rsd[j] = v;
            }
    __syncthreads();
    // Rc and R = Rc Rs: R[i,j] = sum_{k=i..j} Rc[i,k] Rs[k,j], every element ONE fma chain in ascending k (the order of
    // mrcqr_triu_mul: the stage call gives the same bits).  A thread owns a 2 x 4 patch (rows i0, i0+1, columns j0..j0+3):
    // per k one 16-byte load of the row pair (lanes contiguous: conflict-free) and the four Rs[k, j0..] (warp-uniform)
    // feed eight chains.  (One chain per thread, then four rows of one column per thread, were bound by shared-memory
    // wavefronts: 17 per 4 fma; the epilogue was two thirds of K4 at n = 128.)
    {
        const int npp = (n + 63) >> 6, ncq = (n + 3) >> 2;
        for (int item = warp; item < npp * ncq; item += K4B_NT / 32) {
            const int pp = item % npp, cq = item / npp;
            const int i0 = 2 * (lane + 32 * pp), j0 = 4 * cq, jmax = min(j0 + 3, n - 1), kw = 64 * pp;
            if (kw > jmax) continue;                                  // warp-uniform: the patch row lies below the diagonal
            double r[2][4];
#pragma unroll
            for (int q = 0; q < 4; ++q) r[0][q] = r[1][q] = 0.0;
            if (R) {
                int k = kw;
#pragma unroll 4
                for (; k < j0; ++k) {                                // all four columns live: Rs[k, j0..j0+3] at W[k*ldw + j0]
                    const double2 c = *reinterpret_cast<const double2*>(W + (size_t)k * ldw + i0);
                    const double2 s01 = *reinterpret_cast<const double2*>(W + (size_t)k * ldw + j0);
                    const double2 s23 = *reinterpret_cast<const double2*>(W + (size_t)k * ldw + j0 + 2);
                    if (i0 <= k) { r[0][0] = fma(c.x, s01.x, r[0][0]); r[0][1] = fma(c.x, s01.y, r[0][1]); r[0][2] = fma(c.x, s23.x, r[0][2]); r[0][3] = fma(c.x, s23.y, r[0][3]); }
                    if (i0 + 1 <= k) { r[1][0] = fma(c.y, s01.x, r[1][0]); r[1][1] = fma(c.y, s01.y, r[1][1]); r[1][2] = fma(c.y, s23.x, r[1][2]); r[1][3] = fma(c.y, s23.y, r[1][3]); }
                }
                for (; k <= jmax; ++k) {                             // the diagonal 4 x 4 corner: column j takes k <= j, Rs[j,j] from rsd
                    const double2 c = *reinterpret_cast<const double2*>(W + (size_t)k * ldw + i0);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int j = j0 + q;
                        if (k <= j && j < n) {
                            const double rs = (k < j) ? W[k * ldw + j] : rsd[j];
                            if (i0 <= k) r[0][q] = fma(c.x, rs, r[0][q]);
                            if (i0 + 1 <= k) r[1][q] = fma(c.y, rs, r[1][q]);
                        }
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int j = j0 + q;
                if (j < n) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int i = i0 + h;
                        if (i < n) {
                            Rc[(size_t)j * n + i] = (i <= j) ? W[j * ldw + i] : 0.0;
                            if (R) R[(size_t)j * n + i] = (i <= j) ? r[h][q] : 0.0;
                        }
                    }
                }
            }
        }
        // patches that lie wholly below the diagonal were skipped above: their zeros
        for (int item = warp; item < npp * ncq; item += K4B_NT / 32) {
            const int pp = item % npp, cq = item / npp;
            const int i0 = 2 * (lane + 32 * pp), j0 = 4 * cq, jmax = min(j0 + 3, n - 1);
            if (64 * pp <= jmax) continue;
            for (int q = 0; q < 4; ++q)
                for (int h = 0; h < 2; ++h) {
                    const int i = i0 + h, j = j0 + q;
                    if (i < n && j < n) { Rc[(size_t)j * n + i] = 0.0; if (R) R[(size_t)j * n + i] = 0.0; }
                }
        }
    }
    {
        int bad = -1;
        prep_cta(W, ldw, n, nB, RcPrep, &bad);
    }
}

// ---- K2 ---------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(SMALL_NT)
mrcqr_k2_sketch_qr(double* __restrict__ As, int s, int n, int use_smem, double* __restrict__ Rs,
                   double* __restrict__ RsPrep, int n16, Status* st)
{
    extern __shared__ __align__(16) double sm[];
    double* betas = sm;                      // n
    double* sig = sm + n;                    // [0]: sigma of the current column, [1]: of the next
    double* W = use_smem ? sm + n + 2 : As;  // s x n, ld = s
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NWARP = SMALL_NT / 32;

    if (use_smem) for (int e = tid; e < s * n; e += SMALL_NT) W[e] = As[e];
    __syncthreads();
    if (warp == 0) {                         // sigma of column 0
        double a = 0.0;
        for (int i = 1 + lane; i < s; i += 32) a = fma(W[i], W[i], a);
        a = warp_sum(a);
        if (lane == 0) sig[0] = a;
    }
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        const double* x = W + (size_t)j * s;
        const double alpha = x[j], sigma = sig[j & 1];
        double beta = alpha, tau = 0.0, inv = 0.0;
        if (sigma != 0.0 && j + 1 < s) {     // LAPACK dgeqr2 / Golub-Van Loan 5.1.1 convention
            const double nrm = sqrt(fma(alpha, alpha, sigma));
            beta = (alpha >= 0.0) ? -nrm : nrm;
            tau = (beta - alpha) / beta;
            inv = 1.0 / (alpha - beta);
        }
        if (tid == 0) betas[j] = beta;
        for (int c = j + 1 + warp; c < n; c += NWARP) {
            double* y = W + (size_t)c * s;
            double w = 0.0;
            for (int i = j + 1 + lane; i < s; i += 32) w = fma(x[i] * inv, y[i], w);
            w = warp_sum(w);
            w = (w + y[j]) * tau;
            double nxt = 0.0;
            for (int i = j + 1 + lane; i < s; i += 32) {
                const double v = fma(-w, x[i] * inv, y[i]);
                y[i] = v;
                if (i > j + 1) nxt = fma(v, v, nxt);
            }
            __syncwarp();
            if (lane == 0) y[j] = y[j] - w;
            if (c == j + 1) { nxt = warp_sum(nxt); if (lane == 0) sig[(j + 1) & 1] = nxt; }
        }
        __syncthreads();
    }
    for (int e = tid; e < n * n; e += SMALL_NT) {
        const int i = e % n, j = e / n;
        double v = 0.0;
        if (i < j && i < s) v = W[(size_t)j * s + i];
        else if (i == j) v = betas[j];
        if (i <= j && betas[i] < 0.0) v = -v;          // sign-normalise row i: diag(Rs) > 0
        Rs[e] = v;
    }
    k2_prepare(Rs, n, RsPrep, n16, st);
}

// ---- K2, register-resident variant (n <= 32*CPW, s <= 32*RPL) -----------------------------------------
// Column c lives in warp c % 32 (slot c / 32), row i in lane i % 32 (slot i / 32): the whole sketch stays
// in registers.  Per Householder step: ONE block barrier; the reflector travels through a double-buffered
// shared vector; the warp that owns column j+1 forms v_{j+1} right after updating it.
// Reflector, unnormalised: v = x - beta e_j (v_j = alpha - beta), H = I - c v v^T, c = 1 / (beta (beta - alpha))
// (= tau / v_j^2 of the LAPACK form): one square root and one reciprocal per column.
// NW warps per CTA (column c -> warp c % NW): a 32 x 16 sketch (n = 16, s = 2n) runs on 16 warps with one row slot
// instead of 32 warps with four, i.e. a cheaper barrier and a quarter of the multiply-adds per reflector; the arithmetic
// of every element is the same (the slots that are gone held exact zeros).
template <int CPW, int RPL, int NW = 32>
__global__ void __launch_bounds__(32 * NW)
mrcqr_k2_sketch_qr_reg(const double* __restrict__ As, int s, int n, double* __restrict__ Rs,
                       double* __restrict__ RsPrep, int n16, Status* st)
{
    __shared__ double vbuf[2][RPL * 32];
    __shared__ double cbuf[2];
    __shared__ double betas[NW * CPW];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double a[CPW][RPL];
#pragma unroll
    for (int k = 0; k < CPW; ++k)
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int c = warp + NW * k, i = lane + 32 * r;
            a[k][r] = (c < n && i < s) ? As[(size_t)c * s + i] : 0.0;
        }
    // forms the reflector of column j (held in slot k of this warp) and publishes it in buffer j & 1
    auto make_v = [&](int k, int j) {
        double alpha_l = 0.0, sig_l = 0.0;
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int i = lane + 32 * r;
            if (i == j) alpha_l = a[k][r];
            if (i > j) sig_l = fma(a[k][r], a[k][r], sig_l);
        }
        const double alpha = __shfl_sync(0xffffffffu, alpha_l, j & 31);
        const double sigma = warp_sum(sig_l);
        double beta = alpha, cf = 0.0;
        if (sigma != 0.0) {
            householder_coeffs(alpha, sigma, beta, cf);
        }
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int i = lane + 32 * r;
            const double v = (i > j) ? a[k][r] : (i == j ? alpha - beta : 0.0);
            vbuf[j & 1][i] = v;
            if (i == j) a[k][r] = beta;                      // R[j,j]
            if (i > j) a[k][r] = 0.0;
        }
        if (lane == 0) { cbuf[j & 1] = cf; betas[j] = beta; }
    };
    if (warp == 0) make_v(0, 0);
    for (int j = 0; j < n; ++j) {
        __syncthreads();
        double v[RPL];
#pragma unroll
        for (int r = 0; r < RPL; ++r) v[r] = vbuf[j & 1][lane + 32 * r];
        const double cf = cbuf[j & 1];
        double w[CPW];
#pragma unroll
        for (int k = 0; k < CPW; ++k) {
            w[k] = 0.0;
#pragma unroll
            for (int r = 0; r < RPL; ++r) w[k] = fma(v[r], a[k][r], w[k]);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
            for (int k = 0; k < CPW; ++k) w[k] += __shfl_xor_sync(0xffffffffu, w[k], o);
#pragma unroll
        for (int k = 0; k < CPW; ++k) {
            const int c = warp + NW * k;
            if (c > j && c < n) {
                const double wt = w[k] * cf;
#pragma unroll
                for (int r = 0; r < RPL; ++r) a[k][r] = fma(-wt, v[r], a[k][r]);
            }
        }
#pragma unroll
        for (int k = 0; k < CPW; ++k)
            if (warp + NW * k == j + 1 && j + 1 < n) make_v(k, j + 1);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < CPW; ++k)
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int c = warp + NW * k, i = lane + 32 * r;
            if (c < n && i < n) {
                double val = (i <= c) ? a[k][r] : 0.0;
                if (i <= c && betas[i] < 0.0) val = -val;    // sign-normalise row i: diag(Rs) > 0
                Rs[(size_t)c * n + i] = val;
            }
        }
    k2_prepare(Rs, n, RsPrep, n16, st);
}

// ---- launchers --------------------------------------------------------------------------------
int launch_prep_R(const double* R, int n, double* Rprep, int n16, Status* st, int err_code, cudaStream_t s)
{
    const int nB = n16 >> 3;
    const size_t total = prep_diag_offset(nB) + (size_t)PREP_DIAG * nB;
    mrcqr_prep_R<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(R, n, Rprep, n16, st, err_code);
    return 1;
}

int launch_triu_mul(const double* Rc, const double* Rs, int n, double* R, cudaStream_t s)
{
    mrcqr_triu_mul<<<(n * n + 255) / 256, 256, 0, s>>>(Rc, Rs, n, R);
    return 1;
}

int launch_k4_cholesky(const double* G16, int n, int n16, double* G_out, double* Rc, double* RcPrep,
                       const double* Rs, double* R, Status* st, cudaStream_t s)
{
    size_t need = ((size_t)9 * n16 + 2 + (size_t)n16 * (n16 + 1)) * sizeof(double);
    const int use_smem = need <= (size_t)SMALL_SMEM_MAX;
    if (use_smem) {
        const size_t smb = ((size_t)n16 * (n16 + 2) + 8 * (size_t)(n16 + 4) + 72 + n16) * sizeof(double);
        cudaFuncSetAttribute(mrcqr_k4_blocked, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smb);
        mrcqr_k4_blocked<<<1, K4B_NT, smb, s>>>(G16, n, n16, G_out, Rc, RcPrep, Rs, R, st);
        return 1;
    }
    return launch_k4_coop(const_cast<double*>(G16), n, n16, G_out, Rc, RcPrep, Rs, R, st, s);
}

int launch_k2_sketch_qr(const double* As, int s_rows, int n, double* Rs, double* RsPrep, int n16,
                        double* betas, Status* st, cudaStream_t s)
{
    if (n <= 64 && s_rows <= 256) {
        if (n <= 16 && s_rows <= 32) mrcqr_k2_sketch_qr_reg<1, 1, 16><<<1, 512, 0, s>>>(As, s_rows, n, Rs, RsPrep, n16, st);
        else if (n <= 16 && s_rows <= 64) mrcqr_k2_sketch_qr_reg<1, 2, 16><<<1, 512, 0, s>>>(As, s_rows, n, Rs, RsPrep, n16, st);
        else if (n <= 32 && s_rows <= 64) mrcqr_k2_sketch_qr_reg<1, 2><<<1, SMALL_NT, 0, s>>>(As, s_rows, n, Rs, RsPrep, n16, st);
        else if (n <= 32 && s_rows <= 128) mrcqr_k2_sketch_qr_reg<1, 4><<<1, SMALL_NT, 0, s>>>(As, s_rows, n, Rs, RsPrep, n16, st);
        else if (s_rows <= 128) mrcqr_k2_sketch_qr_reg<2, 4><<<1, SMALL_NT, 0, s>>>(As, s_rows, n, Rs, RsPrep, n16, st);
        else mrcqr_k2_sketch_qr_reg<2, 8><<<1, SMALL_NT, 0, s>>>(As, s_rows, n, Rs, RsPrep, n16, st);
        return 1;
    }
    if (k2_blocked_usable(s_rows, n) && betas)
        return launch_k2_blocked(const_cast<double*>(As), s_rows, n, betas, Rs, RsPrep, n16, st, s);
    size_t need = ((size_t)n + 2 + (size_t)s_rows * n) * sizeof(double);
    const int use_smem = need <= (size_t)SMALL_SMEM_MAX;
    const size_t smem = use_smem ? need : ((size_t)n + 2) * sizeof(double);
    cudaFuncSetAttribute(mrcqr_k2_sketch_qr, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    mrcqr_k2_sketch_qr<<<1, SMALL_NT, smem, s>>>(const_cast<double*>(As), s_rows, n, use_smem, Rs, RsPrep, n16, st);
    return 1;
}

} // namespace mrcqr
