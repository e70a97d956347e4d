// k4_coop.cu -- K4 for n16 > 160 (G does not fit one CTA's shared memory): blocked right-looking Cholesky
// G = Rc^T Rc (Algorithm 1 step 2) on a cooperative grid, 8 columns per step, one grid barrier
// per step.  Column j of the working upper triangle belongs to CTA j mod G.  Per step every CTA
//   (1) loads and factors the 8x8 diagonal block itself (warp 0; rsqrt pivots; identical arithmetic everywhere),
//   (2) computes the WHOLE 8-row panel Rc[k0:k0+8, j] for all trailing columns j (one thread per column:
//       redundant across CTAs, 8 x n values, so that no second barrier is needed),
//   (3) applies the rank-8 update to the trailing columns it owns; after the barrier it writes their panel rows.
// A pivot <= 0 or NaN is reported, never shifted away.  Epilogue (grid-wide): Rc, the
// prepared Rc and R = Rc Rs (Algorithm 2 step 9).
#include "mrcqr_internal.cuh"
#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace mrcqr {

constexpr int KC_NT = 512;

__global__ void __launch_bounds__(KC_NT, 1)
mrcqr_k4_coop(double* __restrict__ W, int n, int n16, double* __restrict__ G_out, double* __restrict__ Rc,
              double* __restrict__ RcPrep, const double* __restrict__ Rs, double* __restrict__ R, Status* st)
{
    cg::grid_group grid = cg::this_grid();
    extern __shared__ __align__(16) double kc_sm[];
    double* Pn = kc_sm;                      // [8][n16]: the current row panel
    double* D = kc_sm + 8 * n16;             // [8][8] diagonal block, D[q*8+p] = element (row p, col q), then Rc block
    double* dinv = D + 64;                   // [8]
    const int tid = threadIdx.x, G = gridDim.x, ld = n16;
    const size_t gtid = (size_t)blockIdx.x * KC_NT + tid, gsz = (size_t)G * KC_NT;

    if (G_out) {
        for (size_t e = gtid; e < (size_t)n * n; e += gsz) G_out[e] = W[(e / n) * ld + e % n];
        grid.sync();
    }
    for (int k0 = 0; k0 < n; k0 += 8) {
        const int kb = min(8, n - k0);
        if (tid < 64) {
            const int p = tid & 7, q = tid >> 3;
            D[tid] = (p <= q && q < kb) ? W[(size_t)(k0 + q) * ld + k0 + p] : 0.0;
        }
        __syncthreads();
        if (tid < 32) {                      // (1) lane j < kb owns column k0 + j of the block
            const int j = tid;
            double c[8];
#pragma unroll
            for (int p = 0; p < 8; ++p) c[p] = (j < kb && p <= j) ? D[j * 8 + p] : 0.0;
#pragma unroll
            for (int p = 0; p < 8; ++p) {
                if (p < kb) {
                    const double piv = __shfl_sync(0xffffffffu, c[p], p);
                    if (blockIdx.x == 0 && j == p && (!(piv > 0.0) || isinf(piv))) report(st, 3, k0 + p);
                    const double ri = rsqrt(piv);
                    const double rp = (j == p) ? piv * ri : c[p] * ri;
                    c[p] = rp;
                    if (j == p) dinv[p] = ri;
#pragma unroll
                    for (int q = p + 1; q < 8; ++q) {
                        const double rq = __shfl_sync(0xffffffffu, rp, q);
                        if (q <= j) c[q] = fma(-rq, rp, c[q]);
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < 8; ++p) if (j < 8) D[j * 8 + p] = (j < kb && p <= j) ? c[p] : 0.0;
        }
        __syncthreads();
        const int t0 = k0 + kb;
        for (int j = k0 + tid; j < n; j += KC_NT) {                     // (2) panel rows of every column j >= k0
            double x[8];
            if (j < t0) {
#pragma unroll
                for (int p = 0; p < 8; ++p) x[p] = D[(j - k0) * 8 + p];  // inside the block: Rc[k0+p, j] (0 below the diagonal)
            } else {
#pragma unroll
                for (int p = 0; p < 8; ++p) {
                    x[p] = 0.0;
                    if (p < kb) {
                        double t = W[(size_t)j * ld + k0 + p];
#pragma unroll
                        for (int q = 0; q < p; ++q) t = fma(-D[p * 8 + q], x[q], t);
                        x[p] = t * dinv[p];
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < 8; ++p) Pn[p * n16 + j] = x[p];
        }
        __syncthreads();
        int j1 = t0 + (((int)blockIdx.x - t0 % G) + G) % G;             // (3) rank-8 update of the owned columns
        for (int j = j1; j < n; j += G) {
            double pj[8];
#pragma unroll
            for (int p = 0; p < 8; ++p) pj[p] = Pn[p * n16 + j];
            for (int i = t0 + tid; i <= j; i += KC_NT) {
                double acc = W[(size_t)j * ld + i];
#pragma unroll
                for (int p = 0; p < 8; ++p) acc = fma(-Pn[p * n16 + i], pj[p], acc);
                W[(size_t)j * ld + i] = acc;
            }
        }
        __threadfence();
        grid.sync();
        // only now may the finished rows replace the input rows other CTAs were still reading in (1), (2)
        for (int j = k0 + (((int)blockIdx.x - k0 % G) + G) % G; j < n; j += G)
            if (tid < kb && k0 + tid <= j) W[(size_t)j * ld + k0 + tid] = Pn[tid * n16 + j];
        __syncthreads();                             // before the next step overwrites Pn
    }
    __threadfence();
    grid.sync();
    // ---- epilogue: W (upper) = Rc
    for (size_t e = gtid; e < (size_t)n * n; e += gsz) {
        const int i = (int)(e % n), j = (int)(e / n);
        double w = 0.0, r = 0.0;
        if (i <= j) {
            w = W[(size_t)j * ld + i];
            if (R) for (int k = i; k <= j; ++k) r = fma(W[(size_t)k * ld + i], Rs[(size_t)j * n + k], r);
        }
        Rc[e] = w;
        if (R) R[e] = r;
    }
    {
        const int nB = n16 >> 3;
        const size_t total = prep_diag_offset(nB) + (size_t)PREP_DIAG * nB;
        int bad = -1;
        for (size_t o = gtid; o < total; o += gsz) RcPrep[o] = prep_value(W, ld, n, nB, o, &bad);
    }
}

int launch_k4_coop(double* G16, int n, int n16, double* G_out, double* Rc, double* RcPrep, const double* Rs,
                   double* R, Status* st, cudaStream_t stream)
{
    int grid = num_sms();
    if (grid > (n + 7) / 8) grid = (n + 7) / 8;
    size_t smem = ((size_t)8 * n16 + 64 + 8) * sizeof(double);
    cudaFuncSetAttribute(mrcqr_k4_coop, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    void* args[] = {&G16, &n, &n16, &G_out, &Rc, &RcPrep, &Rs, &R, &st};
    cudaLaunchCooperativeKernel((const void*)mrcqr_k4_coop, dim3(grid), dim3(KC_NT), args, smem, stream);
    return 1;
}

} // namespace mrcqr
