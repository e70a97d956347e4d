// k2_blocked.cu -- K2 for n > 64: blocked Householder QR of the s x n sketch on the whole GPU
// (Algorithm 2 steps 5-6; FP64 arithmetic on the precision-p values, R5).
//
// The single-CTA unblocked kernel needs one block barrier and ~2 k cycles per column and streams a
// sketch that no longer fits shared memory (0.7 / 4.7 / 39 ms at n = 128 / 256 / 512).  Here the sketch
// is factored in panels of 8 columns by a cooperative grid (one CTA per SM, 256 threads, thread = row):
//   F  every CTA factors the panel REDUNDANTLY in registers (identical arithmetic, so no exchange is
//      needed): column j first receives the reflectors 0..j-1 of the panel in compact form
//        y_i = v_i^T a_j,   z_i = c_i (y_i - sum_{l<i} S_il z_l),   a_j -= sum_i z_i v_i,   S = V^T V,
//      (the same numbers as applying H_0 .. H_{j-1} one after the other), then its own reflector
//      v_j = a_j - beta e_j, H_j = I - c_j v_j v_j^T, c_j = 1 / (beta (beta - alpha));
//   A  every CTA applies the 8 reflectors to the trailing columns it owns (column c belongs to CTA
//      c mod G) with the same compact form: ONE block reduction of 8 dot products per column;
//   one grid barrier per panel.
// Block reductions sum a batch of up to 16 values at once: a butterfly exchange that halves the batch in
// every round (16 shuffles instead of 80), warp partials through shared memory, fixed order.
// R is left in the upper triangle of the (workspace) sketch; CTA 0 extracts it, sign-normalises the rows
// to diag(R_s) > 0 and writes the prepared R_s.
#include "mrcqr_internal.cuh"
#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace mrcqr {

constexpr int KB_NT = 256;            // threads per CTA (thread t owns rows t, t + 256, ...)
constexpr int KB_NW = KB_NT / 32;
constexpr int KB_B = 8;               // panel width

// Sum of each of the KP (8 or 16) values of v over the 256 threads; every thread receives all totals in tot[].
// red: shared scratch [KB_NW][16] + [16].  Fixed order: butterfly inside a warp, warps 0..7 in order.
template <int KP>
__device__ __forceinline__ void block_sum(double (&v)[KP], double* red, double (&tot)[KP])
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int h = KP / 2, bit = 16; h >= 1; h >>= 1, bit >>= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int q = 0; q < KP / 2; ++q) {
            if (q < h) {
                const double send = up ? v[q] : v[q + h];
                const double keep = up ? v[q + h] : v[q];
                v[q] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
            }
        }
    }
    // KP = 16: bits 16, 8, 4, 2 consumed, lanes l and l^1 hold partial sums of the same value; KP = 8: bits 16, 8, 4
    if (KP == 16) v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
    else { v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2); v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1); }
    // value index held by this lane: the kept half at every round (bit set -> upper half)
    int idx = 0;
    if (KP == 16) idx = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
    else idx = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
    __syncthreads();                                   // previous use of red is over
    if ((KP == 16 && (lane & 1) == 0) || (KP == 8 && (lane & 3) == 0)) red[warp * 16 + idx] = v[0];
    __syncthreads();
    if (threadIdx.x < KP) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < KB_NW; ++w) t += red[w * 16 + threadIdx.x];
        red[KB_NW * 16 + threadIdx.x] = t;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < KP; ++q) tot[q] = red[KB_NW * 16 + q];
}

template <int RPT>
__global__ void __launch_bounds__(KB_NT, 1)
mrcqr_k2_blocked(double* __restrict__ As, int s, int n, double* __restrict__ betas_g, double* __restrict__ Rs,
                 double* __restrict__ RsPrep, int n16, Status* st)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double red[KB_NW * 16 + 16];
    const int tid = threadIdx.x, G = gridDim.x;

    for (int j0 = 0; j0 < n; j0 += KB_B) {
        const int bw = min(KB_B, n - j0);
        double P[KB_B][RPT];                         // the panel: thread = row
        int rel[RPT];                                // row - j0 (row >= s: a value that matches no pivot)
#pragma unroll
        for (int q = 0; q < RPT; ++q) {
            const int row = tid + KB_NT * q;
            rel[q] = row < s ? row - j0 : -(1 << 30);
#pragma unroll
            for (int c = 0; c < KB_B; ++c) P[c][q] = (c < bw && row < s) ? As[(size_t)(j0 + c) * s + row] : 0.0;
        }
        double vd[KB_B], cf[KB_B], S[KB_B][KB_B];
#pragma unroll
        for (int i = 0; i < KB_B; ++i) {
            vd[i] = 0.0; cf[i] = 0.0;
#pragma unroll
            for (int l = 0; l < KB_B; ++l) S[i][l] = 0.0;
        }
        // reflector i of the panel at this thread's row q: below the pivot the stored column, at the pivot vd, above 0
#define KB_V(i, q) (rel[q] > (i) ? P[i][q] : (rel[q] == (i) ? vd[i] : 0.0))
        // z_i = c_i (y_i - sum_{l<i} S_il z_l): the coefficients of H_{cnt-1} ... H_0 applied in sequence
#define KB_RECUR(y, z, cnt)                                                           \
        _Pragma("unroll") for (int i = 0; i < KB_B; ++i) {                            \
            z[i] = 0.0;                                                               \
            if (i < (cnt)) {                                                          \
                double acc_ = y[i];                                                   \
                _Pragma("unroll") for (int l = 0; l < i; ++l) acc_ = fma(-S[i][l], z[l], acc_); \
                z[i] = cf[i] * acc_;                                                  \
            }                                                                         \
        }
#pragma unroll
        for (int j = 0; j < KB_B; ++j) {
            if (j < bw) {                            // uniform
                if (j > 0) {
                    double vals[16], tot[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) vals[i] = 0.0;
#pragma unroll
                    for (int q = 0; q < RPT; ++q) {
                        const double vprev = KB_V(j - 1, q);
#pragma unroll
                        for (int i = 0; i < j; ++i) {
                            const double vi = KB_V(i, q);
                            vals[i] = fma(vi, P[j][q], vals[i]);                       // y_i = v_i^T a_j
                            if (i < j - 1) vals[8 + i] = fma(vi, vprev, vals[8 + i]);   // S_{j-1,i} = v_i^T v_{j-1}
                        }
                    }
                    block_sum<16>(vals, red, tot);
#pragma unroll
                    for (int i = 0; i < j - 1; ++i) S[j - 1][i] = tot[8 + i];
                    double z[KB_B];
                    KB_RECUR(tot, z, j)
#pragma unroll
                    for (int q = 0; q < RPT; ++q)
#pragma unroll
                        for (int i = 0; i < j; ++i) P[j][q] = fma(-z[i], KB_V(i, q), P[j][q]);
                }
                double v2[8], t2[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) v2[i] = 0.0;
#pragma unroll
                for (int q = 0; q < RPT; ++q) {
                    if (rel[q] > j) v2[0] = fma(P[j][q], P[j][q], v2[0]);
                    if (rel[q] == j) v2[1] = P[j][q];
                }
                block_sum<8>(v2, red, t2);
                const double sigma = t2[0], alpha = t2[1];
                double beta = alpha, c = 0.0;
                if (sigma != 0.0) {
                    householder_coeffs(alpha, sigma, beta, c);
                }
                vd[j] = alpha - beta; cf[j] = c;
#pragma unroll
                for (int q = 0; q < RPT; ++q) if (rel[q] == j) P[j][q] = beta;         // R[j,j] (the reflector's pivot lives in vd)
                if (blockIdx.x == 0 && tid == 0) betas_g[j0 + j] = beta;
            }
        }
        if (bw > 1) {                                // last row of S: v_i^T v_{bw-1}
            double vals[8], tot[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) vals[i] = 0.0;
#pragma unroll
            for (int q = 0; q < RPT; ++q)
#pragma unroll
                for (int j = 1; j < KB_B; ++j)
                    if (j == bw - 1) {
                        const double vlast = KB_V(j, q);
#pragma unroll
                        for (int i = 0; i < j; ++i) vals[i] = fma(KB_V(i, q), vlast, vals[i]);
                    }
            block_sum<8>(vals, red, tot);
#pragma unroll
            for (int j = 1; j < KB_B; ++j)
                if (j == bw - 1) {
#pragma unroll
                    for (int i = 0; i < j; ++i) S[j][i] = tot[i];
                }
        }
        // ---- apply H_{bw-1} ... H_0 to the trailing columns this CTA owns
        int c0 = j0 + bw;
        c0 += ((int)blockIdx.x - c0 % G + G) % G;
        for (int c = c0; c < n; c += G) {
            double a[RPT], vals[8], tot[8], z[KB_B];
#pragma unroll
            for (int i = 0; i < 8; ++i) vals[i] = 0.0;
#pragma unroll
            for (int q = 0; q < RPT; ++q) {
                const int row = tid + KB_NT * q;
                a[q] = row < s ? As[(size_t)c * s + row] : 0.0;
#pragma unroll
                for (int i = 0; i < KB_B; ++i) if (i < bw) vals[i] = fma(KB_V(i, q), a[q], vals[i]);
            }
            block_sum<8>(vals, red, tot);
            KB_RECUR(tot, z, bw)
#pragma unroll
            for (int q = 0; q < RPT; ++q) {
#pragma unroll
                for (int i = 0; i < KB_B; ++i) if (i < bw) a[q] = fma(-z[i], KB_V(i, q), a[q]);
                const int row = tid + KB_NT * q;
                if (row < s) As[(size_t)c * s + row] = a[q];
            }
        }
#undef KB_V
#undef KB_RECUR
        __threadfence();
        grid.sync();
        // only now may the R entries of the panel (rows <= pivot) replace the unfactored panel in the sketch: every CTA
        // loaded it at the top of this iteration, and nothing orders those loads before this point except the barrier
        if (blockIdx.x == 0) {
#pragma unroll
            for (int q = 0; q < RPT; ++q)
#pragma unroll
                for (int c = 0; c < KB_B; ++c)
                    if (c < bw && rel[q] >= -j0 && rel[q] <= c) As[(size_t)(j0 + c) * s + tid + KB_NT * q] = P[c][q];
        }
    }
    if (blockIdx.x == 0) {
        __syncthreads();                             // the last panel's write-back above, by other threads of this CTA
        for (int e = tid; e < n * n; e += KB_NT) {
            const int i = e % n, j = e / n;
            double v = 0.0;
            if (i < j) v = As[(size_t)j * s + i];
            else if (i == j) v = betas_g[j];
            if (i <= j && betas_g[i] < 0.0) v = -v;    // sign-normalise row i: diag(Rs) > 0
            Rs[e] = v;
        }
        k2_prepare(Rs, n, RsPrep, n16, st);
    }
}

bool k2_blocked_usable(int s_rows, int n) { return n > 64 && s_rows <= 16 * KB_NT; }

// `As` is factored IN PLACE (the caller passes a workspace copy); betas: n doubles of workspace.
int launch_k2_blocked(double* As, int s_rows, int n, double* betas, double* Rs, double* RsPrep, int n16,
                      Status* st, cudaStream_t stream)
{
    int grid = num_sms();
    void* args[] = {&As, &s_rows, &n, &betas, &Rs, &RsPrep, &n16, &st};
    const int rpt = (s_rows + KB_NT - 1) / KB_NT;
    const void* fn = rpt <= 1 ? (const void*)mrcqr_k2_blocked<1> : rpt <= 2 ? (const void*)mrcqr_k2_blocked<2>
                   : rpt <= 4 ? (const void*)mrcqr_k2_blocked<4> : rpt <= 8 ? (const void*)mrcqr_k2_blocked<8>
                   : (const void*)mrcqr_k2_blocked<16>;
    cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(KB_NT), args, 0, stream);
    return 1;
}

} // namespace mrcqr
