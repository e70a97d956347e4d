// k35_rows.cu -- the two passes over A that dominate MRCQR ("TRSM x2" is 56-74 %
// of the paper's runtime):
//   K3  mrcqr_k3_gram   Algorithm 2 step 7 fused with Algorithm 1 step 1:
//                       per row y = a Rs^-1 (solve_tile), G += y^T y on DMMA; Y never leaves the SM.
//   K5  mrcqr_k5_formq  Algorithm 1 step 3: y recomputed bit-identically,
//                       q = y Rc^-1, Q streamed out.
// Persistent CTAs, static tile -> CTA map (tile i belongs to CTA i mod grid, visited in ascending
// order), so every sum has a fixed order: results are deterministic run to run.
#include "rows.cuh"

namespace mrcqr {

constexpr int GRAM_MAXS = 6;          // 16x16 super-blocks of G a warp accumulates per sweep (48 doubles)
constexpr int GRAM_CHAIN = 256;       // max DMMA k-steps chained into one accumulator before a flush

RowCfg row_config(int n)
{
    RowCfg c;
    c.n16 = round_up(n, 16);
    if (c.n16 <= 64)       { c.TM = 128; c.NW = 4; }
    else if (c.n16 <= 128) { c.TM = 128; c.NW = 8; }
    else if (c.n16 <= 256) { c.TM = 64;  c.NW = 8; }
    else                   { c.TM = 32;  c.NW = 4; }
    c.smem_bytes = c.n16 * (c.TM + 4) * 8;
    c.ctas_per_sm = 0;
    return c;
}

__device__ __forceinline__ void sb_to_pq(int sb, int& p, int& q)
{
    int qq = 0;
    while ((qq + 1) * (qq + 2) / 2 <= sb) ++qq;
    q = qq; p = sb - qq * (qq + 1) / 2;
}

// G partial of this CTA: n16 x n16 col-major, blocks (I <= J) of the upper triangle only.
template <int TM, int NW, bool VEC>
__global__ void __launch_bounds__(NW * 32)
mrcqr_k3_gram(int64_t m, int n, int n16, int64_t lda, const double* __restrict__ A,
              const double* __restrict__ RsPrep, double* __restrict__ partials,
              int64_t ntiles, double* __restrict__ Ydump)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int LDT = TM + 4, NT = NW * 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int P = n16 >> 4, NS = P * (P + 1) / 2;
    const int per_warp = (NS - warp + NW - 1) / NW;            // super-blocks of this warp
    const int sweeps = (per_warp + GRAM_MAXS - 1) / GRAM_MAXS;
    const bool persist = ((NS + NW - 1) / NW) <= GRAM_MAXS;    // uniform over the CTA
    double* part = partials + (size_t)blockIdx.x * n16 * n16;
    constexpr int FLUSH_TILES = GRAM_CHAIN * 4 / TM;

    double acc[GRAM_MAXS][4][2];
#pragma unroll
    for (int u = 0; u < GRAM_MAXS; ++u)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[u][b][0] = acc[u][b][1] = 0.0;
    bool first_flush = true;
    int since_flush = 0;

    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t row0 = tile * TM;
        __syncthreads();                                        // previous tile fully consumed
        load_tile<TM, NT, VEC>(Ysm, A, lda, m, n, n16, row0);
        __syncthreads();
        solve_tile<TM, NW>(Ysm, RsPrep, n16);
        __syncthreads();
        if (Ydump) store_tile<TM, NT, false>(Ysm, Ydump, m, m, n, row0);
        const bool last_tile = (tile + gridDim.x >= ntiles);
        ++since_flush;
        for (int sw = 0; sw < sweeps; ++sw) {
            int pp[GRAM_MAXS], qq[GRAM_MAXS];
            const int cnt = min(GRAM_MAXS, per_warp - sw * GRAM_MAXS);
#pragma unroll
            for (int u = 0; u < GRAM_MAXS; ++u) {
                pp[u] = qq[u] = 0;
                if (u < cnt) sb_to_pq(warp + NW * (sw * GRAM_MAXS + u), pp[u], qq[u]);
            }
            for (int ks = 0; ks < TM / 4; ++ks) {
                const double* yk = Ysm + g * LDT + 4 * ks + t;          // fragment (i = g, row = t)
#pragma unroll
                for (int u = 0; u < GRAM_MAXS; ++u) {
                    if (u < cnt) {
                        const double fa0 = yk[(16 * pp[u]) * LDT], fa1 = yk[(16 * pp[u] + 8) * LDT];
                        double fb0 = fa0, fb1 = fa1;
                        if (pp[u] != qq[u]) { fb0 = yk[(16 * qq[u]) * LDT]; fb1 = yk[(16 * qq[u] + 8) * LDT]; }
                        dmma884(acc[u][0], fa0, fb0);
                        dmma884(acc[u][1], fa0, fb1);
                        if (pp[u] != qq[u]) dmma884(acc[u][2], fa1, fb0);
                        dmma884(acc[u][3], fa1, fb1);
                    }
                }
            }
            const bool flush = !persist || last_tile || since_flush >= FLUSH_TILES;
            if (flush) {
#pragma unroll
                for (int u = 0; u < GRAM_MAXS; ++u) {
                    if (u < cnt) {
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            if (b == 2 && pp[u] == qq[u]) continue;
                            const int I = 2 * pp[u] + (b >> 1), J = 2 * qq[u] + (b & 1);
                            double* dst = part + (size_t)(8 * J + 2 * t) * n16 + 8 * I + g;
                            if (first_flush) { dst[0] = acc[u][b][0]; dst[n16] = acc[u][b][1]; }
                            else { dst[0] += acc[u][b][0]; dst[n16] += acc[u][b][1]; }
                            acc[u][b][0] = acc[u][b][1] = 0.0;
                        }
                    }
                }
            }
        }
        if (!persist || since_flush >= FLUSH_TILES) { first_flush = false; since_flush = 0; }
    }
}

template <int TM, int NW, bool VEC>
__global__ void __launch_bounds__(NW * 32)
mrcqr_k5_formq(int64_t m, int n, int n16, int64_t lda, const double* __restrict__ A,
               const double* __restrict__ RsPrep, const double* __restrict__ RcPrep,
               int64_t ldq, double* __restrict__ Q, int64_t ntiles, double* __restrict__ Ydump)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int NT = NW * 32;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t row0 = tile * TM;
        __syncthreads();
        load_tile<TM, NT, VEC>(Ysm, A, lda, m, n, n16, row0);
        __syncthreads();
        solve_tile<TM, NW>(Ysm, RsPrep, n16);                  // y = a Rs^-1, same code as K3
        if (Ydump) { __syncthreads(); store_tile<TM, NT, false>(Ysm, Ydump, m, m, n, row0); __syncthreads(); }
        solve_tile<TM, NW>(Ysm, RcPrep, n16);                  // q = y Rc^-1
        __syncthreads();
        store_tile<TM, NT, VEC>(Ysm, Q, ldq, m, n, row0);
    }
}

// G16[i,j] (i <= j) = sum over CTA partials in a fixed two-level order; mirrored to the lower part.
__global__ void mrcqr_reduce_partials(const double* __restrict__ partials, int np, int n16, double* __restrict__ G16)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n16 * n16) return;
    const int i = e % n16, j = e / n16;
    if (i > j) return;
    const size_t stride = (size_t)n16 * n16;
    double total = 0.0;
    for (int c0 = 0; c0 < np; c0 += 16) {
        double sub = 0.0;
        const int c1 = min(np, c0 + 16);
        for (int c = c0; c < c1; ++c) sub += partials[(size_t)c * stride + e];
        total += sub;
    }
    G16[e] = total;
    G16[(size_t)i * n16 + j] = total;
}

// ------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------
int num_sms()
{
    static int sms = 0;
    if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); }
    return sms;
}

size_t k3_partials_bytes(int n)
{
    RowCfg c = row_config(n);
    // at most 4 resident CTAs per SM are ever launched
    return (size_t)num_sms() * 4 * (size_t)c.n16 * c.n16 * sizeof(double);
}

template <typename K>
static int grid_for(K kernel, int threads, int smem, int64_t ntiles)
{
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    int occ = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem);
    if (occ < 1) occ = 1;
    if (occ > 4) occ = 4;
    int64_t g = (int64_t)occ * num_sms();
    return (int)(g < ntiles ? g : ntiles);
}

static bool vec_ok(const void* p, int64_t ld) { return ((uintptr_t)p % 16 == 0) && (ld % 2 == 0); }

#define MRCQR_ROW_DISPATCH(CALL)                                                     \
    if (c.TM == 128 && c.NW == 4) { if (vec) { CALL(128, 4, true) } else { CALL(128, 4, false) } }      \
    else if (c.TM == 128 && c.NW == 8) { if (vec) { CALL(128, 8, true) } else { CALL(128, 8, false) } } \
    else if (c.TM == 64) { if (vec) { CALL(64, 8, true) } else { CALL(64, 8, false) } }                 \
    else { if (vec) { CALL(32, 4, true) } else { CALL(32, 4, false) } }

int launch_k3_gram(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                   double* partials, int* n_partials_out, double* Ydump, cudaStream_t s)
{
    RowCfg c = row_config(n);
    const int64_t ntiles = (m + c.TM - 1) / c.TM;
    const bool vec = vec_ok(A, lda);
#define K3_CALL(TM_, NW_, V_)                                                                       \
    { auto k = mrcqr_k3_gram<TM_, NW_, V_>;                                                         \
      int grid = grid_for(k, NW_ * 32, c.smem_bytes, ntiles); *n_partials_out = grid;               \
      k<<<grid, NW_ * 32, c.smem_bytes, s>>>(m, n, c.n16, lda, A, RsPrep, partials, ntiles, Ydump); }
    MRCQR_ROW_DISPATCH(K3_CALL)
#undef K3_CALL
    return 1;
}

int launch_k5_formq(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                    const double* RcPrep, int64_t ldq, double* Q, double* Ydump, cudaStream_t s)
{
    RowCfg c = row_config(n);
    const int64_t ntiles = (m + c.TM - 1) / c.TM;
    const bool vec = vec_ok(A, lda) && vec_ok(Q, ldq);
#define K5_CALL(TM_, NW_, V_)                                                                       \
    { auto k = mrcqr_k5_formq<TM_, NW_, V_>;                                                        \
      int grid = grid_for(k, NW_ * 32, c.smem_bytes, ntiles);                                       \
      k<<<grid, NW_ * 32, c.smem_bytes, s>>>(m, n, c.n16, lda, A, RsPrep, RcPrep, ldq, Q, ntiles, Ydump); }
    MRCQR_ROW_DISPATCH(K5_CALL)
#undef K5_CALL
    return 1;
}

int launch_reduce_partials(const double* partials, int n_partials, int n, int n16, double* G16, cudaStream_t s)
{
    (void)n;
    const int total = n16 * n16;
    mrcqr_reduce_partials<<<(total + 255) / 256, 256, 0, s>>>(partials, n_partials, n16, G16);
    return 1;
}

} // namespace mrcqr
