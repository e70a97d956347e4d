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
    c.smem_bytes = c.n16 * (c.TM + 4) * 8 + 2 * c.n16 * 64;   // tile + diagonal blocks of Rs and Rc
    c.ctas_per_sm = 0;
    return c;
}

__device__ __forceinline__ void sb_to_pq(int sb, int& p, int& q)
{
    int qq = 0;
    while ((qq + 1) * (qq + 2) / 2 <= sb) ++qq;
    q = qq; p = sb - qq * (qq + 1) / 2;
}

// ---- Gram accumulation, "row pair" scheme (n16 <= 16 * NW) -----------------------------------------
// Warp w owns the 8x8 blocks (r, r..nB-1) and (r2, r2..nB-1) of the upper triangle, r = w,
// r2 = nB-1-w: nB+1 blocks for every warp (perfect balance), accumulators stay in registers for the
// CTA's whole life, one fragment load per block column serves both rows.
template <int TM, int NBMAX>
struct GramPair {
    static constexpr int NH = NBMAX / 2;
    double acc1[NBMAX][2];      // block (r,  r + cc),      cc = 0 .. nB-1-r
    double acc2[NH][2];         // block (r2, nB-1 - e),    e  = 0 .. nB-1-r2 (= r)   -- indexed from the end
    __device__ __forceinline__ void zero()
    {
#pragma unroll
        for (int b = 0; b < NBMAX; ++b) acc1[b][0] = acc1[b][1] = 0.0;
#pragma unroll
        for (int b = 0; b < NH; ++b) acc2[b][0] = acc2[b][1] = 0.0;
    }
    // r < r2, or r == r2 (odd nB, middle row: acc2 unused); warps with r > r2 own nothing.
    // Every register array is indexed by unrolled loop counters only (no local memory).
    __device__ __forceinline__ void accumulate(const double* Ysm, int nB, int r, int r2)
    {
        constexpr int LDT = TM + 4;
        const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
        if (r > r2) return;
        const int ne = (r2 != r) ? (nB - r2) : 0;
        const double* y0 = Ysm + g * LDT + t;
#pragma unroll 2
        for (int ks = 0; ks < TM / 4; ++ks) {
            const double* yk = y0 + 4 * ks;
            double f[NBMAX], fe[NH];
#pragma unroll
            for (int cc = 0; cc < NBMAX; ++cc) f[cc] = (r + cc < nB) ? yk[(8 * (r + cc)) * LDT] : 0.0;
#pragma unroll
            for (int e = 0; e < NH; ++e) fe[e] = (e < ne) ? yk[(8 * (nB - 1 - e)) * LDT] : 0.0;
            const double fr2 = yk[(8 * r2) * LDT];
#pragma unroll
            for (int cc = 0; cc < NBMAX; ++cc)
                if (r + cc < nB) dmma884(acc1[cc], f[0], f[cc]);
#pragma unroll
            for (int e = 0; e < NH; ++e)
                if (e < ne) dmma884(acc2[e], fr2, fe[e]);
        }
    }
    __device__ __forceinline__ void flush(double* part, int n16, int nB, int r, int r2, bool first)
    {
        const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
        if (r > r2) return;
        const int ne = (r2 != r) ? (nB - r2) : 0;
#pragma unroll
        for (int cc = 0; cc < NBMAX; ++cc) {
            if (r + cc < nB) {
                double* dst = part + (size_t)(8 * (r + cc) + 2 * t) * n16 + 8 * r + g;
                if (first) { dst[0] = acc1[cc][0]; dst[n16] = acc1[cc][1]; }
                else { dst[0] += acc1[cc][0]; dst[n16] += acc1[cc][1]; }
                acc1[cc][0] = acc1[cc][1] = 0.0;
            }
        }
#pragma unroll
        for (int e = 0; e < NH; ++e) {
            if (e < ne) {
                double* dst = part + (size_t)(8 * (nB - 1 - e) + 2 * t) * n16 + 8 * r2 + g;
                if (first) { dst[0] = acc2[e][0]; dst[n16] = acc2[e][1]; }
                else { dst[0] += acc2[e][0]; dst[n16] += acc2[e][1]; }
                acc2[e][0] = acc2[e][1] = 0.0;
            }
        }
    }
};

// G partial of this CTA: n16 x n16 col-major, blocks (I <= J) of the upper triangle only.
template <int TM, int NW, bool VEC>
__global__ void __launch_bounds__(NW * 32, (TM == 128 && NW == 4) ? 3 : 1)
mrcqr_k3_gram(int64_t m, int n, int n16, int64_t lda, const double* __restrict__ A,
              const double* __restrict__ RsPrep, double* __restrict__ partials,
              int64_t ntiles, double* __restrict__ Ydump)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int LDT = TM + 4, NT = NW * 32;
    constexpr bool PAIR = (TM == 128);                         // n16 <= 16 * NW for both TM = 128 shapes
    double* Dsm = Ysm + (size_t)n16 * LDT;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int nB = n16 >> 3;
    double* part = partials + (size_t)blockIdx.x * n16 * n16;
    constexpr int FLUSH_TILES = GRAM_CHAIN * 4 / TM;
    load_diag_blocks<NT>(Dsm, RsPrep, n16);

    if (PAIR) {
        GramPair<TM, 2 * NW> gp;
        gp.zero();
        const int r = warp, r2 = nB - 1 - warp;
        bool first = true;
        int since = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int64_t row0 = tile * TM;
            __syncthreads();
            load_tile<TM, NT, VEC>(Ysm, A, lda, m, n, n16, row0);
            __syncthreads();
            solve_tile<TM, NW>(Ysm, RsPrep, Dsm, n16);
            __syncthreads();
            if (Ydump) store_tile<TM, NT, false>(Ysm, Ydump, m, m, n, row0);
            gp.accumulate(Ysm, nB, r, r2);
            ++since;
            if (since >= FLUSH_TILES || tile + gridDim.x >= ntiles) {
                gp.flush(part, n16, nB, r, r2, first);
                first = false; since = 0;
            }
        }
        return;
    }

    // ---- super-block sweeps (n16 > 128): 16x16 super-blocks, flushed to the L2-resident partial every tile
    const int P = n16 >> 4, NS = P * (P + 1) / 2;
    const int per_warp = (NS - warp + NW - 1) / NW;
    const int sweeps = (per_warp + GRAM_MAXS - 1) / GRAM_MAXS;
    bool first_tile = true;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t row0 = tile * TM;
        __syncthreads();
        load_tile<TM, NT, VEC>(Ysm, A, lda, m, n, n16, row0);
        __syncthreads();
        solve_tile<TM, NW>(Ysm, RsPrep, Dsm, n16);
        __syncthreads();
        if (Ydump) store_tile<TM, NT, false>(Ysm, Ydump, m, m, n, row0);
        for (int sw = 0; sw < sweeps; ++sw) {
            double acc[GRAM_MAXS][4][2];
            int pp[GRAM_MAXS], qq[GRAM_MAXS];
            const int cnt = min(GRAM_MAXS, per_warp - sw * GRAM_MAXS);
#pragma unroll
            for (int u = 0; u < GRAM_MAXS; ++u) {
                pp[u] = qq[u] = 0;
                if (u < cnt) sb_to_pq(warp + NW * (sw * GRAM_MAXS + u), pp[u], qq[u]);
#pragma unroll
                for (int b = 0; b < 4; ++b) acc[u][b][0] = acc[u][b][1] = 0.0;
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
#pragma unroll
            for (int u = 0; u < GRAM_MAXS; ++u) {
                if (u < cnt) {
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        if (b == 2 && pp[u] == qq[u]) continue;
                        const int I = 2 * pp[u] + (b >> 1), J = 2 * qq[u] + (b & 1);
                        double* dst = part + (size_t)(8 * J + 2 * t) * n16 + 8 * I + g;
                        if (first_tile) { dst[0] = acc[u][b][0]; dst[n16] = acc[u][b][1]; }
                        else { dst[0] += acc[u][b][0]; dst[n16] += acc[u][b][1]; }
                    }
                }
            }
        }
        first_tile = false;
    }
}

template <int TM, int NW, bool VEC>
__global__ void __launch_bounds__(NW * 32, (TM == 128 && NW == 4) ? 3 : 1)
mrcqr_k5_formq(int64_t m, int n, int n16, int64_t lda, const double* __restrict__ A,
               const double* __restrict__ RsPrep, const double* __restrict__ RcPrep,
               int64_t ldq, double* __restrict__ Q, int64_t ntiles, double* __restrict__ Ydump)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int LDT = TM + 4, NT = NW * 32;
    double* DsmS = Ysm + (size_t)n16 * LDT;
    double* DsmC = DsmS + (size_t)n16 * 8;
    load_diag_blocks<NT>(DsmS, RsPrep, n16);
    load_diag_blocks<NT>(DsmC, RcPrep, n16);
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t row0 = tile * TM;
        __syncthreads();
        load_tile<TM, NT, VEC>(Ysm, A, lda, m, n, n16, row0);
        __syncthreads();
        solve_tile<TM, NW>(Ysm, RsPrep, DsmS, n16);            // y = a Rs^-1, same code as K3
        if (Ydump) { __syncthreads(); store_tile<TM, NT, false>(Ysm, Ydump, m, m, n, row0); __syncthreads(); }
        solve_tile<TM, NW>(Ysm, RcPrep, DsmC, n16);            // q = y Rc^-1
        __syncthreads();
        store_tile<TM, NT, VEC>(Ysm, Q, ldq, m, n, row0);
    }
}

// G16[i,j] (i <= j) = sum over the CTA partials in a FIXED order (deterministic split-m reduction):
// partials are taken in groups of 16 consecutive CTAs summed in order; thread q of an element adds the
// groups q, q+8, q+16, ... in order; the 8 per-thread sums are combined by a fixed binary tree.
// 32 elements x 8 group lanes per CTA; mirrored to the lower triangle.
__global__ void __launch_bounds__(256)
mrcqr_reduce_partials(const double* __restrict__ partials, int np, int n16, double* __restrict__ G16)
{
    __shared__ double sm[8][33];
    const int el = threadIdx.x & 31, q = threadIdx.x >> 5;
    const int e = blockIdx.x * 32 + el;
    const size_t stride = (size_t)n16 * n16;
    const int i = e % n16, j = e / n16;
    const bool live = (e < n16 * n16) && (i <= j);
    double total = 0.0;
    if (live) {
        for (int c0 = 16 * q; c0 < np; c0 += 16 * 8) {
            double sub = 0.0;
            const int c1 = min(np, c0 + 16);
            for (int c = c0; c < c1; ++c) sub += partials[(size_t)c * stride + e];
            total += sub;
        }
    }
    sm[q][el] = total;
    __syncthreads();
    if (q == 0 && live) {
        const double t = ((sm[0][el] + sm[1][el]) + (sm[2][el] + sm[3][el])) + ((sm[4][el] + sm[5][el]) + (sm[6][el] + sm[7][el]));
        G16[e] = t;
        G16[(size_t)i * n16 + j] = t;
    }
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
    mrcqr_reduce_partials<<<(total + 31) / 32, 256, 0, s>>>(partials, n_partials, n16, G16);
    return 1;
}

} // namespace mrcqr
