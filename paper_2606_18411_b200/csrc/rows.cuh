// rows.cuh -- device building blocks of the two row-streaming passes (K3: precondition + Gram,
// K5: form Q).  A CTA owns a tile of TM consecutive rows of A, held column-major in shared memory
// as Ysm[col * LDT + row], LDT = TM + 4 (LDT = 4 mod 16 makes every DMMA fragment load hit 16
// distinct 8-byte banks per half warp).
//
// solve_tile() is THE forward substitution  Y <- Y * R^-1  (Algorithm 2 step 7, and
// Algorithm 1 step 3).  K3 and K5 both call this one function with the same template
// arguments and the same prepared factor, and every floating-point operation in it is an explicit
// DMMA, fma or multiply, so the Y a row gets in K5 is bit-identical to the Y K3 fed to the Gram
// matrix.  The result for a row does not depend on which tile slot,
// warp or CTA holds it: each row's arithmetic touches only that row's data and R.
#pragma once
#include "mrcqr_internal.cuh"

namespace mrcqr {

// D(8x8) += A(8x4, row) * B(4x8, col), FP64 tensor-core op (SASS: DMMA.8x8x4 on sm_100a).
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// 16-byte asynchronous global -> shared copy (SASS: LDGSTS), src_bytes < 16 zero-fills the rest.
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, int src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Cooperative load of rows [row0, row0+TM) x n columns of A into the tile; zero fill for rows >= m
// and for the padding columns n..n16-1.  VEC (A, lda, row0 16-byte aligned): every thread fires all
// of its 16-byte cp.async copies back to back, so the whole tile is in flight at once (no register
// staging, memory-level parallelism = tile size); the caller waits with cp_async_wait_all().
template <int TM, int NT, bool VEC>
__device__ __forceinline__ void load_tile(double* Ysm, const double* __restrict__ A, int64_t lda,
                                          int64_t m, int n, int n16, int64_t row0)
{
    constexpr int LDT = TM + 4;
    if (VEC) {
        constexpr int H = TM / 2;
        const int64_t left = m - row0;                  // rows available in this tile (may exceed TM)
#pragma unroll 8
        for (int e = threadIdx.x; e < n * H; e += NT) {
            const int col = e / H, r2 = (e % H) * 2;
            const int64_t avail = left - r2;
            const int bytes = avail >= 2 ? 16 : (avail == 1 ? 8 : 0);
            const double* src = A + (size_t)col * (size_t)lda + row0 + (bytes ? r2 : 0);
            cp_async16(Ysm + col * LDT + r2, src, bytes);
        }
        for (int e = threadIdx.x; e < (n16 - n) * H; e += NT) {
            const int col = n + e / H, r2 = (e % H) * 2;
            *reinterpret_cast<double2*>(Ysm + col * LDT + r2) = make_double2(0.0, 0.0);
        }
        cp_async_wait_all();
    } else {
        for (int e = threadIdx.x; e < n16 * TM; e += NT) {
            int col = e / TM, rr = e % TM;
            int64_t r = row0 + rr;
            double v = 0.0;
            if (col < n && r < m) v = __ldcs(A + (size_t)col * (size_t)lda + r);
            Ysm[col * LDT + rr] = v;
        }
    }
}

// Cooperative store of the tile (first n columns, rows < m) to a column-major m x n matrix.
template <int TM, int NT, bool VEC>
__device__ __forceinline__ void store_tile(const double* Ysm, double* __restrict__ Q, int64_t ldq,
                                           int64_t m, int n, int64_t row0)
{
    constexpr int LDT = TM + 4;
    if (VEC) {
        constexpr int H = TM / 2;
        for (int e = threadIdx.x; e < n * H; e += NT) {
            int col = e / H, r2 = (e % H) * 2;
            int64_t r = row0 + r2;
            double2 v = *reinterpret_cast<const double2*>(Ysm + col * LDT + r2);
            double* dst = Q + (size_t)col * (size_t)ldq + r;
            if (r + 1 < m) __stcs(reinterpret_cast<double2*>(dst), v);
            else if (r < m) __stcs(dst, v.x);
        }
    } else {
        for (int e = threadIdx.x; e < n * TM; e += NT) {
            int col = e / TM, rr = e % TM;
            int64_t r = row0 + rr;
            if (r < m) __stcs(Q + (size_t)col * (size_t)ldq + r, Ysm[col * LDT + rr]);
        }
    }
}

// Copies the 8x8 diagonal blocks of a prepared factor into shared memory: Dsm[J*64 + jj*8 + j] =
// Rp[8J+j, 8J+jj] (column-major 8x8 per block), so the substitution reads them as broadcast LDS.128.
template <int NT>
__device__ __forceinline__ void load_diag_blocks(double* Dsm, const double* __restrict__ Rp, int n16)
{
    for (int e = threadIdx.x; e < n16 * 8; e += NT) {
        const int J = e >> 6, jj = (e >> 3) & 7, j = e & 7;
        Dsm[e] = __ldg(Rp + (size_t)(8 * J + jj) * n16 + 8 * J + j);
    }
}

// 8x8 substitution of block J for the rows of this warp, one thread per row:
//   y_j = t_j / R[j,j],  t_jj -= y_j R[j,jj]  (jj > j), coefficients from the shared diagonal blocks.
template <int TM, int RG>
__device__ __forceinline__ void diag_block(double* Ysm, const double* Dsm, int J, int rbase, int lane)
{
    constexpr int LDT = TM + 4;
    double d[8][8];
    const double2* dp = reinterpret_cast<const double2*>(Dsm + J * 64);
#pragma unroll
    for (int jj = 0; jj < 8; ++jj)
#pragma unroll
        for (int h = 0; h <= jj / 2; ++h) {
            const double2 v = dp[jj * 4 + h];
            d[jj][2 * h] = v.x; d[jj][2 * h + 1] = v.y;
        }
    if (lane < 8 * RG) {
        double* yr = Ysm + (8 * J) * LDT + rbase + lane;
        double y[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) y[j] = yr[j * LDT];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            y[j] = y[j] * d[j][j];                                     // times 1/R[j,j]
#pragma unroll
            for (int jj = j + 1; jj < 8; ++jj) y[jj] = fma(y[j], d[jj][j], y[jj]);   // -R[j,jj]
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) yr[j * LDT] = y[j];
    }
}

// In-place Y <- Y * R^-1 on the rows owned by this warp (8*RG rows starting at warp*8*RG).
// Rp is the prepared factor (see mrcqr_internal.cuh): strict upper = -R, diagonal = 1/R[j,j];
// Dsm its diagonal blocks in shared memory (load_diag_blocks).
// Left-looking over PAIRS of 8-column blocks (J0, J1 = J0 + 1), so every A fragment read from shared
// memory feeds two DMMAs (shared-memory bandwidth, not the FP64 pipe, was the first limit):
//   T_J0, T_J1 += Y_K * (-R[K,J0]), Y_K * (-R[K,J1])   K < J0      DMMA.8x8x4, fragments prefetched
//   Y_J0 = T_J0 * R[J0,J0]^-1                                      8x8 substitution, thread per row
//   T_J1 += Y_J0 * (-R[J0,J1]);  Y_J1 = T_J1 * R[J1,J1]^-1
// Fragment conventions (fixed, so the summation order is fixed): in a DMMA lane (g, t) supplies
// k = t and k = t + 4; accumulator column 2t+e of the hardware layout carries matrix column t + 4e
// of the block (B fragment lane g loads column (g>>1) + 4(g&1)), which makes the accumulator's
// shared-memory loads and stores bank-conflict free with LDT = 4 mod 16.
template <int TM, int NW>
__device__ __forceinline__ void solve_tile(double* Ysm, const double* __restrict__ Rp,
                                           const double* Dsm, int n16)
{
    constexpr int LDT = TM + 4;
    constexpr int RG = TM / (8 * NW);                 // 8-row groups per warp
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int rbase = warp * (8 * RG);
    const int nB = n16 >> 3;
    const int csel = (g >> 1) + 4 * (g & 1);           // matrix column carried by hardware column g
    const double* ya = Ysm + t * LDT + rbase + g;      // A fragment base: (m = g, k = t)

    for (int J0 = 0; J0 < nB; J0 += 2) {
        const int J1 = J0 + 1;
        double cA[RG][2], cB[RG][2];
        double* colA = Ysm + (8 * J0 + t) * LDT + rbase + g;           // accumulator element e: + 4e*LDT
        double* colB = colA + 8 * LDT;
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
            cA[rg][0] = colA[8 * rg]; cA[rg][1] = colA[4 * LDT + 8 * rg];
            cB[rg][0] = colB[8 * rg]; cB[rg][1] = colB[4 * LDT + 8 * rg];
        }
        const double* rA = Rp + (size_t)(8 * J0 + csel) * n16 + t;     // B fragments: (k = t, n = g)
        const double* rB = rA + (size_t)8 * n16;
        if (J0 > 0) {
            double a0[RG], a1[RG];
            double bA0 = __ldg(rA), bA1 = __ldg(rA + 4), bB0 = __ldg(rB), bB1 = __ldg(rB + 4);
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) { a0[rg] = ya[8 * rg]; a1[rg] = ya[4 * LDT + 8 * rg]; }
            for (int K = 0; K < J0; ++K) {
                const int Kn = (K + 1 < J0) ? K + 1 : K;               // prefetch (re-reads the last one)
                const double nA0 = __ldg(rA + 8 * Kn), nA1 = __ldg(rA + 8 * Kn + 4);
                const double nB0 = __ldg(rB + 8 * Kn), nB1 = __ldg(rB + 8 * Kn + 4);
                const double* yn = ya + 8 * Kn * LDT;
                double n0[RG], n1[RG];
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) { n0[rg] = yn[8 * rg]; n1[rg] = yn[4 * LDT + 8 * rg]; }
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) dmma884(cA[rg], a0[rg], bA0);
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) dmma884(cB[rg], a0[rg], bB0);
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) dmma884(cA[rg], a1[rg], bA1);
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) dmma884(cB[rg], a1[rg], bB1);
                bA0 = nA0; bA1 = nA1; bB0 = nB0; bB1 = nB1;
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) { a0[rg] = n0[rg]; a1[rg] = n1[rg]; }
            }
        }
        // ---- block J0
        const double xB0 = __ldg(rB + 8 * J0), xB1 = __ldg(rB + 8 * J0 + 4);    // -R[J0, J1] fragments
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) { colA[8 * rg] = cA[rg][0]; colA[4 * LDT + 8 * rg] = cA[rg][1]; }
        __syncwarp();
        diag_block<TM, RG>(Ysm, Dsm, J0, rbase, lane);
        __syncwarp();
        // ---- cross term and block J1
        {
            const double* yj = ya + 8 * J0 * LDT;
            double a0[RG], a1[RG];
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) { a0[rg] = yj[8 * rg]; a1[rg] = yj[4 * LDT + 8 * rg]; }
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) dmma884(cB[rg], a0[rg], xB0);
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) dmma884(cB[rg], a1[rg], xB1);
        }
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) { colB[8 * rg] = cB[rg][0]; colB[4 * LDT + 8 * rg] = cB[rg][1]; }
        __syncwarp();
        diag_block<TM, RG>(Ysm, Dsm, J1, rbase, lane);
        __syncwarp();
    }
}

} // namespace mrcqr
