// rows.cuh -- device building blocks of the two row-streaming passes (K3: precondition + Gram,
// K5: form Q).
//
// Geometry.  A warp owns a SLAB of SR = 8*RG consecutive rows of A, held column-major in shared
// memory as slab[col * LDS_ + row], LDS_ = SR + 4 (LDS_ = 4 or 12 mod 16 makes every DMMA fragment
// access below hit 16 distinct 8-byte banks per half warp).  A CTA tile is NW slabs.
//
// solve_slab() is THE forward substitution  Y <- Y * R^-1  (Algorithm 2 step 7, and
// Algorithm 1 step 3).  K3 and K5 both call this one function with the same template
// arguments and the same prepared factor, and every floating-point operation in it is an explicit
// DMMA, fma or multiply, so the Y a row gets in K5 is bit-identical to the Y K3 fed to the Gram
// matrix.  The result for a row does not depend on which slab slot,
// warp or CTA holds it: each row's arithmetic touches only that row's data and R.
//
// The solve is register resident: a panel of up to 8 column blocks (64 columns) of the slab lives in
// DMMA accumulator registers.  Columns left of the panel contribute through a left-looking sweep
// (A fragments = solved Y from the slab, B fragments = -R in fragment order from L1/L2); inside the
// panel the sweep is right-looking and the accumulator registers of a solved block ARE the A
// fragments of its updates (fragment conventions below), so the panel never leaves the register
// file except for the 8x8 diagonal substitutions, which run one thread per row through the slab.
#pragma once
#include "mrcqr_internal.cuh"

namespace mrcqr {

// Diagonal 8x8 blocks of the two prepared factors (FAC 0: R_s, FAC 1: R_c), 36 doubles per block:
// [0..8) 1/R[j,j], then -R[j,jj] for j < jj, j-major.  Constant memory: the thread-per-row
// substitution reads them with warp-uniform addresses, off the shared-memory pipe.
#ifndef MRCQR_NO_CONST_DIAG
__constant__ __align__(16) double c_diag[2][PREP_MAX_NB * PREP_DIAG];
#endif

__host__ __device__ constexpr int diag_off(int j, int jj) { return 8 + j * 7 - j * (j - 1) / 2 + (jj - j - 1); }

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
// the same with an L2 eviction policy (createpolicy): for data that is read once while other lines should stay in L2
__device__ __forceinline__ void cp_async16_hint(void* smem_dst, const void* gmem_src, int src_bytes, uint64_t policy)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(d), "l"(gmem_src), "r"(src_bytes), "l"(policy) : "memory");
}
__device__ __forceinline__ uint64_t l2_evict_first_policy()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}

// Warp-cooperative load of rows [row0, row0+SR) x n columns of A into this warp's slab; zero fill
// for rows >= m.  The padding columns n..n16-1 are zeroed once by zero_pad_columns().  VEC (A, lda
// 16-byte aligned): every lane fires all of its 16-byte cp.async copies back to back, so the whole
// slab is in flight at once; the caller waits with cp_async_wait_all() + __syncwarp().
template <int SR, bool VEC>
__device__ __forceinline__ void load_slab(double* slab, const double* __restrict__ A, int64_t lda,
                                          int64_t m, int n, int64_t row0, int lane)
{
    constexpr int LDS_ = SR + 4;
    if (VEC) {
        constexpr int H = SR / 2;                       // 16-byte chunks per column
        const int64_t left = m - row0;
#pragma unroll 8
        for (int e = lane; e < n * H; e += 32) {
            const int col = e / H, r2 = (e % H) * 2;
            const int64_t avail = left - r2;
            const int bytes = avail >= 2 ? 16 : (avail == 1 ? 8 : 0);
            const double* src = A + (size_t)col * (size_t)lda + row0 + (bytes ? r2 : 0);
            cp_async16(slab + col * LDS_ + r2, src, bytes);
        }
    } else {
        for (int e = lane; e < n * SR; e += 32) {
            const int col = e / SR, rr = e % SR;
            const int64_t r = row0 + rr;
            slab[col * LDS_ + rr] = (r < m) ? __ldcs(A + (size_t)col * (size_t)lda + r) : 0.0;
        }
    }
}

// load_slab<SR, true> with every line marked evict-first in L2 (a source that is read exactly once)
template <int SR>
__device__ __forceinline__ void load_slab_once(double* slab, const double* __restrict__ A, int64_t lda,
                                               int64_t m, int n, int64_t row0, int lane, uint64_t policy)
{
    constexpr int LDS_ = SR + 4, H = SR / 2;
    const int64_t left = m - row0;
#pragma unroll 8
    for (int e = lane; e < n * H; e += 32) {
        const int col = e / H, r2 = (e % H) * 2;
        const int64_t avail = left - r2;
        const int bytes = avail >= 2 ? 16 : (avail == 1 ? 8 : 0);
        const double* src = A + (size_t)col * (size_t)lda + row0 + (bytes ? r2 : 0);
        cp_async16_hint(slab + col * LDS_ + r2, src, bytes, policy);
    }
}

template <int SR>
__device__ __forceinline__ void zero_pad_columns(double* slab, int n, int n16, int lane)
{
    constexpr int LDS_ = SR + 4;
    for (int e = lane; e < (n16 - n) * SR; e += 32) slab[(n + e / SR) * LDS_ + e % SR] = 0.0;
}

// Warp-cooperative store of the slab (first n columns, rows < m) to a column-major m x n matrix.
template <int SR, bool VEC>
__device__ __forceinline__ void store_slab(const double* slab, double* __restrict__ Q, int64_t ldq,
                                           int64_t m, int n, int64_t row0, int lane)
{
    constexpr int LDS_ = SR + 4;
    if (VEC) {
        constexpr int H = SR / 2;
#pragma unroll 4
        for (int e = lane; e < n * H; e += 32) {
            const int col = e / H, r2 = (e % H) * 2;
            const int64_t r = row0 + r2;
            const double2 v = *reinterpret_cast<const double2*>(slab + col * LDS_ + r2);
            double* dst = Q + (size_t)col * (size_t)ldq + r;
            if (r + 1 < m) __stcs(reinterpret_cast<double2*>(dst), v);
            else if (r < m) __stcs(dst, v.x);
        }
    } else {
        for (int e = lane; e < n * SR; e += 32) {
            const int col = e / SR, rr = e % SR;
            const int64_t r = row0 + rr;
            if (r < m) __stcs(Q + (size_t)col * (size_t)ldq + r, slab[col * LDS_ + rr]);
        }
    }
}

// 8x8 substitution of one diagonal block for one row, in registers:
//   y_jj = t_jj / R[jj,jj] + sum_{j<jj} y_j * (-R[j,jj] / R[jj,jj]),
// i.e. the columns are scaled first (8 independent multiplies) and the substitution is unit upper
// triangular: the dependent chain is 7 fma deep instead of 16 operations.  c: the block's 36 prepared
// coefficients (constant memory, warp-uniform).
__device__ __forceinline__ void diag_substitute(double (&y)[8], const double* c)
{
#pragma unroll
    for (int j = 0; j < 8; ++j) y[j] = y[j] * c[j];
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
        for (int jj = j + 1; jj < 8; ++jj) y[jj] = fma(y[j], c[diag_off(j, jj)], y[jj]);
}

// Fragment conventions (fixed, so the summation order is fixed).  DMMA.8x8x4: lane (g, t) = (lane/4,
// lane%4) supplies A[m=g][k=t], B[k=t][n=g] and owns C[m=g][n=2t], C[m=g][n=2t+1].  Hardware column
// n = g carries matrix column csel(g) = (g>>1) + 4(g&1) of an 8-column block, so accumulator element
// e of lane (g, t) is matrix column t + 4e: exactly the two A-fragment values (k = t, k = t + 4) the
// same lane must supply when that block later multiplies -R[K, J].
// Prepared factor, fragment order: fragpair(K, J)[lane] = (-R[8K+t, 8J+csel(g)], -R[8K+t+4, 8J+csel(g)]).
__device__ __forceinline__ const double2* fragpair(const double2* __restrict__ frag, int Kg, int Jg, int lane)
{
    return frag + ((size_t)(Jg * (Jg - 1) / 2 + Kg) * 32 + lane);
}

// ---- where the prepared factor of a solve lives ---------------------------------------------------------
// ConstFactor: off-diagonal fragment pairs in global memory (read-only path, L1 / L2 resident), the diagonal blocks of
// factor FAC in constant memory.  SmemFactor: the whole prepared factor (layout of mrcqr_internal.cuh) in shared memory
// (the batched one-CTA-per-problem kernel, where every problem has factors of its own).  Same arithmetic either way.
#ifndef MRCQR_NO_CONST_DIAG
template <int FAC>
struct ConstFactor {
    const double2* __restrict__ frag;
    __device__ __forceinline__ double2 pair(int Kg, int Jg, int lane) const { return __ldg(fragpair(frag, Kg, Jg, lane)); }
    __device__ __forceinline__ const double* diag(int Kg) const { return &c_diag[FAC][Kg * PREP_DIAG]; }
    __device__ __forceinline__ void substitute(double (&y)[8], int P0, int K) const { diag_substitute(y, diag(P0 + K)); }
    __device__ __forceinline__ double2 pair_in(int P0, int K, int J, int lane) const { return pair(P0 + K, P0 + J, lane); }
};
#endif
#ifndef MRCQR_NO_CONST_DIAG
// PanelFactor: one 64-column panel starting at block P0 (the panel passes): off-diagonal pairs from global memory, the
// panel's own diagonal blocks at the START of c_pdiag[FAC] (uploaded per launch), so that block K of the panel has
// compile-time constant-bank offsets and the coefficients are instruction operands, not loads.
__constant__ double c_pdiag[2][8 * PREP_DIAG];
template <int FAC>
struct PanelFactor {
    const double2* __restrict__ frag; int P0;
    __device__ __forceinline__ double2 pair(int Kg, int Jg, int lane) const { return __ldg(fragpair(frag, Kg, Jg, lane)); }
    __device__ __forceinline__ const double* diag(int Kg) const { return &c_pdiag[FAC][(Kg - P0) * PREP_DIAG]; }
    __device__ __forceinline__ void substitute(double (&y)[8], int, int K) const { diag_substitute(y, &c_pdiag[FAC][K * PREP_DIAG]); }
    __device__ __forceinline__ double2 pair_in(int P0_, int K, int J, int lane) const { return pair(P0_ + K, P0_ + J, lane); }
};
// FusedFactor: all panels of a solve in ONE launch (mrcqr_panel_fused): the panel index p is a run-time value, so the
// substitution of block K of panel p is picked by a warp-uniform switch among NPMAX copies whose coefficients are
// compile-time offsets into c_diag[FAC] (instruction operands again, not indexed constant loads).
template <int FAC, int NPMAX>
struct FusedFactor {
    const double2* __restrict__ frag; int p;
    const double* dbase;                      // &c_diag[FAC][B0 * PREP_DIAG]: the panels start at block B0 (a ragged panel may come first)
    const double2* __restrict__ own;          // fragpair(frag, P0, P0, lane): the panel's own pairs start here
    unsigned jstride;                         // 32 P0: pair (P0 + K, P0 + J) sits at own + J jstride + 32 (J (J - 1) / 2 + K)
    __device__ __forceinline__ FusedFactor(const double2* f, int B0, int p_, int lane)
        : frag(f), p(p_), dbase(&c_diag[FAC][B0 * PREP_DIAG]),
          own(f + ((size_t)(B0 + 8 * p_) * (B0 + 8 * p_ - 1) / 2 + B0 + 8 * p_) * 32 + lane), jstride(32u * (unsigned)(B0 + 8 * p_)) {}
    __device__ __forceinline__ double2 pair(int Kg, int Jg, int lane) const { return __ldg(fragpair(frag, Kg, Jg, lane)); }
    // in-panel pair with compile-time K, J: one multiply-add on the address instead of the triangular index arithmetic
    __device__ __forceinline__ double2 pair_in(int, int K, int J, int) const
    { return __ldg(own + (size_t)jstride * (unsigned)J + (unsigned)(32 * (J * (J - 1) / 2 + K))); }
    __device__ __forceinline__ void substitute(double (&y)[8], int, int K) const
    {
        switch (p) {
            case 0: diag_substitute(y, dbase + (0 + K) * PREP_DIAG); break;
            case 1: diag_substitute(y, dbase + (8 + K) * PREP_DIAG); break;
            case 2: diag_substitute(y, dbase + (16 + K) * PREP_DIAG); break;
            case 3: diag_substitute(y, dbase + (24 + K) * PREP_DIAG); break;
            case 4: if (NPMAX > 4) diag_substitute(y, dbase + (32 + K) * PREP_DIAG); break;
            case 5: if (NPMAX > 4) diag_substitute(y, dbase + (40 + K) * PREP_DIAG); break;
            case 6: if (NPMAX > 4) diag_substitute(y, dbase + (48 + K) * PREP_DIAG); break;
            default: if (NPMAX > 4) diag_substitute(y, dbase + (56 + K) * PREP_DIAG); break;
        }
    }
};
#endif
struct SmemFactor {
    const double* prep; int nB;
    __device__ __forceinline__ double2 pair(int Kg, int Jg, int lane) const
    { return *reinterpret_cast<const double2*>(prep + 2 * ((size_t)(Jg * (Jg - 1) / 2 + Kg) * 32 + lane)); }
    __device__ __forceinline__ const double* diag(int Kg) const { return prep + prep_diag_offset(nB) + Kg * PREP_DIAG; }
    __device__ __forceinline__ void substitute(double (&y)[8], int P0, int K) const { diag_substitute(y, diag(P0 + K)); }
    __device__ __forceinline__ double2 pair_in(int P0, int K, int J, int lane) const { return pair(P0 + K, P0 + J, lane); }
};

// ---- where a block goes between its DMMA (accumulator) form and its one-thread-per-row form -------
// SlabXpose: through the block's own columns of the slab (leading dimension SR + 4); the solved block
// stays there (in-place solve).
template <int RG>
struct SlabXpose {
    static constexpr int SR = 8 * RG, LDS_ = SR + 4;
    static constexpr bool REUSE = false;      // every block has its own columns: no barrier before the next step
    double* slab; int lane, g, t;
    __device__ __forceinline__ SlabXpose(double* s, int l) : slab(s), lane(l), g(l >> 2), t(l & 3) {}
    __device__ __forceinline__ double* accp(int Kg, int rg, int e) const { return slab + (8 * Kg + t + 4 * e) * LDS_ + 8 * rg + g; }
    __device__ __forceinline__ double* rowp(int Kg, int j) const { return slab + (8 * Kg + j) * LDS_ + lane; }
    __device__ __forceinline__ bool row_active() const { return SR >= 32 || lane < SR; }
};
// ScratchXpose: through ONE per-warp scratch block (8 columns, leading dimension SR + 4) that every block of the panel
// reuses; the solved block goes to the sink (e.g. straight to global memory in row form), not to a slab.
template <int RG>
struct ScratchXpose {
    static constexpr int SR = 8 * RG, LDS_ = SR + 4;
    static constexpr bool REUSE = true;
    double* scr; int lane, g, t;
    __device__ __forceinline__ ScratchXpose(double* s, int l) : scr(s), lane(l), g(l >> 2), t(l & 3) {}
    __device__ __forceinline__ double* accp(int, int rg, int e) const { return scr + (t + 4 * e) * LDS_ + 8 * rg + g; }
    __device__ __forceinline__ double* rowp(int, int j) const { return scr + j * LDS_ + lane; }
    __device__ __forceinline__ bool row_active() const { return SR >= 32 || lane < SR; }
};
struct NoSink { __device__ __forceinline__ void operator()(int, const double (&)[8]) const {} };
// RowSink: a solved block leaves for a column-major matrix straight from its row form (lane = row of the slab: 256
// contiguous bytes per column and warp); out = &Q[row0 + lane], columns >= n and rows >= m are not written.
struct RowSink {
    double* out; int64_t ldq; int n; bool row_ok;
    __device__ __forceinline__ void operator()(int Kg, const double (&y)[8]) const
    {
        if (!row_ok) return;
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if (8 * Kg + j < n) __stcs(out + (size_t)(8 * Kg + j) * (size_t)ldq, y[j]);
    }
};

// The right-looking sweep inside a panel of PB column blocks starting at global block P0, on the
// accumulator registers acc[rg][J][e] (matrix column 8(P0+J) + t + 4e of row 8 rg + g).
// Step K: block K is final; it goes through X to one thread per row for its 8x8 substitution and
// comes back as A fragments.  The updates of the
// blocks J > K+1 by block K are DELAYED into step K+1, where they are independent of (and overlap
// with) the dependent fma chain of that step's substitution; only J = K+1 is updated at once.
// sink(Kg, y) sees every solved block in row form (lane = row of the slab).
// This is the ONLY place the solve's arithmetic lives: K3 and K5 both run it.
// KEEP: the solved blocks are also left in acc (fragment form), so that a second solve of the same panel can start from
// the registers.  DROP_LAST: the last block is not written back to its transposition buffer after its substitution (the
// sink has taken it and no later block needs its fragments).  Neither changes a single floating-point operation.
template <int RG, int PB, bool KEEP = false, bool DROP_LAST = false, typename X, typename F, typename SINK>
__device__ __forceinline__ void panel_core(double (&acc)[RG][PB][2], const X& xp, const F& fac,
                                           int P0, int lane, const SINK& sink)
{
    double ap0[RG], ap1[RG];                                  // A fragments of block K-1
#pragma unroll
    for (int K = 0; K < PB; ++K) {
        // the pair this step's critical update needs is requested before the transposition (the __syncwarp()s below
        // keep the compiler from hoisting it): an L1 miss then hides under the substitution
        // (panel passes only: K3 / K5 run more warps on fewer registers and lose by the longer live range)
        double2 bnext = make_double2(0.0, 0.0);
        if (X::REUSE && K + 1 < PB) bnext = fac.pair_in(P0, K, K + 1, lane);
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) { *xp.accp(P0 + K, rg, 0) = acc[rg][K][0]; *xp.accp(P0 + K, rg, 1) = acc[rg][K][1]; }
        __syncwarp();
        double y[8];
        if (xp.row_active()) {
#pragma unroll
            for (int j = 0; j < 8; ++j) y[j] = *xp.rowp(P0 + K, j);
        }
        if (K > 0) {
#pragma unroll
            for (int J = K + 1; J < PB; ++J) {
                const double2 b = fac.pair_in(P0, K - 1, J, lane);
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], ap0[rg], b.x);
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], ap1[rg], b.y);
            }
        }
        if (xp.row_active()) {
            fac.substitute(y, P0, K);
            if (!(DROP_LAST && K == PB - 1)) {
#pragma unroll
                for (int j = 0; j < 8; ++j) *xp.rowp(P0 + K, j) = y[j];
            }
            sink(P0 + K, y);
        }
        if (!(DROP_LAST && K == PB - 1)) {
            __syncwarp();
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) { ap0[rg] = *xp.accp(P0 + K, rg, 0); ap1[rg] = *xp.accp(P0 + K, rg, 1); }
        }
        if (X::REUSE || KEEP) {
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) { acc[rg][K][0] = ap0[rg]; acc[rg][K][1] = ap1[rg]; }
        }
        if (K + 1 < PB) {
            if (!X::REUSE) bnext = fac.pair_in(P0, K, K + 1, lane);
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][K + 1], ap0[rg], bnext.x);
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][K + 1], ap1[rg], bnext.y);
        }
        if (X::REUSE) __syncwarp();
    }
}

// One panel of PB column blocks starting at global block P0 of an in-place slab solve.
template <int RG, int PB, typename F>
__device__ __forceinline__ void solve_panel(double* slab, const F& fac, int P0, int lane)
{
    constexpr int SR = 8 * RG, LDS_ = SR + 4;
    const int g = lane >> 2, t = lane & 3;
    double* yw = slab + t * LDS_ + g;                 // (row g of group 0, column t of block 0)
    double acc[RG][PB][2];
#pragma unroll
    for (int J = 0; J < PB; ++J)
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
            acc[rg][J][0] = yw[(8 * (P0 + J)) * LDS_ + 8 * rg];
            acc[rg][J][1] = yw[(8 * (P0 + J) + 4) * LDS_ + 8 * rg];
        }
    // ---- left-looking: T_J += Y_K * (-R[K, J]) for the solved blocks K < P0
    for (int Kg = 0; Kg < P0; ++Kg) {
        double a0[RG], a1[RG];
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
            a0[rg] = yw[(8 * Kg) * LDS_ + 8 * rg];
            a1[rg] = yw[(8 * Kg + 4) * LDS_ + 8 * rg];
        }
#pragma unroll
        for (int J = 0; J < PB; ++J) {
            const double2 b = fac.pair(Kg, P0 + J, lane);
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], a0[rg], b.x);
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], a1[rg], b.y);
        }
    }
    panel_core<RG, PB>(acc, SlabXpose<RG>(slab, lane), fac, P0, lane, NoSink());
}

// In-place Y <- Y * R^-1 on this warp's slab (8*RG rows x 8*nB columns) against the prepared factor `fac`.
// NBT > 0: nB known at compile time (only the panel shapes that occur are instantiated); the arithmetic is the same
// either way.
template <int RG, int NBT, typename F>
__device__ __forceinline__ void solve_slab_f(double* slab, const F& fac, int nB, int lane)
{
    if (NBT > 0) {
        constexpr int FULL = NBT / 8, REST = NBT % 8;
#pragma unroll
        for (int p = 0; p < FULL; ++p) solve_panel<RG, 8>(slab, fac, 8 * p, lane);
        if (REST > 0) solve_panel<RG, (REST > 0 ? REST : 2)>(slab, fac, 8 * FULL, lane);
        return;
    }
    for (int P0 = 0; P0 < nB; P0 += 8) {
        const int pb = nB - P0;
        if (pb >= 8)      solve_panel<RG, 8>(slab, fac, P0, lane);
        else if (pb == 6) solve_panel<RG, 6>(slab, fac, P0, lane);
        else if (pb == 4) solve_panel<RG, 4>(slab, fac, P0, lane);
        else              solve_panel<RG, 2>(slab, fac, P0, lane);
    }
}

#ifndef MRCQR_NO_CONST_DIAG
// The form K3 / K5 use: frag = prepared factor in fragment order (global), FAC selects its diagonal blocks in constant memory.
template <int RG, int FAC, int NBT = 0>
__device__ __forceinline__ void solve_slab(double* slab, const double2* __restrict__ frag, int nB, int lane)
{
    solve_slab_f<RG, NBT>(slab, ConstFactor<FAC>{frag}, nB, lane);
}
#endif

} // namespace mrcqr
