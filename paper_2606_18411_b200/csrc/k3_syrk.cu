// k3_syrk.cu -- Gram matrix of a STORED Y (Algorithm 1 step 1) for n16 > 128.
//
// For n <= 128 the Gram matrix is accumulated inside K3 while Y is still in shared memory.  Beyond
// that the upper triangle of G (131 k doubles at n = 512) no longer fits the register file of one SM,
// so stage 2a runs in the paper's own order (TrsmPre writes A_1 = A Rs^-1, here into
// the Q buffer), this kernel forms G = Y^T Y from it, and stage 2b solves in place (SURVEY.md 8(f)
// "store-Y": 3 m n^2 flops instead of 4 m n^2; Y costs one write and 1 + reads of 8 m n bytes).
//
// G is cut into 128 x 128 blocks (I <= J); a CTA owns one block and a strided set of the 32-row chunks
// (deterministic split of m: chunk c belongs to CTA c mod k of its block), streams 32-row chunks of the two 128-column panels of Y through a
// triple-buffered shared-memory tile (cp.async, one barrier per chunk) and accumulates on DMMA: 8 warps as 4 x 2, each
// 32 x 64 of the block (4 x 8 accumulators, 12 fragment loads per 32 DMMA).  Accumulator chains are
// flushed to the CTA's partial every 1024 rows (reading R7); a reduction kernel adds the
// partials of a block in a fixed order.  Bit-reproducible: every element of a CTA's partial has ONE owner
// thread for the whole kernel; its later flushes are result-less atomic adds (RED.ADD.F64: same rounding as DADD,
// applied in program order for one thread and one address, see gram_flush in gram_roles.cuh), so the order of the
// additions is fixed although the instruction is an atomic.
// n16 not a multiple of 128: the last 128-column panel holds fewer than 16 live 8-column blocks.  Up to 10 live blocks
// mrcqr_syrk_ragged runs instead: the same kernel with the dead block columns of the last block column compiled out
// (template arguments, never run-time predicates around a DMMA) and CTA counts per block CLASS (sy_class) from a cost
// model with a floor for blocks that have little to multiply (m = 2^21: n = 136 4.72 -> 2.89 ms, n = 192 4.71 -> 3.94,
// n = 272 10.6 -> 7.3); with more live blocks the full kernel is as fast.
#include "mrcqr_internal.cuh"
#include "gram_roles.cuh"

namespace mrcqr {

constexpr int SY_B = 128;             // block edge (columns)
constexpr int SY_KC = 32;             // rows per chunk
constexpr int SY_LD = SY_KC + 4;      // 36: conflict-free DMMA fragment loads
constexpr int SY_THREADS = 256;
constexpr int SY_FLUSH = 32;          // chunks per accumulator chain (1024 rows = 256 DMMA k-steps)

__device__ __forceinline__ void sy_dmma(double (&c)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ void sy_cp16(void* dst, const void* src, int bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src), "r"(bytes) : "memory");
}

struct SyrkParams {
    int64_t m, ldy;
    int n, n16, P, pairs;
    int ks0, ks1, ks2, ks3;           // CTAs (strided sets of 32-row chunks) per block of class 0..3 (sy_class); separate
                                      // members read through sy_ks: an indexed array would move the kernel parameters to
                                      // local memory and make everything derived from them look divergent to the compiler
    int nb_last;                      // live 8-column blocks of the last 128-column panel (16: n16 is a multiple of 128)
    int vec;
};

// Blocks (I <= J) fall into four cost classes: 0 diagonal, 1 the last diagonal block, 2 off-diagonal, 3 off-diagonal in the
// last block column.  When the last 128-column panel holds fewer than 16 live 8-column blocks (n16 not a multiple of 128)
// the blocks of classes 1 and 3 cost less (mrcqr_syrk_ragged skips the dead block columns) and get fewer CTAs.
__host__ __device__ __forceinline__ int sy_class(int i, int j, int P) { return (i == j ? 0 : 2) + (j == P - 1 ? 1 : 0); }
__host__ __device__ __forceinline__ int sy_ks(const SyrkParams& p, int cls) { return cls == 0 ? p.ks0 : (cls == 1 ? p.ks1 : (cls == 2 ? p.ks2 : p.ks3)); }

// CTA b -> (pair, index within the pair); CTAs are ordered by pair, a pair owns sy_ks(class) consecutive CTAs
__host__ __device__ __forceinline__ void sy_locate(const SyrkParams& p, int b, int& pair, int& ks_id, int& ks_n)
{
    int off = 0;
    for (int q = 0; q < p.pairs; ++q) {
        int j = 0;
        while ((j + 1) * (j + 2) / 2 <= q) ++j;
        const int i = q - j * (j + 1) / 2;
        const int k = sy_ks(p, sy_class(i, j, p.P));
        if (b < off + k) { pair = q; ks_id = b - off; ks_n = k; return; }
        off += k;
    }
    pair = p.pairs - 1; ks_id = 0; ks_n = 1;
}
__host__ __device__ __forceinline__ int sy_pair_offset(const SyrkParams& p, int pair)
{
    int off = 0;
    for (int q = 0; q < pair; ++q) {
        int j = 0;
        while ((j + 1) * (j + 2) / 2 <= q) ++j;
        off += sy_ks(p, sy_class(q - j * (j + 1) / 2, j, p.P));
    }
    return off;
}

__device__ __forceinline__ void sy_pair(int p, int& I, int& J)      // p -> (I <= J), column-major over the upper triangle
{
    int j = 0;
    while ((j + 1) * (j + 2) / 2 <= p) ++j;
    J = j; I = p - j * (j + 1) / 2;
}

// loads rows [r0, r0+32) of the 128-column panel `pan` of Y into dst[col][SY_LD]; zero fill outside m x n.
// VEC: thread (col0 = tid / 16, r2 = 2 (tid % 16)) copies 16 bytes of the columns col0, col0 + 16, ...:
// the source pointer advances by a constant, colmask (bit k: column col0 + 16 k exists) is per kernel.
__device__ __forceinline__ void sy_load_panel(double* dst, const SyrkParams& p, const double* __restrict__ Y,
                                              int pan, int64_t r0, int tid, unsigned colmask)
{
    const int64_t left = p.m - r0;
    if (p.vec) {
        const int col0 = tid >> 4, r2 = (tid & 15) * 2;
        const int64_t avail = left - r2;
        const int rb = avail >= 2 ? 16 : (avail == 1 ? 8 : 0);
        const double* src = Y + (size_t)(pan * SY_B + col0) * (size_t)p.ldy + r0 + r2;
        double* d = dst + col0 * SY_LD + r2;
        const size_t step = (size_t)16 * (size_t)p.ldy;
#pragma unroll
        for (int k = 0; k < SY_B / 16; ++k) {
            const int bytes = ((colmask >> k) & 1u) ? rb : 0;
            sy_cp16(d + k * 16 * SY_LD, bytes ? src + k * step : Y, bytes);
        }
    } else {
        for (int e = tid; e < SY_B * SY_KC; e += SY_THREADS) {
            const int col = e / SY_KC, rr = e % SY_KC;
            const int gc = pan * SY_B + col;
            dst[col * SY_LD + rr] = (gc < p.n && rr < left) ? Y[(size_t)gc * (size_t)p.ldy + r0 + rr] : 0.0;
        }
    }
}

__global__ void __launch_bounds__(SY_THREADS, 1)
mrcqr_syrk(SyrkParams p, const double* __restrict__ Y, double* __restrict__ partials)
{
    extern __shared__ __align__(16) double sy_sm[];        // [3 stages][2 panels][128 * SY_LD]
    constexpr int PAN = SY_B * SY_LD;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    int pair, ks_id, ks_n;
    sy_locate(p, blockIdx.x, pair, ks_id, ks_n);
    int I, J;
    sy_pair(pair, I, J);
    const bool diag = (I == J);
    const int wi = warp & 3, wj = warp >> 2;
    // This CTA's chunks are ks_id, ks_id + ks_n, ks_id + 2 ks_n, ... of the m / 32 chunks (a strided, not a contiguous,
    // range): every block type then sweeps the rows at the same pace (the split equalises their finishing times), the CTAs
    // of the diagonal and of the off-diagonal blocks that need the same panel chunk ask for it within microseconds of each
    // other, and the second one finds it in L2 (contiguous ranges read every panel of Y twice from DRAM).
    const int64_t chunks = (p.m + SY_KC - 1) / SY_KC;
    const int nchunks = chunks > ks_id ? (int)((chunks - ks_id + ks_n - 1) / ks_n) : 0;
    auto chunk_row = [&](int c) { return ((int64_t)ks_id + (int64_t)c * ks_n) * SY_KC; };
    double* part = partials + (size_t)blockIdx.x * SY_B * SY_B;

    unsigned maskI = 0, maskJ = 0;
#pragma unroll
    for (int k = 0; k < SY_B / 16; ++k) {
        if (I * SY_B + (tid >> 4) + 16 * k < p.n) maskI |= 1u << k;
        if (J * SY_B + (tid >> 4) + 16 * k < p.n) maskJ |= 1u << k;
    }
    auto issue = [&](int c) {                        // chunk c -> stage c % 3
        double* st = sy_sm + (size_t)(c % 3) * 2 * PAN;
        sy_load_panel(st, p, Y, I, chunk_row(c), tid, maskI);
        if (!diag) sy_load_panel(st + PAN, p, Y, J, chunk_row(c), tid, maskJ);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    // three stages, ONE barrier per chunk: the barrier of iteration c also proves that every warp is done
    // with chunk c-1, whose stage chunk c+2 is about to overwrite
    if (nchunks > 0) issue(0);
    if (nchunks > 1) issue(1);
    bool first = true;
    if (diag) {
        // diagonal block: only the upper triangle, 136 8x8 blocks split 18,18,18,18,16,16,16,16 over the warps
        // (gram_roles.cuh, the ownership table of K3 at n = 128)
        constexpr int MAXOWN = gram_maxown<16, 8>();
        double acc[MAXOWN][2];
#pragma unroll
        for (int b = 0; b < MAXOWN; ++b) acc[b][0] = acc[b][1] = 0.0;
        for (int c = 0; c < nchunks; ++c) {
            if (c + 1 < nchunks) asm volatile("cp.async.wait_group 1;" ::: "memory");
            else asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();
            if (c + 2 < nchunks) issue(c + 2);
            const double* pI = sy_sm + (size_t)(c % 3) * 2 * PAN;
            const bool fl = ((c + 1) % SY_FLUSH == 0 || c + 1 == nchunks);
#define SY_ROLE(R_) { gram_accumulate<16, 8, R_, SY_KC, 1, MAXOWN>(acc, pI, 0, lane); \
                      if (fl) gram_flush<16, 8, R_, MAXOWN>(acc, part, SY_B, first, lane); }
            switch (warp) {
                case 0: SY_ROLE(0) break; case 1: SY_ROLE(1) break; case 2: SY_ROLE(2) break; case 3: SY_ROLE(3) break;
                case 4: SY_ROLE(4) break; case 5: SY_ROLE(5) break; case 6: SY_ROLE(6) break; default: SY_ROLE(7) break;
            }
#undef SY_ROLE
            if (fl) first = false;
        }
        if (nchunks == 0)                            // an empty range still owns a (zero) partial
            for (int e = tid; e < SY_B * SY_B; e += SY_THREADS) part[e] = 0.0;
        return;
    }
    double acc[4][8][2];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    auto flush = [&]() {
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                double* dst = part + (size_t)(64 * wj + 8 * b + 2 * t) * SY_B + 32 * wi + 8 * a + g;
                if (first) { dst[0] = acc[a][b][0]; dst[SY_B] = acc[a][b][1]; }
                else { atomicAdd(dst, acc[a][b][0]); atomicAdd(dst + SY_B, acc[a][b][1]); }   // single-owner RED.ADD.F64: order fixed (header comment)
                acc[a][b][0] = acc[a][b][1] = 0.0;
            }
        first = false;
    };
    for (int c = 0; c < nchunks; ++c) {
        if (c + 1 < nchunks) asm volatile("cp.async.wait_group 1;" ::: "memory");
        else asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        if (c + 2 < nchunks) issue(c + 2);
        {
            const double* pI = sy_sm + (size_t)(c % 3) * 2 * PAN;
            const double* pJ = pI + PAN;
            const double* fi = pI + (32 * wi + g) * SY_LD + t;
            const double* fj = pJ + (64 * wj + g) * SY_LD + t;
#pragma unroll 2
            for (int ks = 0; ks < SY_KC / 4; ++ks) {
                double fI[4], fJ[8];
#pragma unroll
                for (int a = 0; a < 4; ++a) fI[a] = fi[(8 * a) * SY_LD + 4 * ks];
#pragma unroll
                for (int b = 0; b < 8; ++b) fJ[b] = fj[(8 * b) * SY_LD + 4 * ks];
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 8; ++b) sy_dmma(acc[a][b], fI[a], fJ[b]);
            }
        }
        if ((c + 1) % SY_FLUSH == 0 || c + 1 == nchunks) flush();
    }
    if (nchunks == 0) flush();                               // an empty range still owns a (zero) partial
}

// ---- ragged last panel (n16 not a multiple of 128): the dead 8-column blocks are compiled out ---------------------
// LIVE / LB are template arguments so that no DMMA sits under a run-time predicate (the compiler guards every mma.sync in
// a conditional with a WARPSYNC and a branch: 38 ms instead of 5 at n = 144 when this was tried with predicates).
template <int ROLE, int MAXOWN, int LIVE>
__device__ __forceinline__ void sy_diag_accumulate_live(double (&acc)[MAXOWN][2], const double* tile, int lane)
{
    const int g = lane >> 2, t = lane & 3;
    const double* y0 = tile + g * SY_LD + t;
#pragma unroll 2
    for (int ks = 0; ks < SY_KC / 4; ++ks) {
        const double* yk = y0 + 4 * ks;
        double f[16];
        static_for<0, LIVE>([&](auto Cc) {
            constexpr int c = decltype(Cc)::value;
            if constexpr (gram_needs<16, 8>(ROLE, c)) f[c] = yk[(8 * c) * SY_LD];
        });
        static_for<0, LIVE>([&](auto Ic) {
            constexpr int I = decltype(Ic)::value;
            static_for<I, LIVE>([&](auto Jc) {
                constexpr int J = decltype(Jc)::value;
                if constexpr (gram_owner<16, 8>(I, J) == ROLE) {
                    constexpr int slot = gram_slot<16, 8>(ROLE, I, J);
                    gram_dmma(acc[slot], f[I], f[J]);
                }
            });
        });
    }
}
template <int ROLE, int MAXOWN, int LIVE>
__device__ __forceinline__ void sy_diag_flush_live(double (&acc)[MAXOWN][2], double* part, bool first, int lane)
{
    const int g = lane >> 2, t = lane & 3;
    static_for<0, LIVE>([&](auto Ic) {
        constexpr int I = decltype(Ic)::value;
        static_for<I, LIVE>([&](auto Jc) {
            constexpr int J = decltype(Jc)::value;
            if constexpr (gram_owner<16, 8>(I, J) == ROLE) {
                constexpr int slot = gram_slot<16, 8>(ROLE, I, J);
                double* dst = part + (size_t)(8 * J + 2 * t) * SY_B + 8 * I + g;
                if (first) { dst[0] = acc[slot][0]; dst[SY_B] = acc[slot][1]; }
                else { atomicAdd(dst, acc[slot][0]); atomicAdd(dst + SY_B, acc[slot][1]); }    // single owner: order fixed (gram_flush)
                acc[slot][0] = acc[slot][1] = 0.0;
            }
        });
    });
}
template <int ROLE, int MAXOWN>
__device__ __forceinline__ void sy_diag_step(double (&acc)[MAXOWN][2], const double* tile, double* part, bool fl, bool first,
                                             int lane, int live)
{
#define SY_LIVE(L_) case L_: sy_diag_accumulate_live<ROLE, MAXOWN, L_>(acc, tile, lane);                       \
                             if (fl) sy_diag_flush_live<ROLE, MAXOWN, L_>(acc, part, first, lane); break;
    switch (live) {
        SY_LIVE(2) SY_LIVE(4) SY_LIVE(6) SY_LIVE(8) SY_LIVE(10)          // SY_RAGGED_MAX_NB = 10: more live blocks run the full kernel
        default: gram_accumulate<16, 8, ROLE, SY_KC, 1, MAXOWN>(acc, tile, 0, lane);
                 if (fl) gram_flush<16, 8, ROLE, MAXOWN>(acc, part, SY_B, first, lane);
    }
#undef SY_LIVE
}
// one chunk of an off-diagonal CTA's warp with LB live block columns (of its 8)
template <int NA, int LB>
__device__ __forceinline__ void sy_off_chunk(double (&acc)[4][8][2], const double* fi, const double* fj)
{
#pragma unroll 2
    for (int ks = 0; ks < SY_KC / 4; ++ks) {
        double fI[NA], fJ[LB];
#pragma unroll
        for (int a = 0; a < NA; ++a) fI[a] = fi[(8 * a) * SY_LD + 4 * ks];
#pragma unroll
        for (int b = 0; b < LB; ++b) fJ[b] = fj[(8 * b) * SY_LD + 4 * ks];
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
            for (int b = 0; b < LB; ++b) sy_dmma(acc[a][b], fI[a], fJ[b]);
    }
}

// The same kernel for a ragged last panel: blocks of the last block column skip their dead 8-column blocks.
__global__ void __launch_bounds__(SY_THREADS, 1)
mrcqr_syrk_ragged(SyrkParams p, const double* __restrict__ Y, double* __restrict__ partials)
{
    extern __shared__ __align__(16) double sy_sm[];        // [3 stages][2 panels][128 * SY_LD]
    constexpr int PAN = SY_B * SY_LD;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    int pair, ks_id, ks_n;
    sy_locate(p, blockIdx.x, pair, ks_id, ks_n);
    int I, J;
    sy_pair(pair, I, J);
    const bool diag = (I == J);
    const int wi = warp & 3, wj = warp >> 2;
    const int nbJ = (J == p.P - 1) ? p.nb_last : 16;          // live 8-column blocks of panel J (a panel I < J is always full)
    const int liveB = nbJ - 8 * wj >= 8 ? 8 : (nbJ - 8 * wj > 0 ? nbJ - 8 * wj : 0);   // ... among this warp's 8 block columns
    // This CTA's chunks are ks_id, ks_id + ks_n, ks_id + 2 ks_n, ... of the m / 32 chunks (a strided, not a contiguous,
    // range): every block type then sweeps the rows at the same pace (the split equalises their finishing times), the CTAs
    // of the diagonal and of the off-diagonal blocks that need the same panel chunk ask for it within microseconds of each
    // other, and the second one finds it in L2 (contiguous ranges read every panel of Y twice from DRAM).
    const int64_t chunks = (p.m + SY_KC - 1) / SY_KC;
    const int nchunks = chunks > ks_id ? (int)((chunks - ks_id + ks_n - 1) / ks_n) : 0;
    auto chunk_row = [&](int c) { return ((int64_t)ks_id + (int64_t)c * ks_n) * SY_KC; };
    double* part = partials + (size_t)blockIdx.x * SY_B * SY_B;

    unsigned maskI = 0, maskJ = 0;
#pragma unroll
    for (int k = 0; k < SY_B / 16; ++k) {
        if (I * SY_B + (tid >> 4) + 16 * k < p.n) maskI |= 1u << k;
        if (J * SY_B + (tid >> 4) + 16 * k < p.n) maskJ |= 1u << k;
    }
    auto issue = [&](int c) {                        // chunk c -> stage c % 3
        double* st = sy_sm + (size_t)(c % 3) * 2 * PAN;
        sy_load_panel(st, p, Y, I, chunk_row(c), tid, maskI);
        if (!diag) sy_load_panel(st + PAN, p, Y, J, chunk_row(c), tid, maskJ);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    // three stages, ONE barrier per chunk: the barrier of iteration c also proves that every warp is done
    // with chunk c-1, whose stage chunk c+2 is about to overwrite
    if (nchunks > 0) issue(0);
    if (nchunks > 1) issue(1);
    bool first = true;
    if (diag) {
        // diagonal block: only the upper triangle, 136 8x8 blocks split 18,18,18,18,16,16,16,16 over the warps
        // (gram_roles.cuh, the ownership table of K3 at n = 128)
        constexpr int MAXOWN = gram_maxown<16, 8>();
        double acc[MAXOWN][2];
#pragma unroll
        for (int b = 0; b < MAXOWN; ++b) acc[b][0] = acc[b][1] = 0.0;
        for (int c = 0; c < nchunks; ++c) {
            if (c + 1 < nchunks) asm volatile("cp.async.wait_group 1;" ::: "memory");
            else asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();
            if (c + 2 < nchunks) issue(c + 2);
            const double* pI = sy_sm + (size_t)(c % 3) * 2 * PAN;
            const bool fl = ((c + 1) % SY_FLUSH == 0 || c + 1 == nchunks);
#define SY_ROLE(R_) sy_diag_step<R_, MAXOWN>(acc, pI, part, fl, first, lane, nbJ);
            switch (warp) {
                case 0: SY_ROLE(0) break; case 1: SY_ROLE(1) break; case 2: SY_ROLE(2) break; case 3: SY_ROLE(3) break;
                case 4: SY_ROLE(4) break; case 5: SY_ROLE(5) break; case 6: SY_ROLE(6) break; default: SY_ROLE(7) break;
            }
#undef SY_ROLE
            if (fl) first = false;
        }
        if (nchunks == 0)                            // an empty range still owns a (zero) partial
            for (int e = tid; e < SY_B * SY_B; e += SY_THREADS) part[e] = 0.0;
        return;
    }
    double acc[4][8][2];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    auto flush = [&]() {
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                if (b >= liveB) continue;                    // dead block column: nothing accumulated, nothing read by the reduction
                double* dst = part + (size_t)(64 * wj + 8 * b + 2 * t) * SY_B + 32 * wi + 8 * a + g;
                if (first) { dst[0] = acc[a][b][0]; dst[SY_B] = acc[a][b][1]; }
                else { atomicAdd(dst, acc[a][b][0]); atomicAdd(dst + SY_B, acc[a][b][1]); }   // single-owner RED.ADD.F64: order fixed (header comment)
                acc[a][b][0] = acc[a][b][1] = 0.0;
            }
        first = false;
    };
    for (int c = 0; c < nchunks; ++c) {
        if (c + 1 < nchunks) asm volatile("cp.async.wait_group 1;" ::: "memory");
        else asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        if (c + 2 < nchunks) issue(c + 2);
        {
            const double* pI = sy_sm + (size_t)(c % 3) * 2 * PAN;
            const double* pJ = pI + PAN;
            const double* fi = pI + (32 * wi + g) * SY_LD + t;
            const double* fj = pJ + (64 * wj + g) * SY_LD + t;
            switch (liveB) {                                 // n16 is a multiple of 16: live counts are even
                case 8: sy_off_chunk<4, 8>(acc, fi, fj); break;
                case 6: sy_off_chunk<4, 6>(acc, fi, fj); break;
                case 4: sy_off_chunk<4, 4>(acc, fi, fj); break;
                case 2: sy_off_chunk<4, 2>(acc, fi, fj); break;
                default: break;
            }
        }
        if ((c + 1) % SY_FLUSH == 0 || c + 1 == nchunks) flush();
    }
    if (nchunks == 0) flush();                               // an empty range still owns a (zero) partial
}

// G16[i,j] (i <= j) = sum over the CTAs (chunk sets) of block (I,J), fixed order (32 lanes of ranges + binary tree)
__global__ void __launch_bounds__(1024)
mrcqr_syrk_reduce(SyrkParams p, const double* __restrict__ partials, double* __restrict__ G16)
{
    __shared__ double sm[32][33];
    const int el = threadIdx.x & 31, q = threadIdx.x >> 5;
    constexpr int CH = SY_B * SY_B / 32;
    const int pair = blockIdx.x / CH, e = (blockIdx.x % CH) * 32 + el;
    int I, J;
    sy_pair(pair, I, J);
    const int i = e % SY_B, j = e / SY_B;
    const int gi = SY_B * I + i, gj = SY_B * J + j;
    const bool live = gi <= gj && gj < p.n16;
    const int ksn = sy_ks(p, sy_class(I, J, p.P)), base = sy_pair_offset(p, pair);
    double total = 0.0;
    if (live)
        for (int c = q; c < ksn; c += 32) total += partials[((size_t)base + c) * SY_B * SY_B + e];
    sm[q][el] = total;
    __syncthreads();
#pragma unroll
    for (int h = 16; h > 0; h >>= 1) {
        if (q < h) sm[q][el] += sm[q + h][el];
        __syncthreads();
    }
    if (q == 0 && live) {
        const double v = sm[0][el];
        G16[(size_t)gj * p.n16 + gi] = v;
        G16[(size_t)gi * p.n16 + gj] = v;
    }
}

// CTAs per block class when the last panel is ragged.  Cost of one 32-row chunk per class in DMMA per k-step and SM
// sub-partition (warp w runs on sub-partition w % 4): 36 for a full diagonal block (the 0.5625 x 64 above), 64 for a full
// off-diagonal one, 4 nb for an off-diagonal block with nb live block columns, and for the last diagonal block the largest
// sub-partition load of the ownership table restricted to the live blocks; never below SY_COST_FLOOR: a CTA with little to
// multiply still waits for its chunks (two in flight, about 2.8 k clk per chunk measured = 22 DMMA slots).
constexpr double SY_COST_FLOOR = 22.0;
constexpr int SY_RAGGED_MAX_NB = 10;         // live blocks of the last panel up to which the ragged kernel is the faster one (measured)
static void syrk_split_ragged(SyrkParams& p, int sms, int64_t chunks)
{
    const int nb = p.nb_last;
    double w[4] = {36.0, 0.0, 64.0, 4.0 * nb};
    int cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = 0; i < 16; ++i)
        for (int j = i; j < nb; ++j) ++cnt[gram_owner<16, 8>(i, j)];
    int mx = 0;
    for (int q = 0; q < 4; ++q) mx = cnt[q] + cnt[q + 4] > mx ? cnt[q] + cnt[q + 4] : mx;
    w[1] = mx * 36.0 / 34.0;
    for (int c = 0; c < 4; ++c) w[c] = w[c] < SY_COST_FLOOR ? SY_COST_FLOOR : w[c];
    const int mult[4] = {p.P - 1, 1, (p.P - 1) * (p.P - 2) / 2, p.P - 1};      // blocks per class
    // k(T) = fewest CTAs per block that finish within T; bisection on T under sum mult k <= SMs, then the SMs left over go,
    // one block class at a time, to the class that finishes last
    auto need = [&](double T, int (&k)[4]) -> int64_t {
        int64_t tot = 0;
        for (int c = 0; c < 4; ++c) {
            k[c] = 1;
            if (mult[c] == 0) continue;
            const int64_t q = (int64_t)(T / w[c]);
            if (q < 1) return (int64_t)1 << 40;
            k[c] = (int)((chunks + q - 1) / q);
            tot += (int64_t)mult[c] * k[c];
        }
        return tot;
    };
    double lo = 0.0, hi = 64.0 * (double)chunks + 1.0;
    int k[4] = {1, 1, 1, 1}, kk[4];
    for (int it = 0; it < 64; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (need(mid, kk) <= sms) hi = mid; else lo = mid;
    }
    if (need(hi, k) > sms) { k[0] = k[1] = k[2] = k[3] = 1; }
    for (;;) {
        int used = 0, worst = -1;
        double tw = -1.0;
        for (int c = 0; c < 4; ++c) {
            if (mult[c] == 0) continue;
            used += mult[c] * k[c];
            const double t = w[c] * (double)((chunks + k[c] - 1) / k[c]);
            if (t > tw && k[c] < chunks) { tw = t; worst = c; }
        }
        if (worst < 0 || used + mult[worst] > sms) break;
        ++k[worst];
    }
    for (int c = 0; c < 4; ++c) k[c] = k[c] > chunks ? (int)chunks : k[c];
    p.ks0 = k[0]; p.ks1 = k[1]; p.ks2 = k[2]; p.ks3 = k[3];
}

static int syrk_grid(const SyrkParams& p)
{
    return (p.P - 1) * p.ks0 + p.ks1 + (p.P - 1) * (p.P - 2) / 2 * p.ks2 + (p.P - 1) * p.ks3;
}

static SyrkParams syrk_params(int64_t m, int n, int n16)
{
    SyrkParams p;
    p.m = m; p.n = n; p.n16 = n16;
    p.P = (n16 + SY_B - 1) / SY_B;
    p.pairs = p.P * (p.P + 1) / 2;
    const int pd = p.P, po = p.pairs - p.P, sms = num_sms();
    const int64_t chunks = (m + SY_KC - 1) / SY_KC;
    // ranges per off-diagonal (ko) and per diagonal (kd) block: every CTA on its own SM (po ko + pd kd <= SMs), the split
    // that minimises the longest CTA, a diagonal block costing 0.5625 of an off-diagonal one per row (18 of 32 block
    // products; measured optimum at C3 among 0.47 .. 0.60)
    int ko = 0, kd = sms / pd > 0 ? sms / pd : 1;
    if (po > 0) {
        double best = 1e300;
        ko = 1; kd = 1;
        for (int o = 1; po * o + pd <= sms; ++o) {
            const int d = (sms - po * o) / pd;
            const double t_off = (double)((chunks + o - 1) / o), t_diag = 0.5625 * (double)((chunks + d - 1) / d);
            const double t = t_off > t_diag ? t_off : t_diag;
            if (t < best) { best = t; ko = o; kd = d; }
        }
    }
    if (ko > chunks) ko = (int)chunks;
    if (kd > chunks) kd = (int)chunks;
    p.ks0 = p.ks1 = kd; p.ks2 = p.ks3 = ko > 0 ? ko : 1;
    p.nb_last = (n16 - SY_B * (p.P - 1)) / 8;
    if (p.nb_last <= SY_RAGGED_MAX_NB) syrk_split_ragged(p, sms, chunks);
    return p;
}

size_t syrk_partials_bytes(int n)
{
    const int n16 = round_up(n, 16);
    const int P = (n16 + SY_B - 1) / SY_B, pairs = P * (P + 1) / 2;
    return (size_t)(num_sms() + pairs) * SY_B * SY_B * sizeof(double);      // one partial per CTA
}

// err[0] = || I - G ||_F for the symmetric n x n matrix held in G16 (upper triangle read), fixed summation order
__global__ void __launch_bounds__(1024)
mrcqr_orth_norm(const double* __restrict__ G16, int n, int n16, double* __restrict__ err)
{
    __shared__ double sm[1024];
    double acc = 0.0;
    for (int e = threadIdx.x; e < n * n; e += 1024) {
        const int i = e % n, j = e / n;
        if (i <= j) {
            const double d = G16[(size_t)j * n16 + i] - (i == j ? 1.0 : 0.0);
            acc = fma(i == j ? 1.0 : 2.0, d * d, acc);
        }
    }
    sm[threadIdx.x] = acc;
    __syncthreads();
    for (int h = 512; h > 0; h >>= 1) {
        if (threadIdx.x < h) sm[threadIdx.x] += sm[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) err[0] = sqrt(sm[0]);
}

int launch_orth_norm(const double* G16, int n, int n16, double* err, cudaStream_t s)
{
    mrcqr_orth_norm<<<1, 1024, 0, s>>>(G16, n, n16, err);
    return 1;
}

int launch_syrk(int64_t m, int n, int64_t ldy, const double* Y, double* partials, int n16, double* G16, cudaStream_t s)
{
    SyrkParams p = syrk_params(m, n, n16);
    p.ldy = ldy;
    p.vec = ((uintptr_t)Y % 16 == 0) && (ldy % 2 == 0);
    const int smem = 3 * 2 * SY_B * SY_LD * (int)sizeof(double);
    cudaFuncSetAttribute(mrcqr_syrk, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (p.nb_last > SY_RAGGED_MAX_NB) mrcqr_syrk<<<syrk_grid(p), SY_THREADS, smem, s>>>(p, Y, partials);
    else {
        cudaFuncSetAttribute(mrcqr_syrk_ragged, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        mrcqr_syrk_ragged<<<syrk_grid(p), SY_THREADS, smem, s>>>(p, Y, partials);
    }
    mrcqr_syrk_reduce<<<p.pairs * (SY_B * SY_B / 32), 1024, 0, s>>>(p, partials, G16);
    return 2;
}

} // namespace mrcqr
