// k35_rows.cu -- the two passes over A that dominate MRCQR ("TRSM x2" is 56-74 %
// of the paper's runtime):
//   K3  mrcqr_k3_gram   Algorithm 2 step 7 fused with Algorithm 1 step 1:
//                       per row y = a Rs^-1 (solve_slab), G += y^T y on DMMA; Y never leaves the SM
//                       (fused form), or is also written to Q's buffer (dump form, n16 >= 48 by default).
//   K5  mrcqr_k5_formq  Algorithm 1 step 3: y recomputed bit-identically (fused form) or
//                       read back (dump form), q = y Rc^-1, Q streamed out.  Warps are fully independent.
//   mrcqr_panel_fused / mrcqr_panel_pass  the triangular solves of the store-Y form (n16 >= 128): 64-column
//                       panels in accumulator registers, all full panels of a solve in one launch.
// Which form runs for which n: api.cu, enqueue_stage23.
// Persistent CTAs, static slab -> warp map, so every sum has a fixed order: results are
// deterministic run to run.
#include "rows.cuh"
#include "gram_roles.cuh"

namespace mrcqr {

constexpr int GRAM_MAXS = 6;          // 16x16 super-blocks of G a warp accumulates per sweep (48 doubles)
constexpr int GRAM_CHAIN = 256;       // max DMMA k-steps chained into one accumulator before a flush
constexpr int SMEM_CAP = 227 * 1024;

RowCfg row_config(int n)
{
    RowCfg c;
    c.n16 = round_up(n, 16);
    if (c.n16 <= 64)       { c.RG = 4; c.NW = 4; }
    else if (c.n16 <= 128) { c.RG = 2; c.NW = 8; }
    else if (c.n16 <= 256) { c.RG = 1; c.NW = 8; }
    else                   { c.RG = 1; c.NW = 4; }
    c.smem_bytes = c.NW * c.n16 * (8 * c.RG + 4) * 8;
    return c;
}

#define MRCQR_ROLE_SWITCH(CALL)                                                                  \
    switch (warp) {                                                                              \
        case 0: CALL(0) break; case 1: CALL(1) break; case 2: CALL(2) break; case 3: CALL(3) break; \
        case 4: if (NW > 4) { CALL(4) } break; case 5: if (NW > 4) { CALL(5) } break;            \
        case 6: if (NW > 4) { CALL(6) } break; default: if (NW > 4) { CALL(7) } break;           \
    }

__device__ __forceinline__ void sb_to_pq(int sb, int& p, int& q)
{
    int qq = 0;
    while ((qq + 1) * (qq + 2) / 2 <= sb) ++qq;
    q = qq; p = sb - qq * (qq + 1) / 2;
}

// G partial of this CTA: n16 x n16 col-major, blocks (I <= J) of the upper triangle only.
// NB > 0: n16 = 8*NB <= 128, compile-time Gram ownership, accumulators live in registers across tiles.
// NB = 0: n16 > 128, 16x16 super-blocks in sweeps, flushed to the L2-resident partial every tile.
template <int RG, int NW, int NB, bool VEC>
__global__ void __launch_bounds__(NW * 32, (RG == 4 && NW == 4) ? (NB == 2 ? 5 : 3) : 1)
mrcqr_k3_gram(int64_t m, int n, int n16, int64_t lda, const double* __restrict__ A,
              const double2* __restrict__ fragS, double* __restrict__ partials,
              int64_t ntiles, double* __restrict__ Ydump, double* __restrict__ Ystore, int64_t ldys)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int SR = 8 * RG, LDS_ = SR + 4, TM = SR * NW;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int nB = n16 >> 3;
    const int slab_stride = n16 * LDS_;
    double* slab = Ysm + (size_t)warp * slab_stride;
    double* part = partials + (size_t)blockIdx.x * n16 * n16;
    zero_pad_columns<SR>(slab, n, n16, lane);

    if (NB > 0) {
        constexpr int NBc = NB > 0 ? NB : 2;
        // WP (n16 <= 32): the Gram of so few blocks is not worth a CTA-wide split (it kept 1-2 of the 4 warps busy
        // between two CTA barriers per tile): every warp accumulates all blocks over ITS OWN slab, with no CTA
        // barrier in the tile loop; the NW accumulator sets are summed in a fixed order (warp 0, through the
        // slabs) only when a chain is flushed.
        constexpr bool WP = (NB == 2 || NB == 4 || NB == 6);
        constexpr int NWG = WP ? 1 : NW;
        constexpr int MAXOWN = gram_maxown<NBc, NWG>();
        constexpr int FLUSH_TILES = WP ? GRAM_CHAIN * 4 / SR : GRAM_CHAIN * 4 / TM;
        double acc[MAXOWN][2];
#pragma unroll
        for (int b = 0; b < MAXOWN; ++b) acc[b][0] = acc[b][1] = 0.0;
        bool first = true;
        int since = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int64_t row0 = tile * TM + warp * SR;
            load_slab<SR, VEC>(slab, A, lda, m, n, row0, lane);
            if (VEC) cp_async_wait_all();
            __syncwarp();
            solve_slab<RG, 0, NBc>(slab, fragS, nB, lane);
            if (Ydump) { __syncwarp(); store_slab<SR, false>(slab, Ydump, m, m, n, row0, lane); }
            if (Ystore) { __syncwarp(); store_slab<SR, VEC>(slab, Ystore, ldys, m, n, row0, lane); }   // store-Y variant
            const bool flush = (++since >= FLUSH_TILES) || (tile + gridDim.x >= ntiles);
            if constexpr (WP) {
                __syncwarp();
                gram_accumulate<NBc, 1, 0, SR, 1, MAXOWN>(acc, slab, slab_stride, lane);
                __syncwarp();
                if (flush) {
#pragma unroll
                    for (int b = 0; b < MAXOWN; ++b) { slab[(2 * b) * 32 + lane] = acc[b][0]; slab[(2 * b + 1) * 32 + lane] = acc[b][1]; }
                    __syncthreads();
                    if (warp == 0) {
#pragma unroll
                        for (int b = 0; b < MAXOWN; ++b)
#pragma unroll
                            for (int w = 1; w < NW; ++w) {
                                acc[b][0] += Ysm[(size_t)w * slab_stride + (2 * b) * 32 + lane];
                                acc[b][1] += Ysm[(size_t)w * slab_stride + (2 * b + 1) * 32 + lane];
                            }
                        gram_flush<NBc, 1, 0, MAXOWN>(acc, part, n16, first, lane);
                    } else {
#pragma unroll
                        for (int b = 0; b < MAXOWN; ++b) acc[b][0] = acc[b][1] = 0.0;
                    }
                    __syncthreads();
                    zero_pad_columns<SR>(slab, n, n16, lane);        // the scratch use above ran over the padding columns
                    __syncwarp();
                    first = false; since = 0;
                }
            } else {
                __syncthreads();
#define GRAM_ACC(R_) gram_accumulate<NBc, NW, R_, SR, NW, MAXOWN>(acc, Ysm, slab_stride, lane);
                MRCQR_ROLE_SWITCH(GRAM_ACC)
#undef GRAM_ACC
                if (flush) {
#define GRAM_FLUSH(R_) gram_flush<NBc, NW, R_, MAXOWN>(acc, part, n16, first, lane);
                    MRCQR_ROLE_SWITCH(GRAM_FLUSH)
#undef GRAM_FLUSH
                    first = false; since = 0;
                }
                __syncthreads();
            }
        }
        return;
    }

    // ---- super-block sweeps (n16 > 128)
    const int P = n16 >> 4, NS = P * (P + 1) / 2;
    const int per_warp = (NS - warp + NW - 1) / NW;
    const int sweeps = (per_warp + GRAM_MAXS - 1) / GRAM_MAXS;
    bool first_tile = true;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t row0 = tile * TM + warp * SR;
        load_slab<SR, VEC>(slab, A, lda, m, n, row0, lane);
        if (VEC) cp_async_wait_all();
        __syncwarp();
        solve_slab<RG, 0>(slab, fragS, nB, lane);
        if (Ydump) { __syncwarp(); store_slab<SR, false>(slab, Ydump, m, m, n, row0, lane); }
        __syncthreads();
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
            for (int w = 0; w < NW; ++w)
                for (int ks = 0; ks < SR / 4; ++ks) {
                    const double* yk = Ysm + (size_t)w * slab_stride + g * LDS_ + 4 * ks + t;   // fragment (i = g, row = t)
#pragma unroll
                    for (int u = 0; u < GRAM_MAXS; ++u) {
                        if (u < cnt) {
                            const double fa0 = yk[(16 * pp[u]) * LDS_], fa1 = yk[(16 * pp[u] + 8) * LDS_];
                            double fb0 = fa0, fb1 = fa1;
                            if (pp[u] != qq[u]) { fb0 = yk[(16 * qq[u]) * LDS_]; fb1 = yk[(16 * qq[u] + 8) * LDS_]; }
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
                        else { atomicAdd(dst, acc[u][b][0]); atomicAdd(dst + n16, acc[u][b][1]); }    // RED.ADD.F64 by the element's ONE owner thread, in program order: deterministic (gram_roles.cuh, gram_flush)
                    }
                }
            }
        }
        first_tile = false;
        __syncthreads();
    }
}

// K5: every warp streams its own slabs (slab i belongs to global warp i mod (grid * NW)); no CTA barrier.
// mode 3: both solves (y = a Rs^-1, q = y Rc^-1); mode 1: only the first (store-Y form of stage 2a for
// n16 > 128, Y goes to the Q buffer); mode 2: only the second, in place on the stored Y.
// warps per CTA by panel size: small panels need few registers, and a 4 KB slab needs many warps in flight
constexpr int k5_max_warps(int nbt) { return nbt == 2 ? 32 : (nbt == 4 ? 16 : 12); }

template <int RG, int NBT, bool VEC>
__global__ void __launch_bounds__(32 * k5_max_warps(NBT), 1)
mrcqr_k5_formq(int64_t m, int n, int n16, int64_t lda, const double* __restrict__ A,
               const double2* __restrict__ fragS, const double2* __restrict__ fragC,
               int64_t ldq, double* __restrict__ Q, int64_t nslabs, double* __restrict__ Ydump, int mode)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int SR = 8 * RG, LDS_ = SR + 4;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int nB = n16 >> 3;
    double* slab = Ysm + (size_t)warp * n16 * LDS_;
    zero_pad_columns<SR>(slab, n, n16, lane);
    const int64_t stride = (int64_t)gridDim.x * nw;
    for (int64_t i = (int64_t)blockIdx.x * nw + warp; i < nslabs; i += stride) {
        const int64_t row0 = i * SR;
        __syncwarp();
        load_slab<SR, VEC>(slab, A, lda, m, n, row0, lane);
        if (VEC) cp_async_wait_all();
        __syncwarp();
        if constexpr (NBT > 0 && NBT <= 8) {
            // one panel (n16 <= 64): the panel goes into accumulator registers ONCE; the second solve starts from the
            // fragments the first one left there, and every block of Q leaves for global memory from its row form, so
            // the slab is not re-read between the solves nor for the store (K5 at n16 = 16 was bound by the
            // shared-memory pipe: 67 % busy).  Same panel_core, same operations as K3's solve_slab: Y stays bit-identical.
            const int g = lane >> 2, t = lane & 3;
            const double* yw = slab + t * LDS_ + g;
            double acc[RG][NBT][2];
#pragma unroll
            for (int J = 0; J < NBT; ++J)
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) {
                    acc[rg][J][0] = yw[(8 * J) * LDS_ + 8 * rg];
                    acc[rg][J][1] = yw[(8 * J + 4) * LDS_ + 8 * rg];
                }
            const SlabXpose<RG> xp(slab, lane);
            const RowSink rs{Q + row0 + lane, ldq, n, row0 + lane < m};
            if ((mode & 2) && Q) {
                if (mode & 1) {
                    panel_core<RG, NBT, true>(acc, xp, ConstFactor<0>{fragS}, 0, lane, NoSink());      // y = a Rs^-1
                    if (Ydump) { __syncwarp(); store_slab<SR, false>(slab, Ydump, m, m, n, row0, lane); }
                    __syncwarp();
                }
                panel_core<RG, NBT, false, true>(acc, xp, ConstFactor<1>{fragC}, 0, lane, rs);         // q = y Rc^-1
            } else {
                if (mode & 1) panel_core<RG, NBT>(acc, xp, ConstFactor<0>{fragS}, 0, lane, NoSink());
                if (Ydump) { __syncwarp(); store_slab<SR, false>(slab, Ydump, m, m, n, row0, lane); __syncwarp(); }
                if (mode & 2) solve_slab<RG, 1, NBT>(slab, fragC, nB, lane);
                __syncwarp();
                if (Q) store_slab<SR, VEC>(slab, Q, ldq, m, n, row0, lane);
            }
        } else {
            if (mode & 1) solve_slab<RG, 0, NBT>(slab, fragS, nB, lane);        // y = a Rs^-1, same code as K3
            if (Ydump) { __syncwarp(); store_slab<SR, false>(slab, Ydump, m, m, n, row0, lane); __syncwarp(); }
            if (mode & 2) solve_slab<RG, 1, NBT>(slab, fragC, nB, lane);        // q = y Rc^-1
            __syncwarp();
            if (Q) store_slab<SR, VEC>(slab, Q, ldq, m, n, row0, lane);          // Q = nullptr: the debug dump wants only Y
        }
    }
}

// ---- panel kernels (store-Y form) -------------------------------------------------------------------------
// mrcqr_panel_pass: one launch solves ONE panel of PB <= 8 column blocks for all rows (today only the ragged FIRST
// panel of a solve, PB = 2, 4 or 6, P0 = 0; the full panels share mrcqr_panel_fused below, which is this kernel with a
// loop over the panels around the body of a round): every warp streams 32-row slabs
// (RG = 4), keeps the panel in accumulator registers, adds the contributions of the already solved
// panels with a left-looking sweep whose A fragments come straight from global memory (lane (g, t)
// reads row g of column t: 64 contiguous bytes per column, every sector fully used; one step
// prefetched ahead), then runs the same in-register panel_core as K3 / K5.
// Memory phases are off the critical path of a warp (round-1 profile of panel 0: 30 % of a warp's time waiting for its
// slab and its stores, 31 % DMMA): the slab buffer is only the LANDING ZONE of the cp.async load -- once the panel is in
// accumulator registers the NEXT round's slab is requested into the same buffer and arrives during the solve; the 8x8
// transposes of panel_core go through a small per-warp scratch block, and every solved block leaves for global memory
// straight from its row form (lane = row: 256 contiguous bytes per column and warp), so there is no store phase.
// The panel's diagonal blocks sit at the start of c_pdiag (uploaded per launch): compile-time constant-bank operands.
// The -R fragments of the left-looking sweep are shared by the 4 warps of the CTA: chunks of PP_KC block rows
// (PP_KC x PB x 512 B) are staged in shared memory by cp.async, double buffered, one barrier per chunk.  The panel's own
// off-diagonal pairs come from L1 / L2 (panel_core requests the one on its critical path a step ahead); staging them in
// shared memory was measured slower either way it fits (once per CTA beside 2-row chunks: 5.45 ms per solve at C3; as two
// more chunks of the pipeline: 5.44; this form: 5.36): every CTA barrier per round costs more than the loads.  Two CTAs per SM.
constexpr int PP_NW = 4;              // warps per CTA
constexpr int PP_KC = 4;              // block rows of R per staged chunk
constexpr int PP_CTAS = 2;            // CTAs per SM

template <int FAC, int PB>
__global__ void __launch_bounds__(PP_NW * 32, PP_CTAS)
mrcqr_panel_pass(int64_t m, int ncols, int P0, const double* __restrict__ own, int64_t ld_own,
                 const double* __restrict__ Yprev, int64_t ldy, const double2* __restrict__ frag,
                 double* __restrict__ dst, int64_t ldd, int64_t nslabs)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int RG = 4, SR = 32, LDS_ = SR + 4;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    double* slab = Ysm + (size_t)warp * (8 * PB) * LDS_;
    double* scr = Ysm + (size_t)PP_NW * (8 * PB) * LDS_ + (size_t)warp * 8 * LDS_;
    double2* Bsm = reinterpret_cast<double2*>(Ysm + (size_t)PP_NW * (8 * PB + 8) * LDS_);   // [2][PB][PP_KC][32]
    zero_pad_columns<SR>(slab, ncols, 8 * PB, lane);       // the loads below never touch the padding columns
    double* yw = slab + t * LDS_ + g;
    const int nchunks = (P0 + PP_KC - 1) / PP_KC;
    auto stage_chunk = [&](int c) {                  // block rows [4c, 4c+4) x the PB block columns of the panel
        double2* dstb = Bsm + (size_t)(c & 1) * PB * PP_KC * 32;
        for (int e = tid; e < PB * PP_KC * 32; e += PP_NW * 32) {
            const int J = e / (PP_KC * 32), kl = (e / 32) % PP_KC, ln = e & 31;
            const int Kg = PP_KC * c + kl;
            if (Kg < P0) cp_async16(dstb + e, fragpair(frag, Kg, P0 + J, ln), 16);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const int64_t rounds = (nslabs + (int64_t)gridDim.x * PP_NW - 1) / ((int64_t)gridDim.x * PP_NW);
    const PanelFactor<FAC> fac{frag, P0};
    {                                                // round 0's slab
        const int64_t i0 = (int64_t)blockIdx.x * PP_NW + warp;
        __syncwarp();
        if (i0 < nslabs) load_slab<SR, true>(slab, own, ld_own, m, ncols, i0 * SR, lane);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    for (int64_t r = 0; r < rounds; ++r) {
        const int64_t i = (r * gridDim.x + blockIdx.x) * PP_NW + warp;
        const bool active = i < nslabs;
        const int64_t row0 = i * SR;
        const int64_t inext = ((r + 1) * gridDim.x + blockIdx.x) * PP_NW + warp;
        __syncthreads();                             // previous round done with both chunk buffers
        if (nchunks > 0) stage_chunk(0);
        const double* yp = Yprev + (size_t)t * (size_t)ldy + row0 + g;
        double a0[RG], a1[RG];
        if (P0 > 0 && active) {
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) { a0[rg] = __ldcs(yp + 8 * rg); a1[rg] = __ldcs(yp + (size_t)4 * ldy + 8 * rg); }
        }
        if (nchunks > 0) asm volatile("cp.async.wait_group 1;" ::: "memory");     // own panel landed (requested a round ago)
        else asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
        double acc[RG][PB][2];
        if (active) {
#pragma unroll
            for (int J = 0; J < PB; ++J)
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) {
                    acc[rg][J][0] = yw[(8 * J) * LDS_ + 8 * rg];
                    acc[rg][J][1] = yw[(8 * J + 4) * LDS_ + 8 * rg];
                }
        }
        __syncwarp();                                // every lane has its fragments: the landing zone is free again
        auto prefetch = [&]() {                      // next round's slab, behind every chunk group of this round
            if (inext < nslabs) load_slab<SR, true>(slab, own, ld_own, m, ncols, inext * SR, lane);
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        if (nchunks == 0) prefetch();
        for (int c = 0; c < nchunks; ++c) {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();                         // chunk c visible; everyone is done with chunk c-1
            if (c + 1 < nchunks) stage_chunk(c + 1);
            else prefetch();
            if (active) {
                const double2* bs = Bsm + (size_t)(c & 1) * PB * PP_KC * 32 + lane;
                const int kend = (P0 - PP_KC * c < PP_KC) ? P0 - PP_KC * c : PP_KC;
                for (int kl = 0; kl < kend; ++kl) {
                    const int Kg = PP_KC * c + kl;
                    double n0[RG], n1[RG];
                    const int Kn = (Kg + 1 < P0) ? Kg + 1 : Kg;
                    const double* yn = yp + (size_t)(8 * Kn) * (size_t)ldy;
#pragma unroll
                    for (int rg = 0; rg < RG; ++rg) { n0[rg] = __ldcs(yn + 8 * rg); n1[rg] = __ldcs(yn + (size_t)4 * ldy + 8 * rg); }
#pragma unroll
                    for (int J = 0; J < PB; ++J) {
                        const double2 b = bs[(J * PP_KC + kl) * 32];
#pragma unroll
                        for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], a0[rg], b.x);
#pragma unroll
                        for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], a1[rg], b.y);
                    }
#pragma unroll
                    for (int rg = 0; rg < RG; ++rg) { a0[rg] = n0[rg]; a1[rg] = n1[rg]; }
                }
            }
        }
        if (active) {
            double* out = dst + row0 + lane;         // lane = row of the slab
            auto sink = [&](int Kg, const double (&y)[8]) {
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int col = 8 * (Kg - P0) + j;
                    if (col < ncols) __stcs(out + (size_t)col * (size_t)ldd, y[j]);
                }
            };
            panel_core<RG, PB>(acc, ScratchXpose<RG>(scr, lane), fac, P0, lane, sink);
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// ---- all panels of a solve in ONE launch (n16 a multiple of 64) ------------------------------------------
// The per-panel launches above re-read the p panels solved before panel p from DRAM (each is m x 64 doubles, far beyond
// L2): 10 panel reads per solve at n = 256 where 4 would do.  Here a warp takes its 32-row slab through ALL panels before
// it moves on: the solved panels it sweeps over were written by itself a few microseconds earlier and come back from L2
// (st.cg / ld.cg: kept in L2, not in L1), so a solve reads its source once and writes its result once.  Same warp
// program per (slab, panel) step as mrcqr_panel_pass; the landing zone receives the NEXT step's panel (same rows, next
// panel; after the last panel the next round's first).  Diagonal blocks: FusedFactor (c_diag, uploaded once per solve).
template <int FAC, int NPMAX, bool RF>
__global__ void __launch_bounds__(PP_NW * 32, PP_CTAS)
mrcqr_panel_fused(int64_t m, int n, int B0arg, int NP, const double* src, int64_t lds,   // src == dst for the in-place solve
                  const double2* __restrict__ frag, double* dst, int64_t ldd, int64_t nslabs)
{
    extern __shared__ __align__(16) double Ysm[];
    constexpr int RG = 4, SR = 32, LDS_ = SR + 4, PB = 8;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    double* slab = Ysm + (size_t)warp * (8 * PB) * LDS_;
    double* scr = Ysm + (size_t)PP_NW * (8 * PB) * LDS_ + (size_t)warp * 8 * LDS_;
    double2* Bsm = reinterpret_cast<double2*>(Ysm + (size_t)PP_NW * (8 * PB + 8) * LDS_);   // [2][PB][PP_KC][32]
    double* yw = slab + t * LDS_ + g;
    const int B0 = RF ? B0arg : 0;                   // RF (ragged first): a panel of B0 = 2, 4 or 6 blocks was solved before this launch
    const int C0 = 8 * B0;                           // first column of the first full panel (a ragged panel of B0 blocks precedes it)
    const int ncols_last = n - C0 - 64 * (NP - 1);
    auto stage_chunk = [&](int c, int P0) {          // block rows [4c, 4c+4) x the PB block columns of panel P0 / 8
        double2* dstb = Bsm + (size_t)(c & 1) * PB * PP_KC * 32;
        for (int e = tid; e < PB * PP_KC * 32; e += PP_NW * 32) {
            const int J = e / (PP_KC * 32), kl = (e / 32) % PP_KC, ln = e & 31;
            const int Kg = PP_KC * c + kl;
            if (Kg < P0) cp_async16(dstb + e, fragpair(frag, Kg, P0 + J, ln), 16);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const uint64_t once = l2_evict_first_policy();
    auto request = [&](int64_t i, int p) {           // panel p of slab i into the landing zone (one commit group)
        if (i < nslabs) {
            const int nc = (p == NP - 1) ? ncols_last : 64;
            if (nc < 64) zero_pad_columns<SR>(slab, nc, 64, lane);
            load_slab_once<SR>(slab, src + (size_t)(C0 + 64 * p) * (size_t)lds, lds, m, nc, i * SR, lane, once);   // read once; the solved panels stay in L2
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const int64_t rounds = (nslabs + (int64_t)gridDim.x * PP_NW - 1) / ((int64_t)gridDim.x * PP_NW);
    __syncwarp();
    request((int64_t)blockIdx.x * PP_NW + warp, 0);
    for (int64_t r = 0; r < rounds; ++r) {
        const int64_t i = (r * gridDim.x + blockIdx.x) * PP_NW + warp;
        const bool active = i < nslabs;
        const int64_t row0 = i * SR;
        const int64_t inext = ((r + 1) * gridDim.x + blockIdx.x) * PP_NW + warp;
        for (int p = 0; p < NP; ++p) {
            const int P0 = B0 + 8 * p, nchunks = (P0 + PP_KC - 1) / PP_KC;
            const int ncols = (p == NP - 1) ? ncols_last : 64;
            const FusedFactor<FAC, NPMAX> fac(frag, B0, p, lane);
            __syncthreads();                         // previous step done with both chunk buffers; its stores are visible
            if (nchunks > 0) stage_chunk(0, P0);
            const double* yp = dst + (size_t)t * (size_t)ldd + row0 + g;
            double a0[RG], a1[RG];
            if (P0 > 0 && active) {
#pragma unroll
                for (int rg = 0; rg < RG; ++rg) { a0[rg] = __ldcg(yp + 8 * rg); a1[rg] = __ldcg(yp + (size_t)4 * ldd + 8 * rg); }
            }
            if (nchunks > 0) asm volatile("cp.async.wait_group 1;" ::: "memory");     // own panel landed (requested a step ago)
            else asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
            double acc[RG][PB][2];
            if (active) {
#pragma unroll
                for (int J = 0; J < PB; ++J)
#pragma unroll
                    for (int rg = 0; rg < RG; ++rg) {
                        acc[rg][J][0] = yw[(8 * J) * LDS_ + 8 * rg];
                        acc[rg][J][1] = yw[(8 * J + 4) * LDS_ + 8 * rg];
                    }
            }
            __syncwarp();                            // every lane has its fragments: the landing zone is free again
            auto prefetch = [&]() { if (p + 1 < NP) request(i, p + 1); else request(inext, 0); };
            if (nchunks == 0) prefetch();
            for (int c = 0; c < nchunks; ++c) {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                __syncthreads();                     // chunk c visible; everyone is done with chunk c-1
                if (c + 1 < nchunks) stage_chunk(c + 1, P0);
                else prefetch();
                if (active) {
                    const double2* bs = Bsm + (size_t)(c & 1) * PB * PP_KC * 32 + lane;
                    const int kend = (RF && P0 - PP_KC * c < PP_KC) ? P0 - PP_KC * c : PP_KC;     // !RF: P0 is a multiple of PP_KC
#pragma unroll (RF ? 1 : (NPMAX == 4 ? 2 : 4))      // up to 4 panels the kernel is bound by its code size more than by the sweep (C3: 5.09 -> 4.95 ms)
                    for (int kl = 0; kl < kend; ++kl) {
                        const int Kg = PP_KC * c + kl;
                        double n0[RG], n1[RG];
                        const int Kn = (Kg + 1 < P0) ? Kg + 1 : Kg;
                        const double* yn = yp + (size_t)(8 * Kn) * (size_t)ldd;
#pragma unroll
                        for (int rg = 0; rg < RG; ++rg) { n0[rg] = __ldcg(yn + 8 * rg); n1[rg] = __ldcg(yn + (size_t)4 * ldd + 8 * rg); }
#pragma unroll
                        for (int J = 0; J < PB; ++J) {
                            const double2 b = bs[(J * PP_KC + kl) * 32];
#pragma unroll
                            for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], a0[rg], b.x);
#pragma unroll
                            for (int rg = 0; rg < RG; ++rg) dmma884(acc[rg][J], a1[rg], b.y);
                        }
#pragma unroll
                        for (int rg = 0; rg < RG; ++rg) { a0[rg] = n0[rg]; a1[rg] = n1[rg]; }
                    }
                }
            }
            if (active) {
                double* o = dst + (size_t)(C0 + 64 * p) * (size_t)ldd + row0 + lane;   // lane = row of the slab
                int left = ncols;                    // columns of the panel not yet stored (blocks arrive in order)
                auto sink = [&](int, const double (&y)[8]) {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {    // one running pointer: no per-column address arithmetic
                        if (j < left) __stcg(o, y[j]);
                        o += ldd;
                    }
                    left -= 8;
                };
                panel_core<RG, PB>(acc, ScratchXpose<RG>(scr, lane), fac, P0, lane, sink);
            }
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// G16[i,j] (i <= j) = sum over the CTA partials in a FIXED order (deterministic split-m reduction):
// thread (element, q) adds the partials q, q+32, q+64, ... in ascending order; the 32 per-thread sums of
// an element are combined by a fixed binary tree in shared memory.  32 elements x 32 lanes per CTA;
// mirrored to the lower triangle.
__global__ void __launch_bounds__(1024)
mrcqr_reduce_partials(const double* __restrict__ partials, int np, int n16, double* __restrict__ G16)
{
    __shared__ double sm[32][33];
    const int el = threadIdx.x & 31, q = threadIdx.x >> 5;
    const int e = blockIdx.x * 32 + el;
    const size_t stride = (size_t)n16 * n16;
    const int i = e % n16, j = e / n16;
    const bool live = (e < n16 * n16) && (i <= j);
    double total = 0.0;
    if (live) {
        // same order of additions as a plain loop; the loads are issued eight at a time so that a thread's chain is
        // np / 256 L2 round trips long, not np / 32 (n = 16, 888 partials: 8.5 -> about 4 us)
        const double* src = partials + e;
        int c = q;
        for (; c + 7 * 32 < np; c += 8 * 32) {
            double v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = src[(size_t)(c + 32 * u) * stride];
#pragma unroll
            for (int u = 0; u < 8; ++u) total += v[u];
        }
        for (; c < np; c += 32) total += src[(size_t)c * stride];
    }
    sm[q][el] = total;
    __syncthreads();
#pragma unroll
    for (int h = 16; h > 0; h >>= 1) {
        if (q < h) sm[q][el] += sm[q + h][el];
        __syncthreads();
    }
    if (q == 0 && live) {
        const double t = sm[0][el];
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
    // one partial per CTA: at most 8 (n16 <= 32) / 4 (n16 <= 128) resident CTAs per SM are launched (grid_for's cap);
    // the n16 > 128 kernel holds a whole SM's shared memory: 1 CTA per SM
    const int per_sm = c.n16 <= 32 ? 8 : (c.n16 <= 128 ? 4 : 1);
    return (size_t)num_sms() * per_sm * (size_t)c.n16 * c.n16 * sizeof(double);
}

int upload_diag(const double* prep, int n16, int fac, cudaStream_t s)
{
    const int nB = n16 >> 3;
    cudaMemcpyToSymbolAsync(c_diag, prep + prep_diag_offset(nB), sizeof(double) * PREP_DIAG * nB,
                            sizeof(double) * (size_t)fac * PREP_MAX_NB * PREP_DIAG, cudaMemcpyDeviceToDevice, s);
    return 1;
}

template <typename K>
static int grid_for(K kernel, int threads, int smem, int64_t ntiles, int cap)
{
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    int occ = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem);
    if (occ < 1) occ = 1;
    if (occ > cap) occ = cap;
    int64_t g = (int64_t)occ * num_sms();
    return (int)(g < ntiles ? g : ntiles);
}

static bool vec_ok(const void* p, int64_t ld) { return ((uintptr_t)p % 16 == 0) && (ld % 2 == 0); }

int launch_k3_gram(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                   double* partials, int* n_partials_out, double* Ydump, double* Ystore, int64_t ldys, cudaStream_t s)
{
    RowCfg c = row_config(n);
    const int TM = 8 * c.RG * c.NW;
    const int64_t ntiles = (m + TM - 1) / TM;
    const bool vec = vec_ok(A, lda) && (!Ystore || vec_ok(Ystore, ldys));
    const double2* frag = reinterpret_cast<const double2*>(RsPrep);
#define K3_GO(RG_, NW_, NB_, V_)                                                                    \
    { auto k = mrcqr_k3_gram<RG_, NW_, NB_, V_>;                                                    \
      int grid = grid_for(k, NW_ * 32, c.smem_bytes, ntiles, c.n16 <= 32 ? 8 : (c.n16 <= 128 ? 4 : 1)); *n_partials_out = grid; \
      k<<<grid, NW_ * 32, c.smem_bytes, s>>>(m, n, c.n16, lda, A, frag, partials, ntiles, Ydump, Ystore, ldys); }
#define K3_CALL(RG_, NW_, NB_) { if (vec) K3_GO(RG_, NW_, NB_, true) else K3_GO(RG_, NW_, NB_, false) }
    switch (c.n16) {
        case 16:  K3_CALL(4, 4, 2) break;   case 32:  K3_CALL(4, 4, 4) break;
        case 48:  K3_CALL(4, 4, 6) break;   case 64:  K3_CALL(4, 4, 8) break;
        case 80:  K3_CALL(2, 8, 10) break;  case 96:  K3_CALL(2, 8, 12) break;
        case 112: K3_CALL(2, 8, 14) break;  case 128: K3_CALL(2, 8, 16) break;
        default:
            if (c.n16 <= 256) K3_CALL(1, 8, 0) else K3_CALL(1, 4, 0)
    }
#undef K3_CALL
#undef K3_GO
    return 1;
}

int launch_k5_formq(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                    const double* RcPrep, int64_t ldq, double* Q, double* Ydump, int mode, cudaStream_t s)
{
    RowCfg c = row_config(n);
    const int SR = 8 * c.RG;
    const int slab_bytes = c.n16 * (SR + 4) * 8;
    int nw = SMEM_CAP / slab_bytes;
    const int wcap = k5_max_warps(c.n16 <= 64 ? c.n16 / 8 : 0);
    if (nw > wcap) nw = wcap;
    if (nw < 1) nw = 1;
    const int smem = nw * slab_bytes;
    const int64_t nslabs = (m + SR - 1) / SR;
    int64_t grid = (nslabs + nw - 1) / nw;
    if (grid > num_sms()) grid = num_sms();
    const bool vec = vec_ok(A, lda) && (!Q || vec_ok(Q, ldq));
    const double2* fS = reinterpret_cast<const double2*>(RsPrep);
    const double2* fC = reinterpret_cast<const double2*>(RcPrep);
#define K5_GO(RG_, NB_, V_)                                                                         \
    { auto k = mrcqr_k5_formq<RG_, NB_, V_>;                                                           \
      cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);                   \
      k<<<(int)grid, nw * 32, smem, s>>>(m, n, c.n16, lda, A, fS, fC, ldq, Q, nslabs, Ydump, mode); }
#define K5_CALL(RG_, NB_) { if (vec) K5_GO(RG_, NB_, true) else K5_GO(RG_, NB_, false) }
    switch (c.n16) {
        case 16:  K5_CALL(4, 2) break;   case 32:  K5_CALL(4, 4) break;
        case 48:  K5_CALL(4, 6) break;   case 64:  K5_CALL(4, 8) break;
        case 80:  K5_CALL(2, 10) break;  case 96:  K5_CALL(2, 12) break;
        case 112: K5_CALL(2, 14) break;  case 128: K5_CALL(2, 16) break;
        default:  K5_CALL(1, 0)
    }
#undef K5_CALL
#undef K5_GO
    return 1;
}

// Y (or Q) <- solve of all panels with factor `fac` (0: Rs, source A; 1: Rc, source = dst in place).
// Requires 16-byte aligned operands and m % 32 == 0 (the caller falls back to the slab kernel otherwise).
bool panel_pass_usable(int64_t m, int n, const double* src, int64_t lds, const double* dstp, int64_t ldd)
{
    (void)n;
    return (m % 32 == 0) && vec_ok(src, lds) && vec_ok(dstp, ldd);
}

int launch_panel_solve(int64_t m, int n, int fac, const double* src, int64_t lds, const double* prep,
                       double* dstp, int64_t ldd, cudaStream_t s)
{
    const int n16 = round_up(n, 16), nB = n16 >> 3;
    const double2* frag = reinterpret_cast<const double2*>(prep);
    const int64_t nslabs = m / 32;
    const int nw = PP_NW;
    int64_t grid = (nslabs + nw - 1) / nw;
    if (grid > PP_CTAS * num_sms()) grid = PP_CTAS * num_sms();
    int launches = 0;
    const int NPF = nB / 8, RB = nB % 8;             // full 8-block panels; blocks of the ragged panel (0, 2, 4 or 6)
    // The ragged panel comes FIRST (blocks [0, RB)): it then needs no left-looking sweep, and the full panels that follow
    // share one launch in which a slab's solved panels come back from L2.  (Ragged last, in a launch of its own, re-read all
    // the solved panels from DRAM for a handful of columns: 1.2 ms for 16 columns at m = 2^21, n = 208.)
    if (RB > 0) {
        const int pb = RB;
        const int ncols = n < 8 * pb ? n : 8 * pb;
        const int smem = nw * (8 * pb + 8) * 36 * 8 + 2 * pb * PP_KC * 512;
        cudaMemcpyToSymbolAsync(c_pdiag, prep + prep_diag_offset(nB), sizeof(double) * PREP_DIAG * pb,
                                sizeof(double) * (size_t)fac * 8 * PREP_DIAG, cudaMemcpyDeviceToDevice, s);
#define PP_GO(FAC_, PB_)                                                                            \
        { auto k = mrcqr_panel_pass<FAC_, PB_>;                                                     \
          cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);               \
          k<<<(int)grid, nw * 32, smem, s>>>(m, ncols, 0, src, lds, dstp, ldd, frag, dstp, ldd, nslabs); }
#define PP_CALL(PB_) { if (fac == 0) PP_GO(0, PB_) else PP_GO(1, PB_) }
        if (pb == 6) PP_CALL(6) else if (pb == 4) PP_CALL(4) else PP_CALL(2)
#undef PP_CALL
#undef PP_GO
        ++launches;
    }
    if (NPF > 0) {
        const int smem = nw * (8 * 8 + 8) * 36 * 8 + 2 * 8 * PP_KC * 512;
#define PF_GO3(FAC_, NPM_, RF_)                                                                     \
        { auto k = mrcqr_panel_fused<FAC_, NPM_, RF_>;                                              \
          cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);               \
          k<<<(int)grid, nw * 32, smem, s>>>(m, n, RB, NPF, src, lds, frag, dstp, ldd, nslabs); }
#define PF_GO(FAC_, NPM_) { if (RB > 0) PF_GO3(FAC_, NPM_, true) else PF_GO3(FAC_, NPM_, false) }
        if (NPF <= 4) { if (fac == 0) PF_GO(0, 4) else PF_GO(1, 4) }
        else { if (fac == 0) PF_GO(0, 8) else PF_GO(1, 8) }
#undef PF_GO3
#undef PF_GO
        ++launches;
    }
    return launches;
}

int launch_reduce_partials(const double* partials, int n_partials, int n, int n16, double* G16, cudaStream_t s)
{
    (void)n;
    const int total = n16 * n16;
    mrcqr_reduce_partials<<<(total + 31) / 32, 1024, 0, s>>>(partials, n_partials, n16, G16);
    return 1;
}

} // namespace mrcqr
