// k1_tc.cu -- K1 for the FP16 sketch (p = half, Algorithm 2 steps 2-4) with
// s <= 128 sampled bins: the pruned first stage of the four-step transform is a DENSE contraction
// and runs on the tensor cores; the pass is then bound by the one read of A.
//
// Split m = m1*m2 with m1 = 256, t = t1*m2 + t2, k = k1 (mod m1):
//     Re X[k] = sum_{t2} [ cos(th) Cc[k1,t2] - sin(th) Cs[k1,t2] ],    th = 2 pi k t2 / m,
//     Cc[k1,t2] = sum_{t1} x~[t1 m2 + t2] cos(2 pi k1 t1 / m1),   Cs likewise with sin.
// Only the s sampled residues k1 = k_i mod m1 are wanted, so (Cc, Cs) = F (2s x m1) * X~ (m1 x m2)
// per column of A, with F the sampled rows of the cosine / sine DFT matrices.  Folding t1 with
// m1 - t1 (cos even, sin odd) halves the contraction length:
//     Cc = x~[0] + sum_{t1=1}^{127} cos(.) (x~[t1] + x~[256-t1]) + (-1)^k1 x~[128],
//     Cs =          sum_{t1=1}^{127} sin(.) (x~[t1] - x~[256-t1]).
// Precision (reading R5): x~ = fl_16(d a) exactly as the paper's DiagMult; the folded
// sums are formed in FP32 and rounded to FP16, F is rounded to FP16, products accumulate in FP32
// (mma.sync.m16n8k16.f16 -> f32); the second stage (twiddles from sincospif on exactly reduced
// integer angles) and all sums over t2 are FP32, the chunk partials are added in FP64 in a fixed
// order.  The result is rounded to FP16 by the finalize kernel.  (The paper's cuFFT half path
// computes every butterfly in half.)
//
// A CTA (8 warps) keeps its rows of F as A fragments in registers for its whole life and streams
// tiles of 256 (t1) x 32 (t2) elements of one column: the raw FP64 rows of the next two tiles arrive by
// bulk asynchronous copies (cp.async.bulk, one 256-byte row per thread, completion on an mbarrier)
// while the current tile is multiplied; the converted / folded FP16 tile is double buffered.
#include "mrcqr_internal.cuh"
#include <cuda_fp16.h>
#include <cuda.h>

namespace mrcqr {

constexpr int TC_M1 = 256;        // first-stage length
constexpr int TC_NT = 32;         // t2 values per tile
constexpr int TC_LDX = 40;        // row stride of the FP16 tiles in halves (80 B: conflict-free ldmatrix)
constexpr int TC_THREADS = 256;

struct K1TcParams {
    int64_t m, lda, m2;
    int n, s, sp;                 // sp = s padded to 32 / 64 / 128
    int tiles_per_col;
    int64_t total_tiles;
    int grid;
};

__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], const void* p)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void ldmatrix_x2_trans(uint32_t (&r)[2], const void* p)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("ldmatrix.sync.aligned.m8n8.x2.trans.shared.b16 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(a));
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi)
{
    const __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const uint32_t*>(&h);
}
// fl_16(d * a) as a float: round to half (RNE), flip the sign bit
__device__ __forceinline__ float diag_half(double a, unsigned neg)
{
    const float v = __half2float(__double2half(a));
    return neg ? -v : v;
}

// ---- mbarrier + bulk asynchronous copy (global -> shared, completion counted in bytes on the mbarrier) ----
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "MBAR_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra MBAR_DONE_%=;\n\t"
        "bra MBAR_WAIT_%=;\n\t"
        "MBAR_DONE_%=:\n\t}"
        ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// TMA: one 3-D box (TC_NT t2 x 256 t1 x 1 column) of FP64 -> shared memory, completion in bytes on the mbarrier
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int x, int y, int z, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(tm), "r"(x), "r"(y), "r"(z),
                   "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

// lo / hi tile of CTA c out of G over T tiles: contiguous, balanced ranges of the column-major tile list
__host__ __device__ __forceinline__ int64_t tc_range_lo(int c, int G, int64_t T) { return ((int64_t)c * T) / G; }

// NTW = n-tiles (8 t2 columns each) per warp; the padded bin count is sp = 32 * NTW: the 8 warps form
// (2 NTW) m-tiles of 16 bins x (4 / NTW) column groups.
template <int NTW>
__global__ void __launch_bounds__(TC_THREADS, 1)
mrcqr_k1_tc(K1TcParams p, const __grid_constant__ CUtensorMap tmapA, const uint32_t* __restrict__ signs32,
            const int64_t* __restrict__ idx, float* __restrict__ partial)
{
    __shared__ __align__(16) __half Xe[2][128 * TC_LDX];
    __shared__ __align__(16) __half Xo[2][128 * TC_LDX];
    __shared__ float x128[2][TC_NT];
    constexpr int MT = 2 * NTW, NG = 4 / NTW, SP = 32 * NTW;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    const int mt = warp % MT, ng = warp / MT;
    const int c16 = tid & 15, rgp = tid >> 4;

    // ---- this lane's two bins (rows g and g+8 of m-tile mt) and their constants ----------------------
    int bin[2]; int64_t kk[2]; int k1[2]; float nyq[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        bin[h] = 16 * mt + g + 8 * h;
        kk[h] = bin[h] < p.s ? idx[bin[h]] : 0;
        k1[h] = (int)(kk[h] & (TC_M1 - 1));
        nyq[h] = (k1[h] & 1) ? -1.0f : 1.0f;
    }
    uint32_t Ac[8][4], As_[8][4];                    // rows of F as mma A fragments (FP16 pairs)
#pragma unroll
    for (int ks = 0; ks < 8; ++ks)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int h = q & 1, t1 = 16 * ks + 2 * t + 8 * (q >> 1);
            float s0, c0, s1, c1;
            sincospif(2.0f * (float)((k1[h] * t1) & (TC_M1 - 1)) / (float)TC_M1, &s0, &c0);
            sincospif(2.0f * (float)((k1[h] * (t1 + 1)) & (TC_M1 - 1)) / (float)TC_M1, &s1, &c1);
            Ac[ks][q] = pack_half2(c0, c1);
            As_[ks][q] = pack_half2(s0, s1);
        }
    float wl[2][NTW][2][2];                          // cos / sin of 2 pi k col / m for this lane's columns
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int nt = 0; nt < NTW; ++nt)
#pragma unroll
            for (int jj = 0; jj < 2; ++jj) {
                const int col = 8 * (ng * NTW + nt) + 2 * t + jj;
                const int64_t r = (kk[h] * col) & (p.m - 1);
                sincospif(2.0f * (float)r / (float)p.m, &wl[h][nt][jj][1], &wl[h][nt][jj][0]);
            }

    const int64_t lo = tc_range_lo(blockIdx.x, p.grid, p.total_tiles);
    const int64_t hi = tc_range_lo(blockIdx.x + 1, p.grid, p.total_tiles);
    const int tpc = p.tiles_per_col;
    // raw FP64 tiles: 2 stages x 256 rows x 256 bytes, each filled by ONE TMA box load (thread 0 issues it)
    extern __shared__ __align__(128) unsigned char raw_sm[];
    __shared__ __align__(8) uint64_t mbar[2];
    if (tid == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    // sign bits of this thread's 16 rows (4 per row pair).  The 16 words of the NEXT tile are requested before the
    // current tile is multiplied and packed after its second stage, so their L2 latency hides under the MMAs.
    unsigned sg_cur = 0u, sw[16];
    auto issue_tile = [&](int64_t id, int stg) {      // tile id -> raw stage stg (one TMA box)
        if (tid == 0) {
            const int j = (int)(id / tpc), tl = (int)(id % tpc);
            mbar_arrive_expect_tx(&mbar[stg], TC_M1 * TC_NT * 8);
            tma_load_3d(raw_sm + (size_t)stg * (TC_M1 * TC_NT * 8), &tmapA, tl * TC_NT, 0, j, &mbar[stg]);
        }
    };
    auto sign_load = [&](int64_t id) {
        const int tl = (int)(id % tpc);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int t1 = rgp + 16 * u, t1m = (t1 == 0) ? 128 : TC_M1 - t1;
            sw[2 * u] = signs32[((int64_t)t1 * p.m2 + (int64_t)tl * TC_NT) >> 5];
            sw[2 * u + 1] = signs32[((int64_t)t1m * p.m2 + (int64_t)tl * TC_NT) >> 5];
        }
    };
    auto sign_pack = [&]() {
        unsigned sg = 0;
#pragma unroll
        for (int u = 0; u < 8; ++u)
            sg |= (((sw[2 * u] >> (2 * c16)) & 3u) | (((sw[2 * u + 1] >> (2 * c16)) & 3u) << 2)) << (4 * u);
        return sg;
    };
    auto convert_tile = [&](int b) {                 // DiagMult + fold + round to FP16: raw[b] -> X[b]
        const double2* raw = reinterpret_cast<const double2*>(raw_sm + (size_t)b * (TC_M1 * TC_NT * 8)) + c16;
        const unsigned sg = sg_cur;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int t1 = rgp + 16 * u, t1m = (t1 == 0) ? 128 : TC_M1 - t1;
            const double2 va = raw[t1 * (TC_NT / 2)], vb = raw[t1m * (TC_NT / 2)];
            const unsigned bits = sg >> (4 * u);
            const float f0 = diag_half(va.x, bits & 1u), f1 = diag_half(va.y, bits & 2u);
            const float g0 = diag_half(vb.x, bits & 4u), g1 = diag_half(vb.y, bits & 8u);
            const bool fold = (t1 != 0);              // t1 = 0: x~[0] alone; its "mirror" slot carries row 128
            const uint32_t e = pack_half2(fold ? f0 + g0 : f0, fold ? f1 + g1 : f1);
            const uint32_t o = fold ? pack_half2(f0 - g0, f1 - g1) : 0u;
            if (!fold) { x128[b][2 * c16] = g0; x128[b][2 * c16 + 1] = g1; }
            *reinterpret_cast<uint32_t*>(&Xe[b][t1 * TC_LDX + 2 * c16]) = e;
            *reinterpret_cast<uint32_t*>(&Xo[b][t1 * TC_LDX + 2 * c16]) = o;
        }
    };

    float accb[2] = {0.0f, 0.0f};
    int seg = 0;
    int curj = (lo < hi) ? (int)(lo / tpc) : 0;
    auto flush = [&]() {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            float a = accb[h];
            a += __shfl_xor_sync(0xffffffffu, a, 1);
            a += __shfl_xor_sync(0xffffffffu, a, 2);
            if (t == 0) partial[((size_t)(blockIdx.x * 2 + seg) * NG + ng) * SP + bin[h]] = a;
            accb[h] = 0.0f;
        }
    };
    if (lo < hi) { issue_tile(lo, 0); sign_load(lo); sg_cur = sign_pack(); }
    if (lo + 1 < hi) issue_tile(lo + 1, 1);
    for (int64_t id = lo; id < hi; ++id) {
        const int b = (int)(id - lo) & 1;
        mbar_wait(&mbar[b], (unsigned)((id - lo) >> 1) & 1u);
        convert_tile(b);
        __syncthreads();                              // X[b] complete; raw[b] and X[b^1] free
        if (id + 2 < hi) issue_tile(id + 2, b);
        if (id + 1 < hi) sign_load(id + 1);
        // ---- first stage on the tensor cores: (Cc, Cs) = F * X~ for this warp's 16 bins x 8 NTW columns
        float accC[NTW][4], accS[NTW][4];
#pragma unroll
        for (int nt = 0; nt < NTW; ++nt)
#pragma unroll
            for (int q = 0; q < 4; ++q) accC[nt][q] = accS[nt][q] = 0.0f;
        const int lrow = (lane & 7) + 8 * ((lane >> 3) & 1);
        const int n0 = 8 * ng * NTW;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            if (NTW == 1) {
                uint32_t r[2];
                ldmatrix_x2_trans(r, &Xe[b][(16 * ks + lrow) * TC_LDX + n0]);
                mma16816(accC[0], Ac[ks], r[0], r[1]);
                ldmatrix_x2_trans(r, &Xo[b][(16 * ks + lrow) * TC_LDX + n0]);
                mma16816(accS[0], As_[ks], r[0], r[1]);
            } else {
#pragma unroll
                for (int np = 0; np < NTW / 2; ++np) {
                    uint32_t r[4];
                    const int off = (16 * ks + lrow) * TC_LDX + n0 + 16 * np + 8 * (lane >> 4);
                    ldmatrix_x4_trans(r, &Xe[b][off]);
                    mma16816(accC[2 * np], Ac[ks], r[0], r[1]);
                    mma16816(accC[2 * np + 1], Ac[ks], r[2], r[3]);
                    ldmatrix_x4_trans(r, &Xo[b][off]);
                    mma16816(accS[2 * np], As_[ks], r[0], r[1]);
                    mma16816(accS[2 * np + 1], As_[ks], r[2], r[3]);
                }
            }
        }
        // ---- second stage: sum over this tile's t2 with the twiddles W_m^{k t2}
        const int j = (int)(id / tpc), tl = (int)(id % tpc);
        if (j != curj) { flush(); ++seg; curj = j; }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            float S1 = 0.0f, S2 = 0.0f;
#pragma unroll
            for (int nt = 0; nt < NTW; ++nt)
#pragma unroll
                for (int jj = 0; jj < 2; ++jj) {
                    const float cc = fmaf(nyq[h], x128[b][n0 + 8 * nt + 2 * t + jj], accC[nt][2 * h + jj]);
                    const float cs = accS[nt][2 * h + jj];
                    const float cl = wl[h][nt][jj][0], sl = wl[h][nt][jj][1];
                    S1 = fmaf(cl, cc, S1); S1 = fmaf(-sl, cs, S1);
                    S2 = fmaf(sl, cc, S2); S2 = fmaf(cl, cs, S2);
                }
            const int64_t r = (kk[h] * ((int64_t)tl * TC_NT)) & (p.m - 1);
            float st, ct;
            sincospif(2.0f * (float)r / (float)p.m, &st, &ct);
            accb[h] += ct * S1 - st * S2;
        }
        if (id + 1 < hi) sg_cur = sign_pack();
    }
    if (lo < hi) flush();
}

// A_s[i, j] = fl_16( sqrt(s/m) * sum of the partials of column j ), CTAs in ascending order, column
// groups in ascending order inside a CTA (fixed order: deterministic).
__global__ void mrcqr_k1_tc_finalize(K1TcParams p, int NG, const float* __restrict__ partial,
                                     double* __restrict__ As, Status* st)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= p.s * p.n) return;
    const int i = e % p.s, j = e / p.s;
    const int64_t tpc = p.tiles_per_col, c_lo = j * tpc, c_hi = c_lo + tpc;
    double acc = 0.0;
    int c0 = (int)((c_lo * p.grid) / p.total_tiles) - 1, c1 = (int)((c_hi * p.grid) / p.total_tiles) + 1;
    if (c0 < 0) c0 = 0;
    if (c1 > p.grid - 1) c1 = p.grid - 1;
    for (int c = c0; c <= c1; ++c) {
        const int64_t lo = tc_range_lo(c, p.grid, p.total_tiles), hi = tc_range_lo(c + 1, p.grid, p.total_tiles);
        if (lo >= hi || lo >= c_hi || hi <= c_lo) continue;
        const int seg = j - (int)(lo / tpc);
        for (int ng = 0; ng < NG; ++ng)
            acc += (double)partial[((size_t)(c * 2 + seg) * NG + ng) * p.sp + i];
    }
    double v = acc * sqrt((double)p.s / (double)p.m);
    v = (double)__half2float(__double2half(v));
    if (isnan(v) || isinf(v)) report(st, 1, j);
    As[e] = v;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*tc_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static tc_encode_fn tc_encode()
{
    static tc_encode_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess) fn = reinterpret_cast<tc_encode_fn>(ptr);
        else cudaGetLastError();
    }
    return fn;
}

bool k1_tc_usable(int64_t m, int n, int64_t lda, const double* A, int prec, int s)
{
    return tc_encode() != nullptr && prec == 16 && s <= 128 && m >= (int64_t)TC_M1 * TC_NT && n <= num_sms() &&
           ((uintptr_t)A % 16 == 0) && (lda % 2 == 0);
}

size_t k1_tc_workspace_bytes() { return (size_t)num_sms() * 2 * 4 * 128 * sizeof(float); }

int launch_k1_tc(int64_t m, int n, int64_t lda, const double* A, int s, const uint64_t* signs,
                 const int64_t* idx, void* work, double* As, Status* st, cudaStream_t stream)
{
    K1TcParams p;
    p.m = m; p.lda = lda; p.m2 = m / TC_M1; p.n = n; p.s = s;
    p.sp = s <= 32 ? 32 : (s <= 64 ? 64 : 128);
    p.tiles_per_col = (int)(p.m2 / TC_NT);
    p.total_tiles = (int64_t)n * p.tiles_per_col;
    p.grid = (int)(p.total_tiles < num_sms() ? p.total_tiles : num_sms());
    float* partial = reinterpret_cast<float*>(work);
    const uint32_t* s32 = reinterpret_cast<const uint32_t*>(signs);
    constexpr int raw_bytes = 2 * TC_M1 * TC_NT * 8;
    CUtensorMap tm;
    {   // A viewed as (t2: m2) x (t1: 256) x (column: n), strides 8, 8 m2, 8 lda bytes; box = 32 x 256 x 1
        const cuuint64_t gdim[3] = {(cuuint64_t)p.m2, (cuuint64_t)TC_M1, (cuuint64_t)n};
        const cuuint64_t gstr[2] = {(cuuint64_t)p.m2 * 8, (cuuint64_t)lda * 8};
        const cuuint32_t box[3] = {TC_NT, TC_M1, 1}, estr[3] = {1, 1, 1};
        if (tc_encode()(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(A), gdim, gstr, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return -1;
    }
#define K1TC_GO(NTW_) { cudaFuncSetAttribute(mrcqr_k1_tc<NTW_>, cudaFuncAttributeMaxDynamicSharedMemorySize, raw_bytes); \
                        mrcqr_k1_tc<NTW_><<<p.grid, TC_THREADS, raw_bytes, stream>>>(p, tm, s32, idx, partial); }
    if (p.sp == 32) K1TC_GO(1) else if (p.sp == 64) K1TC_GO(2) else K1TC_GO(4)
#undef K1TC_GO
    mrcqr_k1_tc_finalize<<<(s * n + 255) / 256, 256, 0, stream>>>(p, 128 / p.sp, partial, As, st);
    return 2;
}

} // namespace mrcqr
