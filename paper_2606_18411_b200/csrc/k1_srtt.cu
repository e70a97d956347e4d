// k1_srtt.cu -- K1: subsampled randomized trigonometric transform, Algorithm 2 steps 2-4
// (PAPER.md:95-97): x~ = fl_p(D a_j), X = DFT_m(x~) down every column, A_s = sqrt(s/m) Re X[S].
//
// The paper runs a full cuFFT and gathers.  Only s real outputs per column are
// wanted, so this kernel uses the four-step split m = m1*m2, t = t1*m2 + t2, k = k1 + m1*k2:
//     X[k] = sum_{t2} W_m^{k t2} Z[k1, t2],     Z[k1, t2] = sum_{t1} x~[t1*m2 + t2] W_m1^{k1 t1},
// and never materialises Z or X in HBM:
//   stage 1  a CTA stages an m1 x W tile (W = 32 or 16 consecutive t2, all t1; 256- or 128-byte coalesced
//            row segments of the column-major A), applying the sign bit and the cast to p on the way
//            in (DiagMult), and runs the 32 length-m1 FFTs in shared memory with
//            radix-4 decimation-in-frequency passes (output left in bit-reversed order).  The input is
//            real, so two ADJACENT t2 of the SAME column ride in one complex transform
//            (z[t1][u] = x~[t1, 2u] + i x~[t1, 2u+1]: exactly the 16-byte pairs the loads fetch): a tile
//            of W complex columns covers 2W consecutive t2 of one column of A, and a column's sketch
//            depends on that column only ("column-wise": a zero column gives an exactly zero
//            sketch column, a column scaled by 2^e an exactly scaled one).
//   stage 2  for each sampled bin k_i only the residue k1 = k_i mod m1 is needed: with P = Z[k1] and
//            Qn = Z[m1 - k1] of the packed transform, the even / odd t2 have E = (P + conj Qn) / 2 and
//            O = -i (P - conj Qn) / 2; the thread that owns the bin multiplies them by W_m^{k_i t2},
//            takes the real part and sums over the tile's t2 into a per-CTA accumulator; a finalize
//            kernel adds the per-chunk partials in a fixed order, scales by sqrt(s/m) and rounds to p.
// Same mathematical result as FFT-then-gather; pass 1 reads A exactly once in every precision.
// T = float serves p = FP16 (inputs and outputs rounded to FP16, FP32 arithmetic) and p = FP32;
// T = double serves p = FP64.  No fast-math intrinsics: twiddles come from sincospi.
#include "mrcqr_internal.cuh"
#include <cstdlib>
#include <cstring>
#include <cuda_fp16.h>

namespace mrcqr {

// W = complex elements per tile row = 2W consecutive t2 of one column (32: a warp instruction covers one tile row;
// 16: two rows, used for FP64 so that m1 = 256 fits the same 68 KB and the per-bin work of stage 2, which scales with
// s * m / m1, halves); the row stride of the tile is W + 1 complex elements (odd: the per-bin gathers of stage 2
// spread over the banks)
constexpr int K1_NT = 256;
constexpr int K1_NWARP = K1_NT / 32;

template <typename T> struct Cx { T x, y; };

template <typename T> __device__ __forceinline__ Cx<T> cmul(Cx<T> a, Cx<T> b)
{
    Cx<T> r;
    r.x = fma(a.x, b.x, -(a.y * b.y));
    r.y = fma(a.x, b.y, a.y * b.x);
    return r;
}
template <typename T> __device__ __forceinline__ Cx<T> cadd(Cx<T> a, Cx<T> b) { return Cx<T>{a.x + b.x, a.y + b.y}; }
template <typename T> __device__ __forceinline__ Cx<T> csub(Cx<T> a, Cx<T> b) { return Cx<T>{a.x - b.x, a.y - b.y}; }
// multiply by -i
template <typename T> __device__ __forceinline__ Cx<T> cmulmi(Cx<T> a) { return Cx<T>{a.y, -a.x}; }

__device__ __forceinline__ void sincospi_t(float a, float* s, float* c) { sincospif(a, s, c); }
__device__ __forceinline__ void sincospi_t(double a, double* s, double* c) { sincospi(a, s, c); }

// fl_p(d * a): sign-bit flip fused with the cast to the sketch precision.
template <typename T, int PREC>
__device__ __forceinline__ T diag_cast(double a, unsigned neg)
{
    T v;
    if (PREC == 16) v = (T)__half2float(__double2half(a));
    else if (PREC == 32) v = (T)__double2float_rn(a);
    else v = (T)a;
    return neg ? -v : v;
}

// s <= K1_INLINE_BINS: mrcqr_factor hands the drawn bins to the register radix-16 kernel as a launch parameter (constant
// bank) instead of copying them to the device first: one host-to-device copy less in front of a call.
constexpr int K1_INLINE_BINS = 256;
struct K1Bins { int64_t v[K1_INLINE_BINS]; };
struct K1Params {
    int64_t m, lda;
    int n, s, m1, log_m1;
    int64_t m2;
    int tiles_per_col, tiles_per_chunk, chunks;
    int vec;                      // A and lda allow 16-byte loads
    int reim;                     // Re+Im variant: 2s sketch rows, Im X[S] below Re X[S]
    int dtab;                     // the per-bin step twiddles W_m^k fit in shared memory (computed once per CTA)
    // mrcqr_factor (register radix-16 form only): the sign words are splitmix64_at(seed, word) evaluated where they are
    // used instead of read from the array a draw kernel wrote (a0: the same bits; one launch less), and the
    // status block is cleared here, by the first kernel of the call
    int gen_signs; uint64_t seed; Status* st_reset;
    int inline_bins;              // the bins are in the K1Bins parameter, idx is not read
};

template <typename T, int PREC, int W, bool REIM>
__global__ void __launch_bounds__(K1_NT, sizeof(T) == 8 ? 2 : 3)      // FP64 tiles: two CTAs per SM by shared memory
mrcqr_k1_srtt(K1Params p, const double* __restrict__ A, const uint32_t* __restrict__ signs32,
              const int64_t* __restrict__ idx, double* __restrict__ partial)
{
    constexpr int K1_W = W, K1_LD = W + 1, SUB = 32 / W;          // SUB tile rows per warp instruction
    extern __shared__ __align__(16) unsigned char smraw[];
    Cx<T>* tile = reinterpret_cast<Cx<T>*>(smraw);                       // [m1][W + 1]
    Cx<T>* tw = tile + (size_t)p.m1 * K1_LD;                             // [m1]  W_m1^e
    constexpr int NACC = REIM ? 2 : 1;                                    // Re (, Im)
    double* colacc = reinterpret_cast<double*>(tw + p.m1);               // [NACC][s]
    Cx<T>* dstep = reinterpret_cast<Cx<T>*>(colacc + NACC * p.s);           // [s]  (cos, sin) of 2 pi k_i / m   (dtab only)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tcol = lane % W, sub = lane / W;
    const int col = blockIdx.x / p.chunks, chunk = blockIdx.x % p.chunks;
    const int m1 = p.m1;
    const double* colA = A + (size_t)col * (size_t)p.lda;

    for (int e = tid; e < m1; e += K1_NT) {
        double sn, cs;
        sincospi(-2.0 * (double)e / (double)m1, &sn, &cs);
        tw[e] = Cx<T>{(T)cs, (T)sn};
    }
    for (int e = tid; e < NACC * p.s; e += K1_NT) colacc[e] = 0.0;
    if (p.dtab)
        for (int i = tid; i < p.s; i += K1_NT) {
            const int64_t k = idx[i];
            Cx<T> d;
            sincospi_t((T)(2.0 * (double)(k & (p.m - 1)) / (double)p.m), &d.y, &d.x);
            dstep[i] = d;
        }

    const int tile_lo = chunk * p.tiles_per_chunk;
    const int tile_hi = min(p.tiles_per_col, tile_lo + p.tiles_per_chunk);
    for (int tl = tile_lo; tl < tile_hi; ++tl) {
        const int64_t t2_0 = (int64_t)tl * (2 * K1_W);
        __syncthreads();
        // ---- load + DiagMult: lane (row, u) fetches the 16-byte pair x[t1, 2u], x[t1, 2u+1] = one complex element;
        //      eight rows per thread (8 loads + 8 sign words) in flight before the first conversion -------------
        if (p.vec) {
            const double2* src = reinterpret_cast<const double2*>(colA + t2_0) + tcol;
            const int64_t m2h = p.m2 >> 1;                          // row stride in double2
            for (int t1b = warp * SUB + sub; t1b < m1; t1b += K1_NWARP * SUB * 8) {
                double2 va[8];
                unsigned sg[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int t1 = t1b + u * K1_NWARP * SUB;
                    va[u] = make_double2(0.0, 0.0); sg[u] = 0;
                    if (t1 < m1) {
                        va[u] = __ldcs(src + (int64_t)t1 * m2h);
                        const int64_t tb = (int64_t)t1 * p.m2 + t2_0 + 2 * tcol;       // even: the pair shares a sign word
                        sg[u] = signs32[tb >> 5] >> (int)(tb & 31);
                    }
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int t1 = t1b + u * K1_NWARP * SUB;
                    if (t1 < m1)
                        tile[(size_t)t1 * K1_LD + tcol] = Cx<T>{diag_cast<T, PREC>(va[u].x, sg[u] & 1u),
                                                                diag_cast<T, PREC>(va[u].y, (sg[u] >> 1) & 1u)};
                }
            }
        }
        else {                                                    // unaligned A: 8-byte loads
            const double* src = colA + t2_0 + 2 * tcol;
#pragma unroll 4
            for (int t1 = warp * SUB + sub; t1 < m1; t1 += K1_NWARP * SUB) {
                const int64_t off = (int64_t)t1 * p.m2;
                const int64_t tb = off + t2_0 + 2 * tcol;
                const unsigned sg = signs32[tb >> 5] >> (int)(tb & 31);
                const double a = __ldcs(src + off), b = __ldcs(src + off + 1);
                tile[t1 * K1_LD + tcol] = Cx<T>{diag_cast<T, PREC>(a, sg & 1u), diag_cast<T, PREC>(b, (sg >> 1) & 1u)};
            }
        }
        __syncthreads();
        // ---- stage 1: m1-point DIF FFT down t1 for each of the W complex lanes ---------------------
        int nb = m1;                                   // current block size
        while (nb >= 4) {
            const int q = nb >> 2, tstride = m1 / nb;
            for (int bf = warp * SUB + sub; bf < (m1 >> 2); bf += K1_NWARP * SUB) {
                const int blk = bf / q, pos = bf % q;
                Cx<T>* base = tile + ((size_t)blk * nb + pos) * K1_LD + tcol;
                Cx<T> a0 = base[0], a1 = base[(size_t)q * K1_LD], a2 = base[(size_t)2 * q * K1_LD], a3 = base[(size_t)3 * q * K1_LD];
                const Cx<T> w1 = tw[pos * tstride], w2 = tw[2 * pos * tstride];
                Cx<T> b0 = cadd(a0, a2), b2 = cmul(csub(a0, a2), w1);
                Cx<T> b1 = cadd(a1, a3), b3 = cmulmi(cmul(csub(a1, a3), w1));
                base[0] = cadd(b0, b1);
                base[(size_t)q * K1_LD] = cmul(csub(b0, b1), w2);
                base[(size_t)2 * q * K1_LD] = cadd(b2, b3);
                base[(size_t)3 * q * K1_LD] = cmul(csub(b2, b3), w2);
            }
            nb >>= 2;
            __syncthreads();
        }
        if (nb == 2) {                                 // odd log2(m1): final radix-2 pass, twiddle 1
            for (int bf = warp * SUB + sub; bf < (m1 >> 1); bf += K1_NWARP * SUB) {
                Cx<T>* base = tile + (size_t)(2 * bf) * K1_LD + tcol;
                Cx<T> a0 = base[0], a1 = base[K1_LD];
                base[0] = cadd(a0, a1);
                base[K1_LD] = csub(a0, a1);
            }
            __syncthreads();
        }
        // ---- stage 2: sampled bins.  Thread (bin i) walks the W complex columns (2W values of t2) of the tile with the
        //      twiddle recurrence we <- we * W_m^{2k} for the even t2 (the odd one is we * W_m^k), re-seeded every 8 steps
        //      from w0 * (W_m^{16k})^j (a few ulp in T); one sincospi per bin and tile; no shuffles: a bin's partial sum
        //      belongs to one thread.
        for (int i = tid; i < p.s; i += K1_NT) {
            const int64_t k = idx[i];
            const int k1 = (int)(k & (m1 - 1));
            const int k1n = (m1 - k1) & (m1 - 1);
            const int br = p.log_m1 ? (int)(__brev((unsigned)k1) >> (32 - p.log_m1)) : 0;
            const int brn = p.log_m1 ? (int)(__brev((unsigned)k1n) >> (32 - p.log_m1)) : 0;
            const Cx<T>* rowP = tile + (size_t)br * K1_LD;
            const Cx<T>* rowQ = tile + (size_t)brn * K1_LD;
            Cx<T> w0, d1, d2, d16;                             // (cos, sin) of 2 pi k t2_0 / m, 2 pi k / m, 2 pi 2k / m, 2 pi 16k / m
            sincospi_t((T)(2.0 * (double)((k * t2_0) & (p.m - 1)) / (double)p.m), &w0.y, &w0.x);
            if (p.dtab) d1 = dstep[i];
            else sincospi_t((T)(2.0 * (double)(k & (p.m - 1)) / (double)p.m), &d1.y, &d1.x);
            d2 = cmul(d1, d1);
            d16 = cmul(d2, d2); d16 = cmul(d16, d16); d16 = cmul(d16, d16);    // four squarings of d1: a few ulp in T
            T va = (T)0, ia = (T)0;
            constexpr int STEP = K1_W < 8 ? K1_W : 8;
#pragma unroll 1
            for (int j8 = 0; j8 < K1_W; j8 += STEP) {
                Cx<T> we = w0;
#pragma unroll
                for (int u = 0; u < STEP; ++u) {
                    const Cx<T> P = rowP[j8 + u], Qn = rowQ[j8 + u];
                    const Cx<T> wo = cmul(we, d1);
                    // 2 E = P + conj Qn (t2 even), 2 O = -i (P - conj Qn) (t2 odd);  Re(e^{-i th} Z) = cos*Zr + sin*Zi
                    va = fma(we.x, P.x + Qn.x, va); va = fma(we.y, P.y - Qn.y, va);
                    va = fma(wo.x, P.y + Qn.y, va); va = fma(wo.y, Qn.x - P.x, va);
                    if (REIM) {                                 // Im(e^{-i th} Z) = cos*Zi - sin*Zr
                        ia = fma(we.x, P.y - Qn.y, ia); ia = fma(-we.y, P.x + Qn.x, ia);
                        ia = fma(wo.x, Qn.x - P.x, ia); ia = fma(-wo.y, P.y + Qn.y, ia);
                    }
                    we = cmul(we, d2);
                }
                w0 = cmul(w0, d16);
            }
            colacc[i] += 0.5 * (double)va;
            if (REIM) colacc[p.s + i] += 0.5 * (double)ia;
        }
    }
    __syncthreads();
    double* out = partial + ((size_t)col * p.chunks + chunk) * NACC * p.s;
    for (int e = tid; e < NACC * p.s; e += K1_NT) out[e] = colacc[e];
}

// =================================================================================================
// K1, register radix-16 form (m1 = 256 = 16 x 16, W = 16): the form every long column takes (m >= 8192).
// The shared-memory radix-4 kernel above moves the tile through shared memory ten times per transform (4 passes read +
// write, staging, stage 2) and was bound by that (round 1: 0.20-0.33 of the HBM peak).  Here a thread owns one 16-point
// butterfly per pass IN REGISTERS:
//   pass 1  thread (b, u) loads x~[t1 = 16 a + b], a = 0..15, of tile column u STRAIGHT FROM GLOBAL MEMORY (a half warp
//           reads 256 contiguous bytes of one row; the 16 loads of the NEXT tile are issued before this tile's butterflies,
//           so the HBM latency hides under two passes and stage 2), applies sign and cast, transforms over a, multiplies
//           by W_256^{b ka} and stores Y[ka][b] to the tile;
//   pass 2  thread (ka, u) transforms the 16 values b = 0..15 in place: Z[k1 = ka + 16 kb] sits in tile row 16 ka + kb;
//   stage 2 as above (thread = bin).
// Three barriers and three shared-memory passes per tile.  ST is the tile's storage type: Cx<T>, or __half2 for the FP16
// sketch, whose transform keeps its intermediates in half like the paper's cufftXt path (FP32
// butterflies, R5) and moves half the shared-memory bytes of the FP32 sketch.
template <typename T> struct K16;
template <> struct K16<float>  { static constexpr float  C = 0.92387953251128674f, S = 0.38268343236508977f, H = 0.70710678118654752f; };
template <> struct K16<double> { static constexpr double C = 0.92387953251128674,  S = 0.38268343236508977,  H = 0.70710678118654752; };

// 4-point forward DFT in place
template <typename T> __device__ __forceinline__ void dft4(Cx<T>& a0, Cx<T>& a1, Cx<T>& a2, Cx<T>& a3)
{
    const Cx<T> s02 = cadd(a0, a2), d02 = csub(a0, a2), s13 = cadd(a1, a3), d13 = cmulmi(csub(a1, a3));
    a0 = cadd(s02, s13); a2 = csub(s02, s13); a1 = cadd(d02, d13); a3 = csub(d02, d13);
}
// 16-point forward DFT in registers: input x[n] in natural order, output X[k] at x[4 (k & 3) + (k >> 2)]
template <typename T> __device__ __forceinline__ void fft16(Cx<T> (&x)[16])
{
    constexpr T C = K16<T>::C, S = K16<T>::S, H = K16<T>::H;
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) dft4(x[n2], x[4 + n2], x[8 + n2], x[12 + n2]);    // x[4 k1 + n2] = sum_n1 x[4 n1 + n2] W4^{n1 k1}
    Cx<T> v;
    v = x[5];  x[5]  = Cx<T>{fma(v.x, C, v.y * S), fma(v.y, C, -(v.x * S))};         // W16^1
    v = x[6];  x[6]  = Cx<T>{(v.x + v.y) * H, (v.y - v.x) * H};                        // W16^2
    v = x[7];  x[7]  = Cx<T>{fma(v.x, S, v.y * C), fma(v.y, S, -(v.x * C))};         // W16^3
    v = x[9];  x[9]  = Cx<T>{(v.x + v.y) * H, (v.y - v.x) * H};                        // W16^2
    v = x[10]; x[10] = Cx<T>{v.y, -v.x};                                               // W16^4 = -i
    v = x[11]; x[11] = Cx<T>{(v.y - v.x) * H, -((v.x + v.y) * H)};                     // W16^6
    v = x[13]; x[13] = Cx<T>{fma(v.x, S, v.y * C), fma(v.y, S, -(v.x * C))};         // W16^3
    v = x[14]; x[14] = Cx<T>{(v.y - v.x) * H, -((v.x + v.y) * H)};                     // W16^6
    v = x[15]; x[15] = Cx<T>{-fma(v.x, C, v.y * S), fma(v.x, S, -(v.y * C))};        // W16^9 = -W16^1
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4(x[4 * k1], x[4 * k1 + 1], x[4 * k1 + 2], x[4 * k1 + 3]);   // x[4 k1 + k2] = X[k1 + 4 k2]
}
__host__ __device__ constexpr int f16pos(int k) { return 4 * (k & 3) + (k >> 2); }

template <typename T> __device__ __forceinline__ void st_tile(Cx<T>* p, Cx<T> v) { *p = v; }
__device__ __forceinline__ void st_tile(__half2* p, Cx<float> v) { *p = __floats2half2_rn(v.x, v.y); }
template <typename T> __device__ __forceinline__ Cx<T> ld_tile(const Cx<T>* p) { return *p; }
__device__ __forceinline__ Cx<float> ld_tile(const __half2* p) { const float2 f = __half22float2(*p); return Cx<float>{f.x, f.y}; }

constexpr int F16_W = 16, F16_NT = 256, F16_M1 = 256, F16_LD = F16_W + 1;
#ifndef F16_DBL_CTAS
#define F16_DBL_CTAS 2
#endif

template <typename T, typename ST, int PREC>
__global__ void __launch_bounds__(F16_NT, sizeof(T) == 8 ? F16_DBL_CTAS : 2)
mrcqr_k1_fft16(K1Params p, const __grid_constant__ K1Bins bins, const double* __restrict__ A,
               const uint32_t* __restrict__ signs32, const int64_t* __restrict__ idx, double* __restrict__ partial)
{
    auto bin_at = [&](int i) -> int64_t { return p.inline_bins ? bins.v[i] : idx[i]; };
    extern __shared__ __align__(16) unsigned char smraw[];
    ST* tile = reinterpret_cast<ST*>(smraw);                                        // [256][17]
    Cx<T>* tw = reinterpret_cast<Cx<T>*>(smraw + (size_t)F16_M1 * F16_LD * sizeof(ST));   // [256]  W_256^e
    double* colacc = reinterpret_cast<double*>(tw + F16_M1);                        // [s]
    Cx<T>* dstep = reinterpret_cast<Cx<T>*>(colacc + p.s);                          // [s]  (cos, sin) of 2 pi k_i / m
    int* kbin = reinterpret_cast<int*>(dstep + p.s);                                // [s]  the bins k_i (< 2^31: m <= 2^31 here)
    unsigned short* perm = reinterpret_cast<unsigned short*>(kbin + p.s);           // [s]  stage-2 order of the bins
    __shared__ int bucket[32];
    const int tid = threadIdx.x, lane = tid & 31;
    const int u = tid & (F16_W - 1), b = tid >> 4;                                  // pass 1: b = t1 mod 16; pass 2: b = ka
    const int col = blockIdx.x / p.chunks, chunk = blockIdx.x % p.chunks;
    const double* colA = A + (size_t)col * (size_t)p.lda;

    const int tile_lo = chunk * p.tiles_per_chunk;
    const int tile_hi = min(p.tiles_per_col, tile_lo + p.tiles_per_chunk);
    double2 v[16];
    unsigned sw = 0;                                                                // sign word of row a = lane % 16 (this half warp's b)
    // rows a = A0 .. A0+7 of tile tl (the request is split in two so that at most 8 rows are in flight beside a butterfly)
    auto fetch = [&](int tl, int A0) {
        const int64_t t2_0 = (int64_t)tl * (2 * F16_W);
        if (p.vec) {
            const double2* src = reinterpret_cast<const double2*>(colA + t2_0) + u;
            const int64_t m2h = p.m2 >> 1;
#pragma unroll
            for (int a = 0; a < 8; ++a) v[A0 + a] = __ldcs(src + (int64_t)(16 * (A0 + a) + b) * m2h);
        } else {
            const double* src = colA + t2_0 + 2 * u;
#pragma unroll
            for (int a = 0; a < 8; ++a) {
                const int64_t off = (int64_t)(16 * (A0 + a) + b) * p.m2;
                v[A0 + a] = make_double2(__ldcs(src + off), __ldcs(src + off + 1));
            }
        }
        if (A0 == 0) {                                                              // m2 % 32 == 0: one word per row and tile
            const int64_t w32 = ((int64_t)(16 * (lane & 15) + b) * p.m2 + t2_0) >> 5;
            sw = p.gen_signs ? (unsigned)(splitmix64_at(p.seed, (uint64_t)(w32 >> 1)) >> (32 * (int)(w32 & 1))) : __ldg(signs32 + w32);
        }
    };
    if (p.st_reset && blockIdx.x == 0 && tid == 0) { p.st_reset->code = 0; p.st_reset->info = 0; }
    // the first tile is requested BEFORE the tables below are built: a CTA of a narrow matrix owns only a few tiles
    // (n = 16: three), and its set-up would otherwise sit in front of the first HBM round trip
    if (tile_lo < tile_hi) { fetch(tile_lo, 0); fetch(tile_lo, 8); }

    for (int e = tid; e < F16_M1; e += F16_NT) {
        double sn, cs;
        sincospi(-2.0 * (double)e / (double)F16_M1, &sn, &cs);
        tw[e] = Cx<T>{(T)cs, (T)sn};
    }
    for (int e = tid; e < p.s; e += F16_NT) colacc[e] = 0.0;
    for (int i = tid; i < p.s; i += F16_NT) {
        const int64_t k = bin_at(i);
        Cx<T> d;
        sincospi_t((T)(2.0 * (double)(k & (p.m - 1)) / (double)p.m), &d.y, &d.x);
        dstep[i] = d;
        kbin[i] = (int)k;
    }
    // Stage 2 reads, per lane, one element of the tile row of its bin: 32 lanes, 32 unrelated rows.  The rows of the lanes
    // that share a shared-memory wavefront (G = 128 bytes / element size: 8, 16 or 32 lanes) should fall into G different
    // banks, i.e. differ in (row mod G).  The bins are therefore dealt to the threads bucket by bucket: bin i of bucket
    // key_i = row_i mod G and rank r inside its bucket goes to position  sum_b min(count_b, r) + #{b < key_i : count_b > r},
    // which walks the buckets round-robin.  Which thread owns a bin does not change the bin's arithmetic.
    if (p.s <= 128) {                                                              // stage 2 is a small part there: identity order
        for (int i = tid; i < p.s; i += F16_NT) perm[i] = (unsigned short)i;
    } else {
        constexpr int G = 128 / (int)sizeof(ST);
        if (tid < 32) bucket[tid] = 0;
        __syncthreads();
        int myrank[16];                                                            // s <= 4096: at most 16 bins per thread here
        int cnt = 0;
        for (int i = tid; i < p.s; i += F16_NT, ++cnt) {
            const int k1 = (int)(bin_at(i) & (F16_M1 - 1));
            const int key = (16 * (k1 & 15) + (k1 >> 4)) & (G - 1);
            myrank[cnt & 15] = atomicAdd(&bucket[key], 1);
        }
        __syncthreads();
        cnt = 0;
        for (int i = tid; i < p.s; i += F16_NT, ++cnt) {
            const int k1 = (int)(bin_at(i) & (F16_M1 - 1));
            const int key = (16 * (k1 & 15) + (k1 >> 4)) & (G - 1);
            const int r = myrank[cnt & 15];
            int pos = 0;
#pragma unroll
            for (int q = 0; q < G; ++q) pos += min(bucket[q], r) + ((q < key && bucket[q] > r) ? 1 : 0);
            perm[pos] = (unsigned short)i;
        }
    }

    for (int tl = tile_lo; tl < tile_hi; ++tl) {
        const int64_t t2_0 = (int64_t)tl * (2 * F16_W);
        Cx<T> x[16];
#pragma unroll
        for (int a = 0; a < 16; ++a) {                                              // DiagMult + cast
            const unsigned bits = __shfl_sync(0xffffffffu, sw, (lane & 16) + a) >> (2 * u);
            x[a] = Cx<T>{diag_cast<T, PREC>(v[a].x, bits & 1u), diag_cast<T, PREC>(v[a].y, (bits >> 1) & 1u)};
        }
        if (tl + 1 < tile_hi) fetch(tl + 1, 0);                                     // first half of the next tile: in flight from here on
        fft16(x);
        __syncthreads();                                                            // stage 2 of the previous tile has read the tile
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) {
            Cx<T> y = x[f16pos(ka)];
            if (ka > 0) y = cmul(y, tw[b * ka]);
            st_tile(tile + (size_t)(16 * ka + b) * F16_LD + u, y);
        }
        __syncthreads();
#pragma unroll
        for (int bb = 0; bb < 16; ++bb) x[bb] = ld_tile(tile + (size_t)(16 * b + bb) * F16_LD + u);
        fft16(x);
#pragma unroll
        for (int kb = 0; kb < 16; ++kb) st_tile(tile + (size_t)(16 * b + kb) * F16_LD + u, x[f16pos(kb)]);
        if (tl + 1 < tile_hi) fetch(tl + 1, 8);                                     // second half: the butterfly registers are free now
        __syncthreads();
        // ---- stage 2: thread = bin; Z[k1] sits in row 16 (k1 & 15) + (k1 >> 4).  With P = Z[k1], Qn = Z[m1 - k1], q = conj(d2),
        //      d1 = W_m^{-k} conjugated (cos, sin of 2 pi k / m), d2 = d1^2 and w0 the twiddle of the tile's first t2:
        //        sum_u Re(conj(w_2u) E_u + conj(w_2u+1) O_u) = Re( conj(w0) (SE + conj(d1) SO) ),
        //        SE = (SP + conj(SQ)) / 2,  SO = -i (SP - conj(SQ)) / 2,  SP = sum_u q^u P_u,  SQ = sum_u d2^u Qn_u,
        //      so the tile costs two Horner recurrences (4 fma per step each) instead of two twiddle recurrences and 8 more
        //      operations per step; the recurrences run over 16 steps: a few ulp in T.
        for (int ps = tid; ps < p.s; ps += F16_NT) {
            const int i = perm[ps];
            const int64_t k = kbin[i];
            const int k1 = (int)(k & (F16_M1 - 1));
            const int k1n = (F16_M1 - k1) & (F16_M1 - 1);
            const ST* rowP = tile + (size_t)(16 * (k1 & 15) + (k1 >> 4)) * F16_LD;
            const ST* rowQ = tile + (size_t)(16 * (k1n & 15) + (k1n >> 4)) * F16_LD;
            Cx<T> w0, d1, d2;
            sincospi_t((T)(2.0 * (double)((k * t2_0) & (p.m - 1)) / (double)p.m), &w0.y, &w0.x);
            d1 = dstep[i];
            d2 = cmul(d1, d1);
            Cx<T> sp = ld_tile(rowP + F16_W - 1), sq = ld_tile(rowQ + F16_W - 1);
#pragma unroll
            for (int q = F16_W - 2; q >= 0; --q) {
                const Cx<T> P = ld_tile(rowP + q), Qn = ld_tile(rowQ + q);
                // sp <- sp * conj(d2) + P ;  sq <- sq * d2 + Qn
                const Cx<T> spn{fma(sp.x, d2.x, fma(sp.y, d2.y, P.x)), fma(sp.y, d2.x, fma(-sp.x, d2.y, P.y))};
                const Cx<T> sqn{fma(sq.x, d2.x, fma(-sq.y, d2.y, Qn.x)), fma(sq.y, d2.x, fma(sq.x, d2.y, Qn.y))};
                sp = spn; sq = sqn;
            }
            // 2 SE = sp + conj(sq), 2 SO = -i (sp - conj(sq));  z = 2 (SE + conj(d1) SO);  result = Re(conj(w0) z) / 2
            const Cx<T> se{sp.x + sq.x, sp.y - sq.y}, so{sp.y + sq.y, sq.x - sp.x};
            const Cx<T> z{se.x + fma(d1.x, so.x, d1.y * so.y), se.y + fma(d1.x, so.y, -(d1.y * so.x))};
            colacc[i] += 0.5 * (double)fma(w0.x, z.x, w0.y * z.y);
        }
    }
    __syncthreads();
    double* out = partial + ((size_t)col * p.chunks + chunk) * p.s;
    for (int e = tid; e < p.s; e += F16_NT) out[e] = colacc[e];
}

// A_s[i, j] = fl_p( sqrt(s/m) * sum_chunks partial ), chunks added in ascending order.
template <int PREC>
__global__ void mrcqr_k1_finalize(K1Params p, const double* __restrict__ partial, double* __restrict__ As, Status* st)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    const int rows = p.reim ? 2 * p.s : p.s, nacc = p.reim ? 2 : 1;
    if (e >= rows * p.n) return;
    const int r = e % rows, j = e / rows;
    const int i = r % p.s, part = r / p.s;                               // Re, Im
    const double* src = partial + ((size_t)j * p.chunks) * nacc * p.s + (size_t)part * p.s + i;
    double acc = 0.0;
    for (int c = 0; c < p.chunks; ++c) acc += src[(size_t)c * nacc * p.s];
    double v = acc * sqrt((double)p.s / (double)p.m);
    if (PREC == 16) v = (double)__half2float(__double2half(v));
    else if (PREC == 32) v = (double)__double2float_rn(v);
    if (isnan(v) || isinf(v)) report(st, 1, j);
    As[e] = v;
}

// The same for a column cut into MANY chunks (a narrow matrix: n = 16 has 86 of them, and a thread that adds them one after
// the other waits for one L2 round trip each: 14 us).  32 elements x 32 chunk groups per CTA: group q adds chunks q, q + 32,
// ... in ascending order, the groups are combined by a fixed binary tree in shared memory (the layout of
// mrcqr_reduce_partials).  Deterministic; the order differs from the plain loop's only in how the chunks are bracketed.
template <int PREC>
__global__ void __launch_bounds__(1024)
mrcqr_k1_finalize_wide(K1Params p, const double* __restrict__ partial, double* __restrict__ As, Status* st)
{
    __shared__ double sm[32][33];
    const int el = threadIdx.x & 31, q = threadIdx.x >> 5;
    const int e = blockIdx.x * 32 + el;
    const int rows = p.reim ? 2 * p.s : p.s, nacc = p.reim ? 2 : 1;
    const bool live = e < rows * p.n;
    double acc = 0.0;
    if (live) {
        const int r = e % rows, j = e / rows;
        const int i = r % p.s, part = r / p.s;
        const size_t cs = (size_t)nacc * p.s;
        const double* src = partial + ((size_t)j * p.chunks) * cs + (size_t)part * p.s + i;
        for (int c = q; c < p.chunks; c += 32) acc += src[(size_t)c * cs];
    }
    sm[q][el] = acc;
    __syncthreads();
#pragma unroll
    for (int h = 16; h > 0; h >>= 1) {
        if (q < h) sm[q][el] += sm[q + h][el];
        __syncthreads();
    }
    if (q == 0 && live) {
        double v = sm[0][el] * sqrt((double)p.s / (double)p.m);
        if (PREC == 16) v = (double)__half2float(__double2half(v));
        else if (PREC == 32) v = (double)__double2float_rn(v);
        if (isnan(v) || isinf(v)) report(st, 1, e / rows);
        As[e] = v;
    }
}

template <int PREC>
static void k1_finalize(const K1Params& p, const double* partial, double* As, Status* st, cudaStream_t stream)
{
    const int total = (p.reim ? 2 : 1) * p.s * p.n;
    if (p.chunks > 8) mrcqr_k1_finalize_wide<PREC><<<(total + 31) / 32, 1024, 0, stream>>>(p, partial, As, st);
    else mrcqr_k1_finalize<PREC><<<(total + 255) / 256, 256, 0, stream>>>(p, partial, As, st);
}

// tile width W of the shared-memory radix-4 form (complex elements = 2W consecutive t2 of one column).  That form now
// serves only short columns (m < 8192) and the Re+Im variant: 32-wide tiles, narrower ones where the column is too short
// for them (m >= 32: 2W <= m / 2).
static int k1_tile_w(int64_t m, int prec, int s, int reim)
{
    (void)prec; (void)s; (void)reim;
    int w = 32;
    while (w > 8 && 4 * (int64_t)w > m) w >>= 1;
    return w;
}

// m2 >= 32: whole sign words per tile row; bins kept as 32-bit integers in shared memory
static bool k1_fft16_usable(int64_t m, int reim) { return !reim && m >= (int64_t)F16_M1 * 2 * F16_W && m <= ((int64_t)1 << 31); }

static K1Params k1_params(int64_t m, int n, int64_t lda, int s, int prec, int reim)
{
    K1Params p;
    p.m = m; p.lda = lda; p.n = n; p.s = s; p.reim = reim;
    p.gen_signs = 0; p.seed = 0; p.st_reset = nullptr; p.inline_bins = 0;
    const bool f16 = k1_fft16_usable(m, reim);
    const int K1_W = f16 ? F16_W : k1_tile_w(m, prec, s, reim);
    const int m1max = f16 ? F16_M1 : ((prec == 64) ? 128 : 256) * (32 / K1_W);    // 68 KB tile (W = 8: 74 KB)
    int64_t m1 = m / (2 * K1_W);
    if (m1 > m1max) m1 = m1max;
    if (m1 < 1) m1 = 1;
    p.m1 = (int)m1; p.m2 = m / m1;
    p.log_m1 = 0; while ((1 << p.log_m1) < p.m1) ++p.log_m1;
    p.tiles_per_col = (int)(p.m2 / (2 * K1_W));
    int chunks = (12 * num_sms() + n - 1) / n;
    if (chunks > p.tiles_per_col) chunks = p.tiles_per_col;
    if (chunks < 1) chunks = 1;
    p.tiles_per_chunk = (p.tiles_per_col + chunks - 1) / chunks;
    p.chunks = (p.tiles_per_col + p.tiles_per_chunk - 1) / p.tiles_per_chunk;
    return p;
}

size_t k1_workspace_bytes(int64_t m, int n, int s, int prec)
{
    size_t fft = 0;
    for (int reim = 0; reim < 2; ++reim) {             // either variant may run in this workspace
        K1Params p = k1_params(m, n, m, s, prec, reim);
        const size_t b = (size_t)n * p.chunks * (reim ? 2 : 1) * (size_t)s * sizeof(double);
        if (b > fft) fft = b;
    }
    return fft;
}

template <typename T, int PREC, int W, bool REIM = false>
static void k1_launch_t(const K1Params& p_in, const double* A, const uint64_t* signs, const int64_t* idx,
                        double* partial, double* As, Status* st, cudaStream_t stream)
{
    K1Params p = p_in;
    size_t smem = (size_t)p.m1 * (W + 1) * sizeof(Cx<T>) + (size_t)p.m1 * sizeof(Cx<T>) + (REIM ? 2 : 1) * (size_t)p.s * sizeof(double);
    p.dtab = smem + (size_t)p.s * sizeof(Cx<T>) <= 200 * 1024;
    if (p.dtab) smem += (size_t)p.s * sizeof(Cx<T>);
    auto k = mrcqr_k1_srtt<T, PREC, W, REIM>;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int grid = p.n * p.chunks;
    k<<<grid, K1_NT, smem, stream>>>(p, A, reinterpret_cast<const uint32_t*>(signs), idx, partial);
    k1_finalize<PREC>(p, partial, As, st, stream);
}

template <typename T, typename ST, int PREC>
static void k1_launch_fft16(const K1Params& p_in, const double* A, const uint64_t* signs, const int64_t* idx,
                            double* partial, double* As, Status* st, cudaStream_t stream, const int64_t* h_bins)
{
    K1Params p = p_in;
    K1Bins bins;                                         // copied into the launch when it is made
    p.inline_bins = (h_bins && p.s <= K1_INLINE_BINS) ? 1 : 0;
    if (p.inline_bins) memcpy(bins.v, h_bins, sizeof(int64_t) * (size_t)p.s);
    size_t smem = (size_t)F16_M1 * F16_LD * sizeof(ST) + (size_t)F16_M1 * sizeof(Cx<T>) + (size_t)p.s * sizeof(double);
    p.dtab = 1;
    smem += (size_t)p.s * (sizeof(Cx<T>) + sizeof(int)) + (size_t)((p.s + 7) & ~7) * sizeof(unsigned short);
    auto k = mrcqr_k1_fft16<T, ST, PREC>;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k<<<p.n * p.chunks, F16_NT, smem, stream>>>(p, bins, A, reinterpret_cast<const uint32_t*>(signs), idx, partial);
    k1_finalize<PREC>(p, partial, As, st, stream);
}

bool k1_generates_signs(int64_t m, int reim) { return k1_fft16_usable(m, reim); }
bool k1_takes_host_bins(int64_t m, int s, int reim) { return k1_fft16_usable(m, reim) && s <= K1_INLINE_BINS; }

int launch_k1_srtt(int64_t m, int n, int64_t lda, const double* A, int prec, int s,
                   const uint64_t* signs, const int64_t* idx, void* k1_work, double* As,
                   Status* st, cudaStream_t stream, int reim, const uint64_t* gen_seed, bool reset_status,
                   const int64_t* h_bins)
{
    double* partial = reinterpret_cast<double*>(k1_work);
    K1Params p = k1_params(m, n, lda, s, prec, reim);
    p.vec = ((uintptr_t)A % 16 == 0) && (lda % 2 == 0);
    if (gen_seed && k1_generates_signs(m, reim)) { p.gen_signs = 1; p.seed = *gen_seed; p.st_reset = reset_status ? st : nullptr; }
    if (k1_fft16_usable(m, reim)) {
        if (prec == 16) k1_launch_fft16<float, __half2, 16>(p, A, signs, idx, partial, As, st, stream, h_bins);
        else if (prec == 32) k1_launch_fft16<float, Cx<float>, 32>(p, A, signs, idx, partial, As, st, stream, h_bins);
        else k1_launch_fft16<double, Cx<double>, 64>(p, A, signs, idx, partial, As, st, stream, h_bins);
        return 2;
    }
    const int w = k1_tile_w(m, prec, s, reim);
#define K1_GO(T_, P_, W_) { if (reim) k1_launch_t<T_, P_, W_, true>(p, A, signs, idx, partial, As, st, stream); \
                            else k1_launch_t<T_, P_, W_, false>(p, A, signs, idx, partial, As, st, stream); }
#define K1_W_SWITCH(T_, P_) { if (w == 8) K1_GO(T_, P_, 8) else if (w == 16) K1_GO(T_, P_, 16) else K1_GO(T_, P_, 32) }
    if (prec == 16) K1_W_SWITCH(float, 16)
    else if (prec == 32) K1_W_SWITCH(float, 32)
    else K1_W_SWITCH(double, 64)
#undef K1_W_SWITCH
#undef K1_GO
    return 2;
}

} // namespace mrcqr
