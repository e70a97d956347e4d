// k_batched.cu -- mrcqr_factor_batched: Algorithm 2 for a BATCH of small tall-skinny problems,
// the repeated-call regime the paper motivates (block Arnoldi, randomized-SVD power iterations, time stepping:
// PAPER.md:39, 172).  A single small factorization is a serial chain of ten dependent kernels (C0: 0.1 ms of latency
// for 0.3 us of memory traffic), which neither a loop nor a CUDA graph can shorten.  Here ONE CTA runs the whole
// chain for one problem out of shared memory and L2, and the grid runs as many problems at once as fit the GPU:
//   a0  draw: sign words on the fly, bins by warp 0 with the same rejection rule as the host draw, rank-sorted;
//   a1-a3  sketch: the defining cosine sum  A_s[i,j] = sqrt(s/m) sum_t d_t fl_p(a_tj) cos(2 pi k_i t / m)  evaluated
//       directly (for m <= 2^16 and s <= 128 the pruned sum costs what an FFT costs and needs no passes): 128-row
//       tiles of A arrive by cp.async (double buffered), are sign-flipped and rounded to p ONCE into a row-major tile,
//       thread = bin walks its rows with a re-seeded twiddle recurrence and n accumulators (arithmetic in T = float for
//       p = half / single, double for p = double; reading R5);
//   a4  Householder QR of the s x n sketch in registers (column -> warp, row -> lane), FP64, diag(R_s) > 0;
//   a5-a6  y = a R_s^-1 with the slab solve of rows.cuh (prepared factor in SHARED memory: every problem has its own) and
//       the warp-private DMMA Gram of gram_roles.cuh, warps summed in a fixed order;
//   a7  Cholesky by warp 0 in shared memory, breakdown reported per problem;
//   a8-a9  q = (a R_s^-1) R_c^-1 streamed out, R = R_c R_s.
// A is read three times as in the large path, the 2nd and 3rd time from L2.  Deterministic: every sum has a fixed order.
#define MRCQR_NO_CONST_DIAG
#include "rows.cuh"
#include "gram_roles.cuh"
#include <cuda_fp16.h>

namespace mrcqr {

constexpr int BT_NT = 256, BT_NW = 8;
constexpr int BT_TR = 128;            // rows per sketch tile
constexpr int BT_SMAX = 128;

struct BatchParams {
    int batch, n, n16, s, prec, vec;
    int64_t m, lda, strideA, ldq, strideQ;
    uint64_t seed;
    const double* A; double* Q; double* R; int* codes;        // codes: batch x 2 ints (code, info), device
    int tr, tr_sh;                                             // rows per sketch tile (min(m, 128), a power of two) and its log2
    // shared-memory layout (byte offsets)
    int o_idx, o_kept, o_as, o_rs, o_prepS, o_prepC, o_w, o_work, total;
};

template <typename T> struct Cx2 { T x, y; };
template <typename T> __device__ __forceinline__ Cx2<T> cmul2(Cx2<T> a, Cx2<T> b)
{
    return Cx2<T>{fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x)};
}

template <typename T, int PREC>
__device__ __forceinline__ T bt_diag_cast(double a, unsigned neg)
{
    T v;
    if (PREC == 16) v = (T)__half2float(__double2half(a));
    else if (PREC == 32) v = (T)__double2float_rn(a);
    else v = (T)a;
    return neg ? -v : v;
}

__device__ __forceinline__ double bt_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Householder R-factor of the s x n sketch As (ld = s) in registers: column c in warp c % 8 (slot c / 8), row i in lane
// i % 32 (slot i / 32).  One block barrier per reflector; unnormalised reflectors H = I - c v v^T, v = x - beta e_j,
// c = 1 / (beta (beta - alpha)).  Rs (n x n, ld = n) receives R with rows negated to diag > 0 (R6).
template <int CPW, int RPL>
__device__ __forceinline__ void bt_householder(const double* As, int s, int n, double* Rs, double* vbuf, double* cbuf, double* betas)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double a[CPW][RPL];
#pragma unroll
    for (int k = 0; k < CPW; ++k)
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int c = warp + BT_NW * k, i = lane + 32 * r;
            a[k][r] = (c < n && i < s) ? As[(size_t)c * s + i] : 0.0;
        }
    auto make_v = [&](int k, int j) {
        double alpha_l = 0.0, sig_l = 0.0;
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int i = lane + 32 * r;
            if (i == j) alpha_l = a[k][r];
            if (i > j) sig_l = fma(a[k][r], a[k][r], sig_l);
        }
        const double alpha = __shfl_sync(0xffffffffu, alpha_l, j & 31);      // row j lives in lane j % 32
        const double sigma = bt_warp_sum(sig_l);
        double beta = alpha, cf = 0.0;
        if (sigma != 0.0) {
            householder_coeffs(alpha, sigma, beta, cf);
        }
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int i = lane + 32 * r;
            const double v = (i > j) ? a[k][r] : (i == j ? alpha - beta : 0.0);
            vbuf[(j & 1) * (RPL * 32) + i] = v;
            if (i == j) a[k][r] = beta;
            if (i > j) a[k][r] = 0.0;
        }
        if (lane == 0) { cbuf[j & 1] = cf; betas[j] = beta; }
    };
    if (warp == 0) make_v(0, 0);
    for (int j = 0; j < n; ++j) {
        __syncthreads();
        double v[RPL];
#pragma unroll
        for (int r = 0; r < RPL; ++r) v[r] = vbuf[(j & 1) * (RPL * 32) + lane + 32 * r];
        const double cf = cbuf[j & 1];
        double w[CPW];
#pragma unroll
        for (int k = 0; k < CPW; ++k) {
            w[k] = 0.0;
#pragma unroll
            for (int r = 0; r < RPL; ++r) w[k] = fma(v[r], a[k][r], w[k]);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
            for (int k = 0; k < CPW; ++k) w[k] += __shfl_xor_sync(0xffffffffu, w[k], o);
#pragma unroll
        for (int k = 0; k < CPW; ++k) {
            const int c = warp + BT_NW * k;
            if (c > j && c < n) {
                const double wt = w[k] * cf;
#pragma unroll
                for (int r = 0; r < RPL; ++r) a[k][r] = fma(-wt, v[r], a[k][r]);
            }
        }
#pragma unroll
        for (int k = 0; k < CPW; ++k)
            if (warp + BT_NW * k == j + 1 && j + 1 < n) make_v(k, j + 1);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < CPW; ++k)
#pragma unroll
        for (int r = 0; r < RPL; ++r) {
            const int c = warp + BT_NW * k, i = lane + 32 * r;
            if (c < n && i < n) {
                double val = (i <= c) ? a[k][r] : 0.0;
                if (i <= c && betas[i] < 0.0) val = -val;
                Rs[(size_t)c * n + i] = val;
            }
        }
    __syncthreads();
}

template <typename T, int PREC, int NB>
__global__ void __launch_bounds__(BT_NT, NB == 2 ? 2 : 1)
mrcqr_factor_batched_kernel(const BatchParams p)
{
    extern __shared__ __align__(16) unsigned char bsm[];
    constexpr int N16 = 8 * NB, SR = 32, LDS_ = SR + 4, RG = 4;
    constexpr int TLD = N16 + 16 / (int)sizeof(T);            // row stride of the converted tile (16-byte aligned rows)
    constexpr int MAXOWN = gram_maxown<NB, 1>();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = p.n, s = p.s;
    const int64_t m = p.m;
    int64_t* idx = reinterpret_cast<int64_t*>(bsm + p.o_idx);            // [s] sorted bins
    int64_t* kept = reinterpret_cast<int64_t*>(bsm + p.o_kept);          // [s] bins in draw order
    double* As = reinterpret_cast<double*>(bsm + p.o_as);                // [n][s]
    double* Rs = reinterpret_cast<double*>(bsm + p.o_rs);                // [n][n]
    double* prepS = reinterpret_cast<double*>(bsm + p.o_prepS);
    double* prepC = reinterpret_cast<double*>(bsm + p.o_prepC);
    double* W = reinterpret_cast<double*>(bsm + p.o_w);                  // [N16][N16 + 1] Gram / Cholesky work
    unsigned char* work = bsm + p.o_work;
    __shared__ double vbuf[2 * 4 * 32];
    __shared__ double cbuf[2];
    __shared__ double betas[32];
    __shared__ uint32_t sgn[BT_TR / 32];
    __shared__ int s_code, s_info;
    constexpr int LDW = N16 + 1;
    const int nbw = (s + 31) / 32;                                       // warps of bins
    const int nbp = nbw <= 1 ? 1 : (nbw <= 2 ? 2 : 4);                   // padded to a power of two (s <= 128)
    const int nrg = BT_NW / nbp;                                         // row groups
    const int bw = warp % nbp, rgi = warp / nbp;
    const int bin = 32 * bw + lane;
    const int TR = p.tr, TSH = p.tr_sh, rows_w = TR / nrg;               // rows of a tile per row group
    const int ntile = (int)(m / TR);

    for (int b = blockIdx.x; b < p.batch; b += gridDim.x) {
        const double* A = p.A + (size_t)b * (size_t)p.strideA;
        double* Q = p.Q + (size_t)b * (size_t)p.strideQ;
        double* R = p.R + (size_t)b * (size_t)n * n;
        const uint64_t seed = p.seed + (uint64_t)b;
        if (tid == 0) { s_code = 0; s_info = 0; }
        // ---- a0: bins (Algorithm 2 step 1; rule of DESIGN.md R1) -----------------------------------
        if (warp == 0) {
            const uint64_t nwords = (uint64_t)((m + 63) / 64), B = (uint64_t)(m / 2 + 1);
            int cnt = 0;
            for (uint64_t k0 = nwords; cnt < s; k0 += 32) {
                const int64_t cand_l = (int64_t)__umul64hi(splitmix64_at(seed, k0 + lane), B);
                for (int c = 0; c < 32 && cnt < s; ++c) {
                    const int64_t cv = __shfl_sync(0xffffffffu, cand_l, c);
                    bool dup = false;
                    for (int e = lane; e < cnt; e += 32) dup |= (kept[e] == cv);
                    if (!__any_sync(0xffffffffu, dup)) {
                        if (lane == 0) kept[cnt] = cv;
                        ++cnt;
                        __syncwarp();
                    }
                }
            }
        }
        __syncthreads();
        for (int e = tid; e < s; e += BT_NT) {                           // rank sort (the bins are distinct)
            const int64_t v = kept[e];
            int rank = 0;
            for (int x = 0; x < s; ++x) rank += (kept[x] < v);
            idx[rank] = v;
        }
        __syncthreads();

        // ---- a1-a3: sketch ---------------------------------------------------------------------------------------
        {
            double* raw = reinterpret_cast<double*>(work);                               // [2][N16][TR + 2]
            const int RLD = TR + 2;
            T* tt = reinterpret_cast<T*>(work + (size_t)2 * N16 * RLD * sizeof(double)); // [TR][TLD]
            auto issue = [&](int tl) {
                double* dst = raw + (size_t)(tl & 1) * N16 * RLD;
                const int64_t t0 = (int64_t)tl * TR;
                if (p.vec) {
                    const int H = TR / 2;
                    for (int e = tid; e < n * H; e += BT_NT) {
                        const int j = e >> (TSH - 1), r2 = (e & (H - 1)) * 2;
                        cp_async16(dst + j * RLD + r2, A + (size_t)j * (size_t)p.lda + t0 + r2, 16);
                    }
                } else {
                    for (int e = tid; e < n * TR; e += BT_NT) {
                        const int j = e >> TSH, r = e & (TR - 1);
                        dst[j * RLD + r] = A[(size_t)j * (size_t)p.lda + t0 + r];
                    }
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
            };
            const bool live = bin < s;
            const int64_t k = live ? idx[bin] : 0;
            Cx2<T> d1, d8;
            Cx2<double> wt, dt;                                             // W_m^{k (t0 + r0)} of the current tile and its step W_m^{k TR}, in double
            {
                double sn, cs;
                sincospi(2.0 * (double)(k & (m - 1)) / (double)m, &sn, &cs);
                d1 = Cx2<T>{(T)cs, (T)sn};
                sincospi(2.0 * (double)((8 * k) & (m - 1)) / (double)m, &sn, &cs);
                d8 = Cx2<T>{(T)cs, (T)sn};
                sincospi(2.0 * (double)((k * (int64_t)(rgi * rows_w)) & (m - 1)) / (double)m, &sn, &cs);
                wt = Cx2<double>{cs, sn};
                sincospi(2.0 * (double)((k * (int64_t)TR) & (m - 1)) / (double)m, &sn, &cs);
                dt = Cx2<double>{cs, sn};
            }
            T acc[N16];
#pragma unroll
            for (int j = 0; j < N16; ++j) acc[j] = (T)0;
            for (int e = tid; e < TR * TLD; e += BT_NT) tt[e] = (T)0;       // padding columns n..N16-1 stay zero
            issue(0);
            for (int tl = 0; tl < ntile; ++tl) {
                const int64_t t0 = (int64_t)tl * TR;
                if (tid < TR / 32) {                                        // sign words of this tile's rows
                    const int64_t tb = t0 + 32 * tid;
                    sgn[tid] = (uint32_t)(splitmix64_at(seed, (uint64_t)(tb >> 6)) >> (tb & 63));
                }
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                __syncthreads();                                            // raw[tl & 1] landed; tt free (previous tile consumed)
                if (tl + 1 < ntile) issue(tl + 1);
                {                                                           // DiagMult + cast, once per element
                    const double* src = raw + (size_t)(tl & 1) * N16 * RLD;
                    for (int e = tid; e < n * TR; e += BT_NT) {
                        const int j = e >> TSH, r = e & (TR - 1);
                        const unsigned neg = (sgn[r >> 5] >> (r & 31)) & 1u;
                        tt[r * TLD + j] = bt_diag_cast<T, PREC>(src[j * RLD + r], neg);
                    }
                }
                __syncthreads();
                if (live) {
                    const int r0 = rgi * rows_w;
                    Cx2<T> w0{(T)wt.x, (T)wt.y};                            // one double rotation per tile instead of a sincospi
                    wt = cmul2(wt, dt);
                    Cx2<T> w = w0;
                    for (int r = 0; r < rows_w; ++r) {
                        if ((r & 7) == 0 && r > 0) { w0 = cmul2(w0, d8); w = w0; }
                        const T* row = tt + (size_t)(r0 + r) * TLD;
                        constexpr int V = 16 / (int)sizeof(T);              // elements per 16-byte load
#pragma unroll
                        for (int j = 0; j < N16; j += V) {
                            if (sizeof(T) == 4) {
                                const float4 x = *reinterpret_cast<const float4*>(row + j);
                                acc[j] = fma(w.x, (T)x.x, acc[j]); acc[j + 1] = fma(w.x, (T)x.y, acc[j + 1]);
                                acc[j + 2] = fma(w.x, (T)x.z, acc[j + 2]); acc[j + 3] = fma(w.x, (T)x.w, acc[j + 3]);
                            } else {
                                const double2 x = *reinterpret_cast<const double2*>(row + j);
                                acc[j] = fma(w.x, (T)x.x, acc[j]); acc[j + 1] = fma(w.x, (T)x.y, acc[j + 1]);
                            }
                        }
                        w = cmul2(w, d1);
                    }
                }
            }
            __syncthreads();                                                // tiles consumed: the region becomes the reduction buffer
            double* red = reinterpret_cast<double*>(work);                  // [nrg][nbp * 32][N16]
            if (live) {
#pragma unroll
                for (int j = 0; j < N16; ++j) red[((size_t)rgi * (nbp * 32) + bin) * N16 + j] = (double)acc[j];
            }
            __syncthreads();
            const double scale = sqrt((double)s / (double)m);
            for (int e = tid; e < s * n; e += BT_NT) {
                const int i = e % s, j = e / s;
                double a = 0.0;
                for (int g2 = 0; g2 < nrg; ++g2) a += red[((size_t)g2 * (nbp * 32) + i) * N16 + j];
                double v = a * scale;
                if (PREC == 16) v = (double)__half2float(__double2half(v));
                else if (PREC == 32) v = (double)__double2float_rn(v);
                if (isnan(v) || isinf(v)) { if (atomicCAS(&s_code, 0, 1) == 0) s_info = j; }
                As[(size_t)j * s + i] = v;
            }
            __syncthreads();
        }

        // ---- a4: sketch QR -> R_s, prepared R_s ---------------------------------------------------------------------
        bt_householder<NB, 4>(As, s, n, Rs, vbuf, cbuf, betas);
        {
            const size_t total = prep_diag_offset(NB) + (size_t)PREP_DIAG * NB;
            int bad = -1;
            for (size_t o = tid; o < total; o += BT_NT) prepS[o] = prep_value(Rs, n, n, NB, o, &bad);
            if (bad >= 0) { if (atomicCAS(&s_code, 0, 2) == 0) s_info = bad; }
        }
        __syncthreads();

        // ---- a5-a6: Y = A Rs^-1 and G = Y^T Y (warp-private accumulators, warps summed in order) ---------------------
        double* slab = reinterpret_cast<double*>(work) + (size_t)warp * N16 * LDS_;
        double* gw = reinterpret_cast<double*>(work) + (size_t)BT_NW * N16 * LDS_;          // [8][N16 * N16]
        const int64_t nslabs = (m + SR - 1) / SR;
        const SmemFactor fS{prepS, NB};
        {
            zero_pad_columns<SR>(slab, n, N16, lane);
            double acc[MAXOWN][2];
#pragma unroll
            for (int q = 0; q < MAXOWN; ++q) acc[q][0] = acc[q][1] = 0.0;
            for (int64_t i = warp; i < nslabs; i += BT_NW) {
                __syncwarp();
                if (p.vec) { load_slab<SR, true>(slab, A, p.lda, m, n, i * SR, lane); cp_async_wait_all(); }
                else load_slab<SR, false>(slab, A, p.lda, m, n, i * SR, lane);
                __syncwarp();
                solve_slab_f<RG, NB>(slab, fS, NB, lane);
                __syncwarp();
                gram_accumulate<NB, 1, 0, SR, 1, MAXOWN>(acc, slab, 0, lane);
            }
            for (int e = lane; e < N16 * N16; e += 32) gw[(size_t)warp * N16 * N16 + e] = 0.0;
            __syncwarp();
            gram_flush<NB, 1, 0, MAXOWN>(acc, gw + (size_t)warp * N16 * N16, N16, true, lane);
        }
        __syncthreads();
        for (int e = tid; e < N16 * N16; e += BT_NT) {
            const int i = e % N16, j = e / N16;
            double a = 0.0;
            if (i <= j)
                for (int w2 = 0; w2 < BT_NW; ++w2) a += gw[(size_t)w2 * N16 * N16 + e];
            W[j * LDW + i] = a;
        }
        __syncthreads();

        // ---- a7: Cholesky G = Rc^T Rc by warp 0 (right-looking; breakdown reported) ----------------------
        if (warp == 0) {
            const int j = lane;
            for (int k = 0; k < n; ++k) {
                const double piv = W[k * LDW + k];
                if (!(piv > 0.0) || isinf(piv)) {
                    if (lane == 0 && atomicCAS(&s_code, 0, 3) == 0) s_info = k;
                    break;
                }
                const double rkk = sqrt(piv), inv = 1.0 / rkk;
                double wkj = 0.0;
                if (j > k && j < n) { wkj = W[j * LDW + k] * inv; W[j * LDW + k] = wkj; }
                if (j == k) W[k * LDW + k] = rkk;
                __syncwarp();
                if (j > k && j < n)
                    for (int i = k + 1; i <= j; ++i) W[j * LDW + i] = fma(-W[i * LDW + k], wkj, W[j * LDW + i]);
                __syncwarp();
            }
        }
        __syncthreads();
        const int code = s_code;
        if (code == 0) {
            // R = Rc Rs (Algorithm 2 step 9) and the prepared Rc
            for (int e = tid; e < n * n; e += BT_NT) {
                const int i = e % n, j = e / n;
                double r = 0.0;
                if (i <= j)
                    for (int k = i; k <= j; ++k) r = fma(W[k * LDW + i], Rs[(size_t)j * n + k], r);
                R[e] = r;
            }
            const size_t total = prep_diag_offset(NB) + (size_t)PREP_DIAG * NB;
            int bad = -1;
            for (size_t o = tid; o < total; o += BT_NT) prepC[o] = prep_value(W, LDW, n, NB, o, &bad);
            __syncthreads();
            // ---- a8: q = (a Rs^-1) Rc^-1 ----------------------------------------------------------------------------
            const SmemFactor fC{prepC, NB};
            zero_pad_columns<SR>(slab, n, N16, lane);
            for (int64_t i = warp; i < nslabs; i += BT_NW) {
                __syncwarp();
                if (p.vec) { load_slab<SR, true>(slab, A, p.lda, m, n, i * SR, lane); cp_async_wait_all(); }
                else load_slab<SR, false>(slab, A, p.lda, m, n, i * SR, lane);
                __syncwarp();
                solve_slab_f<RG, NB>(slab, fS, NB, lane);
                solve_slab_f<RG, NB>(slab, fC, NB, lane);
                __syncwarp();
                if (p.vec) store_slab<SR, true>(slab, Q, p.ldq, m, n, i * SR, lane);
                else store_slab<SR, false>(slab, Q, p.ldq, m, n, i * SR, lane);
            }
        }
        if (tid == 0) { p.codes[2 * b] = code; p.codes[2 * b + 1] = s_info; }
        __syncthreads();
    }
}

static BatchParams batched_layout(BatchParams p, int tsize)
{
    const int n16 = p.n16, s = p.s;
    auto al16 = [](int x) { return (x + 15) / 16 * 16; };
    int o = 0;
    p.o_idx = o;   o += al16(8 * s);
    p.o_kept = o;  o += al16(8 * s);
    p.o_as = o;    o += al16(8 * s * p.n);
    p.o_rs = o;    o += al16(8 * p.n * p.n);
    p.o_prepS = o; o += al16(8 * n16 * n16);
    p.o_prepC = o; o += al16(8 * n16 * n16);
    p.o_w = o;     o += al16(8 * n16 * (n16 + 1));
    p.o_work = o;
    const int nbw = (s + 31) / 32, nbp = nbw <= 1 ? 1 : (nbw <= 2 ? 2 : 4), nrg = BT_NW / nbp;
    const int k1 = 2 * n16 * (p.tr + 2) * 8 + p.tr * (n16 + 16 / tsize) * tsize;
    const int red = nrg * nbp * 32 * n16 * 8;
    const int k3 = BT_NW * n16 * 36 * 8 + BT_NW * n16 * n16 * 8;
    int w = k1 > red ? k1 : red;
    if (k3 > w) w = k3;
    p.total = o + al16(w);
    return p;
}

bool batched_fused_usable(int64_t m, int n, int s)
{
    return n <= 32 && s <= BT_SMAX && m >= 32 && m <= (1 << 16) && (double)m * s * round_up(n, 16) <= (double)(1u << 27);
}

// Enqueues the fused kernel; codes_dev: batch x 2 ints.  Returns the number of launches (0: shape not supported).
int launch_factor_batched(int batch, int64_t m, int n, int64_t lda, int64_t strideA, const double* A, int64_t ldq,
                          int64_t strideQ, double* Q, double* R, int prec, int s, uint64_t seed, int* codes_dev,
                          cudaStream_t st)
{
    if (!batched_fused_usable(m, n, s)) return 0;
    BatchParams p{};
    p.batch = batch; p.n = n; p.n16 = round_up(n, 16); p.s = s; p.prec = prec;
    p.m = m; p.lda = lda; p.strideA = strideA; p.ldq = ldq; p.strideQ = strideQ; p.seed = seed;
    p.A = A; p.Q = Q; p.R = R; p.codes = codes_dev;
    p.tr = m >= BT_TR ? BT_TR : (int)m;
    p.tr_sh = 0; while ((1 << p.tr_sh) < p.tr) ++p.tr_sh;
    p.vec = ((uintptr_t)A % 16 == 0) && (lda % 2 == 0) && (strideA % 2 == 0) &&
            ((uintptr_t)Q % 16 == 0) && (ldq % 2 == 0) && (strideQ % 2 == 0);
    p = batched_layout(p, prec == 64 ? 8 : 4);
#define BT_GO(T_, P_, NB_)                                                                                      \
    { auto k = mrcqr_factor_batched_kernel<T_, P_, NB_>;                                                        \
      cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, p.total);                            \
      int occ = 1;                                                                                              \
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, BT_NT, p.total);                                   \
      if (occ < 1) occ = 1;                                                                                     \
      int grid = occ * num_sms();                                                                               \
      if (grid > batch) grid = batch;                                                                           \
      k<<<grid, BT_NT, p.total, st>>>(p); }
#define BT_NB(T_, P_) { if (p.n16 == 16) BT_GO(T_, P_, 2) else BT_GO(T_, P_, 4) }
    if (prec == 16) BT_NB(float, 16) else if (prec == 32) BT_NB(float, 32) else BT_NB(double, 64)
#undef BT_NB
#undef BT_GO
    return 1;
}

} // namespace mrcqr
