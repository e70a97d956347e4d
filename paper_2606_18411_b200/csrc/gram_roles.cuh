// gram_roles.cuh -- accumulation of the upper triangle of G = Y^T Y in 8x8 DMMA blocks with compile-time
// block ownership, shared by K3 (k35_rows.cu, the fused Gram for n16 <= 128) and by the diagonal 128 x 128
// blocks of the SYRK (k3_syrk.cu).
#pragma once
#include "mrcqr_internal.cuh"
#include <type_traits>

namespace mrcqr {

// D(8x8) += A(8x4, row) * B(4x8, col), FP64 tensor-core op (SASS: DMMA.8x8x4 on sm_100a).
__device__ __forceinline__ void gram_dmma(double (&c)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// ---- Gram accumulation with compile-time block ownership (n16 <= 128) --------------------------------
// The upper triangle of G in 8x8 blocks (I <= J) is split over the NWG warps of a CTA so that a warp's
// blocks form rectangles / triangles: a warp that owns a set of blocks loads one fragment per distinct
// block row / column it touches and reuses it across its blocks (2-D register blocking; shared-memory
// traffic, not the FP64 pipe, was the limit of a row-wise split).
template <int NB, int NWG>
__host__ __device__ constexpr int gram_owner(int I, int J)
{
    if (NB == 8 && NWG == 4) {                       // 9 blocks per warp
        if (J < 4) return (I == 0 && J == 3) ? 2 : 0;
        if (I >= 4) return (I == 4 && J == 7) ? 3 : 1;
        return I < 2 ? 2 : 3;
    }
    if (NB == 16 && NWG == 8) {                      // 18,18,18,18,16,16,16,16 blocks
        const int a = I >> 2, b = J >> 2;
        if (a == b) return a;
        if (a == 0 && b == 1) return (I & 3) < 2 ? 0 : 1;
        if (a == 2 && b == 3) return (I & 3) < 2 ? 2 : 3;
        if (a == 0 && b == 2) return 4;
        if (a == 0 && b == 3) return 5;
        if (a == 1 && b == 2) return 6;
        return 7;
    }
    return (I < NB - 1 - I ? I : NB - 1 - I) % NWG;  // block rows r and NB-1-r: NB+1 blocks per warp
}
template <int NB, int NWG>
__host__ __device__ constexpr int gram_slot(int role, int I, int J)   // index of (I,J) among role's blocks
{
    int cnt = 0;
    for (int i = 0; i < NB; ++i)
        for (int j = i; j < NB; ++j) {
            if (i == I && j == J) return cnt;
            if (gram_owner<NB, NWG>(i, j) == role) ++cnt;
        }
    return cnt;
}
template <int NB, int NWG>
__host__ __device__ constexpr bool gram_needs(int role, int c)
{
    for (int i = 0; i < NB; ++i)
        for (int j = i; j < NB; ++j)
            if (gram_owner<NB, NWG>(i, j) == role && (i == c || j == c)) return true;
    return false;
}
template <int NB, int NWG>
__host__ __device__ constexpr int gram_maxown()
{
    int mx = 0;
    for (int r = 0; r < NWG; ++r) { const int c = gram_slot<NB, NWG>(r, NB, NB); if (c > mx) mx = c; }
    return mx;
}

// compile-time loop: f(std::integral_constant<int, B>) ... f(std::integral_constant<int, E-1>)
template <int B, int E, typename F>
__device__ __forceinline__ void static_for(F&& f)
{
    if constexpr (B < E) { f(std::integral_constant<int, B>{}); static_for<B + 1, E>(f); }
}

template <int NB, int NWG, int ROLE, int SR, int NSLAB, int MAXOWN>
__device__ __forceinline__ void gram_accumulate(double (&acc)[MAXOWN][2], const double* tile, int slab_stride, int lane)
{
    constexpr int LDS_ = SR + 4;
    const int g = lane >> 2, t = lane & 3;
    for (int w = 0; w < NSLAB; ++w) {
        const double* y0 = tile + (size_t)w * slab_stride + g * LDS_ + t;
#pragma unroll 2
        for (int ks = 0; ks < SR / 4; ++ks) {
            const double* yk = y0 + 4 * ks;
            double f[NB];
            static_for<0, NB>([&](auto Cc) {
                constexpr int c = decltype(Cc)::value;
                if constexpr (gram_needs<NB, NWG>(ROLE, c)) f[c] = yk[(8 * c) * LDS_];
            });
            static_for<0, NB>([&](auto Ic) {
                constexpr int I = decltype(Ic)::value;
                static_for<I, NB>([&](auto Jc) {
                    constexpr int J = decltype(Jc)::value;
                    if constexpr (gram_owner<NB, NWG>(I, J) == ROLE) {
                        constexpr int slot = gram_slot<NB, NWG>(ROLE, I, J);
                        gram_dmma(acc[slot], f[I], f[J]);
                    }
                });
            });
        }
    }
}

// Every element of a partial belongs to ONE thread for the whole kernel, so later flushes add with a result-less
// atomicAdd (RED.ADD.F64: fire and forget, same rounding as DADD, applied in program order for one thread and one
// address: still deterministic) instead of a load-add-store whose load latency every warp would wait out.
template <int NB, int NWG, int ROLE, int MAXOWN>
__device__ __forceinline__ void gram_flush(double (&acc)[MAXOWN][2], double* part, int n16, bool first, int lane)
{
    const int g = lane >> 2, t = lane & 3;
    static_for<0, NB>([&](auto Ic) {
        constexpr int I = decltype(Ic)::value;
        static_for<I, NB>([&](auto Jc) {
            constexpr int J = decltype(Jc)::value;
            if constexpr (gram_owner<NB, NWG>(I, J) == ROLE) {
                constexpr int slot = gram_slot<NB, NWG>(ROLE, I, J);
                double* dst = part + (size_t)(8 * J + 2 * t) * n16 + 8 * I + g;
                if (first) { dst[0] = acc[slot][0]; dst[n16] = acc[slot][1]; }
                else { atomicAdd(dst, acc[slot][0]); atomicAdd(dst + n16, acc[slot][1]); }
                acc[slot][0] = acc[slot][1] = 0.0;
            }
        });
    });
}


} // namespace mrcqr
