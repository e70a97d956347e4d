// orth_static.cu -- mrcqr_orth_error_noalloc: ||I - Q^T Q||_F without any allocation.
//
// The ordinary entry point (mrcqr_orth_error, api.cu) takes the partials of the split-m Gram accumulation,
// the n16 x n16 Gram matrix and the norm from the context's workspace, which it grows with cudaMalloc on
// first use.  Callers that cannot allocate (stream capture, serving loops, harnesses that forbid it) get the
// same kernels in the same order here, with that scratch in the file-scope device array below.
//
//   * Size: NA_DOUBLES * 8 = 20 054 016 bytes (19.1 MiB), held by every GPU that loads the library until the
//     process exits.  It fits n <= MRCQR_NOALLOC_N_MAX = 128 (one 128 x 128 block, one partial per SYRK CTA,
//     at most NA_PARTIALS = 152 CTAs: the launcher uses one per SM) and any m.  Anything larger is refused
//     with MRCQR_ERR_TOO_LARGE before a kernel is launched.
//   * Every call shares the array and finds the last call's contents in it.  Nothing has to start at zero:
//     each SYRK CTA stores (not adds) its first flush over its whole partial, the reduction reads only what
//     this call's CTAs wrote and writes every element of G16 that is read afterwards.
//   * Calls that overlap on the GPU (two streams, two host threads) RACE on the array: serialise them.
//   * The call allocates nothing, frees nothing, reads nothing back and does not synchronise: it enqueues its
//     kernels on the stream and returns; err (and G) are DEVICE outputs, valid once the stream reaches them.
//
// In host code `na_scratch` is a host-side stand-in for the symbol, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
#include "../mrcqr_internal.cuh"
#include "../../../include/mrcqr.h"
#include <mutex>

namespace mrcqr {

constexpr int NA_N16 = 128;                                   // MRCQR_NOALLOC_N_MAX
constexpr int NA_PARTIALS = 152;                              // >= SMs + 1 of every sm_100a part (B200: 148)
constexpr size_t NA_BLOCK = (size_t)NA_N16 * NA_N16;          // doubles of one 128 x 128 block
constexpr size_t NA_DOUBLES = (NA_PARTIALS + 1) * NA_BLOCK;   // partials, then G16

static __device__ __align__(256) double na_scratch[NA_DOUBLES];

constexpr int NA_MAX_DEVICES = 64;
static double* na_ptr[NA_MAX_DEVICES];                        // device address of na_scratch, per device
static std::mutex na_mutex;

// device address of the scratch array on the CURRENT device (asked once per device), or nullptr
static double* na_device_scratch()
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) return nullptr;
    std::lock_guard<std::mutex> lock(na_mutex);
    if (!na_ptr[dev]) {
        double* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, na_scratch) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        na_ptr[dev] = p;
    }
    return na_ptr[dev];
}

// G (n x n, ld n, full symmetric) <- the leading n x n of G16 (ld n16)
__global__ void __launch_bounds__(256)
mrcqr_noalloc_copy_g(const double* __restrict__ G16, int n, int n16, double* __restrict__ G)
{
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x)
        G[e] = G16[(size_t)(e / n) * n16 + e % n];
}

} // namespace mrcqr

using namespace mrcqr;

extern "C" int mrcqr_orth_error_noalloc(int64_t m, int n, int64_t ldq, const double* Q, double* err, double* G, void* stream)
{
    if (n < 1) return -2;
    if (m < n) return -1;
    if (ldq < m) return -3;
    if (!Q) return -4;
    if (!err) return -5;
    const int n16 = round_up(n, 16);
    if (n > MRCQR_NOALLOC_N_MAX || n16 > NA_N16) return MRCQR_ERR_TOO_LARGE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return MRCQR_ERR_CUDA; }
    if (syrk_partials_bytes(n) > NA_PARTIALS * NA_BLOCK * sizeof(double)) return MRCQR_ERR_TOO_LARGE;   // a part with > 151 SMs
    double* scratch = na_device_scratch();
    if (!scratch) return MRCQR_ERR_CUDA;
    double* part = scratch;
    double* G16 = scratch + NA_PARTIALS * NA_BLOCK;
    cudaStream_t st = (cudaStream_t)stream;
    launch_syrk(m, n, ldq, Q, part, n16, G16, st);            // mrcqr_syrk + mrcqr_syrk_reduce (k3_syrk.cu)
    launch_orth_norm(G16, n, n16, err, st);
    if (G) mrcqr_noalloc_copy_g<<<(n * n + 255) / 256, 256, 0, st>>>(G16, n, n16, G);
    return cudaGetLastError() == cudaSuccess ? 0 : MRCQR_ERR_CUDA;
}
