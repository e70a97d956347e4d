// mrcqr_internal.cuh -- shared declarations of the CUDA path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstddef>

namespace mrcqr {

// device status block (8 ints): [0] = first error code, [1] = info (pivot index), rest scratch
struct Status { int code; int info; int pad[6]; };

__device__ __forceinline__ void report(Status* st, int code, int info)
{
    if (atomicCAS(&st->code, 0, code) == 0) st->info = info;
}

inline int round_up(int x, int q) { return (x + q - 1) / q * q; }

// ---- tile geometry of the row-streaming kernels (K3 / K5), chosen from n only -----------------
// n16 = n padded to a multiple of 16 (8-wide DMMA blocks, 16-wide Gram super-blocks).
struct RowCfg { int n16; int TM; int NW; int smem_bytes; int ctas_per_sm; };
RowCfg row_config(int n);

// "prepared" upper-triangular factor consumed by the tile solve: n16 x n16 col-major, ld = n16,
//   strictly upper part = -R[k,j], diagonal = 1/R[j,j], padding = identity, strictly lower = 0.
// Built once per factor by prep_R; both K3 and K5 read the same buffer (bit-identical Y).

// launchers (each returns the number of kernel launches it enqueued)
int launch_prep_R(const double* R, int n, double* Rprep, int n16, Status* st, int err_code, cudaStream_t s);
int launch_k3_gram(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                   double* partials, int* n_partials_out, double* Ydump, cudaStream_t s);
int launch_reduce_partials(const double* partials, int n_partials, int n, int n16, double* G16, cudaStream_t s);
int launch_k4_cholesky(const double* G16, int n, int n16, double* G_out, double* Rc, double* RcPrep,
                       Status* st, cudaStream_t s);
int launch_k5_formq(int64_t m, int n, int64_t lda, const double* A, const double* RsPrep,
                    const double* RcPrep, int64_t ldq, double* Q, double* Ydump, cudaStream_t s);
int launch_triu_mul(const double* Rc, const double* Rs, int n, double* R, cudaStream_t s);
int launch_k2_sketch_qr(const double* As, int s_rows, int n, double* work, double* Rs, Status* st, cudaStream_t s);

// K1: sampled transform.  Returns launches.  As (s x n, ld = s) receives precision-p values in FP64.
size_t k1_workspace_bytes(int64_t m, int n, int s, int prec);
int launch_k1_srtt(int64_t m, int n, int64_t lda, const double* A, int prec, int s,
                   const uint64_t* signs, const int64_t* idx, void* k1_work, double* As,
                   Status* st, cudaStream_t stream);

size_t k3_partials_bytes(int n);
int num_sms();

} // namespace mrcqr
