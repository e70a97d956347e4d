// api.cu -- the C ABI declared in include/mrcqr.h: argument checking, the library-owned workspace,
// the seeded draw (Algorithm 2 step 1) and the composition of the kernels K1..K5.
#include "../../include/mrcqr.h"
#include "mrcqr_internal.cuh"
#include <algorithm>
#include <mutex>
#include <cstring>
#include <vector>

namespace mrcqr {

// device side of the draw: sign words, plus reset of the status block (first kernel of a call)
__global__ void mrcqr_draw_signs(uint64_t seed, int64_t nwords, uint64_t* __restrict__ signs, Status* st)
{
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w == 0 && st) { st->code = 0; st->info = 0; }
    if (w < nwords) signs[w] = splitmix64_at(seed, (uint64_t)w);
}

__global__ void mrcqr_reset_status(Status* st) { st->code = 0; st->info = 0; }

// same as mrcqr_draw_signs with the seed read from device memory (graph replay: the seed is data, not a launch parameter)
__global__ void mrcqr_draw_signs_p(const uint64_t* __restrict__ seedp, int64_t nwords, uint64_t* __restrict__ signs, Status* st)
{
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t seed = *seedp;
    if (w == 0 && st) { st->code = 0; st->info = 0; }
    if (w < nwords) signs[w] = splitmix64_at(seed, (uint64_t)w);
}

static void draw_bins_host(int64_t m, int s, uint64_t seed, int64_t* idx)
{
    const uint64_t nw = (uint64_t)((m + 63) / 64), B = (uint64_t)(m / 2 + 1);
    std::vector<int64_t> sorted;                 // kept candidates, ascending (binary search = "is new")
    sorted.reserve((size_t)s);
    for (uint64_t k = nw; (int)sorted.size() < s; ++k) {
        const unsigned __int128 prod = (unsigned __int128)splitmix64_at(seed, k) * (unsigned __int128)B;
        const int64_t cand = (int64_t)(uint64_t)(prod >> 64);
        auto it = std::lower_bound(sorted.begin(), sorted.end(), cand);
        if (it == sorted.end() || *it != cand) sorted.insert(it, cand);
    }
    std::memcpy(idx, sorted.data(), sizeof(int64_t) * (size_t)s);
}

// ---- workspace -----------------------------------------------------------------------------------
struct Layout {
    size_t status, signs, idx, As, Rs, RsPrep, RcPrep, G16, Rc, Rtmp, betas, k1, k3, total;
};

static size_t al(size_t x) { return (x + 255) / 256 * 256; }

static Layout make_layout(int64_t m, int n, int s, int prec)
{
    Layout L;
    const size_t n16 = (size_t)round_up(n, 16);
    size_t o = 0;
    L.status = o; o += al(sizeof(Status));
    L.signs = o;  o += al((size_t)((m + 63) / 64) * 8);
    L.idx = o;    o += al((size_t)std::max(s, 1) * 8);
    L.As = o;     o += al((size_t)2 * std::max(s, 1) * n * 8);       // 2s rows in the Re+Im variant
    L.Rs = o;     o += al((size_t)n * n * 8);
    L.RsPrep = o; o += al(n16 * n16 * 8);
    L.RcPrep = o; o += al(n16 * n16 * 8);
    L.G16 = o;    o += al(n16 * n16 * 8);
    L.Rc = o;     o += al((size_t)n * n * 8);
    L.Rtmp = o;   o += al((size_t)2 * n * n * 8);                        // CholQR2: R1, R2
    L.betas = o;  o += al((size_t)n * 8);
    L.k1 = o;     o += al(s > 0 ? k1_workspace_bytes(m, n, s, prec) : 0);
    L.k3 = o;     o += al(std::max(k3_partials_bytes(n), syrk_partials_bytes(n)));   // Gram partials of either stage-2 form
    L.total = o;
    return L;
}

constexpr int ASYNC_RING = 8;          // pinned bin buffers of mrcqr_factor_async calls in flight
struct Ctx {
    char* ws = nullptr; size_t ws_bytes = 0;
    int* h_status = nullptr;                 // pinned, 2 ints
    int64_t* h_idx = nullptr; size_t h_idx_cap = 0;   // pinned staging of the bins
    double* hA = nullptr; double* hQ = nullptr; double* hR = nullptr; size_t hA_bytes = 0, hR_bytes = 0; // host-path device buffers
    int last_info = 0, last_launches = 0;
    bool last_graph = false;                 // the last mrcqr_factor call replayed a CUDA graph
    cudaStream_t host_stream = nullptr;      // mrcqr_factor_host: a non-blocking stream of the library's own
    int* bcodes = nullptr; int* h_bcodes = nullptr; size_t bcodes_cap = 0;   // mrcqr_factor_batched: (code, info) per problem, device + pinned
    bool timing = false; cudaEvent_t ev[8] = {}; bool ev_ok = false; float stage_ms[8] = {};
    bool have_device = false, probed = false;
    int store_y = -1;                        // mrcqr_set_store_y: -1 by measured threshold, 0 never for n16 <= 128, 1 always
    bool last_store_y = false;               // what the last mrcqr_factor did
    bool reim = false;                       // mrcqr_set_sketch_reim: Re+Im sketch (2s rows)
    // mrcqr_set_graph: the whole enqueue sequence of mrcqr_factor captured once per (shape, buffers) and replayed
    bool use_graph = false;
    cudaGraphExec_t gexec = nullptr; int glaunches = 0; uint64_t* h_seed = nullptr;
    struct { int64_t m, lda; int n, prec, s; const void *A, *Q, *R, *ws, *hidx; int store_y; bool reim; } gkey = {};
    // mrcqr_factor_async: calls in flight.  Each one owns a slot of a ring of pinned bin buffers until the event recorded
    // behind its host-to-device copy has completed; the run-time status stays in the device status block (first error
    // wins) until mrcqr_wait reads and clears it.
    int64_t* h_ring = nullptr; size_t h_ring_cap = 0; int ring_pos = 0;
    cudaEvent_t ring_ev[ASYNC_RING] = {}; bool ring_busy[ASYNC_RING] = {};
    int async_pending = 0; cudaStream_t async_stream = nullptr; size_t async_status_off = 0; bool in_async = false;
};
// Every entry point works on the calling thread's CURRENT context: the process default one, or the handle made current
// with mrcqr_set_current (mrcqr_create / mrcqr_destroy).  A context owns its workspace, staging buffers, settings,
// status and graph cache, so two host threads with a handle and a stream each may factor at the same time.
static Ctx g_default;
static thread_local Ctx* t_current = nullptr;
static inline Ctx& ctx() { return t_current ? *t_current : g_default; }
#define g (ctx())

// The diagonal-block coefficients of the row kernels are constant-bank operands (rows.cuh: c_diag, c_pdiag), a device-wide
// resource: the stretch "upload the prepared diagonal blocks ... last kernel that reads them" of one factorization must not
// interleave with another context's.  The gate orders such stretches ON THE DEVICE (a stream waits for the event the
// previous stretch recorded) and on the host (a mutex held while the stretch is enqueued); everything before it (K1, K2)
// and the batched kernel (coefficients in shared memory) overlap freely.
// While the process has only its default context (mrcqr_create never called) two stretches cannot be in flight at once
// (one workspace: its calls are ordered already), and the two stream operations per stretch are skipped: they are part
// of the gaps between the kernels of a small factorization.  mrcqr_create synchronises the device once and turns them on.
struct ConstGate {
    std::recursive_mutex mu;                 // recursive: a call that spans two stretches (the debug dump) nests them
    cudaEvent_t ev = nullptr;
    bool pending = false;
    bool multi = false;                      // a second context exists (or existed)
    void acquire(cudaStream_t st)
    {
        mu.lock();
        if (!multi) return;
        if (!ev) cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        cudaStreamIsCapturing(st, &cs);
        if (pending && cs == cudaStreamCaptureStatusNone) cudaStreamWaitEvent(st, ev, 0);
    }
    void release(cudaStream_t st)
    {
        if (multi) {
            cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
            cudaStreamIsCapturing(st, &cs);
            if (cs == cudaStreamCaptureStatusNone) { cudaEventRecord(ev, st); pending = true; }
        }
        mu.unlock();
    }
    void enable()
    {
        std::lock_guard<std::recursive_mutex> lk(mu);
        if (!multi) { cudaDeviceSynchronize(); cudaGetLastError(); multi = true; }
    }
};
static ConstGate g_gate;
struct GateScope {
    cudaStream_t st;
    explicit GateScope(cudaStream_t s) : st(s) { g_gate.acquire(st); }
    ~GateScope() { g_gate.release(st); }
};

static void drop_graph()
{
    if (g.gexec) { cudaGraphExecDestroy(g.gexec); g.gexec = nullptr; }
}

static bool device_ok()
{
    if (!g.probed) {
        int cnt = 0;
        g.have_device = (cudaGetDeviceCount(&cnt) == cudaSuccess && cnt > 0);
        if (!g.have_device) cudaGetLastError();
        g.probed = true;
    }
    return g.have_device;
}

static bool ensure_ws(size_t bytes)
{
    if (!g.h_status && cudaMallocHost(&g.h_status, 64) != cudaSuccess) return false;   // [0..1] status, [2..3] a double
    // a synchronous entry point while mrcqr_factor_async calls are in flight: they finish first (the workspace is shared);
    // their status is dropped with the pending count, as the header says
    if (g.async_pending > 0 && !g.in_async) { cudaStreamSynchronize(g.async_stream); g.async_pending = 0; }
    if (bytes <= g.ws_bytes) return true;
    if (g.ws) { cudaDeviceSynchronize(); drop_graph(); cudaFree(g.ws); g.ws = nullptr; g.ws_bytes = 0; }
    if (cudaMalloc(&g.ws, bytes) != cudaSuccess) { cudaGetLastError(); return false; }
    g.ws_bytes = bytes;
    return true;
}

static bool ensure_hidx(size_t count)
{
    if (count <= g.h_idx_cap) return true;
    if (g.h_idx) cudaFreeHost(g.h_idx);
    g.h_idx_cap = 0;
    if (cudaMallocHost(&g.h_idx, count * sizeof(int64_t)) != cudaSuccess) { g.h_idx = nullptr; return false; }
    g.h_idx_cap = count;
    return true;
}

// reads the status block back and synchronises; returns the final code of the call
static int finish(const Layout& L, cudaStream_t st, int launches)
{
    g.last_launches = launches;
    g.last_graph = false;
    cudaMemcpyAsync(g.h_status, g.ws + L.status, 8, cudaMemcpyDeviceToHost, st);
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MRCQR_ERR_CUDA;
    g.last_info = g.h_status[1];
    return g.h_status[0];
}

static bool is_pow2(int64_t m) { return m > 0 && (m & (m - 1)) == 0; }
static bool prec_ok(int p) { return p == 16 || p == 32 || p == 64; }
constexpr int N_MAX = 512;
constexpr int S_MAX = 4096;
constexpr int STORE_Y_AUTO_N16 = 48;     // n16 from which storing Y is the faster form of stage 2 (measured, see enqueue_stage23)
constexpr int STORE_Y_SYRK_N16 = 128;    // ... and from which the stored Y goes through the panel solves and the SYRK

// enqueue helpers shared by the stage calls and mrcqr_factor ----------------------------------------
static int enqueue_sketch(const Layout& L, int64_t m, int n, int64_t lda, const double* A, int prec, int s,
                          const uint64_t* signs, const int64_t* idx, double* As_out, double* Rs, cudaStream_t st)
{
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    double* As = reinterpret_cast<double*>(g.ws + L.As);
    const int rows = g.reim ? 2 * s : s;
    int k = launch_k1_srtt(m, n, lda, A, prec, s, signs, idx, g.ws + L.k1, As, stat, st, g.reim);
    if (As_out) cudaMemcpyAsync(As_out, As, sizeof(double) * (size_t)rows * n, cudaMemcpyDeviceToDevice, st);
    k += launch_k2_sketch_qr(As, rows, n, Rs, reinterpret_cast<double*>(g.ws + L.RsPrep), round_up(n, 16),
                             reinterpret_cast<double*>(g.ws + L.betas), stat, st);
    return k;
}

static int enqueue_gram(const Layout& L, int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                        double* G_out, double* Rc, double* Ydump, cudaStream_t st)
{
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    const int n16 = round_up(n, 16);
    double* RsPrep = reinterpret_cast<double*>(g.ws + L.RsPrep);
    double* RcPrep = reinterpret_cast<double*>(g.ws + L.RcPrep);
    double* G16 = reinterpret_cast<double*>(g.ws + L.G16);
    double* part = reinterpret_cast<double*>(g.ws + L.k3);
    int np = 0;
    GateScope gate(st);
    int k = launch_prep_R(Rs, n, RsPrep, n16, stat, MRCQR_ERR_SINGULAR, st);
    k += upload_diag(RsPrep, n16, 0, st);
    k += launch_k3_gram(m, n, lda, A, RsPrep, part, &np, Ydump, nullptr, 0, st);
    k += launch_reduce_partials(part, np, n, n16, G16, st);
    k += launch_k4_cholesky(G16, n, n16, G_out, Rc, RcPrep, nullptr, nullptr, stat, st);
    k += upload_diag(RcPrep, n16, 1, st);
    return k;
}

static int enqueue_formq(const Layout& L, int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                         const double* Rc, bool prep_rs, bool prep_rc, int64_t ldq, double* Q, double* R,
                         double* Ydump, cudaStream_t st)
{
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    const int n16 = round_up(n, 16);
    double* RsPrep = reinterpret_cast<double*>(g.ws + L.RsPrep);
    double* RcPrep = reinterpret_cast<double*>(g.ws + L.RcPrep);
    int k = 0;
    GateScope gate(st);
    if (prep_rs) { k += launch_prep_R(Rs, n, RsPrep, n16, stat, MRCQR_ERR_SINGULAR, st); k += upload_diag(RsPrep, n16, 0, st); }
    if (prep_rc) { k += launch_prep_R(Rc, n, RcPrep, n16, stat, MRCQR_ERR_BREAKDOWN, st); k += upload_diag(RcPrep, n16, 1, st); }
    k += launch_k5_formq(m, n, lda, A, RsPrep, RcPrep, ldq, Q, Ydump, 3, st);
    if (R) k += launch_triu_mul(Rc, Rs, n, R, st);
    return k;
}

} // namespace mrcqr

// =================================================================================================
// C ABI
// =================================================================================================
using namespace mrcqr;

extern "C" int mrcqr_draw(int64_t m, int s, uint64_t seed, uint64_t* signs_host, int64_t* idx_host)
{
    if (m < 1) return -1;
    if (s < 0 || (int64_t)s > m / 2 + 1) return -2;
    if (!signs_host) return -4;
    if (!idx_host && s > 0) return -5;
    const int64_t nw = (m + 63) / 64;
    for (int64_t w = 0; w < nw; ++w) signs_host[w] = splitmix64_at(seed, (uint64_t)w);
    if (s > 0) draw_bins_host(m, s, seed, idx_host);
    return 0;
}

// The draw exactly as mrcqr_factor performs it: sign words by the device kernel, bins on the host and copied.
extern "C" int mrcqr_draw_device(int64_t m, int s, uint64_t seed, uint64_t* signs, int64_t* idx, void* stream)
{
    if (m < 1) return -1;
    if (s < 0 || (int64_t)s > m / 2 + 1) return -2;
    if (!signs) return -4;
    if (!idx && s > 0) return -5;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    if (!ensure_hidx((size_t)std::max(s, 1))) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t nw = (m + 63) / 64;
    mrcqr_draw_signs<<<(unsigned)((nw + 255) / 256), 256, 0, st>>>(seed, nw, signs, nullptr);
    if (s > 0) {
        draw_bins_host(m, s, seed, g.h_idx);
        cudaMemcpyAsync(idx, g.h_idx, sizeof(int64_t) * (size_t)s, cudaMemcpyHostToDevice, st);
    }
    g.last_launches = 1; g.last_graph = false;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MRCQR_ERR_CUDA;
    return 0;
}

extern "C" size_t mrcqr_workspace_bytes(int64_t m, int n, int s, mrcqr_prec_t prec)
{
    if (m < 1 || n < 1 || n > N_MAX || !prec_ok((int)prec) || !device_ok()) return 0;
    if (s <= 0) s = 3 * n;
    return make_layout(m, n, s, (int)prec).total;
}

extern "C" int mrcqr_last_info(void) { return g.last_info; }
extern "C" int mrcqr_last_launch_count(void) { return g.last_launches; }
extern "C" int mrcqr_last_used_graph(void) { return g.last_graph ? 1 : 0; }

static void free_ctx(Ctx& c)
{
    if (!c.probed || !c.have_device) { c = Ctx(); return; }
    cudaDeviceSynchronize();
    if (c.gexec) { cudaGraphExecDestroy(c.gexec); c.gexec = nullptr; }
    if (c.h_seed) cudaFreeHost(c.h_seed);
    if (c.ws) cudaFree(c.ws);
    if (c.h_status) cudaFreeHost(c.h_status);
    if (c.h_idx) cudaFreeHost(c.h_idx);
    if (c.h_ring) cudaFreeHost(c.h_ring);
    for (int i = 0; i < ASYNC_RING; ++i) if (c.ring_ev[i]) cudaEventDestroy(c.ring_ev[i]);
    if (c.ev_ok) for (int i = 0; i < 8; ++i) cudaEventDestroy(c.ev[i]);
    if (c.hA) cudaFree(c.hA);
    if (c.hQ) cudaFree(c.hQ);
    if (c.hR) cudaFree(c.hR);
    if (c.host_stream) cudaStreamDestroy(c.host_stream);
    if (c.bcodes) cudaFree(c.bcodes);
    if (c.h_bcodes) cudaFreeHost(c.h_bcodes);
    c = Ctx();
}

extern "C" void mrcqr_shutdown(void) { free_ctx(ctx()); }

extern "C" int mrcqr_create(mrcqr_handle_t* handle)
{
    if (!handle) return -1;
    g_gate.enable();
    *handle = reinterpret_cast<mrcqr_handle_t>(new Ctx());
    return 0;
}

extern "C" int mrcqr_destroy(mrcqr_handle_t handle)
{
    if (!handle) return -1;
    Ctx* c = reinterpret_cast<Ctx*>(handle);
    if (t_current == c) t_current = nullptr;
    free_ctx(*c);
    delete c;
    return 0;
}

extern "C" int mrcqr_set_current(mrcqr_handle_t handle)
{
    t_current = reinterpret_cast<Ctx*>(handle);       // NULL: the process default context
    return 0;
}

extern "C" int mrcqr_sketch(int64_t m, int n, int64_t lda, const double* A, mrcqr_prec_t prec, int s,
                            const uint64_t* signs, const int64_t* idx, double* As_out, double* Rs,
                            void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (!is_pow2(m) || m < n || m < 32) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!prec_ok((int)prec)) return -5;
    if (s < n || (int64_t)s > m / 2 + 1 || s > S_MAX || (g.reim && 2 * s > S_MAX)) return -6;
    if (!signs) return -7;
    if (!idx) return -8;
    if (!Rs) return -10;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    Layout L = make_layout(m, n, s, (int)prec);
    if (!ensure_ws(L.total)) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    mrcqr_reset_status<<<1, 1, 0, st>>>(stat);
    int k = 1 + enqueue_sketch(L, m, n, lda, A, (int)prec, s, signs, idx, As_out, Rs, st);
    return finish(L, st, k);
}

extern "C" int mrcqr_precondition_gram(int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                                       double* G_out, double* Rc, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (m < n) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!Rs) return -5;
    if (!Rc) return -7;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    Layout L = make_layout(m, n, 0, 64);
    if (!ensure_ws(L.total)) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    mrcqr_reset_status<<<1, 1, 0, st>>>(reinterpret_cast<Status*>(g.ws + L.status));
    int k = 1 + enqueue_gram(L, m, n, lda, A, Rs, G_out, Rc, nullptr, st);
    return finish(L, st, k);
}

extern "C" int mrcqr_form_q(int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                            const double* Rc, int64_t ldq, double* Q, double* R, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (m < n) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!Rs) return -5;
    if (!Rc) return -6;
    if (ldq < m) return -7;
    if (!Q) return -8;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    Layout L = make_layout(m, n, 0, 64);
    if (!ensure_ws(L.total)) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    mrcqr_reset_status<<<1, 1, 0, st>>>(reinterpret_cast<Status*>(g.ws + L.status));
    int k = 1 + enqueue_formq(L, m, n, lda, A, Rs, Rc, true, true, ldq, Q, R, nullptr, st);
    return finish(L, st, k);
}

extern "C" int mrcqr_debug_dump_y(int64_t m, int n, int64_t lda, const double* A, const double* Rs,
                                  double* Y_stage2a, double* Y_stage2b, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (m < n) return -1;
    if (lda < m) return -3;
    if (!A || !Rs || !Y_stage2a || !Y_stage2b) return -4;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    Layout L = make_layout(m, n, 0, 64);
    if (!ensure_ws(L.total)) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    mrcqr_reset_status<<<1, 1, 0, st>>>(reinterpret_cast<Status*>(g.ws + L.status));
    double* Rc = reinterpret_cast<double*>(g.ws + L.Rc);
    GateScope gate(st);                              // stage 2b below reuses the coefficients stage 2a uploaded
    int k = 1 + enqueue_gram(L, m, n, lda, A, Rs, nullptr, Rc, Y_stage2a, st);
    k += enqueue_formq(L, m, n, lda, A, Rs, Rc, false, false, m, nullptr, nullptr, Y_stage2b, st);   // Q = nullptr: not stored
    int rc = finish(L, st, k);
    return rc;
}

static bool timing_events()
{
    if (!g.ev_ok) {
        for (int i = 0; i < 8; ++i) if (cudaEventCreate(&g.ev[i]) != cudaSuccess) return false;
        g.ev_ok = true;
    }
    return true;
}

extern "C" int mrcqr_set_timing(int on) { g.timing = (on != 0); return 0; }
extern "C" int mrcqr_set_store_y(int mode) { g.store_y = mode < 0 ? -1 : (mode != 0); return 0; }
extern "C" int mrcqr_last_used_store_y(void) { return g.last_store_y ? 1 : 0; }
extern "C" int mrcqr_set_sketch_reim(int on) { g.reim = (on != 0); return 0; }
extern "C" int mrcqr_set_graph(int on) { g.use_graph = (on != 0); if (!on) drop_graph(); return 0; }

extern "C" int mrcqr_last_timing(float* ms_out_host)
{
    if (!ms_out_host) return -1;
    for (int i = 0; i < 7; ++i) ms_out_host[i] = g.stage_ms[i];
    return 0;
}

// Stage 2 + 3 of Algorithm 2 (steps 7-9) on device buffers, the prepared R_s already in the workspace:
// precondition + Gram, Cholesky (+ R = Rc Rs), form Q.  Shared by mrcqr_factor and the CholQR entry points.
static int enqueue_stage23(const Layout& L, int64_t m, int n, int64_t lda, const double* A, int64_t ldq, double* Q,
                           double* R, const double* Rs, cudaStream_t st, bool tm)
{
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    double* Rc = reinterpret_cast<double*>(g.ws + L.Rc);
    int k = 0;
    {
        const int n16 = round_up(n, 16);
        double* RsPrep = reinterpret_cast<double*>(g.ws + L.RsPrep);
        double* RcPrep = reinterpret_cast<double*>(g.ws + L.RcPrep);
        double* G16 = reinterpret_cast<double*>(g.ws + L.G16);
        double* part = reinterpret_cast<double*>(g.ws + L.k3);
        int np = 0;
        GateScope gate(st);
        k += upload_diag(RsPrep, n16, 0, st);
        if (tm) cudaEventRecord(g.ev[3], st);
        // Stage 2 has three forms (include/mrcqr.h, mrcqr_set_store_y):
        //   fused   K3 keeps Y = A Rs^-1 on chip, K5 recomputes it bit-identically (north_star's form; 4 m n^2 flops)
        //   dump    K3 also writes Y into Q's buffer, K5 solves it in place against Rc (3 m n^2 flops, same Q bit for bit)
        //   syrk    panel solve writes Y, the SYRK forms G from it, panel solve in place (3 m n^2 flops; the only form for
        //           n16 > 128, where the Gram matrix no longer fits one SM)
        // Default (-1): the fastest measured one.  m = 2^21, ms per factorization, fused / dump / syrk:
        //   n16 = 16: 0.309 / 0.334 / 1.58   32: 0.620 / 0.632 / 1.85   48: 1.094 / 1.030 / -   64: 1.79 / 1.69 / 2.66
        //   80: 3.13 / 2.86 / 3.78   96: 3.94 / 3.57 / 4.30   112: 5.10 / 4.60 / 4.80   128: 6.69 / 5.93 / 5.09
        // i.e. fused while HBM binds (n16 <= 32), dump for 48 <= n16 <= 112, syrk from 128 on.
        const bool panels_ok = panel_pass_usable(m, n, A, lda, Q, ldq);
        const bool want_y = n16 > 128 || g.store_y > 0 || (g.store_y < 0 && n16 >= STORE_Y_AUTO_N16);
        const bool syrk_form = n16 > 128 || (want_y && n16 >= STORE_Y_SYRK_N16 && panels_ok);
        const bool panels = syrk_form && panels_ok;
        const bool dump_form = want_y && !syrk_form;
        g.last_store_y = want_y;
        if (syrk_form) {
            if (panels) k += launch_panel_solve(m, n, 0, A, lda, RsPrep, Q, ldq, st);
            else k += launch_k5_formq(m, n, lda, A, RsPrep, RcPrep, ldq, Q, nullptr, 1, st);
            if (tm) cudaEventRecord(g.ev[4], st);
            k += launch_syrk(m, n, ldq, Q, part, n16, G16, st);
        } else {
            k += launch_k3_gram(m, n, lda, A, RsPrep, part, &np, nullptr, dump_form ? Q : nullptr, ldq, st);
            if (tm) cudaEventRecord(g.ev[4], st);
            k += launch_reduce_partials(part, np, n, n16, G16, st);
        }
        if (tm) cudaEventRecord(g.ev[5], st);
        k += launch_k4_cholesky(G16, n, n16, nullptr, Rc, RcPrep, Rs, R, stat, st);     // + step 9: R = Rc Rs
        k += upload_diag(RcPrep, n16, 1, st);
        if (tm) cudaEventRecord(g.ev[6], st);
        if (panels) k += launch_panel_solve(m, n, 1, Q, ldq, RcPrep, Q, ldq, st);                // q = y Rc^-1 in place
        else if (syrk_form || dump_form) k += launch_k5_formq(m, n, ldq, Q, RsPrep, RcPrep, ldq, Q, nullptr, 2, st);
        else k += launch_k5_formq(m, n, lda, A, RsPrep, RcPrep, ldq, Q, nullptr, 3, st);        // Alg.1 step 3
        if (tm) cudaEventRecord(g.ev[7], st);
    }
    return k;
}

// enqueues steps 1-9 on st.  seed_dev != nullptr: the seed and the bins are read from seed_dev / the pinned
// staging buffers when the work RUNS (graph capture); otherwise they are taken now.
static int enqueue_factor(const Layout& L, int64_t m, int n, int64_t lda, const double* A, int64_t ldq, double* Q,
                          double* R, int prec, int s, uint64_t seed, const uint64_t* seed_dev, cudaStream_t st, bool tm,
                          const int64_t* h_bins = nullptr, bool reset_status = true)
{
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    Status* stat0 = reset_status ? stat : nullptr;      // the first kernel clears the status block (not between async calls)
    if (!h_bins) h_bins = g.h_idx;
    uint64_t* signs = reinterpret_cast<uint64_t*>(g.ws + L.signs);
    int64_t* idx = reinterpret_cast<int64_t*>(g.ws + L.idx);
    double* Rs = reinterpret_cast<double*>(g.ws + L.Rs);
    // Algorithm 2 step 1: bins on the host (s values), sign words on the device (m bits)
    // ... or, for s <= 256 in front of the register radix-16 K1, not copied at all: they ride in the launch parameters
    const bool bins_inline = !seed_dev && k1_takes_host_bins(m, s, g.reim);
    if (!bins_inline) cudaMemcpyAsync(idx, h_bins, sizeof(int64_t) * (size_t)s, cudaMemcpyHostToDevice, st);
    const int64_t nw = (m + 63) / 64;
    // sign words: by the draw kernel, or (register radix-16 form of K1, seed known now) by K1 itself where it uses them
    const bool k1_draws = !seed_dev && k1_generates_signs(m, g.reim);
    int k = 0;
    if (seed_dev) { mrcqr_draw_signs_p<<<(unsigned)((nw + 255) / 256), 256, 0, st>>>(seed_dev, nw, signs, stat0); k = 1; }
    else if (!k1_draws) { mrcqr_draw_signs<<<(unsigned)((nw + 255) / 256), 256, 0, st>>>(seed, nw, signs, stat0); k = 1; }
    double* As = reinterpret_cast<double*>(g.ws + L.As);
    if (tm) cudaEventRecord(g.ev[0], st);
    k += launch_k1_srtt(m, n, lda, A, prec, s, signs, idx, g.ws + L.k1, As, stat, st, g.reim,
                        k1_draws ? &seed : nullptr, reset_status, bins_inline ? h_bins : nullptr);   // steps 2-4
    if (tm) cudaEventRecord(g.ev[1], st);
    k += launch_k2_sketch_qr(As, g.reim ? 2 * s : s, n, Rs, reinterpret_cast<double*>(g.ws + L.RsPrep), round_up(n, 16),
                             reinterpret_cast<double*>(g.ws + L.betas), stat, st);                              // steps 5-6
    if (tm) cudaEventRecord(g.ev[2], st);
    k += enqueue_stage23(L, m, n, lda, A, ldq, Q, R, Rs, st, tm);                              // steps 7-9
    return k;
}

static int factor_device(int64_t m, int n, int64_t lda, const double* A, int64_t ldq, double* Q, double* R,
                         int prec, int s, uint64_t seed, cudaStream_t st)
{
    Layout L = make_layout(m, n, s, prec);
    if (!ensure_ws(L.total) || !ensure_hidx((size_t)s)) return MRCQR_ERR_CUDA;
    draw_bins_host(m, s, seed, g.h_idx);
    const bool tm = g.timing && timing_events();
    if (g.use_graph && !tm) {
        if (!g.h_seed && cudaMallocHost(&g.h_seed, 64) != cudaSuccess) { cudaGetLastError(); g.h_seed = nullptr; }
        const bool same = g.gexec && g.gkey.m == m && g.gkey.lda == lda && g.gkey.n == n && g.gkey.prec == prec &&
                          g.gkey.s == s && g.gkey.A == A && g.gkey.Q == Q && g.gkey.R == R && g.gkey.ws == g.ws &&
                          g.gkey.hidx == g.h_idx && g.gkey.store_y == g.store_y && g.gkey.reim == g.reim;
        if (g.h_seed && !same) {
            drop_graph();
            uint64_t* seed_dev = reinterpret_cast<uint64_t*>(g.ws + L.status) + 2;        // Status::pad
            cudaGraph_t graph = nullptr;
            if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                cudaMemcpyAsync(seed_dev, g.h_seed, sizeof(uint64_t), cudaMemcpyHostToDevice, st);
                g.glaunches = enqueue_factor(L, m, n, lda, A, ldq, Q, R, prec, s, 0, seed_dev, st, false);
                cudaMemcpyAsync(g.h_status, g.ws + L.status, 8, cudaMemcpyDeviceToHost, st);
                if (cudaStreamEndCapture(st, &graph) != cudaSuccess || !graph ||
                    cudaGraphInstantiate(&g.gexec, graph, 0) != cudaSuccess) g.gexec = nullptr;
                if (graph) cudaGraphDestroy(graph);
            }
            cudaGetLastError();
            if (g.gexec) {
                g.gkey.m = m; g.gkey.lda = lda; g.gkey.n = n; g.gkey.prec = prec; g.gkey.s = s; g.gkey.A = A; g.gkey.Q = Q;
                g.gkey.R = R; g.gkey.ws = g.ws; g.gkey.hidx = g.h_idx; g.gkey.store_y = g.store_y; g.gkey.reim = g.reim;
            }
        }
        if (g.gexec) {
            *g.h_seed = seed;
            g.last_launches = g.glaunches;
            g.last_graph = true;
            cudaError_t le;
            { GateScope gate(st); le = cudaGraphLaunch(g.gexec, st); }
            if (le != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MRCQR_ERR_CUDA;
            g.last_info = g.h_status[1];
            return g.h_status[0];
        }
    }
    const int k = enqueue_factor(L, m, n, lda, A, ldq, Q, R, prec, s, seed, nullptr, st, tm);
    const int rc = finish(L, st, k);
    if (tm) for (int i = 0; i < 7; ++i) cudaEventElapsedTime(&g.stage_ms[i], g.ev[i], g.ev[i + 1]);
    return rc;
}

extern "C" int mrcqr_factor(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R,
                            mrcqr_prec_t sketch_prec, int s, uint64_t seed, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (!is_pow2(m) || m < n || m < 32) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!Q) return -5;
    if (!R) return -6;
    if (!prec_ok((int)sketch_prec)) return -7;
    if (s <= 0) s = 3 * n;
    if (s < n || (int64_t)s > m / 2 + 1 || s > S_MAX || (g.reim && 2 * s > S_MAX)) return -8;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    return factor_device(m, n, lda, A, lda, Q, R, (int)sketch_prec, s, seed, (cudaStream_t)stream);
}

// ---- calls in flight (repeated-call mode) ---------------------------------------------------------
// mrcqr_factor_async enqueues the same work as mrcqr_factor and returns; mrcqr_wait synchronises and reports.
static int wait_async(int* info_host)
{
    if (g.async_pending == 0) { if (info_host) *info_host = 0; return 0; }
    cudaStream_t st = g.async_stream;
    Status* stat = reinterpret_cast<Status*>(g.ws + g.async_status_off);
    cudaMemcpyAsync(g.h_status, stat, 8, cudaMemcpyDeviceToHost, st);
    mrcqr_reset_status<<<1, 1, 0, st>>>(stat);
    g.async_pending = 0;
    for (int i = 0; i < ASYNC_RING; ++i) g.ring_busy[i] = false;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MRCQR_ERR_CUDA;
    g.last_info = g.h_status[1];
    if (info_host) *info_host = g.h_status[1];
    return g.h_status[0];
}

extern "C" int mrcqr_wait(int* info_host) { return device_ok() ? wait_async(info_host) : MRCQR_ERR_CUDA; }

extern "C" int mrcqr_factor_async(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R,
                                  mrcqr_prec_t sketch_prec, int s, uint64_t seed, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (!is_pow2(m) || m < n || m < 32) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!Q) return -5;
    if (!R) return -6;
    if (!prec_ok((int)sketch_prec)) return -7;
    if (s <= 0) s = 3 * n;
    if (s < n || (int64_t)s > m / 2 + 1 || s > S_MAX || (g.reim && 2 * s > S_MAX)) return -8;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    Layout L = make_layout(m, n, s, (int)sketch_prec);
    // The calls in flight share the context's workspace, ordered by their stream: another stream, or a workspace that
    // has to grow (or whose status block would move), first drains what is pending (its status is kept: see below).
    int carried = 0, carried_info = 0;
    if (g.async_pending > 0 && (st != g.async_stream || L.total > g.ws_bytes || L.status != g.async_status_off)) {
        carried = wait_async(&carried_info);
        if (carried == MRCQR_ERR_CUDA) return carried;
    }
    g.in_async = true;
    const bool ws_ok = ensure_ws(L.total);
    g.in_async = false;
    if (!ws_ok) return MRCQR_ERR_CUDA;
    if ((size_t)s > g.h_ring_cap) {                              // (re)allocate the ring: nothing is in flight on a smaller one
        if (g.async_pending > 0) { const int c = wait_async(&carried_info); if (c == MRCQR_ERR_CUDA) return c; if (!carried) carried = c; }
        if (g.h_ring) cudaFreeHost(g.h_ring);
        g.h_ring = nullptr; g.h_ring_cap = 0;
        const size_t cap = std::max<size_t>((size_t)s, 256);
        if (cudaMallocHost(&g.h_ring, sizeof(int64_t) * cap * ASYNC_RING) != cudaSuccess) { cudaGetLastError(); g.h_ring = nullptr; return MRCQR_ERR_CUDA; }
        g.h_ring_cap = cap;
    }
    const int slot = g.ring_pos;
    g.ring_pos = (g.ring_pos + 1) % ASYNC_RING;
    if (!g.ring_ev[slot] && cudaEventCreateWithFlags(&g.ring_ev[slot], cudaEventDisableTiming) != cudaSuccess) return MRCQR_ERR_CUDA;
    if (g.ring_busy[slot] && cudaEventSynchronize(g.ring_ev[slot]) != cudaSuccess) return MRCQR_ERR_CUDA;   // its copy has run
    int64_t* bins = g.h_ring + (size_t)slot * g.h_ring_cap;
    draw_bins_host(m, s, seed, bins);
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    if (g.async_pending == 0) {
        mrcqr_reset_status<<<1, 1, 0, st>>>(stat);
        if (carried) {                                           // an error of the drained calls is not lost
            g.h_status[4] = carried; g.h_status[5] = carried_info;      // pinned; rewritten only after another drain (a sync)
            cudaMemcpyAsync(stat, g.h_status + 4, 8, cudaMemcpyHostToDevice, st);
        }
    }
    const int k = enqueue_factor(L, m, n, lda, A, lda, Q, R, (int)sketch_prec, s, seed, nullptr, st, false, bins, false);
    // the bins are on the device once the first kernels have run; the slot is free from this event on
    cudaEventRecord(g.ring_ev[slot], st);
    g.ring_busy[slot] = true;
    g.async_stream = st; g.async_status_off = L.status; ++g.async_pending;
    g.last_launches = k; g.last_graph = false;
    return cudaGetLastError() == cudaSuccess ? 0 : MRCQR_ERR_CUDA;
}

// ||I - Q^T Q||_F on the device: DMMA SYRK of Q (deterministic row split, chains flushed every 1024 rows) + norm
static int orth_error_device(int64_t m, int n, int64_t ldq, const double* Q, double* err_host, cudaStream_t st)
{
    Layout L = make_layout(m, n, 0, 64);
    if (!ensure_ws(L.total)) return MRCQR_ERR_CUDA;
    const int n16 = round_up(n, 16);
    double* G16 = reinterpret_cast<double*>(g.ws + L.G16);
    double* part = reinterpret_cast<double*>(g.ws + L.k3);
    double* err = reinterpret_cast<double*>(g.ws + L.betas);          // n doubles of scratch: [0] receives the norm
    mrcqr_reset_status<<<1, 1, 0, st>>>(reinterpret_cast<Status*>(g.ws + L.status));
    int k = 1 + launch_syrk(m, n, ldq, Q, part, n16, G16, st);
    k += launch_orth_norm(G16, n, n16, err, st);
    cudaMemcpyAsync(g.h_status + 2, err, sizeof(double), cudaMemcpyDeviceToHost, st);
    const int rc = finish(L, st, k);
    if (rc == 0) std::memcpy(err_host, g.h_status + 2, sizeof(double));
    return rc;
}

extern "C" int mrcqr_orth_error(int64_t m, int n, int64_t ldq, const double* Q, double* err_host, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (m < n) return -1;
    if (ldq < m) return -3;
    if (!Q) return -4;
    if (!err_host) return -5;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    return orth_error_device(m, n, ldq, Q, err_host, (cudaStream_t)stream);
}

extern "C" int mrcqr_factor_auto(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R,
                                 mrcqr_prec_t first_prec, int s, uint64_t seed, double tol,
                                 int* prec_used_host, double* orth_host, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (!is_pow2(m) || m < n || m < 32) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!Q) return -5;
    if (!R) return -6;
    if (!prec_ok((int)first_prec)) return -7;
    if (s <= 0) s = 3 * n;
    if (s < n || (int64_t)s > m / 2 + 1 || s > S_MAX || (g.reim && 2 * s > S_MAX)) return -8;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    if (!(tol > 0.0)) tol = 1e-13;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = 0;
    for (int p = (int)first_prec; p <= 64; p *= 2) {         // half -> single -> double
        rc = factor_device(m, n, lda, A, lda, Q, R, p, s, seed, st);
        if (rc < 0 || rc == MRCQR_ERR_CUDA) return rc;
        double orth = -1.0;
        if (rc == 0) {
            const int rc2 = orth_error_device(m, n, lda, Q, &orth, st);
            if (rc2 != 0) return rc2;
        }
        if (prec_used_host) *prec_used_host = p;
        if (orth_host) *orth_host = orth;
        if (rc == 0 && orth <= tol) return 0;                 // NaN fails the comparison: escalates
        if (rc == 0) rc = MRCQR_ERR_NOT_ORTHOGONAL;
    }
    return rc;                                               // the outcome at the highest precision
}

__global__ void mrcqr_set_identity(double* __restrict__ M, int n)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n * n) M[e] = (e % n == e / n) ? 1.0 : 0.0;
}

// Algorithm 1 on A itself: the stage-2/3 kernels with R_s = I
static int cholqr_device(int64_t m, int n, int64_t lda, const double* A, int64_t ldq, double* Q, double* R, cudaStream_t st)
{
    Layout L = make_layout(m, n, 0, 64);
    if (!ensure_ws(L.total)) return MRCQR_ERR_CUDA;
    Status* stat = reinterpret_cast<Status*>(g.ws + L.status);
    double* Rs = reinterpret_cast<double*>(g.ws + L.Rs);
    mrcqr_reset_status<<<1, 1, 0, st>>>(stat);
    mrcqr_set_identity<<<(n * n + 255) / 256, 256, 0, st>>>(Rs, n);
    int k = 2 + launch_prep_R(Rs, n, reinterpret_cast<double*>(g.ws + L.RsPrep), round_up(n, 16), stat, MRCQR_ERR_SINGULAR, st);
    k += enqueue_stage23(L, m, n, lda, A, ldq, Q, R, Rs, st, false);
    return finish(L, st, k);
}

extern "C" int mrcqr_cholqr(int64_t m, int n, int64_t lda, const double* A, double* Q, double* R, int passes, void* stream)
{
    if (n < 1 || n > N_MAX) return -2;
    if (m < n) return -1;
    if (lda < m) return -3;
    if (!A) return -4;
    if (!Q) return -5;
    if (!R) return -6;
    if (passes != 1 && passes != 2) return -7;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = cholqr_device(m, n, lda, A, lda, Q, R, st);
    if (rc != 0 || passes == 1) return rc;
    // CholQR2: Algorithm 1 again on Q (in place), R = R2 R1; R1, R2 live in the workspace
    Layout L = make_layout(m, n, 0, 64);
    double* R1 = reinterpret_cast<double*>(g.ws + L.Rtmp);
    double* R2 = R1 + (size_t)n * n;
    cudaMemcpyAsync(R1, R, sizeof(double) * (size_t)n * n, cudaMemcpyDeviceToDevice, st);
    rc = cholqr_device(m, n, lda, Q, lda, Q, R2, st);
    if (rc == 0) {
        launch_triu_mul(R2, R1, n, R, st);
        if (cudaStreamSynchronize(st) != cudaSuccess) rc = MRCQR_ERR_CUDA;
    }
    return rc;
}

extern "C" int mrcqr_kappa_probe(int64_t m, int n, int64_t lda, const double* A, double* Qwork, double* Rwork,
                                 double* kappa_lb_host, int* prec_host, void* stream)
{
    if (!kappa_lb_host) return -7;
    int rc = mrcqr_cholqr(m, n, lda, A, Qwork, Rwork, 1, stream);
    if (rc < 0 || rc == MRCQR_ERR_CUDA) return rc;
    const double u = 1.1102230246251565e-16;                   // 2^-53
    double lb = 1.0 / sqrt(u);                                 // CholQR broke down: kappa^2 u >~ 1
    if (rc == 0) {
        double qf = 0.0;
        rc = mrcqr_orth_error(m, n, lda, Qwork, &qf, stream);
        if (rc != 0) return rc;
        const double q = qf / sqrt((double)n);                 // ||.||_2 >= ||.||_F / sqrt(n): keeps eq. (2) a LOWER bound
        lb = sqrt(q / (u * (1.0 + q)));
    }
    *kappa_lb_host = lb;
    if (prec_host) *prec_host = lb < 1e4 ? 16 : (lb < 1e8 ? 32 : 64);
    return 0;
}

// Algorithm 2 for `batch` independent problems of one shape (the repeated-call regime).
extern "C" int mrcqr_factor_batched(int batch, int64_t m, int n, int64_t lda, int64_t strideA, const double* A,
                                    int64_t strideQ, double* Q, double* R, mrcqr_prec_t sketch_prec, int s,
                                    uint64_t seed, int* codes_host, void* stream)
{
    if (batch < 1) return -1;
    if (!is_pow2(m) || m < n || m < 32) return -2;
    if (n < 1 || n > N_MAX) return -3;
    if (lda < m) return -4;
    if (batch > 1 && strideA < (int64_t)(n - 1) * lda + m) return -5;
    if (!A) return -6;
    if (batch > 1 && strideQ < (int64_t)(n - 1) * lda + m) return -7;
    if (!Q) return -8;
    if (!R) return -9;
    if (!prec_ok((int)sketch_prec)) return -10;
    if (s <= 0) s = 3 * n;
    if (s < n || (int64_t)s > m / 2 + 1 || s > S_MAX || (g.reim && 2 * s > S_MAX)) return -11;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    int first = 0;
    if (!g.reim && batched_fused_usable(m, n, s)) {
        if ((size_t)batch > g.bcodes_cap) {
            if (g.bcodes) cudaFree(g.bcodes);
            if (g.h_bcodes) cudaFreeHost(g.h_bcodes);
            g.bcodes = g.h_bcodes = nullptr; g.bcodes_cap = 0;
            if (cudaMalloc(&g.bcodes, sizeof(int) * 2 * (size_t)batch) != cudaSuccess ||
                cudaMallocHost(&g.h_bcodes, sizeof(int) * 2 * (size_t)batch) != cudaSuccess) { cudaGetLastError(); return MRCQR_ERR_CUDA; }
            g.bcodes_cap = (size_t)batch;
        }
        const int k = launch_factor_batched(batch, m, n, lda, strideA, A, lda, strideQ, Q, R, (int)sketch_prec, s, seed, g.bcodes, st);
        g.last_launches = k; g.last_graph = false;
        cudaMemcpyAsync(g.h_bcodes, g.bcodes, sizeof(int) * 2 * (size_t)batch, cudaMemcpyDeviceToHost, st);
        if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MRCQR_ERR_CUDA;
        for (int b = 0; b < batch; ++b) {
            if (codes_host) codes_host[b] = g.h_bcodes[2 * b];
            if (!first && g.h_bcodes[2 * b]) { first = g.h_bcodes[2 * b]; g.last_info = g.h_bcodes[2 * b + 1]; }
        }
        return first;
    }
    // shapes beyond one CTA's reach: the problems are large enough for the ordinary path, one after the other
    int launches = 0, info = 0;
    for (int b = 0; b < batch; ++b) {
        const int rc = factor_device(m, n, lda, A + (size_t)b * (size_t)strideA, lda, Q + (size_t)b * (size_t)strideQ,
                                     R + (size_t)b * (size_t)n * n, (int)sketch_prec, s, seed + (uint64_t)b, st);
        if (rc < 0 || rc == MRCQR_ERR_CUDA) return rc;
        launches += g.last_launches;
        if (codes_host) codes_host[b] = rc;
        if (!first && rc) { first = rc; info = g.last_info; }
    }
    g.last_launches = launches;
    if (first) g.last_info = info;
    return first;
}

extern "C" int mrcqr_factor_host(int64_t m, int n, int64_t lda, const double* A_host, double* Q_host,
                                 double* R_host, mrcqr_prec_t sketch_prec, int s, uint64_t seed)
{
    if (n < 1 || n > N_MAX) return -2;
    if (!is_pow2(m) || m < n || m < 32) return -1;
    if (lda < m) return -3;
    if (!A_host) return -4;
    if (!Q_host) return -5;
    if (!R_host) return -6;
    if (!prec_ok((int)sketch_prec)) return -7;
    if (s <= 0) s = 3 * n;
    if (s < n || (int64_t)s > m / 2 + 1 || s > S_MAX || (g.reim && 2 * s > S_MAX)) return -8;
    if (!device_ok()) return MRCQR_ERR_CUDA;
    // device copies are packed (ld = m): only the m x n part of a host matrix with lda > m is touched
    const size_t bytes = sizeof(double) * (size_t)m * n, rbytes = sizeof(double) * (size_t)n * n;
    if (bytes > g.hA_bytes) {
        if (g.hA) cudaFree(g.hA);
        if (g.hQ) cudaFree(g.hQ);
        g.hA = g.hQ = nullptr; g.hA_bytes = 0;
        if (cudaMalloc(&g.hA, bytes) != cudaSuccess || cudaMalloc(&g.hQ, bytes) != cudaSuccess) { cudaGetLastError(); return MRCQR_ERR_CUDA; }
        g.hA_bytes = bytes;
    }
    if (rbytes > g.hR_bytes) {
        if (g.hR) cudaFree(g.hR);
        g.hR = nullptr; g.hR_bytes = 0;
        if (cudaMalloc(&g.hR, rbytes) != cudaSuccess) { cudaGetLastError(); return MRCQR_ERR_CUDA; }
        g.hR_bytes = rbytes;
    }
    if (!g.host_stream && cudaStreamCreateWithFlags(&g.host_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); g.host_stream = nullptr; return MRCQR_ERR_CUDA;
    }
    cudaStream_t st = g.host_stream;
    const size_t row = sizeof(double) * (size_t)m, hpitch = sizeof(double) * (size_t)lda;
    if (cudaMemcpy2DAsync(g.hA, row, A_host, hpitch, row, (size_t)n, cudaMemcpyHostToDevice, st) != cudaSuccess) return MRCQR_ERR_CUDA;
    int rc = factor_device(m, n, m, g.hA, m, g.hQ, g.hR, (int)sketch_prec, s, seed, st);
    if (rc != 0) return rc;
    cudaMemcpy2DAsync(Q_host, hpitch, g.hQ, row, row, (size_t)n, cudaMemcpyDeviceToHost, st);
    cudaMemcpyAsync(R_host, g.hR, rbytes, cudaMemcpyDeviceToHost, st);
    if (cudaStreamSynchronize(st) != cudaSuccess) return MRCQR_ERR_CUDA;
    return 0;
}
