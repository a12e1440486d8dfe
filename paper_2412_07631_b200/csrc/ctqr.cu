// ctqr.cu -- C-ABI (include/ctqr.h) and the host-side drivers of the hot path:
//   a4 in-core blocked Householder QR with look-ahead, a6 batched Q^T B, a7 blocked TRSM
//   (Eq. 2-3; TRSM task list L62-73).
// and a5, the out-of-core scheduler (factor_ooc, streamed solve, optional file tier).
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <stdarg.h>
#include <stdlib.h>
#include <errno.h>
#include <fcntl.h>
#include <sys/mman.h>
#include <sys/stat.h>
#include <unistd.h>
#include <string.h>
#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <thread>
#include <unordered_map>
#include <vector>

#include "../../include/ctqr.h"
#include "common.cuh"
#include "kernels.h"
#include "solve_small.cuh"
#include "solve_small2.cuh"
#include "solve_mid.cuh"

using namespace ctqr;

template <typename T> static GemmLaunch gemm_plan(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems, int64_t sstride, bool aligned);
template <> GemmLaunch gemm_plan<double>(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems, int64_t sstride, bool aligned) { return gemm_plan_f64(ta, M, N, K, impl, sms, partial, max_elems, sstride, aligned); }
template <> GemmLaunch gemm_plan<float>(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems, int64_t sstride, bool aligned) { return gemm_plan_f32(ta, M, N, K, impl, sms, partial, max_elems, sstride, aligned); }
template <typename T> static bool gemm_aligned(const GemmArgs<T>& g) {
    return ((uintptr_t)g.A % 16 == 0) && ((uintptr_t)g.B % 16 == 0) && ((g.lda * (int64_t)sizeof(T)) % 16 == 0) &&
           ((g.ldb * (int64_t)sizeof(T)) % 16 == 0);
}
template <typename T> static cudaError_t gemm_run(bool ta, const GemmArgs<T>& g, const GemmLaunch& L, int impl, cudaStream_t st);
template <> cudaError_t gemm_run<double>(bool ta, const GemmArgs<double>& g, const GemmLaunch& L, int impl, cudaStream_t st) { return gemm_run_f64(ta, g, L, impl, st); }
template <> cudaError_t gemm_run<float>(bool ta, const GemmArgs<float>& g, const GemmLaunch& L, int impl, cudaStream_t st) { return gemm_run_f32(ta, g, L, impl, st); }
// direct product C <- alpha op(A) B + beta C
template <typename T> static cudaError_t gemm_direct(bool ta, const GemmArgs<T>& g, int impl, int sms, cudaStream_t st) {
    return gemm_run<T>(ta, g, gemm_plan<T>(ta, g.M, g.N, g.K, impl, sms, false, 0, 0, gemm_aligned(g)), impl, st);
}
static cudaError_t panel_launch(int ib, int rpt, PanelArgs<double>& pa, int G, cudaStream_t st) { return panel_launch_f64(ib, rpt, pa, G, st); }
static cudaError_t panel_launch(int ib, int rpt, PanelArgs<float>& pa, int G, cudaStream_t st) { return panel_launch_f32(ib, rpt, pa, G, st); }

// ------------------------------------------------------------------------------------------
// error plumbing
// ------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";
static int set_err(int code, const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
    return code;
}
#define CK(call)                                                                                  \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return set_err(CTQR_ERR_CUDA, "%s failed at %s:%d: %s", #call, __FILE__, __LINE__,     \
                           cudaGetErrorString(e_));                                               \
    } while (0)
#define CKI(call) do { int r_ = (call); if (r_ != 0) return r_; } while (0)

extern "C" const char* ct_qr_last_error(void) { return g_err; }
// error plumbing for the library's other translation units (refine.cu); not part of the ABI
extern "C" __attribute__((visibility("hidden"))) int ctqr_internal_set_error(int code, const char* what, const char* detail) {
    return set_err(code, "%s%s%s", what, (detail && detail[0]) ? ": " : "", detail ? detail : "");
}
extern "C" const char* ct_qr_strerror(int code) {
    if (code < 0) return "invalid argument (the -code-th argument)";
    switch (code) {
        case CTQR_OK: return "success";
        case CTQR_ERR_CUDA: return "CUDA runtime failure or no device";
        case CTQR_ERR_NOMEM: return "out of memory / device budget too small";
        case CTQR_ERR_IO: return "file tier I/O failure";
        case CTQR_ERR_SINGULAR: return "R has a zero on its diagonal";
        case CTQR_ERR_STATE: return "handle state does not allow this call";
        default: return "unknown error";
    }
}
extern "C" int ct_qr_version(void) { return 100; }

// ------------------------------------------------------------------------------------------
// Process-wide cache of the small per-handle device buffers (T, tau, workspaces, LL slots, the solve
// staging buffer; not the matrix storage, not the super-panel buffers).  cudaMalloc / cudaFree cost
// 0.1 - 100 ms each and cudaFree synchronises the device; a service that factors or reloads one
// geometry after another would pay that for ~20 buffers per handle.  Blocks of
// at most kCacheMaxBlock bytes go back to a size-ordered free list (at most kCacheMaxTotal bytes are
// kept) and are handed out again to the next request of up to half their size; contents are
// unspecified, as after cudaMalloc.  Callers free only buffers no kernel is using (handles are
// destroyed after a device synchronise, workspaces are replaced between synchronous calls).
// ------------------------------------------------------------------------------------------
namespace {
constexpr size_t kCacheMaxBlock = (size_t)256 << 20, kCacheMaxTotal = (size_t)1 << 30;
struct DevCache {
    std::mutex mu;
    std::multimap<uint64_t, void*> free_;          // key = device << 32 | bytes  (bytes <= 256 MiB)
    std::unordered_map<void*, uint64_t> key_;      // every block this cache may take back
    size_t cached = 0;
} g_cache;
}
static cudaError_t dev_alloc_raw(void** p, size_t bytes) {
    cudaError_t e = cudaMalloc(p, bytes);
    if (e == cudaSuccess) return e;
    cudaGetLastError();
    std::vector<void*> drop;                        // out of memory: give the cached blocks back and retry once
    {
        std::lock_guard<std::mutex> lk(g_cache.mu);
        for (auto& kv : g_cache.free_) { drop.push_back(kv.second); g_cache.key_.erase(kv.second); }
        g_cache.free_.clear(); g_cache.cached = 0;
    }
    if (drop.empty()) return e;
    for (void* q : drop) cudaFree(q);
    return cudaMalloc(p, bytes);
}
template <typename P>
static cudaError_t dev_alloc(P** p, size_t bytes) {
    void* q = nullptr;
    int dev = 0; cudaGetDevice(&dev);
    if (bytes > 0 && bytes <= kCacheMaxBlock) {
        std::lock_guard<std::mutex> lk(g_cache.mu);
        auto it = g_cache.free_.lower_bound(((uint64_t)dev << 32) | bytes);
        if (it != g_cache.free_.end() && (it->first >> 32) == (uint64_t)dev && (it->first & 0xffffffffu) <= 2 * bytes + 4096) {
            q = it->second; g_cache.cached -= (size_t)(it->first & 0xffffffffu); g_cache.free_.erase(it);
            *p = (P*)q;
            return cudaSuccess;
        }
    }
    cudaError_t e = dev_alloc_raw(&q, bytes);
    if (e != cudaSuccess) return e;
    if (q && bytes <= kCacheMaxBlock) {
        std::lock_guard<std::mutex> lk(g_cache.mu);
        g_cache.key_[q] = ((uint64_t)dev << 32) | bytes;
    }
    *p = (P*)q;
    return cudaSuccess;
}
static void dev_free(void* p) {
    if (!p) return;
    {
        std::lock_guard<std::mutex> lk(g_cache.mu);
        auto it = g_cache.key_.find(p);
        if (it != g_cache.key_.end()) {
            const size_t bytes = (size_t)(it->second & 0xffffffffu);
            if (g_cache.cached + bytes <= kCacheMaxTotal) {
                g_cache.free_.emplace(it->second, p); g_cache.cached += bytes;
                return;
            }
            g_cache.key_.erase(it);
        }
    }
    cudaFree(p);
}

extern "C" int64_t ct_qr_trim_cache(void) {
    std::vector<void*> drop;
    size_t bytes = 0;
    {
        std::lock_guard<std::mutex> lk(g_cache.mu);
        for (auto& kv : g_cache.free_) { drop.push_back(kv.second); g_cache.key_.erase(kv.second); }
        bytes = g_cache.cached;
        g_cache.free_.clear(); g_cache.cached = 0;
    }
    for (void* q : drop) cudaFree(q);
    return (int64_t)bytes;
}
// large allocations (matrix storage, super-panel buffers, accessor temporaries): plain cudaMalloc that gives the
// cached small blocks back and retries once before reporting out-of-memory
static cudaError_t big_alloc(void** p, size_t bytes) { return dev_alloc_raw(p, bytes); }
// free device memory as a budget: what cudaMemGetInfo reports plus what the cache could give back
static size_t free_device_bytes() {
    size_t freeb = 0, totb = 0;
    if (cudaMemGetInfo(&freeb, &totb) != cudaSuccess) { cudaGetLastError(); return 0; }
    std::lock_guard<std::mutex> lk(g_cache.mu);
    return freeb + g_cache.cached;
}

// ------------------------------------------------------------------------------------------
// handle
// ------------------------------------------------------------------------------------------
struct ctqr_handle_s {
    ctqr_dtype_t dtype = CTQR_F64;
    size_t w = 8;
    int64_t m = 0, n = 0, lda = 0;     // lda: leading dimension of dA
    int nb = 128, ib = 16, P = 0, lookahead = 1, gemm_impl = 0;
    int sms = 148;
    void* dA = nullptr; bool own_A = false;   // factored matrix (device, in-core path)
    void* dT = nullptr;                // P blocks of nb x nb (ld nb)
    void* dRd = nullptr;               // P blocks of nb x nb (ld nb): diagonal blocks of R
    void* dRinv = nullptr;             // their inverses (nb == 128 only), filled at the first solve
    bool rinv_ready = false;
    void* dNm = nullptr; bool nm_ready = false; void* dLLt = nullptr;   // N_i = R_ii^{-1} R_{i,i+1} and the LL slots of the pipelined small-S TRSM
    void* dGt = nullptr; bool gt_ready = false;   // Mt[j] = T_(j-1) (V_(j-1)^T V_j) of the pipelined small-S Q^T B (fp64), built at first use
    void* dTau = nullptr;              // n
    // workspaces: [0] update stream, [1] panel stream
    void* dWp[2] = {nullptr, nullptr}; size_t wp_elems[2] = {0, 0};
    void* dW[2] = {nullptr, nullptr};  size_t w_elems[2] = {0, 0};
    // two-panel (256-wide) trailing updates: W / T^T W (256 x nc each), two merged T factors, merge scratch
    void* dW2[2] = {nullptr, nullptr}; size_t w2_elems = 0; void* dT2 = nullptr; void* dMerge = nullptr;
    // fp32 only: TF32 hi / lo split of the pair's reflector block (rows below the first diagonal block; one [hi | lo]
    // buffer per T2 slot, leading dimension ldvs) and of T2^T W, for the TMA-fed tcgen05 update (gemm_umma_tma.cuh)
    void* dVs[2] = {nullptr, nullptr}; int64_t ldvs = 0; void* dWs = nullptr; size_t ws_elems = 0;
    void* dCw = nullptr; size_t cw_bytes = 0;   // staging buffer of the solves (B in, X out), grow-only: no allocation per batch
    void* dPart = nullptr;             // LL slots of the panel kernel
    int solve_pairs = 0;                             // option: 0 by size, 1 from 256 right-hand sides on, -1 never
    void* dT12 = nullptr;                            // off-diagonal blocks -T_k (V_k^T V_k+1) T_k+1 of the merged T factors of the pairs
    std::vector<unsigned char> t12_have;             // (2i, 2i+1), kept from the factorisation's merges for the large-batch Q^T B
    void* dLLm = nullptr;                        // LL slots of the medium-S Q^T B kernel (solve_mid.cuh), built at first use
    void* dLLs = nullptr; unsigned ll_seq = 0;   // LL slots / step numbers of the fused small-S solve kernels
    unsigned bar_count = 0;            // step numbers handed to the panel kernel (never reused)
    int* dFlag = nullptr;
    cudaStream_t sU = nullptr, sP = nullptr, sC = nullptr, sD = nullptr, user = nullptr;
    cudaEvent_t evP = nullptr, evL = nullptr, evU = nullptr;
    cudaEvent_t evS[3] = {nullptr, nullptr, nullptr};   // timing events of the solve calls, created once per handle
    std::vector<cudaEvent_t> ev;       // event pool
    ctqr_stats_t st;
    int64_t launches = 0;
    // opt->profile: per-launch event spans of the trailing-update contractions
    struct Span { cudaEvent_t a, b; double flops; int kind; };
    int profile = 0;
    void* dTickets = nullptr; int ticket_pos = 0;   // zeroed counter pairs for the SM-confined fp64 launches (kTicketRing of them)
    int trsm_exact = 0;    // 1: opt->trsm_exact; 2: forced by the conditioning guard of the diagonal blocks
    int reserve_sms = -1;  // SMs left to the look-ahead panel chain during the bulk update (fp32 tcgen05 path): -1 auto, 0 off
    std::vector<Span> spans;
    // out of core: [a, b] brackets on the compute stream around every wait for a copy (exposed copy time) and on the
    // copy streams around every copy (busy time)
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> wait_spans, copy_spans;
    std::vector<cudaEvent_t> tpool; size_t tpool_used = 0;
    cudaEvent_t timing_event() {
        if (tpool_used == tpool.size()) { cudaEvent_t e; cudaEventCreate(&e); tpool.push_back(e); }
        return tpool[tpool_used++];
    }
    // host matrix staged in core: column chunks arriving on the copy stream while the first panels are already factored;
    // (one past the last column of the chunk, event recorded after its copy); emptied once every event has been waited for
    std::vector<std::pair<int64_t, cudaEvent_t>> arrive;
    bool factored = false;
    // opt->lower_bandwidth: A(i, j) == 0 for i - j > kl, so the reflectors of the
    // columns [.., jend) end at row min(m, kl + jend) and every product over rows stops there
    int64_t kl = 0;
    // out-of-core state
    bool ooc = false; void* hA = nullptr; int64_t hlda = 0; int n_super = 1;
    // file-backed tier: the matrix / factor lives in a file mapped MAP_SHARED (the OS page cache is the
    // host-RAM block cache over the disk of PAPER.md L58)
    void* fmap = nullptr; size_t fmap_len = 0; int ffd = -1;
    void* spbuf[2] = {nullptr, nullptr};   // super-panel buffers, alive only during factor_ooc
    void* dVb[2] = {nullptr, nullptr}; int64_t ldvb = 0;   // double buffer for streamed panels (m x nb each)
    void* dVp[2] = {nullptr, nullptr};                    // double buffer for streamed panel PAIRS (m x 256 each; out-of-core
                                                          // left-looking updates, workspace outside the tile budget)
    cudaEvent_t evVin[2] = {nullptr, nullptr}, evVfree[2] = {nullptr, nullptr};
    ~ctqr_handle_s() {
        if (own_A && dA) cudaFree(dA);
        if (fmap) { msync(fmap, fmap_len, MS_SYNC); munmap(fmap, fmap_len); }
        if (ffd >= 0) close(ffd);
        dev_free(dT); dev_free(dRd); dev_free(dRinv); dev_free(dTau); dev_free(dGt); dev_free(dNm); dev_free(dLLt);
        for (int i = 0; i < 2; ++i) { dev_free(dWp[i]); dev_free(dW[i]); dev_free(dW2[i]); }
        dev_free(dT2); dev_free(dMerge); dev_free(dCw); dev_free(dWs);
        for (int i = 0; i < 2; ++i) if (dVs[i]) cudaFree(dVs[i]);
        dev_free(dPart); dev_free(dLLs); dev_free(dLLm); dev_free(dT12); dev_free(dFlag); dev_free(dTickets);
        for (int i = 0; i < 2; ++i) cudaFree(spbuf[i]);
        for (auto e : ev) cudaEventDestroy(e);
        for (auto e : tpool) cudaEventDestroy(e);
        if (sU) cudaStreamDestroy(sU);
        if (sP) cudaStreamDestroy(sP);
        if (sC) cudaStreamDestroy(sC);
        if (sD) cudaStreamDestroy(sD);
        for (int i = 0; i < 2; ++i) dev_free(dVb[i]);
        for (int i = 0; i < 2; ++i) if (dVp[i]) cudaFree(dVp[i]);
    }
};
typedef ctqr_handle_s H;

template <typename T> static inline T* P_(void* p) { return reinterpret_cast<T*>(p); }

// one past the last row that the reflectors of the columns [.., jend) can touch
static inline int64_t row_end(const H& h, int64_t jend) { return h.kl > 0 ? std::min(h.m, h.kl + jend) : h.m; }

static bool is_device_ptr(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// ------------------------------------------------------------------------------------------
// larfb: C <- (I - V T^T V^T) C   (with C = B it is row a6)
//   V: mk x kw explicit unit-lower-trapezoid (ld ldv), T: kw x kw upper (ld ldt), C: mk x nc.
// ------------------------------------------------------------------------------------------
// SM confinement of a stream-K launch (fp64: two CTAs per SM, so a smaller grid alone leaves no SM empty; see
// GemmLaunch::reserve).  Hands the launch a fresh pair of zeroed counters; the ring is re-zeroed on the
// launching stream when it wraps (all users are on that stream).
constexpr int kTicketRing = 4096;
template <typename T>
static int confine(H& h, GemmLaunch& L, int reserve_sms, cudaStream_t st) {
    if (sizeof(T) != 8 || reserve_sms <= 0 || L.kind != 1 || !h.dTickets) return 0;
    if (h.ticket_pos == kTicketRing) {
        CK(cudaMemsetAsync(h.dTickets, 0, (size_t)kTicketRing * 2 * sizeof(unsigned), st));
        h.ticket_pos = 0;
    }
    L.reserve = reserve_sms;
    L.tickets = reinterpret_cast<unsigned*>(h.dTickets) + 2 * (size_t)h.ticket_pos++;
    return 0;
}
template <typename T>
static int gemm_direct_confined(H& h, bool ta, const GemmArgs<T>& g, int sms, int reserve_sms, cudaStream_t st) {
    GemmLaunch L = gemm_plan<T>(ta, g.M, g.N, g.K, h.gemm_impl, sms, false, 0, 0, gemm_aligned(g));
    CKI(confine<T>(h, L, reserve_sms, st));
    CK(gemm_run<T>(ta, g, L, h.gemm_impl, st));
    return 0;
}

template <typename T>
static int larfb(H& h, int ws, cudaStream_t st, const T* V, int64_t ldv, int64_t mk, int kw, const T* Tm, int ldt,
                 T* C, int64_t ldc, int64_t nc, bool prof = false, int reserve_sms = 0) {
    if (nc <= 0 || mk <= 0 || kw <= 0) return 0;
    // reserve_sms: leave that many SMs to the look-ahead panel chain running on the other stream (only
    // meaningful for one-CTA-per-SM kernels: a smaller persistent grid then leaves whole SMs empty)
    const int sms = std::max(8, h.sms - reserve_sms);
    const int64_t ldw = round_up(kw, 4);
    // W = V^T C as partial products over K (stream-K or split grid), summed by the T^T W kernel
    const int64_t sstride = ldw * nc;
    if ((size_t)sstride > h.wp_elems[ws] || (size_t)sstride > h.w_elems[ws])
        return set_err(CTQR_ERR_NOMEM, "larfb workspace too small (kw=%d nc=%lld)", kw, (long long)nc);
    T* Wp = P_<T>(h.dWp[ws]);
    T* W = P_<T>(h.dW[ws]);
    GemmArgs<T> g1{};
    g1.M = kw; g1.N = nc; g1.K = mk; g1.A = V; g1.lda = ldv; g1.B = C; g1.ldb = ldc;
    g1.C = Wp; g1.ldc = ldw; g1.alpha = T(1); g1.beta = T(0); g1.split_stride = sstride;
    GemmLaunch L1 = gemm_plan<T>(true, kw, nc, mk, h.gemm_impl, sms, true,
                                 (int64_t)h.wp_elems[ws], sstride, gemm_aligned(g1));
    CKI(confine<T>(h, L1, reserve_sms, st));
    prof = prof && h.profile;
    const double fl = 2.0 * (double)mk * (double)kw * (double)nc;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (prof) { e0 = h.timing_event(); e1 = h.timing_event(); CK(cudaEventRecord(e0, st)); }
    CK(gemm_run<T>(true, g1, L1, h.gemm_impl, st));
    if (prof) { CK(cudaEventRecord(e1, st)); h.spans.push_back({e0, e1, fl, 0}); }
    const T* W2 = W;
    if (L1.kind == 1 && kw == 128 && nc <= 512 && L1.seg.BN % 8 == 0 && ldt % (16 / (int)sizeof(T)) == 0 &&
        (uintptr_t)Tm % 16 == 0) {
        // narrow right-hand side (the solve, the look-ahead block): partial sum and T^T W in one small kernel
        CK(mm128_launch<T>(true, Tm, ldt, Wp, 0, L1.seg, nc, W, ldw, st));
    } else if (L1.kind == 1 && kw == 128 && nc >= 128 && ldt % (16 / (int)sizeof(T)) == 0 && (uintptr_t)Tm % 16 == 0) {
        // full-width panel: W <- sum of the partial tiles, then T^T W as one more tensor-core
        // contraction (T is stored with explicit zeros below the diagonal), written over the partials
        CK(partial_sum_launch<T>(Wp, L1.seg, kw, nc, W, ldw, st));
        GemmArgs<T> gt{};
        gt.M = kw; gt.N = nc; gt.K = kw; gt.A = Tm; gt.lda = ldt; gt.B = W; gt.ldb = ldw;
        gt.C = Wp; gt.ldc = ldw; gt.alpha = T(1); gt.beta = T(0);
        CKI(gemm_direct_confined<T>(h, true, gt, sms, reserve_sms, st));
        W2 = Wp;
        h.launches += 1;
    } else {
        CK(ttw_launch<T>(Wp, L1.seg, sstride, ldw, Tm, ldt, kw, nc, W, ldw, st));
    }
    GemmArgs<T> g2{};
    g2.M = mk; g2.N = nc; g2.K = kw; g2.A = V; g2.lda = ldv; g2.B = W2; g2.ldb = ldw;
    g2.C = C; g2.ldc = ldc; g2.alpha = T(-1); g2.beta = T(1);
    if (prof) { e0 = h.timing_event(); e1 = h.timing_event(); CK(cudaEventRecord(e0, st)); }
    CKI(gemm_direct_confined<T>(h, false, g2, sms, reserve_sms, st));
    if (prof) { CK(cudaEventRecord(e1, st)); h.spans.push_back({e0, e1, fl, 1}); }
    h.launches += 3;
    return 0;
}

// out-of-core copy brackets -> stats (after the streams have been synchronised); releases the timing events
static void resolve_copy_spans(H& h) {
    h.st.copy_exposed_ms = h.st.copy_busy_ms = 0;
    for (auto& s : h.wait_spans) { float ms = 0; cudaEventElapsedTime(&ms, s.first, s.second); h.st.copy_exposed_ms += ms; }
    for (auto& s : h.copy_spans) { float ms = 0; cudaEventElapsedTime(&ms, s.first, s.second); h.st.copy_busy_ms += ms; }
    h.wait_spans.clear(); h.copy_spans.clear();
    h.tpool_used = 0;
}

// sum the profiled spans into the stats (after the streams have been synchronised)
static void resolve_spans(H& h) {
    h.st.vtc_ms = h.st.upd_ms = h.st.vtc_flops = h.st.upd_flops = 0; h.st.vtc_launches = h.st.upd_launches = 0;
    for (auto& s : h.spans) {
        float ms = 0; cudaEventElapsedTime(&ms, s.a, s.b);
        if (s.kind == 0) { h.st.vtc_ms += ms; h.st.vtc_flops += s.flops; h.st.vtc_launches++; }
        else             { h.st.upd_ms += ms; h.st.upd_flops += s.flops; h.st.upd_launches++; }
    }
    h.spans.clear();
    resolve_copy_spans(h);
}

// [st] wait for `ev` (a copy), bracketed by timing events: the time the stream really stalls is the exposed copy time
static int wait_copy(H& h, cudaStream_t st, cudaEvent_t ev) {
    cudaEvent_t a = h.timing_event(), b = h.timing_event();
    CK(cudaEventRecord(a, st));
    CK(cudaStreamWaitEvent(st, ev, 0));
    CK(cudaEventRecord(b, st));
    h.wait_spans.push_back({a, b});
    return 0;
}

// ------------------------------------------------------------------------------------------
// panel factorisation (a1 + a2) of columns [j0, j0+nbw) of the device matrix A (rows j0..m)
// ------------------------------------------------------------------------------------------
template <typename T>
static int launch_panel(H& h, int ib, cudaStream_t st, PanelArgs<T>& pa, int rpt, int G) {
    pa.bar_base = h.bar_count;
    cudaError_t e = panel_launch(ib, rpt, pa, G, st);
    if (e != cudaSuccess)
        return set_err(CTQR_ERR_CUDA, "panel kernel launch failed (ib=%d rpt=%d G=%d): %s", ib, rpt, G, cudaGetErrorString(e));
    h.bar_count += (unsigned)pa.ibw;          // one step number per column, never reused by this handle
    h.launches += 1;
    return 0;
}

// rows-per-thread variants compiled for (dtype, ib), most rows first
template <typename T>
static const int* panel_rpts(int ib) {
    static const int rpts_f64_16[] = {4, 2, 1, 0}, rpts_f32_16[] = {8, 4, 2, 1, 0};
    static const int rpts_8[] = {8, 2, 0}, rpts_f64_32[] = {2, 1, 0}, rpts_f32_32[] = {4, 2, 1, 0};
    return ib == 16 ? (sizeof(T) == 8 ? rpts_f64_16 : rpts_f32_16)
         : ib == 8  ? rpts_8 : (sizeof(T) == 8 ? rpts_f64_32 : rpts_f32_32);
}
// widest inner block <= h.ib whose register-resident kernel can hold `rows` rows on this device
template <typename T>
static int panel_ib_for(const H& h, int64_t rows) {
    for (int ib = h.ib; ib >= 8; ib /= 2)
        if (ceil_div(rows, (int64_t)kPanelThreads * panel_rpts<T>(ib)[0]) <= h.sms) return ib;
    return 0;
}

template <typename T>
static int panel_inner(H& h, int ib, cudaStream_t st, T* A, int64_t lda, int64_t m, int64_t j0, int64_t jb, int ibw, T* Rd, T* Tin) {
    constexpr int NT = kPanelThreads;
    PanelArgs<T> pa{};
    pa.A = A; pa.lda = lda; pa.m = m; pa.j0 = j0; pa.jb = jb; pa.ibw = ibw;
    pa.tau = P_<T>(h.dTau); pa.Rd = Rd; pa.ldrd = h.nb; pa.Tin = Tin; pa.ldtin = h.nb;
    pa.part = P_<T>(h.dPart);
    const int64_t rows = m - jb;
    const int gmax = h.sms;
    const int* list = panel_rpts<T>(ib);
    // largest rpt whose grid still has >= 8 CTAs (enough parallelism), else the smallest that fits
    int pick = 0;
    for (const int* r = list; *r; ++r) {
        int64_t g = ceil_div(rows, (int64_t)NT * *r);
        if (g <= gmax && (g >= 8 || r[1] == 0)) { pick = *r; break; }
    }
    if (!pick)
        for (const int* r = list; *r; ++r)
            if (ceil_div(rows, (int64_t)NT * *r) <= gmax) { pick = *r; break; }
    if (!pick)
        return set_err(CTQR_ERR_NOMEM, "panel of %lld rows does not fit the register-resident kernel (ib=%d)",
                       (long long)rows, ib);
    return launch_panel<T>(h, ib, st, pa, pick, (int)std::max<int64_t>(1, ceil_div(rows, (int64_t)NT * pick)));
}

template <typename T>
static int panel_factor(H& h, cudaStream_t st, T* A, int64_t lda, int64_t m, int64_t j0, int nbw, int k) {
    T* Rd = P_<T>(h.dRd) + (size_t)k * h.nb * h.nb;
    T* Tk = P_<T>(h.dT) + (size_t)k * h.nb * h.nb;
    // inner width for this panel: h.ib unless the panel is too tall for that kernel's registers
    const int ib = panel_ib_for<T>(h, m - j0);
    if (!ib)
        return set_err(CTQR_ERR_NOMEM, "panel of %lld rows does not fit the register-resident panel kernel",
                       (long long)(m - j0));
    for (int64_t jb = j0; jb < j0 + nbw; jb += ib) {
        const int ibw = (int)std::min<int64_t>(ib, j0 + nbw - jb);
        T* Tin = Tk + (jb - j0) + (jb - j0) * (int64_t)h.nb;      // diagonal block of T_k
        CKI(panel_inner<T>(h, ib, st, A, lda, m, j0, jb, ibw, Rd, Tin));
        const int64_t ncp = j0 + nbw - (jb + ibw);
        if (ncp > 0)
            CKI(larfb<T>(h, 1, st, A + jb + jb * lda, lda, m - jb, ibw, Tin, h.nb,
                         A + jb + (jb + ibw) * lda, lda, ncp));
    }
    if (nbw <= ib) return 0;            // single inner block: its T is the panel's T
    // T_k from the Gram matrix of the finished panel
    const T* V = A + j0 + j0 * lda;
    const int64_t mk = m - j0;
    const int64_t ldg = round_up(nbw, 4);
    const int64_t gstride = ldg * nbw;
    GemmArgs<T> g{};
    g.M = nbw; g.N = nbw; g.K = mk; g.A = V; g.lda = lda; g.B = V; g.ldb = lda;
    g.C = P_<T>(h.dWp[1]); g.ldc = ldg; g.alpha = T(1); g.beta = T(0); g.split_stride = gstride;
    const GemmLaunch LG = gemm_plan<T>(true, nbw, nbw, mk, h.gemm_impl, h.sms, true,
                                       (int64_t)h.wp_elems[1], gstride, gemm_aligned(g));
    CK(gemm_run<T>(true, g, LG, h.gemm_impl, st));
    CK(larft_launch<T>(P_<T>(h.dWp[1]), LG.seg, gstride, (int)ldg, nbw, ib, Tk, h.nb, st));
    h.launches += 2;
    return 0;
}

static cudaEvent_t new_event(H& h, bool timing) {
    cudaEvent_t e = nullptr;
    if (cudaEventCreateWithFlags(&e, timing ? cudaEventDefault : cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;                 // cudaEventRecord(nullptr, ..) then fails and the caller's CK reports it
    }
    h.ev.push_back(e);
    return e;
}

// `st` must not touch the columns [.., col_end) before their host-to-device chunks have landed (h.arrive, see factor_typed)
static int wait_columns(H& h, cudaStream_t st, int64_t col_end) {
    for (auto& a : h.arrive) {
        CK(cudaStreamWaitEvent(st, a.second, 0));
        if (a.first >= col_end) break;
    }
    return 0;
}

// ------------------------------------------------------------------------------------------
// a4: right-looking blocked QR of the columns [c0, c1) (c0 a multiple of nb) with look-ahead:
// panel k+1 is factored on the high-priority stream sP while the bulk of update k runs on sU.
// A is the VIRTUAL base of the buffer holding those columns: element (i, j) lives at
// A[i + j * lda] and only c0 <= j < c1 is ever touched.  Earlier panels must already have been
// applied.  Everything is enqueued; on return sU waits for the last panel.  No host sync.
// ------------------------------------------------------------------------------------------
template <typename T>
static int factor_range_single(H& h, T* A, int64_t lda, int64_t c0, int64_t c1) {
    const int nb = h.nb;
    const int k0 = (int)(c0 / nb), k1 = (int)ceil_div(c1, nb);
    if (!h.evP) { h.evP = new_event(h, false); h.evL = new_event(h, false); h.evU = new_event(h, false); }
    cudaEvent_t evP = h.evP, evL = h.evL, evU = h.evU;
    if (!h.arrive.empty()) { CKI(wait_columns(h, h.sU, c1)); h.arrive.clear(); }   // no copy overlap on this path
    CK(cudaEventRecord(evU, h.sU));
    CK(cudaStreamWaitEvent(h.sP, evU, 0));
    if (!h.lookahead) {
        for (int k = k0; k < k1; ++k) {
            const int64_t j0 = (int64_t)k * nb;
            const int nbw = (int)std::min<int64_t>(nb, c1 - j0);
            const int64_t me = row_end(h, j0 + nbw);
            CKI(panel_factor<T>(h, h.sU, A, lda, me, j0, nbw, k));
            const int64_t nc = c1 - (j0 + nbw);
            CKI(larfb<T>(h, 0, h.sU, A + j0 + j0 * lda, lda, me - j0, nbw,
                         P_<T>(h.dT) + (size_t)k * nb * nb, nb, A + j0 + (j0 + nbw) * lda, lda, nc, true));
        }
        return 0;
    }
    CKI(panel_factor<T>(h, h.sP, A, lda, row_end(h, std::min<int64_t>(c0 + nb, c1)), c0, (int)std::min<int64_t>(nb, c1 - c0), k0));
    CK(cudaEventRecord(evP, h.sP));
    for (int k = k0; k < k1; ++k) {
        const int64_t j0 = (int64_t)k * nb;
        const int nbw = (int)std::min<int64_t>(nb, c1 - j0);
        const int64_t jn = j0 + nbw;                        // first trailing column
        if (jn >= c1) break;
        const int nbn = (int)std::min<int64_t>(nb, c1 - jn); // width of panel k+1
        const int64_t me = row_end(h, jn), men = row_end(h, jn + nbn);   // row ends of panels k and k+1
        const T* V = A + j0 + j0 * lda;
        const T* Tk = P_<T>(h.dT) + (size_t)k * nb * nb;
        CK(cudaStreamWaitEvent(h.sU, evP, 0));              // V_k, T_k ready
        CKI(larfb<T>(h, 0, h.sU, V, lda, me - j0, nbw, Tk, nb, A + j0 + jn * lda, lda, nbn, true));
        CK(cudaEventRecord(evL, h.sU));
        CK(cudaStreamWaitEvent(h.sP, evL, 0));
        CKI(panel_factor<T>(h, h.sP, A, lda, men, jn, nbn, k + 1));
        CK(cudaEventRecord(evP, h.sP));
        // Bulk update.  The fp32 contractions are one-CTA-per-SM persistent kernels, so a smaller grid
        // leaves whole SMs empty: the first part of the bulk runs on (SMs - R) while the look-ahead
        // panel chain (R co-resident CTAs of the cooperative panel kernel + its small kernels, on the
        // high-priority stream) uses the rest; the remainder of the bulk then takes every SM.
        // The fp64 kernels run two CTAs per SM, so there the CTAs that land on the R reserved SMs retire
        // at once and the rest draw their worker index from a counter (GemmLaunch::reserve).
        const int64_t ncb = c1 - jn - nbn;
        int R = 0; int64_t nA = ncb;
        if (h.gemm_impl == 0 && h.reserve_sms != 0 && ncb > 0) {
            const int64_t mk1 = men - jn;
            const int ibn = panel_ib_for<T>(h, mk1);
            const int Gp = ibn ? (int)ceil_div(mk1, (int64_t)kPanelThreads * panel_rpts<T>(ibn)[0]) : h.sms;
            R = h.reserve_sms > 0 ? h.reserve_sms : Gp + 2;
            if (R > (int)(h.sms * 0.45)) R = 0;          // tall panels: the chain is negligible against the update
            if (R > 0) {
                const double t_panel = 0.25e-3 + 1.5e-8 * (double)mk1;                   // s, calibrated at c3 (flat optimum, both precisions)
                const double rate = (sizeof(T) == 4 ? 69e12 : 25e12) * (double)(h.sms - R) / (double)h.sms;   // flop/s of the pair of products
                nA = (int64_t)(t_panel * rate / (4.0 * (double)(me - j0) * nbw));
                nA = std::min<int64_t>(ncb, round_up(std::max<int64_t>(nA, 128), 128));
                if (ncb - nA < 256) nA = ncb;
            }
        }
        T* Cb = A + j0 + (jn + nbn) * lda;
        CKI(larfb<T>(h, 0, h.sU, V, lda, me - j0, nbw, Tk, nb, Cb, lda, nA, true, R));
        if (nA < ncb) CKI(larfb<T>(h, 0, h.sU, V, lda, me - j0, nbw, Tk, nb, Cb + nA * lda, lda, ncb - nA, true, 0));
    }
    CK(cudaStreamWaitEvent(h.sU, evP, 0));
    return 0;
}

// ------------------------------------------------------------------------------------------
// Two panels per trailing update (in core, nb = 128).  C <- C - V W with K = nb = 128 is the
// slowest contraction of the factorisation (8 k-tiles per output tile, C read and written
// once per panel); applying panels k, k+1 together as ONE 256-wide compact-WY block
//     Q = H_k H_{k+1} = I - [V_k V_{k+1}] T2 [V_k V_{k+1}]^T,
//     T2 = [[T_k, -T_k (V_k^T V_{k+1}) T_{k+1}], [0, T_{k+1}]]        (the larft recurrence, one block step)
// halves the passes over C and doubles K (measured: the fp64 kernel alone 24.3 -> 27.8 TFLOP/s).
// The look-ahead chain then factors TWO panels (with the narrow larfb between them) and merges
// their T factors while the bulk of the previous pair's update runs.  V_{k+1} is zero in the
// rows of panel k's diagonal block, where the matrix holds R_{k,k+1}: the products touching those
// rows are issued separately (W_bot = V_{k+1}^T C[nb:], and the top nb rows of C take only V_k).
// ------------------------------------------------------------------------------------------
template <typename T>
static int ensure_pair_ws(H& h, int64_t nc) {
    const size_t need = (size_t)256 * (size_t)nc;
    if (h.dW2[0] && h.w2_elems >= need) return 0;
    for (int i = 0; i < 2; ++i) { if (h.dW2[i]) dev_free(h.dW2[i]); h.dW2[i] = nullptr; }
    for (int i = 0; i < 2; ++i)
        if (dev_alloc(&h.dW2[i], need * sizeof(T)) != cudaSuccess) { cudaGetLastError(); h.w2_elems = 0; return 1; }
    h.w2_elems = need;
    if (sizeof(T) == 4 && h.gemm_impl == 0) {
        const size_t need_ws = (size_t)2 * 256 * (size_t)nc;
        if (h.ws_elems < need_ws) {
            dev_free(h.dWs); h.dWs = nullptr; h.ws_elems = 0;
            if (dev_alloc(&h.dWs, need_ws * sizeof(float)) != cudaSuccess) { cudaGetLastError(); return 1; }
            h.ws_elems = need_ws;
        }
        if (!h.dVs[0]) {
            h.ldvs = round_up(h.m, 32);
            for (int i = 0; i < 2; ++i)
                if (big_alloc(&h.dVs[i], (size_t)2 * h.ldvs * 256 * sizeof(float)) != cudaSuccess) {
                    cudaGetLastError();
                    if (h.dVs[0]) { cudaFree(h.dVs[0]); h.dVs[0] = nullptr; }
                    return 1;
                }
        }
    }
    if (!h.dT2) {
        if (dev_alloc(&h.dT2, (size_t)2 * 256 * 256 * sizeof(T)) != cudaSuccess) { cudaGetLastError(); return 1; }
        CK(cudaMemsetAsync(h.dT2, 0, (size_t)2 * 256 * 256 * sizeof(T), h.sU));
    }
    if (!h.dMerge && dev_alloc(&h.dMerge, (size_t)2 * 128 * 128 * sizeof(T)) != cudaSuccess) { cudaGetLastError(); return 1; }
    if (!h.dT12 && h.P >= 2) {
        if (dev_alloc(&h.dT12, (size_t)(h.P / 2) * 128 * 128 * sizeof(T)) != cudaSuccess) { cudaGetLastError(); h.dT12 = nullptr; }
        else h.t12_have.assign((size_t)(h.P / 2), 0);           // (without it the solve applies one panel at a time)
    }
    return 0;
}

// T2[slot] for the panels starting at columns j0 and j0 + 128 (both factored, both 128 wide); stream st
template <typename T>
static int pair_merge(H& h, cudaStream_t st, const T* A, int64_t lda, int64_t m, int64_t j0, int slot) {
    const int nb = 128;
    const int k = (int)(j0 / nb);
    const T* Tk = P_<T>(h.dT) + (size_t)k * nb * nb;
    const T* Tk1 = Tk + (size_t)nb * nb;
    T* T2 = P_<T>(h.dT2) + (size_t)slot * 256 * 256;
    T* G = P_<T>(h.dMerge), *X = G + 128 * 128;
    // G = V_k[nb:, :]^T V_{k+1}  (stream-K partial tiles, summed in a fixed order)
    GemmArgs<T> g{};
    g.M = nb; g.N = nb; g.K = m - j0 - nb; g.A = A + (j0 + nb) + j0 * lda; g.lda = lda;
    g.B = A + (j0 + nb) + (j0 + nb) * lda; g.ldb = lda;
    g.C = P_<T>(h.dWp[1]); g.ldc = nb; g.alpha = T(1); g.beta = T(0); g.split_stride = (int64_t)nb * nb;
    const GemmLaunch LG = gemm_plan<T>(true, nb, nb, g.K, h.gemm_impl, h.sms, true, (int64_t)h.wp_elems[1],
                                       g.split_stride, gemm_aligned(g));
    if (LG.kind != 1) return set_err(CTQR_ERR_STATE, "pair merge needs the stream-K product");
    CK(gemm_run<T>(true, g, LG, h.gemm_impl, st));
    CK(partial_sum_launch<T>(P_<T>(h.dWp[1]), LG.seg, nb, nb, G, nb, st));
    // X = G T_{k+1};  T2[0:nb, nb:2nb] = -T_k X
    GemmArgs<T> g2{};
    g2.M = nb; g2.N = nb; g2.K = nb; g2.A = G; g2.lda = nb; g2.B = Tk1; g2.ldb = nb; g2.C = X; g2.ldc = nb;
    g2.alpha = T(1); g2.beta = T(0);
    CK(gemm_direct<T>(false, g2, h.gemm_impl, h.sms, st));
    GemmArgs<T> g3{};
    g3.M = nb; g3.N = nb; g3.K = nb; g3.A = Tk; g3.lda = nb; g3.B = X; g3.ldb = nb; g3.C = T2 + (size_t)nb * 256; g3.ldc = 256;
    g3.alpha = T(-1); g3.beta = T(0);
    CK(gemm_direct<T>(false, g3, h.gemm_impl, h.sms, st));
    CK(copy2d_launch<T>(Tk, nb, T2, 256, nb, nb, st));
    CK(copy2d_launch<T>(Tk1, nb, T2 + nb + (size_t)nb * 256, 256, nb, nb, st));
    h.launches += 6;
    if (h.dT12 && (k & 1) == 0 && (size_t)(k / 2) < h.t12_have.size()) {
        // the solve applies Q^T to large batches pair by pair as well: keep this pair's off-diagonal block
        CK(copy2d_launch<T>(T2 + (size_t)nb * 256, 256, P_<T>(h.dT12) + (size_t)(k / 2) * nb * nb, nb, nb, nb, st));
        h.t12_have[k / 2] = 1;
        h.launches += 1;
    }
    if constexpr (sizeof(T) == 4) {
        if (h.dVs[slot]) {
            // both contractions of this pair's trailing updates read [V_k V_{k+1}] once per output tile: split it into TF32
            // hi / lo once, here on the panel stream (gemm_umma_tma.cuh); rows from j0 (the rows of the first diagonal block
            // in the second panel's columns hold R_{k,k+1}: split along, never used)
            float* hi = P_<float>(h.dVs[slot]);
            CK(split_tf32_launch(A + j0 + j0 * lda, lda, m - j0, 2 * nb, hi, hi + (size_t)h.ldvs * 256, h.ldvs, st));
            h.launches += 1;
        }
    }
    return 0;
}

// C[j0:m, 0:nc] <- (H_k H_{k+1})^T C for the pair at columns j0, j0 + 128; T2 = its merged factor; stream sU
template <typename T>
static int larfb_pair(H& h, cudaStream_t st, const T* A, int64_t lda, int64_t m, int64_t j0, int slot, T* C,
                      int64_t ldc, int64_t nc, int reserve_sms, int64_t min_nc = 1024) {
    const T* T2 = P_<T>(h.dT2) + (size_t)slot * 256 * 256;
    if (nc <= 0) return 0;
    const int nb = 128;
    const int k = (int)(j0 / nb);
    const T* V1 = A + j0 + j0 * lda;
    const T* V2 = A + (j0 + nb) + (j0 + nb) * lda;
    const int64_t mk = m - j0;
    if (nc < min_nc || (size_t)256 * (size_t)nc > h.w2_elems) {
        // narrow right-hand side: the two panels one after the other (same product, small kernels)
        CKI(larfb<T>(h, 0, st, V1, lda, mk, nb, P_<T>(h.dT) + (size_t)k * nb * nb, nb, C, ldc, nc, true, reserve_sms));
        CKI(larfb<T>(h, 0, st, V2, lda, mk - nb, nb, P_<T>(h.dT) + (size_t)(k + 1) * nb * nb, nb, C + nb, ldc, nc, true,
                     reserve_sms));
        return 0;
    }
    const int sms = std::max(8, h.sms - reserve_sms);
    T* Wp = P_<T>(h.dWp[0]);
    T* W = P_<T>(h.dW2[0]);
    T* W2 = P_<T>(h.dW2[1]);
    const bool prof = h.profile;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    // W[0:nb] = V_k^T C,  W[nb:2nb] = V_{k+1}^T C[nb:]
    for (int half = 0; half < 2; ++half) {
        GemmArgs<T> g1{};
        g1.M = nb; g1.N = nc; g1.K = mk - half * nb; g1.A = half ? V2 : V1; g1.lda = lda; g1.B = C + half * nb; g1.ldb = ldc;
        g1.C = Wp; g1.ldc = nb; g1.alpha = T(1); g1.beta = T(0); g1.split_stride = (int64_t)nb * nc;
        GemmLaunch L1 = gemm_plan<T>(true, nb, nc, g1.K, h.gemm_impl, sms, true, (int64_t)h.wp_elems[0], g1.split_stride,
                                     gemm_aligned(g1));
        if (L1.kind != 1) return set_err(CTQR_ERR_STATE, "pair update needs the stream-K product");
        CKI(confine<T>(h, L1, reserve_sms, st));
        if (prof) { e0 = h.timing_event(); e1 = h.timing_event(); CK(cudaEventRecord(e0, st)); }
        bool pre = false;
#ifndef CTQR_NO_VTC_TMA
        if constexpr (sizeof(T) == 4) {
            if (h.dVs[slot]) {
                // fp32: V pre-split by the merge and TMA-fed, the streamed C split on the fly (vtc_tma_kernel)
                const float* vh = P_<float>(h.dVs[slot]) + (half ? (size_t)nb + (size_t)nb * h.ldvs : 0);
                cudaError_t ev = vtc_presplit_launch(g1, vh, vh + (size_t)h.ldvs * 256, h.ldvs, L1, st);
                if (ev == cudaSuccess) pre = true;
                else if (ev != cudaErrorNotSupported) CK(ev);
            }
        }
#endif
        if (!pre) CK(gemm_run<T>(true, g1, L1, h.gemm_impl, st));
        if (prof) { CK(cudaEventRecord(e1, st)); h.spans.push_back({e0, e1, 2.0 * (double)g1.K * nb * (double)nc, 0}); }
        CK(partial_sum_launch<T>(Wp, L1.seg, nb, nc, W + half * nb, 256, st));
    }
    // W2 = T2^T W
    GemmArgs<T> gt{};
    gt.M = 256; gt.N = nc; gt.K = 256; gt.A = T2; gt.lda = 256; gt.B = W; gt.ldb = 256; gt.C = W2; gt.ldc = 256;
    gt.alpha = T(1); gt.beta = T(0);
    CKI(gemm_direct_confined<T>(h, true, gt, sms, reserve_sms, st));
    // top nb rows: only V_k reaches them;  the rest: K = 256
    GemmArgs<T> ga{};
    ga.M = nb; ga.N = nc; ga.K = nb; ga.A = V1; ga.lda = lda; ga.B = W2; ga.ldb = 256; ga.C = C; ga.ldc = ldc;
    ga.alpha = T(-1); ga.beta = T(1);
    CKI(gemm_direct_confined<T>(h, false, ga, sms, reserve_sms, st));
    GemmArgs<T> gb{};
    gb.M = mk - nb; gb.N = nc; gb.K = 256; gb.A = A + (j0 + nb) + j0 * lda; gb.lda = lda; gb.B = W2; gb.ldb = 256;
    gb.C = C + nb; gb.ldc = ldc; gb.alpha = T(-1); gb.beta = T(1);
    bool done = false;
    if constexpr (sizeof(T) == 4) {
        if (h.dVs[slot] && h.dWs && (size_t)2 * 256 * (size_t)nc <= h.ws_elems && ldc % 4 == 0) {
            // fp32: operands pre-split once (V by the merge, T2^T W here), TMA-fed tcgen05 kernel, 128 x 128 tiles
            float* whi = P_<float>(h.dWs); float* wlo = whi + (size_t)256 * nc;
            const float* vhi = P_<float>(h.dVs[slot]) + nb; const float* vlo = vhi + (size_t)h.ldvs * 256;   // rows below the first diagonal block
            CK(split_tf32_launch(W2, 256, 256, nc, whi, wlo, 256, st));
            if (prof) { e0 = h.timing_event(); e1 = h.timing_event(); CK(cudaEventRecord(e0, st)); }
            CK(upd_presplit_launch(gb.M, nc, 256, -1.f, vhi, vlo, h.ldvs, whi, wlo, 256, 1.f, gb.C, ldc, sms, st));
            if (prof) { CK(cudaEventRecord(e1, st)); h.spans.push_back({e0, e1, 2.0 * (double)gb.M * 256 * (double)nc, 1}); }
            h.launches += 1;
            done = true;
        }
    }
    if (!done) {
        if (prof) { e0 = h.timing_event(); e1 = h.timing_event(); CK(cudaEventRecord(e0, st)); }
        CKI(gemm_direct_confined<T>(h, false, gb, sms, reserve_sms, st));
        if (prof) { CK(cudaEventRecord(e1, st)); h.spans.push_back({e0, e1, 2.0 * (double)gb.M * 256 * (double)nc, 1}); }
    }
    h.launches += 7;
    return 0;
}

template <typename T>
static int factor_range_pairs(H& h, T* A, int64_t lda, int64_t c0, int64_t c1) {
    const int nb = 128;
    if (!h.evP) { h.evP = new_event(h, false); h.evL = new_event(h, false); h.evU = new_event(h, false); }
    cudaEvent_t evP = h.evP, evL = h.evL, evU = h.evU;
    CK(cudaEventRecord(evU, h.sU));
    CK(cudaStreamWaitEvent(h.sP, evU, 0));
    // the look-ahead chain of one pair on sP: panel, narrow larfb onto the next panel's columns, panel, merge
    auto chain = [&](int64_t j0, int slot) -> int {
        const int k = (int)(j0 / nb);
        const int64_t m = row_end(h, j0 + 2 * nb);          // row end of the pair (its first panel ends nb rows earlier: zeros)
        CKI(panel_factor<T>(h, h.sP, A, lda, m, j0, nb, k));
        CKI(larfb<T>(h, 1, h.sP, A + j0 + j0 * lda, lda, m - j0, nb, P_<T>(h.dT) + (size_t)k * nb * nb, nb,
                     A + j0 + (j0 + nb) * lda, lda, nb));
        CKI(panel_factor<T>(h, h.sP, A, lda, m, j0 + nb, nb, k + 1));
        CKI(pair_merge<T>(h, h.sP, A, lda, m, j0, slot));
        CK(cudaEventRecord(evP, h.sP));
        return 0;
    };
    int slot = 0;
    // host matrix still arriving in column chunks (factor_typed): the first chain needs the first pair's columns only, the
    // first trailing update then follows the copy chunk by chunk; every later step is ordered behind those waits
    const bool arriving = !h.arrive.empty() && c0 == 0;
    if (arriving) CKI(wait_columns(h, h.sP, 2 * nb));
    else if (!h.arrive.empty()) { CKI(wait_columns(h, h.sU, c1)); h.arrive.clear(); }
    CKI(chain(c0, slot));
    for (int64_t j0 = c0;; j0 += 2 * nb, slot ^= 1) {
        const int64_t jn = j0 + 2 * nb;                     // first trailing column
        const int64_t rem = c1 - jn;
        const int64_t m = row_end(h, jn);                   // row end of this pair
        CK(cudaStreamWaitEvent(h.sU, evP, 0));              // V, T2 of this pair ready
        if (arriving && j0 == c0 && rem >= 2 * nb) {
            // first pair: look-ahead block, next chain, then the bulk in the order the chunks arrive
            CKI(wait_columns(h, h.sU, jn + 2 * nb));
            CKI(larfb_pair<T>(h, h.sU, A, lda, m, j0, slot, A + j0 + jn * lda, lda, 2 * nb, 0));
            CK(cudaEventRecord(evL, h.sU));
            CK(cudaStreamWaitEvent(h.sP, evL, 0));
            CKI(chain(jn, slot ^ 1));
            int64_t ca = jn + 2 * nb;
            for (auto& a : h.arrive) {
                const int64_t cb = std::min<int64_t>(a.first, c1);
                if (cb <= ca) continue;
                CK(cudaStreamWaitEvent(h.sU, a.second, 0));
                CKI(larfb_pair<T>(h, h.sU, A, lda, m, j0, slot, A + j0 + ca * lda, lda, cb - ca, 0));
                ca = cb;
            }
            h.arrive.clear();
            continue;
        }
        if (!h.arrive.empty()) { CKI(wait_columns(h, h.sU, c1)); h.arrive.clear(); }
        if (rem < 2 * nb) {
            // no further full pair: finish this update, then the single-panel driver takes the tail
            CKI(larfb_pair<T>(h, h.sU, A, lda, m, j0, slot, A + j0 + jn * lda, lda, rem, 0));
            if (rem > 0) CKI(factor_range_single<T>(h, A, lda, jn, c1));
            return 0;
        }
        // look-ahead block: the columns of the next pair
        CKI(larfb_pair<T>(h, h.sU, A, lda, m, j0, slot, A + j0 + jn * lda, lda, 2 * nb, 0));
        CK(cudaEventRecord(evL, h.sU));
        CK(cudaStreamWaitEvent(h.sP, evL, 0));
        CKI(chain(jn, slot ^ 1));
        // bulk: first part beside the chain on SMs - R (see factor_range_single), then everything
        const int64_t ncb = rem - 2 * nb;
        int R = 0; int64_t nA = ncb;
        if (h.reserve_sms != 0 && ncb > 0) {
            const int64_t mk1 = row_end(h, jn + 2 * nb) - jn;
            const int ibn = panel_ib_for<T>(h, mk1);
            const int Gp = ibn ? (int)ceil_div(mk1, (int64_t)kPanelThreads * panel_rpts<T>(ibn)[0]) : h.sms;
            R = h.reserve_sms > 0 ? h.reserve_sms : Gp + 2;
            if (R > (int)(h.sms * 0.45)) R = 0;
            if (R > 0) {
                const double t_chain = 2.0 * (0.25e-3 + 1.5e-8 * (double)mk1) + 0.15e-3;
                const double rate = (sizeof(T) == 4 ? 100e12 : 31e12) * (double)(h.sms - R) / (double)h.sms;
                nA = (int64_t)(t_chain * rate / (4.0 * (double)(m - j0) * 2 * nb));
                nA = std::min<int64_t>(ncb, round_up(std::max<int64_t>(nA, 1024), 128));
                if (ncb - nA < 1024) nA = ncb;
            }
        }
        T* Cb = A + j0 + (jn + 2 * nb) * lda;
        CKI(larfb_pair<T>(h, h.sU, A, lda, m, j0, slot, Cb, lda, nA, R));
        if (nA < ncb) CKI(larfb_pair<T>(h, h.sU, A, lda, m, j0, slot, Cb + nA * lda, lda, ncb - nA, 0));
    }
}

template <typename T>
static int factor_range(H& h, T* A, int64_t lda, int64_t c0, int64_t c1) {
    const bool aligned = (uintptr_t)A % 16 == 0 && (lda * (int64_t)sizeof(T)) % 16 == 0;
    if (h.lookahead && h.nb == 128 && h.gemm_impl == 0 && aligned && c0 % 128 == 0 && c1 - c0 >= 4 * 128 &&
        h.m - c0 >= 1024 && ensure_pair_ws<T>(h, c1 - c0) == 0)
        return factor_range_pairs<T>(h, A, lda, c0, c1);
    return factor_range_single<T>(h, A, lda, c0, c1);
}

template <typename T> static int band_check(H& h, const T* A, int64_t lda, int64_t c0, int64_t c1);
template <typename T> static int band_check_enqueue(H& h, const T* A, int64_t lda, int64_t c0, int64_t c1);
static int band_check_result(H& h);

template <typename T>
static int factor_incore(H& h, T* A, int64_t lda) {
    cudaEvent_t t0 = new_event(h, true), t1 = new_event(h, true);
    CK(cudaEventRecord(t0, h.sU));
    // the band promise is verified inside the timed window (factor_ms includes the check), before anything is factored
    if (h.kl > 0) {
        if (!h.arrive.empty()) { CKI(wait_columns(h, h.sU, h.n)); h.arrive.clear(); }
        CKI(band_check<T>(h, A, lda, 0, h.n));
    }
    CKI(factor_range<T>(h, A, lda, 0, h.n));
    CK(cudaEventRecord(t1, h.sU));
    CK(cudaStreamSynchronize(h.sU));
    CK(cudaStreamSynchronize(h.sP));
    float ms = 0; CK(cudaEventElapsedTime(&ms, t0, t1));
    h.st.factor_ms = ms;
    resolve_spans(h);
    return 0;
}

// ------------------------------------------------------------------------------------------
// a5: out-of-core tile scheduler (section 2.2: blocks, task list, prefetch of
// the operands of the next tasks during the current one; here the slow tier is pinned host
// memory and the overlap is copy streams + events instead of an I/O thread).
//
// Left-looking over column SUPER-PANELS of ns columns (ns a multiple of nb, two buffers):
//   for s = 0 .. Ps-1:           (sC = H2D copy stream, sD = D2H copy stream, sU/sP compute)
//     [sC] SP_s <- host A[:, c0:c1)                       (issued while SP_{s-1} is being factored)
//     for every earlier panel k, in order:   SP_s[j0:m, :] <- (I - V_k T_k^T V_k^T) SP_s[j0:m, :]
//          V_k comes from the other device buffer when k belongs to SP_{s-1} (still resident),
//          else it is streamed host -> Vb[k & 1] on sC (double-buffered against the larfb on sU)
//     [sU,sP] right-looking factorisation of SP_s with look-ahead (factor_range)
//     [sD] host A[:, c0:c1) <- SP_s                       (in place; overlaps the work on SP_{s+1})
// T_k, tau and the diagonal R blocks stay resident.  Host-link bytes: every super-panel in and
// out once plus the earlier reflectors once per later super-panel = m n w (P_s + 3)/2.
// ------------------------------------------------------------------------------------------
template <typename T>
static int stream_panel_in(H& h, int slot, const T* hsrc, int64_t hld, int64_t rows, int cols, void* dst = nullptr) {
    // [sC] wait until the larfb that last read Vb[slot] (or the pair buffer of that slot: they share the events) is done,
    // copy, signal
    CK(cudaStreamWaitEvent(h.sC, h.evVfree[slot], 0));
    cudaEvent_t ca = h.timing_event(), cb = h.timing_event();
    CK(cudaEventRecord(ca, h.sC));
    CK(cudaMemcpy2DAsync(dst ? dst : h.dVb[slot], h.ldvb * sizeof(T), hsrc, hld * sizeof(T), rows * sizeof(T), cols,
                         cudaMemcpyHostToDevice, h.sC));
    CK(cudaEventRecord(cb, h.sC));
    h.copy_spans.push_back({ca, cb});
    CK(cudaEventRecord(h.evVin[slot], h.sC));
    h.st.h2d_bytes += (double)rows * cols * sizeof(T);
    return 0;
}

static int ensure_stream_bufs(H& h) {
    if (h.dVb[0]) return 0;
    h.ldvb = round_up(h.m, 16 / (int64_t)h.w);
    for (int i = 0; i < 2; ++i) {
        if (dev_alloc(&h.dVb[i], (size_t)h.ldvb * h.nb * h.w) != cudaSuccess) {
            cudaGetLastError();
            return set_err(CTQR_ERR_NOMEM, "cannot allocate the panel stream buffers");
        }
        h.evVin[i] = new_event(h, false); h.evVfree[i] = new_event(h, false);
        CK(cudaEventRecord(h.evVfree[i], h.sU));
    }
    if (!h.sC) CK(cudaStreamCreateWithFlags(&h.sC, cudaStreamNonBlocking));
    if (!h.sD) CK(cudaStreamCreateWithFlags(&h.sD, cudaStreamNonBlocking));
    return 0;
}


template <typename T>
static int factor_ooc(H& h, T* hA, int64_t hlda, int64_t ns) {
    const int64_t m = h.m, n = h.n;
    const int nb = h.nb;
    const int Ps = (int)ceil_div(n, ns);
    const int64_t lds = round_up(m, 16 / (int64_t)sizeof(T));
    CKI(ensure_stream_bufs(h));
    T* sp[2] = {nullptr, nullptr};
    for (int i = 0; i < 2; ++i) {
        if (big_alloc(&h.spbuf[i], (size_t)lds * std::min<int64_t>(ns, n) * sizeof(T)) != cudaSuccess) {
            cudaGetLastError();
            return set_err(CTQR_ERR_NOMEM, "cannot allocate the super-panel buffers (%lld columns)", (long long)ns);
        }
        sp[i] = P_<T>(h.spbuf[i]);         // owned by the handle: freed below, or by the destructor on an error path
    }
    // Left-looking updates two panels at a time (the 256-wide compact-WY block of factor_range_pairs: K = 256 updates,
    // pre-split TMA-fed operands in fp32) when every earlier panel is 128 wide and the pair workspaces can be had:
    // [V_k V_(k+1)] split buffers, W blocks, and two m x 256 stream buffers -- workspace, outside the tile budget
    // (about 12 m 256 w bytes in fp32, 2 m 256 w in fp64).  Otherwise one panel at a time, as before.
    bool pairs = h.lookahead && nb == 128 && h.gemm_impl == 0 && ns % (2 * nb) == 0 && ns >= 1024 && Ps > 1 &&
                 (lds * (int64_t)sizeof(T)) % 16 == 0 && ensure_pair_ws<T>(h, std::min<int64_t>(ns, n)) == 0;
    if (pairs) {
        for (int i = 0; i < 2 && pairs; ++i)
            if (!h.dVp[i] && big_alloc(&h.dVp[i], (size_t)h.ldvb * 2 * nb * sizeof(T)) != cudaSuccess) { cudaGetLastError(); pairs = false; }
    }
    std::vector<cudaEvent_t> evIn(Ps), evOut(Ps), evDone(Ps), evFree(Ps);
    for (int s = 0; s < Ps; ++s) {
        evIn[s] = new_event(h, false); evOut[s] = new_event(h, false);
        evDone[s] = new_event(h, false); evFree[s] = new_event(h, false);
    }
    cudaEvent_t t0 = new_event(h, true), t1 = new_event(h, true);
    CK(cudaEventRecord(t0, h.sU));
    CK(cudaStreamWaitEvent(h.sC, t0, 0));
    auto load_sp = [&](int s) -> int {
        const int64_t c0 = (int64_t)s * ns, c1 = std::min<int64_t>(n, c0 + ns);
        if (s >= 2) {                                     // buffer reuse: SP_{s-2} written back and no longer read
            CK(cudaStreamWaitEvent(h.sC, evOut[s - 2], 0));
            CK(cudaStreamWaitEvent(h.sC, evFree[s - 2], 0));
        }
        cudaEvent_t ca = h.timing_event(), cb = h.timing_event();
        CK(cudaEventRecord(ca, h.sC));
        CK(cudaMemcpy2DAsync(sp[s & 1], lds * sizeof(T), hA + c0 * hlda, hlda * sizeof(T), m * sizeof(T), c1 - c0,
                             cudaMemcpyHostToDevice, h.sC));
        CK(cudaEventRecord(cb, h.sC));
        h.copy_spans.push_back({ca, cb});
        CK(cudaEventRecord(evIn[s], h.sC));
        h.st.h2d_bytes += (double)m * (c1 - c0) * sizeof(T);
        return 0;
    };
    if (h.kl > 0 && Ps > 1) {
        // The band promise is verified on the WHOLE matrix before anything is written back over the caller's host
        // matrix (or file): the part below the band of every super-panel (rows > kl + c0) is streamed through the two
        // super-panel buffers and checked; a violation returns -6 with the input untouched.  Extra host-link bytes:
        // about w (m - kl)^2 / 2, i.e. n / (m (P_s + 3)) of the factorisation's traffic for [A0; c I] (6 % at
        // configs[4] with 7 super-panels).
        cudaEvent_t evC[2] = {new_event(h, false), new_event(h, false)}, evK[2] = {new_event(h, false), new_event(h, false)};
        CK(cudaMemsetAsync(h.dFlag, 0x7f, sizeof(int), h.sU));
        for (int i = 0; i < 2; ++i) CK(cudaEventRecord(evK[i], h.sU));
        for (int s = 0; s < Ps; ++s) {
            const int64_t c0 = (int64_t)s * ns, c1 = std::min<int64_t>(n, c0 + ns);
            const int64_t r0 = h.kl + c0 + 1;             // first row that can lie below the band in these columns
            if (r0 >= m) break;
            const int b = s & 1;
            CK(cudaStreamWaitEvent(h.sC, evK[b], 0));
            CK(cudaMemcpy2DAsync(sp[b], lds * sizeof(T), hA + r0 + c0 * hlda, hlda * sizeof(T), (m - r0) * sizeof(T), c1 - c0,
                                 cudaMemcpyHostToDevice, h.sC));
            CK(cudaEventRecord(evC[b], h.sC));
            h.st.h2d_bytes += (double)(m - r0) * (c1 - c0) * sizeof(T);
            CK(cudaStreamWaitEvent(h.sU, evC[b], 0));
            CKI(band_check_enqueue<T>(h, sp[b] - r0 - c0 * lds, lds, c0, c1));
            CK(cudaEventRecord(evK[b], h.sU));
        }
        CKI(band_check_result(h));
        CK(cudaStreamWaitEvent(h.sC, evK[0], 0));
        CK(cudaStreamWaitEvent(h.sC, evK[1], 0));
    }
    int rc = load_sp(0);
    for (int s = 0; s < Ps && rc == 0; ++s) {
        const int64_t c0 = (int64_t)s * ns, c1 = std::min<int64_t>(n, c0 + ns);
        T* Cv = sp[s & 1] - c0 * lds;                     // virtual base of SP_s
        CKI(wait_copy(h, h.sU, evIn[s]));
        if (h.kl > 0 && Ps == 1) { rc = band_check<T>(h, Cv, lds, c0, c1); if (rc) break; }   // single super-panel: nothing written back yet
        // ---- earlier reflectors, streamed from the host (super-panels 0 .. s-2) ----
        const int kres = s >= 1 ? (int)(((int64_t)(s - 1) * ns) / nb) : 0;   // first panel of SP_{s-1}
        const int kcur = (int)(c0 / nb);
        for (int k = 0; k < kres && rc == 0; ++k) {
            const int64_t j0 = (int64_t)k * nb;
            if (pairs && k + 1 < kres && (j0 + nb) / ns == j0 / ns) {
                // two panels of one earlier super-panel at a time: the m x 256 block at (j0, j0) is the pair's [V_k V_(k+1)]
                const int slot = (k >> 1) & 1;
                CK(cudaStreamWaitEvent(h.sC, evOut[(int)(j0 / ns)], 0));
                const int64_t me = row_end(h, j0 + 2 * nb);
                rc = stream_panel_in<T>(h, slot, hA + j0 + j0 * hlda, hlda, me - j0, 2 * nb, h.dVp[slot]);
                if (rc) break;
                CKI(wait_copy(h, h.sU, h.evVin[slot]));
                const T* Vv = P_<T>(h.dVp[slot]) - j0 - j0 * h.ldvb;          // virtual base: (j0, j0) is the buffer's origin
                rc = pair_merge<T>(h, h.sU, Vv, h.ldvb, me, j0, slot);
                if (rc == 0) rc = larfb_pair<T>(h, h.sU, Vv, h.ldvb, me, j0, slot, Cv + j0 + c0 * lds, lds, c1 - c0, 0);
                CK(cudaEventRecord(h.evVfree[slot], h.sU));
                ++k;
                continue;
            }
            const int slot = k & 1;
            CK(cudaStreamWaitEvent(h.sC, evOut[(int)(j0 / ns)], 0));          // factor of that SP is on the host
            const int64_t mk = row_end(h, j0 + nb) - j0;                     // V_k is zero below (band promise)
            rc = stream_panel_in<T>(h, slot, hA + j0 + j0 * hlda, hlda, mk, nb);
            if (rc) break;
            CKI(wait_copy(h, h.sU, h.evVin[slot]));
            rc = larfb<T>(h, 0, h.sU, P_<T>(h.dVb[slot]), h.ldvb, mk, nb, P_<T>(h.dT) + (size_t)k * nb * nb, nb,
                          Cv + j0 + c0 * lds, lds, c1 - c0, true);
            CK(cudaEventRecord(h.evVfree[slot], h.sU));
        }
        // ---- reflectors of SP_{s-1}, still resident in the other buffer ----
        if (s >= 1 && rc == 0) {
            const T* Pv = sp[(s - 1) & 1] - (int64_t)(s - 1) * ns * lds;
            for (int k = kres; k < kcur && rc == 0; ++k) {
                const int64_t j0 = (int64_t)k * nb;
                if (pairs && k + 1 < kcur) {
                    const int slot = (k >> 1) & 1;
                    const int64_t me = row_end(h, j0 + 2 * nb);
                    rc = pair_merge<T>(h, h.sU, Pv, lds, me, j0, slot);
                    if (rc == 0) rc = larfb_pair<T>(h, h.sU, Pv, lds, me, j0, slot, Cv + j0 + c0 * lds, lds, c1 - c0, 0);
                    ++k;
                    continue;
                }
                rc = larfb<T>(h, 0, h.sU, Pv + j0 + j0 * lds, lds, row_end(h, j0 + nb) - j0, nb, P_<T>(h.dT) + (size_t)k * nb * nb, nb,
                              Cv + j0 + c0 * lds, lds, c1 - c0, true);
            }
            CK(cudaEventRecord(evFree[s - 1], h.sU));
        }
        if (rc) break;
        // ---- prefetch the next super-panel while this one is factored ----
        if (s + 1 < Ps) { rc = load_sp(s + 1); if (rc) break; }
        rc = factor_range<T>(h, Cv, lds, c0, c1);
        if (rc) break;
        CK(cudaEventRecord(evDone[s], h.sU));
        CK(cudaStreamWaitEvent(h.sD, evDone[s], 0));
        cudaEvent_t da = h.timing_event(), db = h.timing_event();
        CK(cudaEventRecord(da, h.sD));
        CK(cudaMemcpy2DAsync(hA + c0 * hlda, hlda * sizeof(T), sp[s & 1], lds * sizeof(T), m * sizeof(T), c1 - c0,
                             cudaMemcpyDeviceToHost, h.sD));
        CK(cudaEventRecord(db, h.sD));
        h.copy_spans.push_back({da, db});
        CK(cudaEventRecord(evOut[s], h.sD));
        h.st.d2h_bytes += (double)m * (c1 - c0) * sizeof(T);
    }
    if (rc == 0) {
        if (Ps >= 2) CKI(wait_copy(h, h.sU, evOut[Ps - 2]));
        CKI(wait_copy(h, h.sU, evOut[Ps - 1]));      // the write-back of the last super-panel has nothing left to hide behind
        CK(cudaEventRecord(t1, h.sU));
    }
    cudaError_t e1 = cudaStreamSynchronize(h.sU), e2 = cudaStreamSynchronize(h.sP);
    cudaError_t e3 = cudaStreamSynchronize(h.sC), e4 = cudaStreamSynchronize(h.sD);
    for (int i = 0; i < 2; ++i) { cudaFree(h.spbuf[i]); h.spbuf[i] = nullptr; }
    if (rc) return rc;
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess)
        return set_err(CTQR_ERR_CUDA, "out-of-core factorisation failed: %s",
                       cudaGetErrorString(e1 != cudaSuccess ? e1 : e2 != cudaSuccess ? e2 : e3 != cudaSuccess ? e3 : e4));
    float ms = 0; CK(cudaEventElapsedTime(&ms, t0, t1));
    h.st.factor_ms = ms;
    resolve_spans(h);
    h.ooc = true; h.hA = hA; h.hlda = hlda; h.n_super = Ps;
    return 0;
}

// ------------------------------------------------------------------------------------------
// allocation of the per-handle state
// ------------------------------------------------------------------------------------------
template <typename T>
static int alloc_state(H& h, int64_t max_nc) {
    const int nb = h.nb;
    const size_t blk = (size_t)nb * nb;
    CK(dev_alloc(&h.dT, blk * h.P * sizeof(T)));
    CK(dev_alloc(&h.dRd, blk * h.P * sizeof(T)));
    CK(cudaMemsetAsync(h.dT, 0, blk * h.P * sizeof(T), h.sU));
    CK(cudaMemsetAsync(h.dRd, 0, blk * h.P * sizeof(T), h.sU));
    CK(dev_alloc(&h.dTau, (size_t)h.n * sizeof(T)));
    if (nb == 128) CK(dev_alloc(&h.dRinv, blk * h.P * sizeof(T)));
    const int64_t slots = (int64_t)h.sms * 2;
    // [0]: trailing update / solve; [1]: in-panel work
    h.w_elems[0] = (size_t)nb * (size_t)max_nc;
    h.wp_elems[0] = (size_t)nb * (size_t)(max_nc + 128 * slots);
    h.w_elems[1] = (size_t)nb * nb;
    h.wp_elems[1] = (size_t)nb * 128 * (size_t)slots;
    for (int i = 0; i < 2; ++i) {
        CK(dev_alloc(&h.dW[i], h.w_elems[i] * sizeof(T)));
        CK(dev_alloc(&h.dWp[i], h.wp_elems[i] * sizeof(T)));
    }
    // LL slots of the panel kernel: [2 parities][G + 1 <= 257][IB <= 32] x 16 bytes, step numbers start at 1
    CK(dev_alloc(&h.dPart, (size_t)2 * 257 * 32 * 16));
    CK(cudaMemsetAsync(h.dPart, 0, (size_t)2 * 257 * 32 * 16, h.sU));
    CK(dev_alloc(&h.dFlag, sizeof(int)));
    CK(dev_alloc(&h.dTickets, (size_t)kTicketRing * 2 * sizeof(unsigned)));
    CK(cudaMemsetAsync(h.dTickets, 0, (size_t)kTicketRing * 2 * sizeof(unsigned), h.sU));
    h.ticket_pos = 0;
    if (nb == 128) {
        // fused small-S solve: [2][sms][nb * kSmallS] partial slots + [2][nb * kSmallS] sum slots (Q^T B),
        // then [P][nb * kSmallS] slots of the fused TRSM, 16 bytes each
        const size_t lls = ((size_t)2 * h.sms + 2 + h.P) * nb * kSmallS * 16;
        CK(dev_alloc(&h.dLLs, lls));
        CK(cudaMemsetAsync(h.dLLs, 0, lls, h.sU));
    }
    h.bar_count = 0;
    return 0;
}

static int ensure_solve_ws(H& h, int64_t S) {
    // the update workspace must hold nb x S (W) and its split partials
    const size_t need_w = (size_t)h.nb * (size_t)S;
    const size_t need_wp = (size_t)h.nb * (size_t)(S + 128 * (int64_t)h.sms * 2);
    if (need_w > h.w_elems[0]) {
        dev_free(h.dW[0]); h.dW[0] = nullptr;
        CK(dev_alloc(&h.dW[0], need_w * h.w)); h.w_elems[0] = need_w;
    }
    if (need_wp > h.wp_elems[0]) {
        dev_free(h.dWp[0]); h.dWp[0] = nullptr;
        CK(dev_alloc(&h.dWp[0], need_wp * h.w)); h.wp_elems[0] = need_wp;
    }
    return 0;
}

// opt->lower_bandwidth: the caller's promise A(i, j) == 0 for i - j > kl is checked before it is used
// (one pass over the part of the matrix below the band; flag = first offending column)
template <typename T>
__global__ void band_check_kernel(const T* __restrict__ A, int64_t lda, int64_t m, int64_t c0, int64_t c1, int64_t kl, int* flag) {
    // A is the virtual base: column j at A + j * lda, only c0 <= j < c1 is read
    for (int64_t j = c0 + blockIdx.x; j < c1; j += gridDim.x) {
        const T* col = A + j * lda;
        bool bad = false;
        for (int64_t i = kl + j + 1 + threadIdx.x; i < m; i += blockDim.x) bad |= (col[i] != T(0));
        if (bad) atomicMin(flag, (int)j);
    }
}
template <typename T>
static int band_check_enqueue(H& h, const T* A, int64_t lda, int64_t c0, int64_t c1) {
    band_check_kernel<T><<<(unsigned)std::min<int64_t>(c1 - c0, (int64_t)h.sms * 8), 256, 0, h.sU>>>(A, lda, h.m, c0, c1, h.kl, h.dFlag);
    CK(cudaGetLastError());
    h.launches += 1;
    return 0;
}
static int band_check_result(H& h) {
    int flag = 0;
    CK(cudaMemcpyAsync(&flag, h.dFlag, sizeof(int), cudaMemcpyDeviceToHost, h.sU));
    CK(cudaStreamSynchronize(h.sU));
    if (flag < h.n)
        return set_err(-6, "lower_bandwidth = %lld but column %d has a non-zero below row %lld",
                       (long long)h.kl, flag, (long long)(h.kl + flag));
    return 0;
}
template <typename T>
static int band_check(H& h, const T* A, int64_t lda, int64_t c0, int64_t c1) {
    CK(cudaMemsetAsync(h.dFlag, 0x7f, sizeof(int), h.sU));
    CKI(band_check_enqueue<T>(h, A, lda, c0, c1));
    return band_check_result(h);
}

// ------------------------------------------------------------------------------------------
// ct_qr_factor
// ------------------------------------------------------------------------------------------
template <typename T>
static int factor_typed(H& h, void* A, int64_t lda, bool a_on_device, const ctqr_options_t& o) {
    const int64_t m = h.m, n = h.n;
    const size_t bytes = (size_t)m * n * sizeof(T);
    const size_t freeb = free_device_bytes();
    const size_t slack = (size_t)2 << 30;                 // workspaces, T, B/X of later solves
    if (a_on_device) {
        CKI(alloc_state<T>(h, n));
        if (o.in_place) { h.dA = A; h.lda = lda; h.own_A = false; }
        else {
            h.lda = round_up(m, 16 / sizeof(T));
            CK(big_alloc(&h.dA, (size_t)h.lda * n * sizeof(T)));
            h.own_A = true;
            CK(cudaMemcpy2DAsync(h.dA, h.lda * sizeof(T), A, lda * sizeof(T), m * sizeof(T), n,
                                 cudaMemcpyDeviceToDevice, h.sU));
        }
        return factor_incore<T>(h, P_<T>(h.dA), h.lda);
    }
    const size_t budget = o.device_budget_bytes > 0 ? (size_t)o.device_budget_bytes
                                                    : (freeb > slack ? freeb - slack : 0);
    if (bytes <= budget && !h.fmap) {
        // host matrix that fits: stage once, factor in core, keep the factor on the device
        CKI(alloc_state<T>(h, n));
        h.lda = round_up(m, 16 / sizeof(T));
        CK(big_alloc(&h.dA, (size_t)h.lda * n * sizeof(T)));
        h.own_A = true;
        h.st.h2d_bytes = (double)bytes;
        const int64_t chunk = round_up(std::max<int64_t>(2048, ceil_div(n, (int64_t)16)), 256);
        if (h.kl > 0 || n < 4 * chunk) {
            // (the band promise is checked on the whole matrix before anything is factored; small matrices: one copy)
            CK(cudaMemcpy2DAsync(h.dA, h.lda * sizeof(T), A, lda * sizeof(T), m * sizeof(T), n, cudaMemcpyHostToDevice, h.sU));
            return factor_incore<T>(h, P_<T>(h.dA), h.lda);
        }
        // The host-to-device copy runs in column chunks on the copy stream while the factorisation already works on the
        // columns that have landed (the first pair's trailing update follows the copy chunk by chunk): the copy, 1 s for
        // 57 GB over the host link, is hidden behind the first panels instead of preceding them.
        if (!h.sC) CK(cudaStreamCreateWithFlags(&h.sC, cudaStreamNonBlocking));
        cudaEvent_t ev0 = new_event(h, false);
        CK(cudaEventRecord(ev0, h.sU));                     // (alloc_state's memsets)
        CK(cudaStreamWaitEvent(h.sC, ev0, 0));
        for (int64_t ca = 0; ca < n; ca += chunk) {
            const int64_t cb = std::min<int64_t>(n, ca + chunk);
            CK(cudaMemcpy2DAsync(P_<T>(h.dA) + ca * h.lda, h.lda * sizeof(T), (const T*)A + ca * lda, lda * sizeof(T), m * sizeof(T),
                                 cb - ca, cudaMemcpyHostToDevice, h.sC));
            cudaEvent_t e = new_event(h, false);
            CK(cudaEventRecord(e, h.sC));
            h.arrive.push_back({cb, e});
        }
        return factor_incore<T>(h, P_<T>(h.dA), h.lda);
    }
    // out of core: budget = 2 super-panel buffers + 2 panel stream buffers
    const int64_t lds = round_up(m, 16 / (int64_t)sizeof(T));
    const int64_t col_bytes = lds * (int64_t)sizeof(T);
    int64_t ns = ((int64_t)budget / col_bytes - 2 * h.nb) / 2;
    ns = (ns / h.nb) * h.nb;
    if (ns > round_up(n, h.nb)) ns = round_up(n, h.nb);
    if (ns < h.nb)
        return set_err(CTQR_ERR_NOMEM, "device budget of %zu bytes cannot hold two %d-column super-panels and two "
                       "panel buffers of %lld rows", budget, h.nb, (long long)m);
    CKI(alloc_state<T>(h, std::min<int64_t>(ns, n)));
    return factor_ooc<T>(h, (T*)A, lda, ns);
}

// handle with its options, streams and device properties (shared by ct_qr_factor and ct_qr_load)
static int new_handle(ctqr_dtype_t dtype, int64_t m, int64_t n, const ctqr_options_t& o, H** out) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return set_err(CTQR_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    H* h = new (std::nothrow) H();
    if (!h) return set_err(CTQR_ERR_NOMEM, "host allocation failed");
    memset(&h->st, 0, sizeof h->st);
    h->dtype = dtype; h->w = dtype == CTQR_F64 ? 8 : 4;
    h->m = m; h->n = n;
    h->nb = o.nb > 0 ? o.nb : 128;
    h->ib = o.ib > 0 ? o.ib : 32;
    if (h->ib != 8 && h->ib != 16 && h->ib != 32) { delete h; return set_err(-6, "ib must be 8, 16 or 32"); }
    if (h->nb > 128 || h->nb % h->ib != 0) { delete h; return set_err(-6, "nb must be a multiple of ib and <= 128"); }
    h->lookahead = o.lookahead < 0 ? 1 : (o.lookahead ? 1 : 0);
    h->gemm_impl = o.gemm_impl;
    h->profile = o.profile ? 1 : 0;
    h->reserve_sms = -1;               // SMs left to the look-ahead chain during the bulk update: chosen per panel
    h->trsm_exact = o.trsm_exact ? 1 : 0;
    h->solve_pairs = o.solve_pairs;
    h->P = (int)ceil_div(n, h->nb);
    h->user = (cudaStream_t)o.stream;
    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete h; return set_err(CTQR_ERR_CUDA, "cudaGetDeviceProperties failed"); }
    h->sms = prop.multiProcessorCount;
    int lo = 0, hi = 0; cudaDeviceGetStreamPriorityRange(&lo, &hi);
    if (cudaStreamCreateWithPriority(&h->sU, cudaStreamNonBlocking, lo) != cudaSuccess ||
        cudaStreamCreateWithPriority(&h->sP, cudaStreamNonBlocking, hi) != cudaSuccess) {
        delete h; return set_err(CTQR_ERR_CUDA, "stream creation failed");
    }
    // order after the caller's stream
    if (cudaStreamSynchronize(h->user) != cudaSuccess) { delete h; return set_err(CTQR_ERR_CUDA, "user stream sync failed"); }
    *out = h;
    return 0;
}

extern "C" int ct_qr_factor(void* A, int64_t m, int64_t n, int64_t lda, ctqr_dtype_t dtype,
                            const ctqr_options_t* opt, ctqr_handle_t* out) {
    g_err[0] = 0;
    const bool use_file = opt && opt->file_path && opt->file_path[0];
    if (!A && !use_file) return set_err(-1, "A is NULL");
    if (m < 1) return set_err(-2, "m < 1");
    if (n < 1 || n > m) return set_err(-3, "need 1 <= n <= m");
    if (lda < m) return set_err(-4, "lda < m");
    if (dtype != CTQR_F32 && dtype != CTQR_F64) return set_err(-5, "bad dtype");
    if (!out) return set_err(-7, "out is NULL");
    ctqr_options_t o; memset(&o, 0, sizeof o); o.lookahead = -1;
    if (opt) o = *opt;
    if (o.lower_bandwidth < 0) return set_err(-6, "lower_bandwidth < 0");
    H* h = nullptr;
    CKI(new_handle(dtype, m, n, o, &h));
    h->kl = (o.lower_bandwidth > 0 && o.lower_bandwidth < m - 1) ? o.lower_bandwidth : 0;   // >= m-1: dense
    if (use_file) {
        // file tier: column-major m x n matrix with leading dimension lda at offset 0 of the file
        const size_t need = (size_t)lda * (size_t)n * h->w;
        h->ffd = open(o.file_path, O_RDWR);
        struct stat sb;
        if (h->ffd < 0 || fstat(h->ffd, &sb) != 0 || (size_t)sb.st_size < need) {
            delete h;
            return set_err(CTQR_ERR_IO, "cannot open %s read-write with at least %zu bytes", o.file_path, need);
        }
        void* mp = mmap(nullptr, need, PROT_READ | PROT_WRITE, MAP_SHARED, h->ffd, 0);
        if (mp == MAP_FAILED) { delete h; return set_err(CTQR_ERR_IO, "mmap of %s failed", o.file_path); }
        h->fmap = mp; h->fmap_len = need;
        A = mp;
    }
    const bool on_dev = !use_file && is_device_ptr(A);
    int rc = (dtype == CTQR_F64) ? factor_typed<double>(*h, A, lda, on_dev, o)
                                 : factor_typed<float>(*h, A, lda, on_dev, o);
    if (rc != 0) { cudaDeviceSynchronize(); delete h; return rc; }
    if (h->fmap) msync(h->fmap, h->fmap_len, MS_ASYNC);
    h->st.update_ms = h->st.vtc_ms + h->st.upd_ms;              // opt->profile only
    h->st.panel_ms = h->profile ? h->st.factor_ms - h->st.update_ms : 0.0;   // time not inside the two bulk contractions
    h->st.m = m; h->st.n = n; h->st.nb = h->nb; h->st.ib = h->ib; h->st.n_panels = h->P;
    h->st.n_superpanels = h->n_super; h->st.out_of_core = h->ooc ? 1 : 0; h->st.singular_col = -1;
    h->st.factor_flops = 2.0 * (double)m * (double)n * (double)n - 2.0 * (double)n * (double)n * (double)n / 3.0;
    h->st.lower_bandwidth = h->kl;
    h->st.factor_flops_performed = h->st.factor_flops;
    if (h->kl > 0) {
        // column j: a reflector of r_j = min(m, kl + j + 1) - j rows applied to the n - j - 1 trailing columns
        double fl = 0;
        for (int64_t j = 0; j < n; ++j) fl += 4.0 * (double)(std::min(m, h->kl + j + 1) - j) * (double)(n - j - 1);
        h->st.factor_flops_performed = fl;
    }
    h->st.kernel_launches = h->launches;
    h->factored = true;
    *out = h;
    return 0;
}

// ------------------------------------------------------------------------------------------
// solve: a6 (Q^T B) and a7 (blocked TRSM)
// ------------------------------------------------------------------------------------------
// Pipelined, TMA-fed small-S Q^T B (solve_small2.cuh).  Returns -1000 when the configuration does not fit.
template <typename T>
static int ensure_mt(H& h) {
    const int nb = 128;
    const T* A = P_<T>(h.dA);
    if (!h.gt_ready) {
        // Mt[j] = T_(j-1) (V_(j-1)^T V_j), once per handle: the Gram block over the rows of panel j as stream-K partial
        // tiles summed in a fixed order, then one 128^3 product
        if (!h.dGt) {
            CK(dev_alloc(&h.dGt, (size_t)h.P * nb * nb * sizeof(T)));
            CK(cudaMemsetAsync(h.dGt, 0, (size_t)h.P * nb * nb * sizeof(T), h.sU));
        }
        if (!h.dMerge) CK(dev_alloc(&h.dMerge, (size_t)2 * 128 * 128 * sizeof(T)));
        T* Gs = P_<T>(h.dMerge);
        for (int j = 1; j < h.P; ++j) {
            const int64_t j0 = (int64_t)j * nb;
            const int kw = (int)std::min<int64_t>(nb, h.n - j0);
            GemmArgs<T> g{};
            g.M = nb; g.N = kw; g.K = row_end(h, j0 + kw) - j0; g.A = A + j0 + (j0 - nb) * h.lda; g.lda = h.lda;
            g.B = A + j0 + j0 * h.lda; g.ldb = h.lda;
            g.C = P_<T>(h.dWp[0]); g.ldc = nb; g.alpha = T(1); g.beta = T(0); g.split_stride = (int64_t)nb * nb;
            const GemmLaunch LG = gemm_plan<T>(true, nb, kw, g.K, h.gemm_impl, h.sms, true, (int64_t)h.wp_elems[0],
                                                    g.split_stride, gemm_aligned(g));
            if (LG.kind != 1) return -1000;
            CK(gemm_run<T>(true, g, LG, h.gemm_impl, h.sU));
            CK(partial_sum_launch<T>(P_<T>(h.dWp[0]), LG.seg, nb, kw, Gs, nb, h.sU));
            GemmArgs<T> g2{};
            g2.M = nb; g2.N = kw; g2.K = nb; g2.A = P_<T>(h.dT) + (size_t)(j - 1) * nb * nb; g2.lda = nb; g2.B = Gs; g2.ldb = nb;
            g2.C = P_<T>(h.dGt) + (size_t)j * nb * nb; g2.ldc = nb; g2.alpha = T(1); g2.beta = T(0);
            CK(gemm_direct<T>(false, g2, h.gemm_impl, h.sms, h.sU));
            h.launches += 3;
        }
        h.gt_ready = true;
    }
    return 0;
}

template <typename T>
static int apply_qt_small2(H& h, T* C, int64_t ldc, int64_t S) {
    const int nb = 128;
    const T* A = P_<T>(h.dA);
    { const int rcm = ensure_mt<T>(h); if (rcm) return rcm; }
    const int64_t nch = ceil_div(h.m, (int64_t)Qt2Chunk<T>::value);
    const int G = (int)std::min<int64_t>(h.sms, nch);
    SmallQt2Args<T> a{};
    a.A = A; a.lda = h.lda; a.m = h.m; a.n = h.n; a.P = h.P; a.Tm = P_<T>(h.dT); a.Mt = P_<T>(h.dGt);
    a.B = C; a.ldb = ldc; a.S = (int)S;
    a.part = reinterpret_cast<uint4*>(h.dLLs);
    a.sums = a.part + (size_t)2 * h.sms * nb * kSmallS;
    a.seq_base = h.ll_seq; h.ll_seq += (unsigned)h.P;
    a.rpc = (int)ceil_div(nch, (int64_t)G) * Qt2Chunk<T>::value;
    a.kl = h.kl;
    // (the update pass has 8 boxes in work at a time, one per warp pair: fewer than 8 stages would let a warp wait for a
    // box two ring turns ahead, which the parity test of an mbarrier cannot tell from the turn before)
    int ns = 10;
    while (ns > 8 && qt2_smem_bytes<T>(a.rpc, ns) > 225 * 1024) --ns;
    const size_t smem = qt2_smem_bytes<T>(a.rpc, ns);
    if (smem > 225 * 1024) return -1000;
    a.nstage = ns;
    CUtensorMap mapV;
    if (tma::map_2d(&mapV, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, (int)sizeof(T), A, h.m, h.n, h.lda, Qt2Chunk<T>::value, 128, CU_TENSOR_MAP_SWIZZLE_128B) != cudaSuccess)
        return -1000;
    static SmemAttr attr;
    CK(ensure_dyn_smem(apply_qt_small2_kernel<T>, smem, attr));
    void* args[] = {(void*)&mapV, (void*)&a};
    CK(cudaLaunchCooperativeKernel((void*)apply_qt_small2_kernel<T>, dim3(G), dim3(kQt2Threads), args, smem, h.sU));
    h.launches += 1;
#ifdef CTQR_SMALL_PROFILE
    {
        unsigned long long ph[16] = {0}, zero[16] = {0};
        cudaStreamSynchronize(h.sU);
        cudaMemcpyFromSymbol(ph, g_small_prof, sizeof(ph));
        cudaMemcpyToSymbol(g_small_prof, zero, sizeof(zero));
        for (int i = 0; i <= 5; ++i) fprintf(stderr, "ph%d %.2f  ", i, ph[i] * 1e-3 / h.P);
        fprintf(stderr, "us/panel (1 gather, 2 reduce, 3 T^T W, 4 update, 5 pass A)\n");
    }
#endif
    return 0;
}

// ------------------------------------------------------------------------------------------
// Medium-S Q^T B (solve_mid.cuh, fp64): the pipelined kernel with NG groups of eight right-hand sides, applied in column
// chunks of 8 NG.  Returns -1000 when the configuration does not fit (shared memory) or more than two chunks are needed.
constexpr int kMidMaxS = 64;
constexpr int64_t kPairTrsmMinS = 512;     // blocked TRSM two diagonal blocks at a time from this many right-hand sides on (n >= 32768)
constexpr int64_t kPairSolveMinS = 512;    // Q^T B two panels at a time from this many right-hand sides on (tall matrices; twice that otherwise)
template <int NG>
static int apply_qt_mid_launch(H& h, double* C, int64_t ldc, int S, int G, int rpc, int ns) {
    const int nb = 128, SM = MidCfg<NG>::SM;
    SmallQt2Args<double> a{};
    a.A = P_<double>(h.dA); a.lda = h.lda; a.m = h.m; a.n = h.n; a.P = h.P; a.Tm = P_<double>(h.dT); a.Mt = P_<double>(h.dGt);
    a.B = C; a.ldb = ldc; a.S = S;
    a.part = reinterpret_cast<uint4*>(h.dLLm);
    a.sums = a.part + (size_t)2 * h.sms * nb * SM;
    a.seq_base = h.ll_seq; h.ll_seq += (unsigned)h.P;
    a.rpc = rpc; a.kl = h.kl; a.nstage = ns;
    CUtensorMap mapV;
    if (tma::map_2d(&mapV, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, a.A, h.m, h.n, h.lda, Qt2Chunk<double>::value, 128, CU_TENSOR_MAP_SWIZZLE_128B) != cudaSuccess)
        return -1000;
    const size_t smem = qt_mid_smem_bytes<NG>(rpc, ns);
    static SmemAttr attr;
    CK(ensure_dyn_smem(apply_qt_mid_kernel<NG>, smem, attr));
    void* args[] = {(void*)&mapV, (void*)&a};
    CK(cudaLaunchCooperativeKernel((void*)apply_qt_mid_kernel<NG>, dim3(G), dim3(kQt2Threads), args, smem, h.sU));
    h.launches += 1;
#ifdef CTQR_SMALL_PROFILE
    {
        unsigned long long ph[16] = {0}, zero[16] = {0};
        cudaStreamSynchronize(h.sU);
        cudaMemcpyFromSymbol(ph, g_small_prof, sizeof(ph));
        cudaMemcpyToSymbol(g_small_prof, zero, sizeof(zero));
        for (int i = 0; i <= 5; ++i) fprintf(stderr, "ph%d %.2f  ", i, ph[i] * 1e-3 / h.P);
        fprintf(stderr, "us/panel, NG %d (1 gather, 2 reduce, 3 T^T W, 4 update, 5 pass A)\n", NG);
    }
#endif
    return 0;
}

static int apply_qt_mid(H& h, double* C, int64_t ldc, int64_t S) {
    const int nb = 128;
    const int64_t nch = ceil_div(h.m, (int64_t)Qt2Chunk<double>::value);
    const int G = (int)std::min<int64_t>(h.sms, nch);
    const int rpc = (int)ceil_div(nch, (int64_t)G) * Qt2Chunk<double>::value;
    const size_t cap = 225 * 1024;
    // ring depth: as many stages as fit, at least the number of boxes the update pass has in work at a time
    auto stages = [&](auto bytes, int lo) { int ns = 8; while (ns > lo && bytes(ns) > cap) --ns; return bytes(ns) <= cap ? ns : 0; };
    const int ns4 = stages([&](int ns) { return qt_mid_smem_bytes<4>(rpc, ns); }, qt_mid_min_stages<4>());
    const int ns2 = stages([&](int ns) { return qt_mid_smem_bytes<2>(rpc, ns); }, qt_mid_min_stages<2>());
    const int chunk = (ns4 && S > 16) ? 32 : 16;            // columns per launch
    if (chunk == 16 && !ns2) return -1000;
    if (ceil_div(S, (int64_t)chunk) > 2) return -1000;
    { const int rcm = ensure_mt<double>(h); if (rcm) return rcm; }
    if (!h.dLLm) {
        const size_t bytes = ((size_t)2 * h.sms + 2) * nb * 32 * 16;      // sized for 32 columns per launch
        CK(dev_alloc(&h.dLLm, bytes));
        CK(cudaMemsetAsync(h.dLLm, 0, bytes, h.sU));
    }
    for (int64_t s0 = 0; s0 < S; s0 += chunk) {
        const int sc = (int)std::min<int64_t>(chunk, S - s0);
        const int rc = (chunk == 32 && sc > 16) ? apply_qt_mid_launch<4>(h, C + s0 * ldc, ldc, sc, G, rpc, ns4)
                                                : apply_qt_mid_launch<2>(h, C + s0 * ldc, ldc, sc, G, rpc, ns2);
        if (rc) return rc;
    }
    return 0;
}

template <typename T>
static int apply_qt_dev(H& h, T* C, int64_t ldc, int64_t S) {
    h.st.apply_qt_path = h.ooc ? 3 : 0;
    if (h.ooc) {
        // factor on the host: stream V_k through the double buffer (sC) against the larfb on sU
        const T* hA = P_<T>(h.hA);
        for (int k = 0; k < h.P; ++k) {
            const int64_t j0 = (int64_t)k * h.nb;
            const int nbw = (int)std::min<int64_t>(h.nb, h.n - j0);
            const int slot = k & 1;
            const int64_t mk = row_end(h, j0 + nbw) - j0;
            CKI(stream_panel_in<T>(h, slot, hA + j0 + j0 * h.hlda, h.hlda, mk, nbw));
            CKI(wait_copy(h, h.sU, h.evVin[slot]));
            CKI(larfb<T>(h, 0, h.sU, P_<T>(h.dVb[slot]), h.ldvb, mk, nbw,
                         P_<T>(h.dT) + (size_t)k * h.nb * h.nb, h.nb, C + j0, ldc, S));
            CK(cudaEventRecord(h.evVfree[slot], h.sU));
        }
        return 0;
    }
    const T* A = P_<T>(h.dA);
    if (S <= kSmallS && h.dLLs && h.gemm_impl == 0 && h.nb == 128 && (h.lda * sizeof(T)) % 16 == 0 && ((uintptr_t)A % 16) == 0 && h.P >= 2) {
        int rc2 = apply_qt_small2<T>(h, C, ldc, S);
        if (rc2 != -1000) { h.st.apply_qt_path = 2; return rc2; }   // -1000: does not fit (shared memory); fall through
    }
    if constexpr (sizeof(T) == 8) {
        if (S > kSmallS && S <= kMidMaxS && h.dLLs && h.gemm_impl == 0 && h.nb == 128 && (h.lda * sizeof(T)) % 16 == 0 &&
            ((uintptr_t)A % 16) == 0 && h.P >= 2) {
            int rc2 = apply_qt_mid(h, C, ldc, S);
            if (rc2 != -1000) { h.st.apply_qt_path = 4; return rc2; }
        }
    }
    if (S <= kSmallS && h.dLLs && h.gemm_impl == 0) {
        // memory-bound regime: one cooperative kernel for all panels (solve_small.cuh)
        SmallQtArgs<T> a{};
        const int64_t nch = ceil_div(h.m, (int64_t)kSmallChunk);
        const int G = (int)std::min<int64_t>(h.sms, nch);
        a.A = A; a.lda = h.lda; a.m = h.m; a.n = h.n; a.nb = h.nb; a.P = h.P; a.Tm = P_<T>(h.dT);
        a.B = C; a.ldb = ldc; a.S = (int)S;
        a.part = reinterpret_cast<uint4*>(h.dLLs);
        a.sums = a.part + (size_t)2 * h.sms * h.nb * kSmallS;
        a.seq_base = h.ll_seq; h.ll_seq += (unsigned)h.P;
        a.rpc = (int)ceil_div(nch, (int64_t)G) * kSmallChunk;
        a.kl = h.kl;
        const size_t smem = ((size_t)h.nb * SmallLd<T>::T_ + 2 * (size_t)h.nb * SmallLd<T>::W + (size_t)kSmallS * (a.rpc + 4)) * sizeof(T);
        if (smem <= 220 * 1024) {
            static SmemAttr attr;
            CK(ensure_dyn_smem(apply_qt_small_kernel<T>, smem, attr));
            void* args[] = {(void*)&a};
            CK(cudaLaunchCooperativeKernel((void*)apply_qt_small_kernel<T>, dim3(G), dim3(kSmallThreads), args, smem, h.sU));
            h.launches += 1;
            h.st.apply_qt_path = 1;
#ifdef CTQR_SMALL_PROFILE
            {
                unsigned long long ph[16] = {0}, zero[16] = {0};
                cudaStreamSynchronize(h.sU);
                cudaMemcpyFromSymbol(ph, g_small_prof, sizeof(ph));
                cudaMemcpyToSymbol(g_small_prof, zero, sizeof(zero));
                for (int i = 1; i <= 8; ++i) fprintf(stderr, "ph%d %.2f  ", i, ph[i] * 1e-3 / h.P);
                fprintf(stderr, "us/panel\n");
            }
#endif
            return 0;
        }
    }
    // Many right-hand sides: two panels at a time, as the factorisation's trailing updates (K = 256 updates; fp32:
    // pre-split TMA-fed operands).  The off-diagonal block of a pair's merged T factor, -T_k (V_k^T V_k+1) T_k+1, was kept
    // by the factorisation's own merge of that pair (no set-up cost here); T2 is assembled per pair from it and the two
    // panel factors.  Pairs the factorisation did not merge (its narrow tail, out-of-core or loaded handles) take one
    // panel at a time.
    // (measured, both precisions: a gain from S = 1024 at configs[2], from S = 512 at configs[3]; a loss of 3-16 % below)
    const bool psize = h.solve_pairs > 0 ? S >= 256
                                         : (h.solve_pairs == 0 && (S >= 2 * kPairSolveMinS || (S >= kPairSolveMinS && h.m >= 65536)));
    const bool pairs = psize && h.nb == 128 && h.gemm_impl == 0 &&
                       h.P >= 2 && h.dT12 && (h.lda * sizeof(T)) % 16 == 0 && ((uintptr_t)A % 16) == 0 &&
                       ((uintptr_t)C % 16) == 0 && (ldc * sizeof(T)) % 16 == 0 &&
                       ensure_pair_ws<T>(h, std::max<int64_t>(S, 1024)) == 0;
    for (int k = 0; k < h.P; ++k) {
        const int64_t j0 = (int64_t)k * h.nb;
        const int nbw = (int)std::min<int64_t>(h.nb, h.n - j0);
        if (pairs && k + 1 < h.P && (k & 1) == 0 && (size_t)(k / 2) < h.t12_have.size() && h.t12_have[k / 2]) {
            const int nb = 128, slot = (k >> 1) & 1;
            const int64_t me = row_end(h, j0 + 2 * nb);
            T* T2 = P_<T>(h.dT2) + (size_t)slot * 256 * 256;
            const T* Tk = P_<T>(h.dT) + (size_t)k * nb * nb;
            CK(copy2d_launch<T>(Tk, nb, T2, 256, nb, nb, h.sU));
            CK(copy2d_launch<T>(Tk + (size_t)nb * nb, nb, T2 + nb + (size_t)nb * 256, 256, nb, nb, h.sU));
            CK(copy2d_launch<T>(P_<T>(h.dT12) + (size_t)(k / 2) * nb * nb, nb, T2 + (size_t)nb * 256, 256, nb, nb, h.sU));
            h.launches += 3;
            if constexpr (sizeof(T) == 4) {
                if (h.dVs[slot]) {
                    float* hi = P_<float>(h.dVs[slot]);
                    CK(split_tf32_launch(A + j0 + j0 * h.lda, h.lda, me - j0, 2 * nb, hi, hi + (size_t)h.ldvs * 256, h.ldvs, h.sU));
                    h.launches += 1;
                }
            }
            CKI(larfb_pair<T>(h, h.sU, A, h.lda, me, j0, slot, C + j0, ldc, S, 0, 256));
            h.st.apply_qt_path = 5;
            ++k;
            continue;
        }
        CKI(larfb<T>(h, 0, h.sU, A + j0 + j0 * h.lda, h.lda, row_end(h, j0 + nbw) - j0, nbw,
                     P_<T>(h.dT) + (size_t)k * h.nb * h.nb, h.nb, C + j0, ldc, S));
    }
    return 0;
}

// Common preamble of the triangular solves: refuse a singular R, build the inverted diagonal blocks once per handle.
// Diagonal tasks X_i = R_ii^{-1} C_i: by default a product with the explicitly inverted 128 x 128 diagonal
// block (inverted once per handle, by back-substitution on the identity, working precision), which turns 128
// dependent steps per right-hand side into one small contraction.  The off-diagonal part of R^{-1} is never
// formed.  A product with an explicit inverse is only conditionally backward stable, so the
// back-substitution kernel is used instead when opt->trsm_exact is set, or when some diagonal block looks
// ill-conditioned: max|R_jj| / min|R_jj| inside the block (a lower bound of its condition number) above
// 1/sqrt(eps) of the working type.
template <typename T>
static int trsm_prepare(H& h) {
    CK(cudaMemsetAsync(h.dFlag, 0x7f, sizeof(int), h.sU));
    CK(find_zero_diag_launch<T>(P_<T>(h.dRd), h.nb, h.n, h.dFlag, h.sU));
    int flag = 0;
    CK(cudaMemcpyAsync(&flag, h.dFlag, sizeof(int), cudaMemcpyDeviceToHost, h.sU));
    CK(cudaStreamSynchronize(h.sU));
    if (flag < h.n) { h.st.singular_col = flag; return set_err(CTQR_ERR_SINGULAR, "R[%d,%d] == 0", flag, flag); }
    if (!h.trsm_exact && h.dRinv && !h.rinv_ready) {
        CK(cudaMemsetAsync(h.dFlag, 0, sizeof(int), h.sU));
        CK(trinv_launch<T>(P_<T>(h.dRd), h.nb, h.n, h.P, P_<T>(h.dRinv), reinterpret_cast<unsigned*>(h.dFlag), h.sU));
        unsigned bits = 0;
        CK(cudaMemcpyAsync(&bits, h.dFlag, sizeof(unsigned), cudaMemcpyDeviceToHost, h.sU));
        CK(cudaStreamSynchronize(h.sU));
        float ratio; memcpy(&ratio, &bits, sizeof ratio);
        h.st.diag_block_cond = ratio;
        h.rinv_ready = true;
        h.launches += 1;
        if (!(ratio <= (sizeof(T) == 8 ? 6.7e7f : 2.9e3f))) h.trsm_exact = 2;      // also catches NaN
    }
    h.st.trsm_exact = h.trsm_exact;
    return 0;
}

template <typename T>
static int trsm_dev(H& h, T* X, int64_t ldx, int64_t S) {
    // X holds C[0:n,:] on entry.  Bottom-up over diagonal blocks:
    //   R_ii X_i = C_i ;  C_j <- C_j - R_ji X_i  for all j < i (one GEMM over rows 0..i0)
    CKI(trsm_prepare<T>(h));
    const bool exact = h.trsm_exact != 0;
    const bool use_inv = !exact && h.dRinv && ldx % (16 / (int64_t)sizeof(T)) == 0;
    // (up to 2 * kSmallS right-hand sides: two launches of the fused kernel read R twice and still beat 2 P launches)
    if (S <= 2 * kSmallS && h.dLLs && h.rinv_ready && !exact && !h.ooc && h.gemm_impl == 0 && h.nb == 128 && h.P >= 2) {
        // memory-bound regime, pipelined: one grid hop per diagonal block (solve_small2.cuh)
        const int nb = 128;
        if (!h.nm_ready) {
            const size_t slots = (size_t)4 * nb * kSmallS * 16;
            if (!h.dNm) CK(dev_alloc(&h.dNm, (size_t)h.P * nb * nb * sizeof(T)));
            if (!h.dLLt) { CK(dev_alloc(&h.dLLt, slots)); CK(cudaMemsetAsync(h.dLLt, 0, slots, h.sU)); }
            CK(cudaMemsetAsync(h.dNm, 0, (size_t)h.P * nb * nb * sizeof(T), h.sU));
            for (int i = 0; i + 1 < h.P; ++i) {
                const int64_t i0 = (int64_t)i * nb;
                GemmArgs<T> gn{};
                gn.M = nb; gn.N = std::min<int64_t>(nb, h.n - i0 - nb); gn.K = nb;
                gn.A = P_<T>(h.dRinv) + (size_t)i * nb * nb; gn.lda = nb;
                gn.B = P_<T>(h.dA) + i0 + (i0 + nb) * h.lda; gn.ldb = h.lda;
                gn.C = P_<T>(h.dNm) + (size_t)i * nb * nb; gn.ldc = nb; gn.alpha = T(1); gn.beta = T(0);
                CK(gemm_direct<T>(false, gn, h.gemm_impl, h.sms, h.sU));
            }
            h.launches += h.P - 1;
            h.nm_ready = true;
        }
        SmallTrsm2Args<T> a{};
        const int64_t nch = ceil_div(h.n, (int64_t)kTrsmChunk);
        const int G = (int)std::min<int64_t>(h.sms, nch);
        a.A = P_<T>(h.dA); a.lda = h.lda; a.n = h.n; a.P = h.P; a.Rinv = P_<T>(h.dRinv); a.Nm = P_<T>(h.dNm);
        a.ldx = ldx;
        a.cslots = reinterpret_cast<uint4*>(h.dLLt);
        a.xslots = a.cslots + (size_t)2 * nb * kSmallS;
        a.rpc = (int)ceil_div(nch, (int64_t)G) * kTrsmChunk;
        const size_t smem = ((size_t)nb * kSmallS + (size_t)kSmallS * kTrsmThreads + (size_t)kSmallS * a.rpc) * sizeof(T);
        if (smem <= 220 * 1024) {
            static SmemAttr attr2;
            CK(ensure_dyn_smem(trsm_small2_kernel<T>, smem, attr2));
            for (int64_t s0 = 0; s0 < S; s0 += kSmallS) {
                a.X = X + s0 * ldx; a.S = (int)std::min<int64_t>(kSmallS, S - s0);
                a.seq_base = h.ll_seq; h.ll_seq += (unsigned)h.P;
                void* args[] = {(void*)&a};
                CK(cudaLaunchCooperativeKernel((void*)trsm_small2_kernel<T>, dim3(G), dim3(kTrsmThreads), args, smem, h.sU));
                h.launches += 1;
            }
            return 0;
        }
    }
    if (S <= kSmallS && h.dLLs && h.rinv_ready && !exact && !h.ooc && h.gemm_impl == 0) {
        // memory-bound regime: one cooperative kernel for all diagonal blocks (solve_small.cuh)
        SmallTrsmArgs<T> a{};
        const int64_t nch = ceil_div(h.n, (int64_t)kTrsmChunk);
        const int G = (int)std::min<int64_t>(h.sms, nch);
        a.A = P_<T>(h.dA); a.lda = h.lda; a.n = h.n; a.nb = h.nb; a.P = h.P; a.Rinv = P_<T>(h.dRinv);
        a.X = X; a.ldx = ldx; a.S = (int)S;
        a.slots = reinterpret_cast<uint4*>(h.dLLs) + ((size_t)2 * h.sms + 2) * h.nb * kSmallS;
        a.seq = ++h.ll_seq;
        a.rpc = (int)ceil_div(nch, (int64_t)G) * kTrsmChunk;
        const size_t smem = ((size_t)h.nb * h.nb + 2 * (size_t)h.nb * kSmallS + (size_t)kSmallS * kTrsmThreads +
                             (size_t)kSmallS * a.rpc) * sizeof(T);
        if (smem <= 220 * 1024) {
            static SmemAttr attr;
            CK(ensure_dyn_smem(trsm_small_kernel<T>, smem, attr));
            void* args[] = {(void*)&a};
            CK(cudaLaunchCooperativeKernel((void*)trsm_small_kernel<T>, dim3(G), dim3(kTrsmThreads), args, smem, h.sU));
            h.launches += 1;
            return 0;
        }
    }
    // Large batches, in core: two diagonal blocks per update of the rows above (K = 256; fp32: operands pre-split and fed
    // by TMA, as in the two-panel trailing update): X_i, then C_(i-1) -= R_(i-1,i) X_i, X_(i-1), then one product with the
    // 256 columns of R.  Same task list, two tasks per step.
    // (measured: TRSM 105 -> 95 ms fp64, 50 -> 46 ms fp32 at configs[3], S = 512; a loss of 2-20 % at configs[2])
    const bool tsize = h.solve_pairs > 0 ? S >= 256 : (h.solve_pairs == 0 && S >= kPairTrsmMinS && h.n >= 32768);
    const bool tpairs = !h.ooc && use_inv && h.nb == 128 && h.gemm_impl == 0 && tsize &&
                        ((uintptr_t)X % 16) == 0 && (h.lda * sizeof(T)) % 16 == 0 &&
                        (sizeof(T) == 8 || ensure_pair_ws<T>(h, std::max<int64_t>(S, 1024)) == 0);
    // X_i = R_ii^{-1} C_i in place for a full block (inverted diagonal blocks): mm128_kernel up to 512 right-hand sides,
    // the contraction (out of place, copied back) beyond
    auto diag_inv = [&](int i) -> int {
        const int64_t i0 = (int64_t)i * 128;
        const T* Ri = P_<T>(h.dRinv) + (size_t)i * 128 * 128;
        if (S <= 512) {
            CK(mm128_launch<T>(false, Ri, 128, X + i0, ldx, SegInfo{}, S, X + i0, ldx, h.sU));
            h.launches += 1;
        } else {
            T* W = P_<T>(h.dW[0]);
            GemmArgs<T> gi{};
            gi.M = 128; gi.N = S; gi.K = 128; gi.A = Ri; gi.lda = 128; gi.B = X + i0; gi.ldb = ldx; gi.C = W; gi.ldc = 128;
            gi.alpha = T(1); gi.beta = T(0);
            CK(gemm_direct<T>(false, gi, h.gemm_impl, h.sms, h.sU));
            CK(copy2d_launch<T>(W, 128, X + i0, ldx, 128, S, h.sU));
            h.launches += 2;
        }
        return 0;
    };
    for (int i = h.P - 1; i >= 0; --i) {
        const int64_t i0 = (int64_t)i * h.nb;
        const int nbw = (int)std::min<int64_t>(h.nb, h.n - i0);
        if (tpairs && i >= 2 && nbw == 128) {
            const int nb = 128;
            const int64_t p0 = i0 - nb;                   // first row / column of the pair (blocks i-1, i)
            const T* A = P_<T>(h.dA);
            CKI(diag_inv(i));
            GemmArgs<T> gs{};
            gs.M = nb; gs.N = S; gs.K = nb; gs.A = A + p0 + i0 * h.lda; gs.lda = h.lda; gs.B = X + i0; gs.ldb = ldx;
            gs.C = X + p0; gs.ldc = ldx; gs.alpha = T(-1); gs.beta = T(1);
            CK(gemm_direct<T>(false, gs, h.gemm_impl, h.sms, h.sU));
            CKI(diag_inv(i - 1));
            h.launches += 1;
            bool done = false;
            if constexpr (sizeof(T) == 4) {
                const int slot2 = (i >> 1) & 1;
                if (h.dVs[slot2] && h.dWs && (size_t)2 * 256 * (size_t)S <= h.ws_elems && ldx % 4 == 0 && S % 8 == 0 && p0 <= h.ldvs) {
                    float* vhi = P_<float>(h.dVs[slot2]); float* vlo = vhi + (size_t)h.ldvs * 256;
                    float* whi = P_<float>(h.dWs); float* wlo = whi + (size_t)256 * S;
                    CK(split_tf32_launch(A + p0 * h.lda, h.lda, p0, 2 * nb, vhi, vlo, h.ldvs, h.sU));
                    CK(split_tf32_launch(X + p0, ldx, 256, S, whi, wlo, 256, h.sU));
                    CK(upd_presplit_launch(p0, S, 256, -1.f, vhi, vlo, h.ldvs, whi, wlo, 256, 1.f, X, ldx, h.sms, h.sU));
                    h.launches += 3;
                    done = true;
                }
            }
            if (!done) {
                GemmArgs<T> g{};
                g.M = p0; g.N = S; g.K = 2 * nb; g.A = A + p0 * h.lda; g.lda = h.lda; g.B = X + p0; g.ldb = ldx;
                g.C = X; g.ldc = ldx; g.alpha = T(-1); g.beta = T(1);
                CK(gemm_direct<T>(false, g, h.gemm_impl, h.sms, h.sU));
                h.launches += 1;
            }
            --i;
            continue;
        }
        const T* Rcol = nullptr; int64_t ldr = 0;        // R[0:i0, i0:i0+nbw]
        const int slot = i & 1;
        if (i0 > 0) {
            if (h.ooc) {
                CKI(stream_panel_in<T>(h, slot, P_<T>(h.hA) + i0 * h.hlda, h.hlda, i0, nbw));
                Rcol = P_<T>(h.dVb[slot]); ldr = h.ldvb;
            } else { Rcol = P_<T>(h.dA) + i0 * h.lda; ldr = h.lda; }
        }
        const T* Xi = X + i0; int64_t ldxi = ldx;         // where the update below reads X_i
        if (use_inv && nbw == 128 && h.nb == 128 && S <= 512) {
            // X_i = R_ii^{-1} C_i in place, one CTA per 8 right-hand sides (small.cuh mm128_kernel)
            CK(mm128_launch<T>(false, P_<T>(h.dRinv) + (size_t)i * h.nb * h.nb, h.nb, X + i0, ldx, SegInfo{}, S, X + i0, ldx, h.sU));
            h.launches += 1;
        } else if (use_inv) {
            // X_i = R_ii^{-1} C_i as a contraction (out of place into W, copied back over C_i)
            T* W = P_<T>(h.dW[0]);
            GemmArgs<T> gi{};
            gi.M = nbw; gi.N = S; gi.K = nbw; gi.A = P_<T>(h.dRinv) + (size_t)i * h.nb * h.nb; gi.lda = h.nb;
            gi.B = X + i0; gi.ldb = ldx; gi.C = W; gi.ldc = h.nb; gi.alpha = T(1); gi.beta = T(0);
            CK(gemm_direct<T>(false, gi, h.gemm_impl, h.sms, h.sU));
            CK(copy2d_launch<T>(W, h.nb, X + i0, ldx, nbw, S, h.sU));
            Xi = W; ldxi = h.nb;
            h.launches += 2;
        } else {
            CK(trsm_diag_launch<T>(P_<T>(h.dRd) + (size_t)i * h.nb * h.nb, h.nb, nbw, X + i0, ldx, S, X + i0, ldx, h.sU));
            h.launches += 1;
        }
        if (i0 > 0) {
            if (h.ooc) CKI(wait_copy(h, h.sU, h.evVin[slot]));
            GemmArgs<T> g{};
            g.M = i0; g.N = S; g.K = nbw; g.A = Rcol; g.lda = ldr; g.B = Xi; g.ldb = ldxi;
            g.C = X; g.ldc = ldx; g.alpha = T(-1); g.beta = T(1);
            CK(gemm_direct<T>(false, g, h.gemm_impl, h.sms, h.sU));
            h.launches += 1;
            if (h.ooc) CK(cudaEventRecord(h.evVfree[slot], h.sU));
        }
    }
    return 0;
}

// X <- R^{-T} C: forward substitution with the transposed factor, top-down over the diagonal blocks,
//   Y_i = R_ii^{-T} C_i ;  C[i0+nb:, :] <- C[i0+nb:, :] - R[i0:i0+nb, i0+nb:n]^T Y_i
// (the same task list as PAPER.md:L62-73 read for R^T; used by the semi-normal-equations refinement
// ct_qr_solve_refined).  In-core factors only.
template <typename T>
static int trsm_t_dev(H& h, T* X, int64_t ldx, int64_t S) {
    if (h.ooc) return set_err(CTQR_ERR_STATE, "the transposed triangular solve needs an in-core factor");
    CKI(trsm_prepare<T>(h));
    const bool use_inv = h.trsm_exact == 0 && h.dRinv && h.rinv_ready;
    T* W = P_<T>(h.dW[0]);
    for (int i = 0; i < h.P; ++i) {
        const int64_t i0 = (int64_t)i * h.nb;
        const int nbw = (int)std::min<int64_t>(h.nb, h.n - i0);
        if (use_inv) {
            GemmArgs<T> gi{};
            gi.M = nbw; gi.N = S; gi.K = nbw; gi.A = P_<T>(h.dRinv) + (size_t)i * h.nb * h.nb; gi.lda = h.nb;
            gi.B = X + i0; gi.ldb = ldx; gi.C = W; gi.ldc = h.nb; gi.alpha = T(1); gi.beta = T(0);
            CK(gemm_direct<T>(true, gi, h.gemm_impl, h.sms, h.sU));
            CK(copy2d_launch<T>(W, h.nb, X + i0, ldx, nbw, S, h.sU));
            h.launches += 2;
        } else {
            CK(trsm_diag_t_launch<T>(P_<T>(h.dRd) + (size_t)i * h.nb * h.nb, h.nb, nbw, X + i0, ldx, S, h.sU));
            h.launches += 1;
        }
        const int64_t rest = h.n - i0 - nbw;
        if (rest > 0) {
            GemmArgs<T> g{};
            g.M = rest; g.N = S; g.K = nbw; g.A = P_<T>(h.dA) + i0 + (i0 + nbw) * h.lda; g.lda = h.lda;
            g.B = X + i0; g.ldb = ldx; g.C = X + i0 + nbw; g.ldc = ldx; g.alpha = T(-1); g.beta = T(1);
            CK(gemm_direct<T>(true, g, h.gemm_impl, h.sms, h.sU));
            h.launches += 1;
        }
    }
    return 0;
}

// stage an m x S host or device matrix into a fresh device buffer (ld = rows rounded up)
template <typename T>
static int stage_in(H& h, const void* src, int64_t lds, int64_t rows, int64_t S, T** out, int64_t* ldo, bool* owned) {
    if (is_device_ptr(src)) { *owned = false; *out = nullptr; *ldo = lds; return 0; }
    const int64_t ld = round_up(rows, 16 / sizeof(T));
    T* d = nullptr;
    CK(cudaMalloc(&d, (size_t)ld * S * sizeof(T)));
    cudaError_t e = cudaMemcpy2DAsync(d, ld * sizeof(T), src, lds * sizeof(T), rows * sizeof(T), S, cudaMemcpyHostToDevice, h.sU);
    if (e != cudaSuccess) { cudaFree(d); return set_err(CTQR_ERR_CUDA, "H2D copy failed: %s", cudaGetErrorString(e)); }
    h.st.h2d_bytes += (double)rows * S * sizeof(T);
    *out = d; *ldo = ld; *owned = true;
    return 0;
}

template <typename T>
static int solve_typed(H& h, const void* B, int64_t ldb, int64_t S, void* X, int64_t ldx, int mode) {
    // mode 0: full solve; 1: apply Q^T in place on B (B is also the output); 2: trsm only (B = C); 3: X = R^{-T} C
    CKI(ensure_solve_ws(h, S));
    h.launches = 0; h.st.h2d_bytes = 0; h.st.d2h_bytes = 0;
    if (!h.evS[0])
        for (int i = 0; i < 3; ++i)
            if (!(h.evS[i] = new_event(h, true))) { h.evS[0] = nullptr; return set_err(CTQR_ERR_CUDA, "cudaEventCreate failed"); }
    cudaEvent_t t0 = h.evS[0], t1 = h.evS[1], t2 = h.evS[2];
    const int64_t m = h.m, n = h.n;
    const int64_t rows_in = (mode >= 2) ? n : m;
    // working buffer Cw (rows_in x S) on the device
    const int64_t ldw = round_up(rows_in, 16 / sizeof(T));
    T* Cw = nullptr;
    bool inplace_dev = (mode == 1) && is_device_ptr(B);
    if (inplace_dev) { Cw = (T*)B; }
    else {
        const size_t need = (size_t)ldw * S * sizeof(T);
        if (need > h.cw_bytes) {                           // kept by the handle: later batches of the same size allocate nothing
            dev_free(h.dCw); h.dCw = nullptr; h.cw_bytes = 0;
            if (dev_alloc(&h.dCw, need) != cudaSuccess) { cudaGetLastError(); return set_err(CTQR_ERR_NOMEM, "cannot allocate %zu bytes for the right-hand sides", need); }
            h.cw_bytes = need;
        }
        Cw = P_<T>(h.dCw);
        const bool bdev = is_device_ptr(B);
        cudaError_t e = cudaMemcpy2DAsync(Cw, ldw * sizeof(T), B, ldb * sizeof(T), rows_in * sizeof(T), S,
                                          bdev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h.sU);
        if (e != cudaSuccess) return set_err(CTQR_ERR_CUDA, "copy of B failed: %s", cudaGetErrorString(e));
        if (!bdev) h.st.h2d_bytes += (double)rows_in * S * sizeof(T);
    }
    const int64_t ldcw = inplace_dev ? ldb : ldw;
    int rc = 0;
    cudaEventRecord(t0, h.sU);
    if (mode < 2) rc = apply_qt_dev<T>(h, Cw, ldcw, S);
    cudaEventRecord(t1, h.sU);
    if (rc == 0 && mode != 1) rc = mode == 3 ? trsm_t_dev<T>(h, Cw, ldcw, S) : trsm_dev<T>(h, Cw, ldcw, S);
    cudaEventRecord(t2, h.sU);
    if (rc == 0) {
        if (mode == 1) {
            if (!inplace_dev) {
                cudaError_t e = cudaMemcpy2DAsync((void*)B, ldb * sizeof(T), Cw, ldw * sizeof(T), m * sizeof(T), S,
                                                  cudaMemcpyDeviceToHost, h.sU);
                if (e != cudaSuccess) rc = set_err(CTQR_ERR_CUDA, "D2H copy failed: %s", cudaGetErrorString(e));
                h.st.d2h_bytes += (double)m * S * sizeof(T);
            }
        } else {
            const bool xdev = is_device_ptr(X);
            cudaError_t e = cudaMemcpy2DAsync(X, ldx * sizeof(T), Cw, ldcw * sizeof(T), n * sizeof(T), S,
                                              xdev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h.sU);
            if (e != cudaSuccess) rc = set_err(CTQR_ERR_CUDA, "copy of X failed: %s", cudaGetErrorString(e));
            if (!xdev) h.st.d2h_bytes += (double)n * S * sizeof(T);
        }
    }
    cudaError_t es = cudaStreamSynchronize(h.sU);
    if (h.sC) { cudaError_t ec = cudaStreamSynchronize(h.sC); if (es == cudaSuccess) es = ec; }
    if (rc == 0 && es != cudaSuccess) rc = set_err(CTQR_ERR_CUDA, "solve failed: %s", cudaGetErrorString(es));
    if (rc == 0) {
        float a = 0, b = 0;
        cudaEventElapsedTime(&a, t0, t1); cudaEventElapsedTime(&b, t1, t2);
        h.st.apply_qt_ms = a; h.st.trsm_ms = b; h.st.solve_ms = a + b;
        h.st.kernel_launches = h.launches;
    }
    if (h.ooc) resolve_copy_spans(h);          // exposed / busy copy time of the streamed solve
    return rc;
}

static int check_handle(ctqr_handle_t h) {
    if (!h) return set_err(-1, "handle is NULL");
    if (!h->factored) return set_err(CTQR_ERR_STATE, "handle holds no factorisation");
    return 0;
}

extern "C" int ct_qr_solve(ctqr_handle_t h, const void* B, int64_t ldb, int64_t S, void* X, int64_t ldx) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!B) return set_err(-2, "B is NULL");
    if (ldb < h->m) return set_err(-3, "ldb < m");
    if (S < 0) return set_err(-4, "S < 0");
    if (!X) return set_err(-5, "X is NULL");
    if (ldx < h->n) return set_err(-6, "ldx < n");
    if (S == 0) return 0;
    if (cudaStreamSynchronize(h->user) != cudaSuccess) return set_err(CTQR_ERR_CUDA, "user stream sync failed");
    return h->dtype == CTQR_F64 ? solve_typed<double>(*h, B, ldb, S, X, ldx, 0)
                                : solve_typed<float>(*h, B, ldb, S, X, ldx, 0);
}

extern "C" int ct_qr_apply_qt(ctqr_handle_t h, void* C, int64_t ldc, int64_t S) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!C) return set_err(-2, "C is NULL");
    if (ldc < h->m) return set_err(-3, "ldc < m");
    if (S < 0) return set_err(-4, "S < 0");
    if (S == 0) return 0;
    if (cudaStreamSynchronize(h->user) != cudaSuccess) return set_err(CTQR_ERR_CUDA, "user stream sync failed");
    return h->dtype == CTQR_F64 ? solve_typed<double>(*h, C, ldc, S, nullptr, 0, 1)
                                : solve_typed<float>(*h, C, ldc, S, nullptr, 0, 1);
}

extern "C" int ct_qr_trsm_t(ctqr_handle_t h, const void* C, int64_t ldc, int64_t S, void* X, int64_t ldx) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!C) return set_err(-2, "C is NULL");
    if (ldc < h->n) return set_err(-3, "ldc < n");
    if (S < 0) return set_err(-4, "S < 0");
    if (!X) return set_err(-5, "X is NULL");
    if (ldx < h->n) return set_err(-6, "ldx < n");
    if (S == 0) return 0;
    if (cudaStreamSynchronize(h->user) != cudaSuccess) return set_err(CTQR_ERR_CUDA, "user stream sync failed");
    return h->dtype == CTQR_F64 ? solve_typed<double>(*h, C, ldc, S, X, ldx, 3)
                                : solve_typed<float>(*h, C, ldc, S, X, ldx, 3);
}

extern "C" int ct_qr_trsm(ctqr_handle_t h, const void* C, int64_t ldc, int64_t S, void* X, int64_t ldx) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!C) return set_err(-2, "C is NULL");
    if (ldc < h->n) return set_err(-3, "ldc < n");
    if (S < 0) return set_err(-4, "S < 0");
    if (!X) return set_err(-5, "X is NULL");
    if (ldx < h->n) return set_err(-6, "ldx < n");
    if (S == 0) return 0;
    if (cudaStreamSynchronize(h->user) != cudaSuccess) return set_err(CTQR_ERR_CUDA, "user stream sync failed");
    return h->dtype == CTQR_F64 ? solve_typed<double>(*h, C, ldc, S, X, ldx, 2)
                                : solve_typed<float>(*h, C, ldc, S, X, ldx, 2);
}

// ------------------------------------------------------------------------------------------
// accessors
// ------------------------------------------------------------------------------------------
template <typename T>
static int copy_out(H& h, const T* dsrc, int64_t lds, void* dst, int64_t ldd, int64_t rows, int64_t cols) {
    const bool ddev = is_device_ptr(dst);
    CK(cudaMemcpy2DAsync(dst, ldd * sizeof(T), dsrc, lds * sizeof(T), rows * sizeof(T), cols,
                         ddev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h.sU));
    CK(cudaStreamSynchronize(h.sU));
    return 0;
}

template <typename T>
static int get_R_typed(H& h, void* R, int64_t ldr) {
    const int64_t n = h.n;
    T* tmp = nullptr;
    CK(big_alloc((void**)&tmp, (size_t)n * n * sizeof(T)));
    cudaError_t e = gather_R_launch<T>(P_<T>(h.dA), h.lda, P_<T>(h.dRd), h.nb, n, tmp, n, h.sU);
    int rc = 0;
    if (e != cudaSuccess) rc = set_err(CTQR_ERR_CUDA, "gather_R failed: %s", cudaGetErrorString(e));
    if (rc == 0) rc = copy_out<T>(h, tmp, n, R, ldr, n, n);
    cudaFree(tmp);
    return rc;
}

// out-of-core factor: off-diagonal blocks of R sit in the host matrix, diagonal blocks in dRd
template <typename T>
static int get_R_ooc(H& h, void* R, int64_t ldr) {
    const int64_t n = h.n; const int nb = h.nb;
    std::vector<T> rd((size_t)h.P * nb * nb), tmp((size_t)n * n, T(0));
    CK(cudaMemcpy(rd.data(), h.dRd, rd.size() * sizeof(T), cudaMemcpyDeviceToHost));
    const T* hA = P_<T>(h.hA);
    for (int64_t c = 0; c < n; ++c) {
        const int64_t pc = c / nb, p0 = pc * nb;
        for (int64_t r = 0; r < p0; ++r) tmp[r + c * n] = hA[r + c * h.hlda];
        for (int64_t r = p0; r <= c; ++r) tmp[r + c * n] = rd[(size_t)pc * nb * nb + (r - p0) + (c - p0) * (int64_t)nb];
    }
    CK(cudaMemcpy2D(R, ldr * sizeof(T), tmp.data(), n * sizeof(T), n * sizeof(T), n,
                    is_device_ptr(R) ? cudaMemcpyHostToDevice : cudaMemcpyHostToHost));
    return 0;
}

extern "C" int ct_qr_get_R(ctqr_handle_t h, void* R, int64_t ldr) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!R) return set_err(-2, "R is NULL");
    if (ldr < h->n) return set_err(-3, "ldr < n");
    if (h->ooc) return h->dtype == CTQR_F64 ? get_R_ooc<double>(*h, R, ldr) : get_R_ooc<float>(*h, R, ldr);
    return h->dtype == CTQR_F64 ? get_R_typed<double>(*h, R, ldr) : get_R_typed<float>(*h, R, ldr);
}

extern "C" int ct_qr_get_V(ctqr_handle_t h, int64_t j0, int64_t ncols, void* V, int64_t ldv) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (j0 < 0 || j0 >= h->n) return set_err(-2, "j0 out of range");
    if (ncols < 1 || j0 + ncols > h->n) return set_err(-3, "ncols out of range");
    if (!V) return set_err(-4, "V is NULL");
    if (ldv < h->m) return set_err(-5, "ldv < m");
    // In-matrix storage already holds explicit V inside each panel's row range; rows above the
    // panel (R entries of earlier block rows) must be reported as zero.
    const size_t w = h->w;
    const bool ddev = is_device_ptr(V);
    for (int64_t c = 0; c < ncols; ++c) {
        const int64_t j = j0 + c, p0 = (j / h->nb) * h->nb;
        char* dst = (char*)V + (size_t)c * ldv * w;
        if (ddev) CK(cudaMemsetAsync(dst, 0, (size_t)p0 * w, h->sU)); else memset(dst, 0, (size_t)p0 * w);
        if (h->ooc)
            CK(cudaMemcpyAsync(dst + (size_t)p0 * w, (char*)h->hA + ((size_t)j * h->hlda + p0) * w, (size_t)(h->m - p0) * w,
                               ddev ? cudaMemcpyHostToDevice : cudaMemcpyHostToHost, h->sU));
        else
            CK(cudaMemcpyAsync(dst + (size_t)p0 * w, (char*)h->dA + ((size_t)j * h->lda + p0) * w, (size_t)(h->m - p0) * w,
                               ddev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->sU));
    }
    CK(cudaStreamSynchronize(h->sU));
    return 0;
}

extern "C" int ct_qr_get_T(ctqr_handle_t h, int64_t panel, void* T, int64_t ldt) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (panel < 0 || panel >= h->P) return set_err(-2, "panel out of range");
    if (!T) return set_err(-3, "T is NULL");
    const int64_t nbw = std::min<int64_t>(h->nb, h->n - panel * h->nb);
    if (ldt < nbw) return set_err(-4, "ldt too small");
    const char* src = (const char*)h->dT + (size_t)panel * h->nb * h->nb * h->w;
    return h->dtype == CTQR_F64 ? copy_out<double>(*h, (const double*)src, h->nb, T, ldt, nbw, nbw)
                                : copy_out<float>(*h, (const float*)src, h->nb, T, ldt, nbw, nbw);
}

extern "C" int ct_qr_get_tau(ctqr_handle_t h, void* tau) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!tau) return set_err(-2, "tau is NULL");
    CK(cudaMemcpyAsync(tau, h->dTau, (size_t)h->n * h->w,
                       is_device_ptr(tau) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->sU));
    CK(cudaStreamSynchronize(h->sU));
    return 0;
}

extern "C" int ct_qr_get_stats(ctqr_handle_t h, ctqr_stats_t* s) {
    g_err[0] = 0;
    if (!h) return set_err(-1, "handle is NULL");
    if (!s) return set_err(-2, "s is NULL");
    *s = h->st;
    return 0;
}

extern "C" int ct_qr_dtype(ctqr_handle_t h) { return h ? (int)h->dtype : -1; }

extern "C" void ct_qr_destroy(ctqr_handle_t h) {
    if (!h) return;
    cudaDeviceSynchronize();
    delete h;
}

// ------------------------------------------------------------------------------------------
// factor persistence (the factor is computed once per
// scanner geometry and reused for every later batch of slices).
//
// File layout (little endian): one 4096-byte header page, then the factored matrix storage
// (column-major, leading dimension hdr.ld, n columns: V below / R above the panel diagonals),
// then P blocks T_k (nb x nb), P diagonal blocks of R (nb x nb), then tau[n].  The matrix
// section starts on a page boundary so that ct_qr_load can map the file and stream panels
// straight from the page cache when the factor does not fit the device budget.
// ------------------------------------------------------------------------------------------
struct FactorFileHeader {
    char magic[8];                    // "CTQRFAC1"
    int32_t version, dtype, nb, ib, P, reserved;
    int64_t m, n, ld;
    uint64_t off_matrix, off_T, off_Rd, off_tau, file_bytes;
    int64_t kl;                       // band promise the factor was computed under (0 = dense); the solve reuses it
};
static const char kFactorMagic[8] = {'C', 'T', 'Q', 'R', 'F', 'A', 'C', '1'};
constexpr size_t kFactorHeaderBytes = 4096;
constexpr size_t kIoChunkBytes = (size_t)256 << 20;   // pinned bounce buffer of save / load, used as two halves

static int write_all(int fd, const void* buf, size_t len, const char* path) {
    const char* p = (const char*)buf;
    while (len > 0) {
        ssize_t k = write(fd, p, len);
        if (k < 0) { if (errno == EINTR) continue; return set_err(CTQR_ERR_IO, "write to %s failed: %s", path, strerror(errno)); }
        p += k; len -= (size_t)k;
    }
    return 0;
}
static int read_all(int fd, void* buf, size_t len, const char* path) {
    char* p = (char*)buf;
    while (len > 0) {
        ssize_t k = read(fd, p, len);
        if (k < 0) { if (errno == EINTR) continue; return set_err(CTQR_ERR_IO, "read from %s failed: %s", path, strerror(errno)); }
        if (k == 0) return set_err(CTQR_ERR_IO, "%s is truncated", path);
        p += k; len -= (size_t)k;
    }
    return 0;
}

// One chunk of a file write running on its own thread (pwrite at an explicit offset, then an asynchronous
// write-back hint so the disk starts on it at once): ct_qr_save overlaps it with the device-to-host copy of the
// next chunk into the other half of the bounce buffer.
struct ChunkWriter {
    std::thread th;
    int err = 0;                       // errno of a failed pwrite (0 = fine); read after wait()
    void start(int fd, const char* buf, size_t len, off_t off) {
        wait();
        err = 0;
        th = std::thread([this, fd, buf, len, off] {
            const char* p = buf; size_t left = len; off_t o = off;
            while (left > 0) {
                ssize_t k = pwrite(fd, p, left, o);
                if (k < 0) { if (errno == EINTR) continue; err = errno; return; }
                p += k; left -= (size_t)k; o += k;
            }
            sync_file_range(fd, off, (off_t)len, SYNC_FILE_RANGE_WRITE);
        });
    }
    void wait() { if (th.joinable()) th.join(); }
    ~ChunkWriter() { wait(); }
};

// device section -> file at offset *off through the two halves of the pinned bounce buffer
static int save_device_section(H& h, int fd, const void* dsrc, size_t bytes, void* bounce, const char* path,
                               ChunkWriter& wr, int& half_idx, off_t* off) {
    const size_t half = kIoChunkBytes / 2;
    for (size_t o = 0; o < bytes; o += half) {
        const size_t len = std::min(half, bytes - o);
        char* buf = (char*)bounce + (size_t)half_idx * half;
        CK(cudaMemcpyAsync(buf, (const char*)dsrc + o, len, cudaMemcpyDeviceToHost, h.sU));
        CK(cudaStreamSynchronize(h.sU));
        wr.wait();                                             // the other half's write (it may still own the disk)
        if (wr.err) return set_err(CTQR_ERR_IO, "write to %s failed: %s", path, strerror(wr.err));
        wr.start(fd, buf, len, *off);
        *off += (off_t)len;
        half_idx ^= 1;
    }
    return 0;
}
static int load_device_section(H& h, int fd, void* ddst, size_t bytes, void* bounce, const char* path) {
    // the two halves of the bounce buffer alternate: the file read of one chunk overlaps the H2D copy of the previous
    const size_t half = kIoChunkBytes / 2;
    cudaEvent_t done[2] = {new_event(h, false), new_event(h, false)};
    bool busy[2] = {false, false};
    int i = 0;
    for (size_t off = 0; off < bytes; off += half, i ^= 1) {
        const size_t len = std::min(half, bytes - off);
        char* buf = (char*)bounce + (size_t)i * half;
        if (busy[i]) CK(cudaEventSynchronize(done[i]));
        CKI(read_all(fd, buf, len, path));
        CK(cudaMemcpyAsync((char*)ddst + off, buf, len, cudaMemcpyHostToDevice, h.sU));
        CK(cudaEventRecord(done[i], h.sU));
        busy[i] = true;
    }
    CK(cudaStreamSynchronize(h.sU));
    return 0;
}

static int save_body(H& h, int fd, const char* path, void* bounce) {
    const size_t w = h.w;
    const size_t blk = (size_t)h.nb * h.nb * w;
    FactorFileHeader hd; memset(&hd, 0, sizeof hd);
    memcpy(hd.magic, kFactorMagic, 8);
    hd.version = 1; hd.dtype = (int32_t)h.dtype; hd.nb = h.nb; hd.ib = h.ib; hd.P = h.P;
    hd.m = h.m; hd.n = h.n; hd.ld = round_up(h.m, 16 / (int64_t)w);
    hd.kl = h.kl;
    hd.off_matrix = kFactorHeaderBytes;
    hd.off_T = hd.off_matrix + (uint64_t)hd.ld * h.n * w;
    hd.off_Rd = hd.off_T + (uint64_t)blk * h.P;
    hd.off_tau = hd.off_Rd + (uint64_t)blk * h.P;
    hd.file_bytes = hd.off_tau + (uint64_t)h.n * w;
    if (posix_fallocate(fd, 0, (off_t)hd.file_bytes) != 0) { /* not fatal: some file systems cannot preallocate */ }
    std::vector<char> page(kFactorHeaderBytes, 0);
    memcpy(page.data(), &hd, sizeof hd);
    CKI(write_all(fd, page.data(), page.size(), path));
    // matrix storage, whole columns at a time (padding rows of the file are zero): the device-to-host copy of one
    // chunk into one half of the bounce buffer overlaps the file write of the previous chunk from the other half
    const size_t col_bytes = (size_t)hd.ld * w;
    const size_t half = kIoChunkBytes / 2;
    const int64_t cols_per = std::max<int64_t>(1, (int64_t)(half / col_bytes));
    std::vector<char> big[2];
    char* bufs[2] = {(char*)bounce, (char*)bounce + half};
    if (col_bytes > half) { for (auto& v : big) v.resize(col_bytes); bufs[0] = big[0].data(); bufs[1] = big[1].data(); }   // pageable
    ChunkWriter wr;
    off_t off = (off_t)hd.off_matrix;
    int hi = 0;
    for (int64_t c0 = 0; c0 < h.n; c0 += cols_per, hi ^= 1) {
        const int64_t nc = std::min<int64_t>(cols_per, h.n - c0);
        char* buf = bufs[hi];
        if (hd.ld != h.m) memset(buf, 0, (size_t)nc * col_bytes);
        if (h.ooc) {
            for (int64_t c = 0; c < nc; ++c)
                memcpy(buf + (size_t)c * col_bytes, (const char*)h.hA + (size_t)(c0 + c) * h.hlda * w, (size_t)h.m * w);
        } else {
            CK(cudaMemcpy2DAsync(buf, col_bytes, (const char*)h.dA + (size_t)c0 * h.lda * w, (size_t)h.lda * w,
                                 (size_t)h.m * w, nc, cudaMemcpyDeviceToHost, h.sU));
            CK(cudaStreamSynchronize(h.sU));
        }
        wr.wait();
        if (wr.err) return set_err(CTQR_ERR_IO, "write to %s failed: %s", path, strerror(wr.err));
        wr.start(fd, buf, (size_t)nc * col_bytes, off);
        off += (off_t)((size_t)nc * col_bytes);
    }
    wr.wait();
    if (wr.err) return set_err(CTQR_ERR_IO, "write to %s failed: %s", path, strerror(wr.err));
    int half_idx = 0;
    CKI(save_device_section(h, fd, h.dT, blk * h.P, bounce, path, wr, half_idx, &off));
    CKI(save_device_section(h, fd, h.dRd, blk * h.P, bounce, path, wr, half_idx, &off));
    CKI(save_device_section(h, fd, h.dTau, (size_t)h.n * w, bounce, path, wr, half_idx, &off));
    wr.wait();
    if (wr.err) return set_err(CTQR_ERR_IO, "write to %s failed: %s", path, strerror(wr.err));
    return 0;
}

extern "C" int ct_qr_save(ctqr_handle_t h, const char* path) {
    g_err[0] = 0;
    CKI(check_handle(h));
    if (!path || !path[0]) return set_err(-2, "path is NULL or empty");
    if (cudaStreamSynchronize(h->user) != cudaSuccess) return set_err(CTQR_ERR_CUDA, "user stream sync failed");
    const int fd = open(path, O_WRONLY | O_CREAT | O_TRUNC, 0644);
    if (fd < 0) return set_err(CTQR_ERR_IO, "cannot create %s: %s", path, strerror(errno));
    void* bounce = nullptr;
    if (cudaMallocHost(&bounce, kIoChunkBytes) != cudaSuccess) {
        cudaGetLastError(); close(fd);
        return set_err(CTQR_ERR_NOMEM, "cannot allocate the pinned bounce buffer");
    }
    int rc = save_body(*h, fd, path, bounce);
    cudaFreeHost(bounce);
    if (rc == 0 && fsync(fd) != 0) rc = set_err(CTQR_ERR_IO, "fsync of %s failed: %s", path, strerror(errno));
    if (close(fd) != 0 && rc == 0) rc = set_err(CTQR_ERR_IO, "close of %s failed: %s", path, strerror(errno));
    if (rc != 0) unlink(path);                 // never leave a partial factor file behind
    return rc;
}

template <typename T>
static int load_typed(H& h, int fd, const FactorFileHeader& hd, const ctqr_options_t& o, const char* path, void* bounce) {
    const size_t w = sizeof(T);
    const size_t blk = (size_t)h.nb * h.nb * w;
    const size_t mat_bytes = (size_t)hd.ld * h.n * w;
    CKI(alloc_state<T>(h, h.nb));              // solve workspaces grow on demand (ensure_solve_ws)
    const size_t freeb = free_device_bytes();
    const size_t slack = (size_t)2 << 30;
    const size_t budget = o.device_budget_bytes > 0 ? (size_t)o.device_budget_bytes : (freeb > slack ? freeb - slack : 0);
    if (mat_bytes <= budget) {
        h.lda = hd.ld;
        if (big_alloc(&h.dA, mat_bytes) != cudaSuccess) { cudaGetLastError(); return set_err(CTQR_ERR_NOMEM, "cannot allocate %zu bytes for the factor", mat_bytes); }
        h.own_A = true;
        if (lseek(fd, (off_t)hd.off_matrix, SEEK_SET) < 0) return set_err(CTQR_ERR_IO, "seek in %s failed", path);
        CKI(load_device_section(h, fd, h.dA, mat_bytes, bounce, path));
        h.st.h2d_bytes = (double)mat_bytes;
    } else {
        // factor larger than the budget: map the file, the solve streams panels from the page cache (a5)
        void* mp = mmap(nullptr, (size_t)hd.file_bytes, PROT_READ, MAP_SHARED, fd, 0);
        if (mp == MAP_FAILED) return set_err(CTQR_ERR_IO, "mmap of %s failed: %s", path, strerror(errno));
        h.fmap = mp; h.fmap_len = (size_t)hd.file_bytes;
        h.ooc = true; h.hA = (char*)mp + hd.off_matrix; h.hlda = hd.ld;
        h.n_super = (int)std::max<int64_t>(1, (int64_t)ceil_div((int64_t)mat_bytes, (int64_t)std::max<size_t>(budget, 1)));
        CKI(ensure_stream_bufs(h));
    }
    if (lseek(fd, (off_t)hd.off_T, SEEK_SET) < 0) return set_err(CTQR_ERR_IO, "seek in %s failed", path);
    CKI(load_device_section(h, fd, h.dT, blk * h.P, bounce, path));
    CKI(load_device_section(h, fd, h.dRd, blk * h.P, bounce, path));
    CKI(load_device_section(h, fd, h.dTau, (size_t)h.n * w, bounce, path));
    CK(cudaStreamSynchronize(h.sU));
    return 0;
}

extern "C" int ct_qr_load(const char* path, const ctqr_options_t* opt, ctqr_handle_t* out) {
    g_err[0] = 0;
    if (!path || !path[0]) return set_err(-1, "path is NULL or empty");
    if (!out) return set_err(-3, "out is NULL");
    ctqr_options_t o; memset(&o, 0, sizeof o); o.lookahead = -1;
    if (opt) o = *opt;
    const int fd = open(path, O_RDONLY);
    if (fd < 0) return set_err(CTQR_ERR_IO, "cannot open %s: %s", path, strerror(errno));
    FactorFileHeader hd;
    struct stat sb;
    int rc = read_all(fd, &hd, sizeof hd, path);
    if (rc == 0 && fstat(fd, &sb) != 0) rc = set_err(CTQR_ERR_IO, "fstat of %s failed", path);
    if (rc == 0) {
        const int64_t w = hd.dtype == CTQR_F64 ? 8 : 4;
        const uint64_t blk = (uint64_t)hd.nb * hd.nb * w;
        const bool ok = memcmp(hd.magic, kFactorMagic, 8) == 0 && hd.version == 1 &&
            (hd.dtype == CTQR_F32 || hd.dtype == CTQR_F64) && hd.n >= 1 && hd.m >= hd.n && hd.ld >= hd.m &&
            hd.nb >= 8 && hd.nb <= 128 && (hd.ib == 8 || hd.ib == 16 || hd.ib == 32) && hd.nb % hd.ib == 0 &&
            hd.P == (int32_t)ceil_div(hd.n, (int64_t)hd.nb) && (hd.ld * w) % 16 == 0 &&
            hd.off_matrix == kFactorHeaderBytes && hd.off_T == hd.off_matrix + (uint64_t)hd.ld * hd.n * w &&
            hd.off_Rd == hd.off_T + blk * hd.P && hd.off_tau == hd.off_Rd + blk * hd.P &&
            hd.file_bytes == hd.off_tau + (uint64_t)hd.n * w && (uint64_t)sb.st_size >= hd.file_bytes;
        if (!ok) rc = set_err(CTQR_ERR_IO, "%s is not a ctqr factor file (bad header or truncated)", path);
    }
    if (rc != 0) { close(fd); return rc; }
    o.nb = hd.nb; o.ib = hd.ib;
    H* h = nullptr;
    rc = new_handle((ctqr_dtype_t)hd.dtype, hd.m, hd.n, o, &h);
    if (rc != 0) { close(fd); return rc; }
    h->kl = (hd.kl > 0 && hd.kl < hd.m - 1) ? hd.kl : 0;
    void* bounce = nullptr;
    if (cudaMallocHost(&bounce, kIoChunkBytes) != cudaSuccess) {
        cudaGetLastError(); close(fd); delete h;
        return set_err(CTQR_ERR_NOMEM, "cannot allocate the pinned bounce buffer");
    }
    rc = hd.dtype == CTQR_F64 ? load_typed<double>(*h, fd, hd, o, path, bounce)
                              : load_typed<float>(*h, fd, hd, o, path, bounce);
    cudaFreeHost(bounce);
    if (rc != 0) { close(fd); cudaDeviceSynchronize(); delete h; return rc; }
    if (h->fmap) h->ffd = fd; else close(fd);  // the mapping keeps the file open for the handle's lifetime
    h->st.m = hd.m; h->st.n = hd.n; h->st.nb = h->nb; h->st.ib = h->ib; h->st.n_panels = h->P;
    h->st.n_superpanels = h->n_super; h->st.out_of_core = h->ooc ? 1 : 0; h->st.singular_col = -1;
    h->st.lower_bandwidth = h->kl;
    h->st.factor_flops = 2.0 * (double)hd.m * (double)hd.n * (double)hd.n - 2.0 * (double)hd.n * (double)hd.n * (double)hd.n / 3.0;
    h->factored = true;
    *out = h;
    return 0;
}

// ------------------------------------------------------------------------------------------
// kernel-level test / probe entry points
// ------------------------------------------------------------------------------------------
// impl == 2 (fp32, op(A) = A only): both operands split once into TF32 hi / lo, then the TMA-fed tcgen05 kernel
static int gemm_presplit(int64_t, int64_t, int64_t, double, const double*, int64_t, const double*, int64_t, double, double*, int64_t, int, int) {
    return set_err(-14, "impl 2 (pre-split tcgen05 kernel) is fp32 only");
}
static int gemm_presplit(int64_t M, int64_t N, int64_t K, double alpha, const float* A, int64_t lda, const float* B, int64_t ldb,
                         double beta, float* C, int64_t ldc, int ta, int sms) {
    if (ta) return set_err(-1, "impl 2 takes op(A) = A only");
    if (M == 0 || N == 0) return 0;
    const int64_t lda2 = round_up(M, 32), ldb2 = round_up(std::max<int64_t>(K, 1), 32);
    float *Ah = nullptr, *Al = nullptr, *Bh = nullptr, *Bl = nullptr;
    cudaError_t e = cudaMalloc(&Ah, (size_t)lda2 * K * 4);
    if (e == cudaSuccess) e = cudaMalloc(&Al, (size_t)lda2 * K * 4);
    if (e == cudaSuccess) e = cudaMalloc(&Bh, (size_t)ldb2 * N * 4);
    if (e == cudaSuccess) e = cudaMalloc(&Bl, (size_t)ldb2 * N * 4);
    if (e == cudaSuccess) e = split_tf32_launch(A, lda, M, K, Ah, Al, lda2, 0);
    if (e == cudaSuccess) e = split_tf32_launch(B, ldb, K, N, Bh, Bl, ldb2, 0);
    if (e == cudaSuccess) e = upd_presplit_launch(M, N, K, (float)alpha, Ah, Al, lda2, Bh, Bl, ldb2, (float)beta, C, ldc, sms, 0);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    cudaFree(Ah); cudaFree(Al); cudaFree(Bh); cudaFree(Bl);
    if (e != cudaSuccess) return set_err(CTQR_ERR_CUDA, "pre-split product failed: %s", cudaGetErrorString(e));
    return 0;
}

template <typename T>
static int gemm_typed(int ta, int64_t M, int64_t N, int64_t K, double alpha, const void* A, int64_t lda,
                      const void* B, int64_t ldb, double beta, void* C, int64_t ldc, int impl) {
    GemmArgs<T> g{};
    g.M = M; g.N = N; g.K = K; g.A = (const T*)A; g.lda = lda; g.B = (const T*)B; g.ldb = ldb;
    g.C = (T*)C; g.ldc = ldc; g.alpha = (T)alpha; g.beta = (T)beta; g.split_stride = 0;
    int dev = 0, sms = 148; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (impl == 2) return gemm_presplit(M, N, K, alpha, (const T*)A, lda, (const T*)B, ldb, beta, (T*)C, ldc, ta, sms);
    CK(gemm_direct<T>(ta != 0, g, impl, sms, 0));
    CK(cudaDeviceSynchronize());
    return 0;
}

extern "C" int ct_qr_gemm(int trans_a, int64_t M, int64_t N, int64_t K, double alpha, const void* A, int64_t lda,
                          const void* B, int64_t ldb, double beta, void* C, int64_t ldc, ctqr_dtype_t dtype, int impl) {
    g_err[0] = 0;
    if (M < 0) return set_err(-2, "M < 0");
    if (N < 0) return set_err(-3, "N < 0");
    if (K < 0) return set_err(-4, "K < 0");
    if (alpha == 0.0) return set_err(-5, "alpha must be non-zero");
    if (!A || !B || !C) return set_err(-6, "NULL operand");
    return dtype == CTQR_F64 ? gemm_typed<double>(trans_a, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, impl)
                             : gemm_typed<float>(trans_a, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, impl);
}

// register-resident arithmetic loops: the measured ceilings the roofline fractions are quoted against
template <int KIND>
__global__ void __launch_bounds__(256) peak_kernel(int iters, double* sink) {
    const int lane = threadIdx.x & 31;
    if (KIND == 0) {
        float a = 1.0f + lane * 1e-6f, b = 0.999f, c[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = (float)i;
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int i = 0; i < 16; ++i) c[i] = fmaf(a, c[i], b);
        float s = 0; for (int i = 0; i < 16; ++i) s += c[i];
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == 1) {
        double a = 1.0 + lane * 1e-9, b = 0.999, c[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = (double)i;
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int i = 0; i < 16; ++i) c[i] = fma(a, c[i], b);
        double s = 0; for (int i = 0; i < 16; ++i) s += c[i];
        if (s == 12345.678) sink[0] = s;
    } else if (KIND == 4 || KIND == 5) {
        // DMMA with a GEMM-like operand pattern: 4 x 4 outer product of fragments per k-step (16 DMMA);
        // KIND 5 additionally reloads the 8 fragments from shared memory every k-step (no barrier).
        __shared__ double sm[4 * 20 * 40];
        for (int i = threadIdx.x; i < 4 * 20 * 40; i += blockDim.x) sm[i] = 1.0 + 1e-9 * i;
        __syncthreads();
        double a[4], b[4], c[4][4][2];
#pragma unroll
        for (int i = 0; i < 4; ++i) { a[i] = 1.0 + lane * 1e-9 + i; b[i] = 0.5 + i; }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) { c[i][j][0] = i; c[i][j][1] = j; }
        const int grp = lane >> 2, tig = lane & 3;
        for (int it = 0; it < iters; ++it) {
            if (KIND == 5) {
                const double* As = sm + ((it & 3) * 4) ;
#pragma unroll
                for (int i = 0; i < 4; ++i) { a[i] = As[(i * 8 + grp) * 20 + tig]; b[i] = As[(32 + i * 8 + grp) * 20 + tig]; }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
        }
        double s = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) s += c[i][j][0] + c[i][j][1];
        if (s == 12345.678) sink[0] = s;
    } else if (KIND == 3) {
        // legacy warp-level TF32 tensor path: mma.sync.m16n8k8 (SASS HMMA.1688.F32.TF32), 4096 flop per warp
        unsigned a[4] = {0x3f800000u + lane, 0x3f800100u, 0x3f800200u, 0x3f800300u}, b[2] = {0x3f000000u, 0x3f000100u};
        float c[16][4];
#pragma unroll
        for (int i = 0; i < 16; ++i) { c[i][0] = i; c[i][1] = -i; c[i][2] = 1; c[i][3] = 2; }
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int i = 0; i < 16; ++i)
                asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                             : "+f"(c[i][0]), "+f"(c[i][1]), "+f"(c[i][2]), "+f"(c[i][3])
                             : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
        float s = 0; for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
        if (s == 12345.678f) sink[0] = s;
    } else {
        double a = 1.0 + lane * 1e-9, b = 0.5, c[16][2];
#pragma unroll
        for (int i = 0; i < 16; ++i) { c[i][0] = i; c[i][1] = -i; }
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int i = 0; i < 16; ++i) dmma884(c[i][0], c[i][1], a, b);
        double s = 0; for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
        if (s == 12345.678) sink[0] = s;
    }
}

extern "C" int ct_qr_peak_probe_cfg(int kind, int iters, int threads, int ctas_per_sm, double* tflops, double* ms_out);
extern "C" int ct_qr_peak_probe(int kind, int iters, double* tflops, double* ms_out) {
    return ct_qr_peak_probe_cfg(kind, iters, 256, 8, tflops, ms_out);
}
extern "C" int ct_qr_peak_probe_cfg(int kind, int iters, int threads, int ctas_per_sm, double* tflops, double* ms_out) {
    g_err[0] = 0;
    if (threads < 32 || threads > 256 || threads % 32) return set_err(-3, "threads must be a multiple of 32 in [32, 256]");
    if (ctas_per_sm < 1 || ctas_per_sm > 16) return set_err(-4, "ctas_per_sm must be in [1, 16]");
    if (kind < 0 || kind > 5) return set_err(-1, "kind must be 0..5");
    if (iters < 1) return set_err(-2, "iters < 1");
    if (!tflops) return set_err(-3, "tflops is NULL");
    int dev = 0; CK(cudaGetDevice(&dev));
    cudaDeviceProp prop; CK(cudaGetDeviceProperties(&prop, dev));
    double* sink = nullptr; CK(cudaMalloc(&sink, 8));
    const int ctas = prop.multiProcessorCount * ctas_per_sm;
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        CK(cudaEventRecord(e0, 0));
        if (kind == 0) peak_kernel<0><<<ctas, threads>>>(iters, sink);
        else if (kind == 1) peak_kernel<1><<<ctas, threads>>>(iters, sink);
        else if (kind == 2) peak_kernel<2><<<ctas, threads>>>(iters, sink);
        else if (kind == 3) peak_kernel<3><<<ctas, threads>>>(iters, sink);
        else if (kind == 4) peak_kernel<4><<<ctas, threads>>>(iters, sink);
        else peak_kernel<5><<<ctas, threads>>>(iters, sink);
        CK(cudaEventRecord(e1, 0));
        CK(cudaEventSynchronize(e1));
        float ms = 0; CK(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    CK(cudaGetLastError());
    // flops per thread-iteration: FMA kinds 16 * 2; DMMA 16 * 512 per warp = 16 * 16 per thread
    const double per_thread = (kind == 2 || kind >= 4) ? 16.0 * 16.0 : (kind == 3) ? 16.0 * 128.0 : 16.0 * 2.0;
    const double flops = per_thread * (double)iters * (double)threads * ctas;
    *tflops = flops / (best * 1e-3) / 1e12;
    if (ms_out) *ms_out = best;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    return 0;
}
