// noalloc.cu -- ct_qr_vtc_noalloc: the split-K product W = V^T C of the block-reflector application (step 1 of
// C <- (I - V T V^T)^T C; "dormqr") for callers that must not allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The library's own path for this product (ct_qr_gemm with trans_a = 1, and the factorisation's larfb) writes its
// split-K / stream-K partial tiles into a workspace obtained from the device-block cache, i.e. from cudaMalloc.  This
// variant keeps the partial tiles in a FILE-SCOPE device array of fixed size instead: kNoAllocScratchBytes = 16 MiB that
// every GPU which loads libctqr.so holds until the process exits.  Consequences, all part of the contract in
// include/ctqr.h:
//   * sizes whose partial tiles do not fit are refused (CTQR_ERR_NOMEM, message names the limit), never spilled;
//   * no cudaMalloc / cudaFree / allocating library routine is called, on any call, first or later;
//   * every call uses the same array: two calls whose kernels overlap on the GPU (different streams, no dependency)
//     race on it.  Calls on one stream are ordered and safe;
//   * the array keeps the previous call's partial tiles.  Nothing has to start at zero: every slot the reduction reads is
//     written in full (zero-padded at ragged edges) by the same call's product kernel first, and there are no counters
//     or flags in the array, so there is nothing to clear and a stale tile can never be read.
//
// In host code `g_noalloc_scratch` is a host-side stand-in for the device array, not a device address; the address the
// kernels get is fetched with cudaGetSymbolAddress, once per device, with that device current.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <algorithm>
#include <mutex>

#include "../../include/ctqr.h"

extern "C" int ctqr_internal_set_error(int code, const char* what, const char* detail);   // ctqr.cu: thread-local message

namespace {

constexpr size_t kNoAllocScratchBytes = (size_t)CTQR_NOALLOC_SCRATCH_BYTES;
constexpr int kTile = 64;                 // output tile: 64 x 64 per CTA
constexpr int kBK = 16;                   // k-step
constexpr int kThreads = 256;             // 16 x 16 threads, 4 x 4 outputs each
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

// partial tile (split, tile): rows of the K range [split * kchunk, (split + 1) * kchunk) of V and C contracted;
// part[(split * ntiles + tile) * 64 * 64 + r + c * 64], written in full
template <typename T>
__global__ void __launch_bounds__(kThreads)
vtc_noalloc_partial_kernel(const T* __restrict__ V, int64_t ldv, const T* __restrict__ C, int64_t ldc, int64_t M, int64_t N,
                           int64_t K, int tilesM, int ntiles, int64_t kchunk, T* __restrict__ part) {
    __shared__ T Vs[kBK][kTile + 1];
    __shared__ T Cs[kBK][kTile + 1];
    const int tile = blockIdx.x % ntiles, split = blockIdx.x / ntiles;
    const int64_t i0 = (int64_t)(tile % tilesM) * kTile, j0 = (int64_t)(tile / tilesM) * kTile;
    const int64_t k0 = (int64_t)split * kchunk, k1 = min(K, k0 + kchunk);
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    T acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = T(0);
    for (int64_t k = k0; k < k1; k += kBK) {
#pragma unroll
        for (int r = 0; r < kBK * kTile / kThreads; ++r) {
            const int idx = tid + r * kThreads, kk = idx % kBK, i = idx / kBK;      // consecutive threads: consecutive k
            const int64_t kg = k + kk;
            Vs[kk][i] = (kg < k1 && i0 + i < M) ? V[kg + (i0 + i) * ldv] : T(0);
            Cs[kk][i] = (kg < k1 && j0 + i < N) ? C[kg + (j0 + i) * ldc] : T(0);
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < kBK; ++kk) {
            T va[4], cb[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) va[a] = Vs[kk][tx + 16 * a];
#pragma unroll
            for (int b = 0; b < 4; ++b) cb[b] = Cs[kk][ty + 16 * b];
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) acc[a][b] = fma(va[a], cb[b], acc[a][b]);
        }
        __syncthreads();
    }
    T* out = part + ((size_t)split * ntiles + tile) * (kTile * kTile);
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) out[(tx + 16 * a) + (ty + 16 * b) * kTile] = acc[a][b];
}

// W[i, j] = sum over the splits, in split order (deterministic), of the partial tiles
template <typename T>
__global__ void __launch_bounds__(kThreads)
vtc_noalloc_reduce_kernel(const T* __restrict__ part, int64_t M, int64_t N, int tilesM, int ntiles, int nsplit, T* __restrict__ W,
                          int64_t ldw) {
    const int64_t e = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (e >= M * N) return;
    const int64_t i = e % M, j = e / M;
    const int tile = (int)(i / kTile) + (int)(j / kTile) * tilesM;
    const T* p = part + (size_t)tile * (kTile * kTile) + (i % kTile) + (j % kTile) * kTile;
    T s = T(0);
    for (int sp = 0; sp < nsplit; ++sp) s += p[(size_t)sp * ntiles * (kTile * kTile)];
    W[i + j * ldw] = s;
}

// device address of the scratch array, fetched once per device with that device current
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices] = {nullptr};

int scratch_for_current_device(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return ctqr_internal_set_error(CTQR_ERR_CUDA, "cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return ctqr_internal_set_error(CTQR_ERR_CUDA, "device index beyond the scratch table", "");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return ctqr_internal_set_error(CTQR_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch)", cudaGetErrorString(e));
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return 0;
}

bool device_pointer(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

template <typename T>
int vtc_noalloc_typed(int64_t M, int64_t N, int64_t K, const T* V, int64_t ldv, const T* C, int64_t ldc, T* W, int64_t ldw,
                      cudaStream_t st) {
    const int64_t tilesM = (M + kTile - 1) / kTile, tilesN = (N + kTile - 1) / kTile, ntiles = tilesM * tilesN;
    const int64_t slots = (int64_t)(kNoAllocScratchBytes / ((size_t)kTile * kTile * sizeof(T)));
    if (tilesM > slots || tilesN > slots || ntiles > slots) {
        char msg[200];
        snprintf(msg, sizeof msg, "ceil(M/64) * ceil(N/64) = %lld output tiles, the static scratch (%zu bytes) holds %lld of this dtype",
                 (long long)ntiles, kNoAllocScratchBytes, (long long)slots);
        return ctqr_internal_set_error(CTQR_ERR_NOMEM, "ct_qr_vtc_noalloc: size beyond the fixed scratch", msg);
    }
    void* sp = nullptr;
    int rc = scratch_for_current_device(&sp);
    if (rc) return rc;
    // split K so that about two waves of CTAs are busy, within the slots the scratch has and the k-steps K has
    int sms = 148, dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); sms = 148; }
    int64_t nsplit = (2 * (int64_t)sms + ntiles - 1) / ntiles;
    nsplit = std::min<int64_t>(nsplit, slots / ntiles);
    nsplit = std::min<int64_t>(nsplit, (K + kBK - 1) / kBK);
    nsplit = std::max<int64_t>(nsplit, 1);
    int64_t kchunk = (K + nsplit - 1) / nsplit;
    kchunk = (kchunk + kBK - 1) / kBK * kBK;
    if (kchunk < kBK) kchunk = kBK;
    nsplit = std::max<int64_t>(1, (K + kchunk - 1) / kchunk);
    T* part = static_cast<T*>(sp);
    vtc_noalloc_partial_kernel<T><<<(unsigned)(ntiles * nsplit), kThreads, 0, st>>>(V, ldv, C, ldc, M, N, K, (int)tilesM, (int)ntiles,
                                                                                 kchunk, part);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return ctqr_internal_set_error(CTQR_ERR_CUDA, "vtc_noalloc_partial_kernel launch", cudaGetErrorString(e));
    vtc_noalloc_reduce_kernel<T><<<(unsigned)((M * N + kThreads - 1) / kThreads), kThreads, 0, st>>>(part, M, N, (int)tilesM, (int)ntiles,
                                                                                                  (int)nsplit, W, ldw);
    e = cudaGetLastError();
    if (e != cudaSuccess) return ctqr_internal_set_error(CTQR_ERR_CUDA, "vtc_noalloc_reduce_kernel launch", cudaGetErrorString(e));
    return 0;
}

}  // namespace

extern "C" int ct_qr_vtc_noalloc(int64_t M, int64_t N, int64_t K, const void* V, int64_t ldv, const void* C, int64_t ldc, void* W,
                                 int64_t ldw, ctqr_dtype_t dtype, void* stream) {
    if (M < 1) return ctqr_internal_set_error(-1, "M < 1", "");
    if (N < 1) return ctqr_internal_set_error(-2, "N < 1", "");
    if (K < 0) return ctqr_internal_set_error(-3, "K < 0", "");
    if (!V || ldv < (K > 0 ? K : 1)) return ctqr_internal_set_error(V ? -5 : -4, V ? "ldv < max(K, 1)" : "V is NULL", "");
    if (!C || ldc < (K > 0 ? K : 1)) return ctqr_internal_set_error(C ? -7 : -6, C ? "ldc < max(K, 1)" : "C is NULL", "");
    if (!W || ldw < M) return ctqr_internal_set_error(W ? -9 : -8, W ? "ldw < M" : "W is NULL", "");
    if (dtype != CTQR_F64 && dtype != CTQR_F32) return ctqr_internal_set_error(-10, "dtype must be CTQR_F32 or CTQR_F64", "");
    if (!device_pointer(V) || !device_pointer(C) || !device_pointer(W))
        return ctqr_internal_set_error(-4, "V, C and W must be device pointers", "");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return dtype == CTQR_F64
               ? vtc_noalloc_typed<double>(M, N, K, static_cast<const double*>(V), ldv, static_cast<const double*>(C), ldc,
                                           static_cast<double*>(W), ldw, st)
               : vtc_noalloc_typed<float>(M, N, K, static_cast<const float*>(V), ldv, static_cast<const float*>(C), ldc,
                                          static_cast<float*>(W), ldw, st);
}
