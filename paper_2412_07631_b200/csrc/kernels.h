// kernels.h -- host-side launchers of the ctqr kernels (each defined in its own translation
// unit so that the library builds in parallel).  Internal to the library; not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctqr {

template <typename T>
struct GemmArgs {
    int64_t M, N, K;
    const T* A; int64_t lda;
    const T* B; int64_t ldb;
    T* C; int64_t ldc;
    T alpha, beta;
    int64_t k_chunk;        // K range per blockIdx.z (multiple of BK); == K when no split
    int64_t split_stride;   // elements between partial outputs
    int a_vec_ok, b_vec_ok; // 16-byte aligned base + leading dimension (vector loads allowed)
};

template <typename T>
struct PanelArgs {
    T* A; int64_t lda; int64_t m;
    int64_t j0;        // first column (= first row) of the enclosing nb-wide panel
    int64_t jb;        // first column (= diagonal row) of this inner block
    int ibw;           // actual width of this inner block (<= IB)
    T* tau;            // tau + jb written
    T* Rd; int ldrd;   // diagonal block of R for the enclosing panel (ldrd x ldrd, zero-initialised)
    T* Tin;            // IB x IB (ld = IB) inner T factor, written by CTA 0
    T* part;           // [2][G][IB] per-CTA partial sums
    T* rowbuf;         // [2][IB] the pivot row broadcast
    unsigned* bar;     // grid barrier counter (monotone)
    unsigned bar_base; // counter value when this launch starts
};

// C <- alpha*op(A)*B + beta*C (see gemm.cuh).  impl: 0 = default for the dtype, 1 = SIMT.
cudaError_t gemm_f64(bool ta, GemmArgs<double> g, int splits, int impl, cudaStream_t st);
cudaError_t gemm_f32(bool ta, GemmArgs<float> g, int splits, int impl, cudaStream_t st);
// output tile (bm, bn) the default kernel will use for an M x N product (for split-K planning)
void gemm_tile_f64(bool ta, int64_t M, int64_t N, int impl, int* bm, int* bn);
void gemm_tile_f32(bool ta, int64_t M, int64_t N, int impl, int* bm, int* bn);

// cooperative register-resident panel kernel; returns cudaErrorInvalidValue for an unsupported (ib, rpt)
cudaError_t panel_launch_f64(int ib, int rpt, PanelArgs<double>& pa, int G, cudaStream_t st);
cudaError_t panel_launch_f32(int ib, int rpt, PanelArgs<float>& pa, int G, cudaStream_t st);
constexpr int kPanelThreads = 256;

template <typename T> cudaError_t larft_launch(const T* Gp, int nsplit, int64_t gstride, int ldg, const T* tau, int nbw, T* Tout, int ldt, cudaStream_t st);
template <typename T> cudaError_t ttw_launch(const T* Wp, int nsplit, int64_t wstride, int64_t ldw, const T* Tm, int ldt, int kw, int64_t N, T* Wout, int64_t ldo, cudaStream_t st);
template <typename T> cudaError_t trsm_diag_launch(const T* R, int ldr, int kw, const T* C, int64_t ldc, int64_t S, T* X, int64_t ldx, cudaStream_t st);
template <typename T> cudaError_t copy2d_launch(const T* src, int64_t lds, T* dst, int64_t ldd, int64_t rows, int64_t cols, cudaStream_t st);
template <typename T> cudaError_t gather_R_launch(const T* A, int64_t lda, const T* Rd, int nb, int64_t n, T* R, int64_t ldr, cudaStream_t st);
template <typename T> cudaError_t find_zero_diag_launch(const T* Rd, int nb, int64_t n, int* result, cudaStream_t st);

}  // namespace ctqr
