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
    T* Tin; int ldtin; // ibw x ibw inner T factor (ld = ldtin), written by CTA 0 into the diagonal block of T_k
    T* part;           // LL slots: [2 parities][G + 1][IB] x 16 bytes (record G = pivot row published by CTA 0)
    unsigned bar_base; // step number before this launch; column j of the launch uses bar_base + j + 1
};

// How the K range of a product was cut, for the kernels that sum the partial outputs.
//   L == 0: classic split grid, every output tile has `nsplit` partials (slot z = blockIdx.z).
//   L  > 0: stream-K (gemm_mma.cuh): the output tile of BN columns with index t has
//           sk_nseg(t, KT, L) partials in slots 0 .. nseg-1 (tilesM == 1 in partial mode).
struct SegInfo { int nsplit; int KT; int64_t L; int BN; };

// A planned product C <- alpha*op(A)*B + beta*C.
struct GemmLaunch {
    int kind;          // 0 = classic kernels (gemm.cuh) with `splits` K slices; 1 = persistent stream-K (gemm_mma.cuh)
    int splits;        // kind 0
    int grid;          // kind 1: CTAs
    int64_t tilesM, tilesN, U, L; int KT; int partial; int G, Gm;   // kind 1: StreamK fields
    int slots;         // partial output buffers needed (each g.split_stride elements apart)
    int cfg;           // kernel configuration index inside the dtype's dispatcher
    SegInfo seg;       // for the consumer of the partials
    // kind 1, optional: keep the kernel off `reserve` SMs (those with the highest %smid).  2 * reserve extra CTAs are
    // launched; a CTA that finds itself on a reserved SM retires at once (at most 2 * reserve do, counted in
    // tickets[0]), every other CTA draws its worker index from tickets[1].  tickets: two zeroed counters per launch.
    int reserve = 0;
    unsigned* tickets = nullptr;
};

// impl: 0 = default for the dtype (fp64: DMMA tensor cores, fp32: 3xTF32 tensor cores),
//       1 = SIMT kernels (DFMA / FFMA).  partial: the product goes to partial buffers that a
//       consumer kernel sums (the partial buffer holds max_elems elements; the classic kernels put
//       slice z at z * sstride, the stream-K kernel uses compact 128 x 64 tiles); otherwise beta*C
//       is added and C written.
// aligned: both operands have 16-byte aligned base pointers and leading dimensions (the stream-K kernel needs it)
GemmLaunch gemm_plan_f64(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems, int64_t sstride, bool aligned);
GemmLaunch gemm_plan_f32(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems, int64_t sstride, bool aligned);
cudaError_t gemm_run_f64(bool ta, GemmArgs<double> g, const GemmLaunch& L, int impl, cudaStream_t st);
cudaError_t gemm_run_f32(bool ta, GemmArgs<float> g, const GemmLaunch& L, int impl, cudaStream_t st);

// fp32 tcgen05 path with pre-split operands (gemm_umma_tma.cuh): TF32 hi / lo bit patterns of a column-major block
// (ld_out a multiple of 4, >= rows; padding rows zeroed), and C <- alpha (Ahi + Alo)(Bhi + Blo) + beta C with
// A m-contiguous (M x K, lda) and B k-contiguous (K x N, ldb), TMA-fed, on `ctas` CTAs (one per SM)
cudaError_t split_tf32_launch(const float* src, int64_t ld, int64_t rows, int64_t cols, float* hi, float* lo, int64_t ld_out, cudaStream_t st);
cudaError_t upd_presplit_launch(int64_t M, int64_t N, int64_t K, float alpha, const float* Ahi, const float* Alo, int64_t lda,
                                const float* Bhi, const float* Blo, int64_t ldb, float beta, float* C, int64_t ldc, int ctas, cudaStream_t st);

// stream-K partial tiles of A^T B (planned by gemm_plan_f32 as the tcgen05 configuration, L.cfg == 21) with A given pre-split
// (K x M, k-contiguous, M <= 128): returns cudaErrorNotSupported when the plan is not that configuration
cudaError_t vtc_presplit_launch(const GemmArgs<float>& g, const float* Ahi, const float* Alo, int64_t lda, const GemmLaunch& L, cudaStream_t st);

// cooperative register-resident panel kernel; returns cudaErrorInvalidValue for an unsupported (ib, rpt)
cudaError_t panel_launch_f64(int ib, int rpt, PanelArgs<double>& pa, int G, cudaStream_t st);
cudaError_t panel_launch_f32(int ib, int rpt, PanelArgs<float>& pa, int G, cudaStream_t st);
constexpr int kPanelThreads = 256;

// panel T from the Gram partials; the ib x ib diagonal blocks of Tk must already hold the inner T factors
template <typename T> cudaError_t larft_launch(const T* Gp, SegInfo seg, int64_t gstride, int ldg, int nbw, int ib, T* Tk, int ldt, cudaStream_t st);
// W <- T^T (sum of partials): scalar kernel for kw <= 32, tensor-core kernel otherwise
template <typename T> cudaError_t ttw_launch(const T* Wp, SegInfo seg, int64_t wstride, int64_t ldw, const T* Tm, int ldt, int kw, int64_t N, T* Wout, int64_t ldo, cudaStream_t st);
// dense (kw x N, ld = ldo) sum of the compact stream-K partial tiles (seg.L > 0)
template <typename T> cudaError_t partial_sum_launch(const T* Wp, SegInfo seg, int kw, int64_t N, T* Wout, int64_t ldo, cudaStream_t st);
template <typename T> cudaError_t trsm_diag_launch(const T* R, int ldr, int kw, const T* C, int64_t ldc, int64_t S, T* X, int64_t ldx, cudaStream_t st);
// X <- R^{-T} X in place on one kw x kw diagonal block (forward substitution with the transposed block)
template <typename T> cudaError_t trsm_diag_t_launch(const T* R, int ldr, int kw, T* X, int64_t ldx, int64_t S, cudaStream_t st);
// inverses of the P diagonal blocks of R (nb x nb each, ld = nb; a narrower last block is padded with zeros)
// out = op(M) * in, M 128 x 128 upper triangular (zeros stored), N <= a few hundred columns; `in` is either a matrix
// (seg.L == 0; may alias out) or the stream-K partial tiles of a 128 x N product (seg.L != 0)
template <typename T> cudaError_t mm128_launch(bool trans, const T* M, int ldm, const T* in, int64_t ldin, SegInfo seg, int64_t N, T* out, int64_t ldo, cudaStream_t st);
// cond_bits (optional, zeroed by the caller): receives the bit pattern of max over blocks of max|R_jj| / min|R_jj| as a float
template <typename T> cudaError_t trinv_launch(const T* Rd, int nb, int64_t n, int P, T* Rinv, unsigned* cond_bits, cudaStream_t st);
template <typename T> cudaError_t copy2d_launch(const T* src, int64_t lds, T* dst, int64_t ldd, int64_t rows, int64_t cols, cudaStream_t st);
template <typename T> cudaError_t gather_R_launch(const T* A, int64_t lda, const T* Rd, int nb, int64_t n, T* R, int64_t ldr, cudaStream_t st);
template <typename T> cudaError_t find_zero_diag_launch(const T* Rd, int nb, int64_t n, int* result, cudaStream_t st);

}  // namespace ctqr
