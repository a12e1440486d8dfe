// small.cu -- launchers of the small kernels (larft, T^T W, diagonal-block TRSM, accessors).
#include "small.cuh"
#include "kernels.h"

namespace ctqr {

template <typename K>
static cudaError_t ensure_smem(K kernel, size_t bytes, SmemAttr& cur) { return ensure_dyn_smem(kernel, bytes, cur); }

template <typename T>
cudaError_t larft_launch(const T* Gp, SegInfo seg, int64_t gstride, int ldg, int nbw, int ib, T* Tk, int ldt,
                         cudaStream_t st) {
    static SmemAttr cur;
    const size_t smem = ((size_t)nbw * (nbw + 1) + (size_t)2 * nbw * (ib + 1)) * sizeof(T);
    cudaError_t e = ensure_smem(larft_kernel<T>, smem, cur);
    if (e != cudaSuccess) return e;
    larft_kernel<T><<<1, 1024, smem, st>>>(Gp, seg, gstride, ldg, nbw, ib, Tk, ldt);
    return cudaGetLastError();
}

template <typename T>
cudaError_t ttw_launch(const T* Wp, SegInfo seg, int64_t wstride, int64_t ldw, const T* Tm, int ldt, int kw, int64_t N,
                       T* Wout, int64_t ldo, cudaStream_t st) {
    if (kw > 32 && kw <= 128 && (seg.L == 0 || seg.BN == 64 || seg.BN == 128)) {
        static SmemAttr cur2;
        const size_t smem2 = (size_t)(128 + 64) * 132 * sizeof(T);
        cudaError_t e2 = ensure_smem(ttw_mma_kernel<T>, smem2, cur2);
        if (e2 != cudaSuccess) return e2;
        ttw_mma_kernel<T><<<(unsigned)ceil_div(N, 64), 256, smem2, st>>>(Wp, seg, wstride, ldw, Tm, ldt, kw, N, Wout, ldo);
        return cudaGetLastError();
    }
    if (seg.L != 0 || kw > 32) return cudaErrorInvalidValue;   // the scalar kernel only sums uniform splits
    const int cw = std::max(1, 64 / kw);
    int tpe = 1;
    while (tpe * 2 * kw * cw <= 256 && tpe < 32) tpe *= 2;
    ttw_kernel<T><<<(unsigned)ceil_div(N, cw), 256, 0, st>>>(Wp, seg.nsplit, wstride, ldw, Tm, ldt, kw, N, Wout, ldo, cw, tpe);
    return cudaGetLastError();
}

template <typename T>
cudaError_t partial_sum_launch(const T* Wp, SegInfo seg, int kw, int64_t N, T* Wout, int64_t ldo, cudaStream_t st) {
    partial_sum_kernel<T><<<(unsigned)ceil_div(N, 2), 256, 0, st>>>(Wp, seg, kw, N, Wout, ldo);
    return cudaGetLastError();
}

template <typename T>
cudaError_t mm128_launch(bool trans, const T* M, int ldm, const T* in, int64_t ldin, SegInfo seg, int64_t N, T* out,
                         int64_t ldo, cudaStream_t st) {
    const size_t smem = ((size_t)128 * Mm128Ld<T>::M + (size_t)128 * Mm128Ld<T>::X +
                         (size_t)(kMm128Threads / 128) * 128 * (kMm128Cols + 1)) * sizeof(T);
    const unsigned grid = (unsigned)ceil_div(N, (int64_t)kMm128Cols);
    const bool partial = seg.L != 0;
    if (partial && (seg.BN % kMm128Cols != 0 || !trans)) return cudaErrorInvalidValue;
    static SmemAttr cur[2];
    if (partial) {
        cudaError_t e = ensure_smem(mm128_kernel<T, true, true>, smem, cur[0]);
        if (e != cudaSuccess) return e;
        mm128_kernel<T, true, true><<<grid, kMm128Threads, smem, st>>>(M, ldm, in, ldin, seg, N, out, ldo);
    } else if (trans) {
        return cudaErrorInvalidValue;
    } else {
        cudaError_t e = ensure_smem(mm128_kernel<T, false, false>, smem, cur[1]);
        if (e != cudaSuccess) return e;
        mm128_kernel<T, false, false><<<grid, kMm128Threads, smem, st>>>(M, ldm, in, ldin, seg, N, out, ldo);
    }
    return cudaGetLastError();
}

template <typename T>
cudaError_t trsm_diag_launch(const T* R, int ldr, int kw, const T* C, int64_t ldc, int64_t S, T* X, int64_t ldx,
                             cudaStream_t st) {
    static SmemAttr cur;
    const size_t smem = (size_t)128 * 129 * sizeof(T);
    cudaError_t e = ensure_smem(trsm_diag_kernel<T, 128>, smem, cur);
    if (e != cudaSuccess) return e;
    trsm_diag_kernel<T, 128><<<(unsigned)ceil_div(S, 16), 256, smem, st>>>(R, ldr, kw, C, ldc, S, X, ldx);
    return cudaGetLastError();
}

template <typename T>
cudaError_t trsm_diag_t_launch(const T* R, int ldr, int kw, T* X, int64_t ldx, int64_t S, cudaStream_t st) {
    static SmemAttr cur;
    const size_t smem = ((size_t)kw * (kw + 1) + (size_t)kw * kTrsmTThreads) * sizeof(T);
    cudaError_t e = ensure_smem(trsm_diag_t_kernel<T>, smem, cur);
    if (e != cudaSuccess) return e;
    trsm_diag_t_kernel<T><<<(unsigned)ceil_div(S, (int64_t)kTrsmTThreads), kTrsmTThreads, smem, st>>>(R, ldr, kw, X, ldx, S);
    return cudaGetLastError();
}

template <typename T>
cudaError_t trinv_launch(const T* Rd, int nb, int64_t n, int P, T* Rinv, unsigned* cond_bits, cudaStream_t st) {
    static SmemAttr cur;
    const size_t smem = (size_t)nb * (nb + 1) * sizeof(T);
    cudaError_t e = ensure_smem(trinv_kernel<T>, smem, cur);
    if (e != cudaSuccess) return e;
    trinv_kernel<T><<<P, 128, smem, st>>>(Rd, nb, n, Rinv, cond_bits);
    return cudaGetLastError();
}

template <typename T>
cudaError_t copy2d_launch(const T* src, int64_t lds, T* dst, int64_t ldd, int64_t rows, int64_t cols, cudaStream_t st) {
    if (rows <= 0 || cols <= 0) return cudaSuccess;
    dim3 grid((unsigned)ceil_div(rows, 256), (unsigned)std::min<int64_t>(cols, 65535));
    copy2d_kernel<T><<<grid, 256, 0, st>>>(src, lds, dst, ldd, rows, cols);
    return cudaGetLastError();
}

template <typename T>
cudaError_t gather_R_launch(const T* A, int64_t lda, const T* Rd, int nb, int64_t n, T* R, int64_t ldr, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(n, 256), (unsigned)std::min<int64_t>(n, 65535));
    gather_R_kernel<T><<<grid, 256, 0, st>>>(A, lda, Rd, nb, n, R, ldr);
    return cudaGetLastError();
}

template <typename T>
cudaError_t find_zero_diag_launch(const T* Rd, int nb, int64_t n, int* result, cudaStream_t st) {
    find_zero_diag_kernel<T><<<(unsigned)ceil_div(n, 256), 256, 0, st>>>(Rd, nb, n, result);
    return cudaGetLastError();
}

#define INST(T)                                                                                                        \
    template cudaError_t trinv_launch<T>(const T*, int, int64_t, int, T*, unsigned*, cudaStream_t);                             \
    template cudaError_t partial_sum_launch<T>(const T*, SegInfo, int, int64_t, T*, int64_t, cudaStream_t);            \
    template cudaError_t larft_launch<T>(const T*, SegInfo, int64_t, int, int, int, T*, int, cudaStream_t);           \
    template cudaError_t ttw_launch<T>(const T*, SegInfo, int64_t, int64_t, const T*, int, int, int64_t, T*, int64_t,  \
                                       cudaStream_t);                                                                  \
    template cudaError_t mm128_launch<T>(bool, const T*, int, const T*, int64_t, SegInfo, int64_t, T*, int64_t, cudaStream_t); \
    template cudaError_t trsm_diag_launch<T>(const T*, int, int, const T*, int64_t, int64_t, T*, int64_t, cudaStream_t); \
    template cudaError_t trsm_diag_t_launch<T>(const T*, int, int, T*, int64_t, int64_t, cudaStream_t);                  \
    template cudaError_t copy2d_launch<T>(const T*, int64_t, T*, int64_t, int64_t, int64_t, cudaStream_t);             \
    template cudaError_t gather_R_launch<T>(const T*, int64_t, const T*, int, int64_t, T*, int64_t, cudaStream_t);     \
    template cudaError_t find_zero_diag_launch<T>(const T*, int, int64_t, int*, cudaStream_t);
INST(float)
INST(double)

}  // namespace ctqr
