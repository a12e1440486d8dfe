// refine.cu -- ct_qr_solve_refined: least-squares solve with a working-precision (normally fp32) factor and
// fp64 iterative refinement ("fp32-factor + fp64 iterative refinement as a precision
// variant bridging the paper's fp32 / fp64 quality gap", Tables 3, 7, 9: L162-167, L271-280, L319-328).
//
// Method (corrected semi-normal equations; the factor enters only through R):
//     x_0 = R^{-1} (Q^T b)                              working precision, Eq. 3
//     repeat:  r = b - A x_k                            fp64
//              g = A^T r                                fp64 (the normal-equations residual, zero at the solution)
//              d = R^{-1} (R^{-T} g)                    working precision, on g scaled to max |g| = 1 per slice
//              x_{k+1} = x_k + d                        fp64
// The fixed point satisfies A^T (b - A x) = 0 exactly, whatever the rounding in R, so the iteration converges to
// the fp64 least-squares solution of the fp64 matrix also for inconsistent (noisy) right-hand sides; the error
// contracts by about cond(A)^2 * u_working per sweep (1e-2 .. 1e-3 for the CT configs in fp32).
//
// This translation unit is written on top of the library's own public entry points (ct_qr_solve, ct_qr_trsm_t,
// ct_qr_trsm, ct_qr_gemm) plus the fp64 kernels below; it does not look inside the handle.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <string.h>
#include <algorithm>
#include <vector>

#include "../../include/ctqr.h"

namespace {

// ---- fp64 kernels ---------------------------------------------------------------------------
// Y[row, s] = beta * Y0[row, s] + alpha * sum_k vals[k] X[colidx[k], s]  for rowptr[row] <= k < rowptr[row + 1]:
// one warp per row, lanes over the row's entries, up to 8 right-hand sides per pass, fixed-order warp reduction
// (deterministic).  Y0 may alias Y; X must not.
constexpr int kSpmmCols = 8;
__global__ void __launch_bounds__(256)
csr_spmm_kernel(int64_t m, const int64_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
                const double* __restrict__ vals, const double* __restrict__ X, int64_t ldx, int64_t S,
                double alpha, double beta, const double* Y0, int64_t ldy0, double* Y, int64_t ldy) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= m) return;
    const int64_t k0 = rowptr[row], k1 = rowptr[row + 1];
    for (int64_t s0 = 0; s0 < S; s0 += kSpmmCols) {
        const int ns = (int)min((int64_t)kSpmmCols, S - s0);
        double acc[kSpmmCols];
#pragma unroll
        for (int s = 0; s < kSpmmCols; ++s) acc[s] = 0.0;
        for (int64_t k = k0 + lane; k < k1; k += 32) {
            const double v = vals[k];
            const double* x = X + colidx[k] + s0 * ldx;
#pragma unroll
            for (int s = 0; s < kSpmmCols; ++s)
                if (s < ns) acc[s] = fma(v, x[(int64_t)s * ldx], acc[s]);
        }
#pragma unroll
        for (int s = 0; s < kSpmmCols; ++s)
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) acc[s] += __shfl_xor_sync(0xffffffffu, acc[s], off);
        if (lane == 0)
#pragma unroll
            for (int s = 0; s < kSpmmCols; ++s)
                if (s < ns) {
                    const double y0 = beta != 0.0 ? beta * Y0[row + (s0 + s) * ldy0] : 0.0;
                    Y[row + (s0 + s) * ldy] = fma(alpha, acc[s], y0);
                }
    }
}

// per column: out[s] = max_i |X[i, s]|  (MODE 0)  or  sum_i X[i, s]^2  (MODE 1); one CTA per column, fixed order
template <int MODE>
__global__ void __launch_bounds__(256) colreduce_kernel(const double* __restrict__ X, int64_t ld, int64_t rows, double* out) {
    __shared__ double sh[256];
    const double* x = X + (int64_t)blockIdx.x * ld;
    double a = 0.0;
    for (int64_t i = threadIdx.x; i < rows; i += 256) a = MODE == 0 ? fmax(a, fabs(x[i])) : fma(x[i], x[i], a);
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int w = 128; w >= 1; w >>= 1) {
        if ((int)threadIdx.x < w) sh[threadIdx.x] = MODE == 0 ? fmax(sh[threadIdx.x], sh[threadIdx.x + w]) : sh[threadIdx.x] + sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[blockIdx.x] = sh[0];
}

// out[i, s] = (T)(in[i, s] / scale[s])   (scale == nullptr or scale[s] == 0: plain conversion)
template <typename T>
__global__ void cast_down_kernel(const double* __restrict__ in, int64_t ldi, int64_t rows, int64_t S, const double* __restrict__ scale,
                                 T* __restrict__ out, int64_t ldo) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows) return;
    for (int64_t s = blockIdx.y; s < S; s += gridDim.y) {
        const double sc = (scale && scale[s] != 0.0) ? scale[s] : 1.0;
        out[i + s * ldo] = (T)(in[i + s * ldi] / sc);
    }
}
// X[i, s] = (accumulate ? X[i, s] : 0) + scale[s] * (double)d[i, s];  D[i, s] = the term that was added (fp64)
template <typename T>
__global__ void add_up_kernel(const T* __restrict__ d, int64_t ldd, int64_t rows, int64_t S, const double* __restrict__ scale,
                              int accumulate, double* __restrict__ X, int64_t ldx, double* __restrict__ D, int64_t ldD) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows) return;
    for (int64_t s = blockIdx.y; s < S; s += gridDim.y) {
        const double sc = (scale && scale[s] != 0.0) ? scale[s] : 1.0;
        const double t = sc * (double)d[i + s * ldd];
        if (D) D[i + s * ldD] = t;
        X[i + s * ldx] = accumulate ? X[i + s * ldx] + t : t;
    }
}

// ---- host helpers -----------------------------------------------------------------------------
struct Bufs {                       // every device allocation of one call; freed on every exit path
    std::vector<void*> p;
    ~Bufs() { for (void* q : p) cudaFree(q); }
    template <typename P> cudaError_t get(P** out, size_t bytes) {
        void* q = nullptr;
        cudaError_t e = cudaMalloc(&q, bytes ? bytes : 1);
        if (e == cudaSuccess) { p.push_back(q); *out = (P*)q; }
        return e;
    }
};
static bool on_device(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}
// device view of an array that may live on the host (staged into `b`)
template <typename P>
static cudaError_t device_view(Bufs& b, const P* src, size_t count, const P** out) {
    if (on_device(src)) { *out = src; return cudaSuccess; }
    P* d = nullptr;
    cudaError_t e = b.get(&d, count * sizeof(P));
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(d, src, count * sizeof(P), cudaMemcpyHostToDevice);
    *out = d;
    return e;
}
struct DevCsr { int64_t m, n; const int64_t* rowptr; const int32_t* colidx; const double* vals; };

static cudaError_t spmm(const DevCsr& A, const double* X, int64_t ldx, int64_t S, double alpha, double beta,
                        const double* Y0, int64_t ldy0, double* Y, int64_t ldy) {
    const int wpb = 8;
    csr_spmm_kernel<<<(unsigned)((A.m + wpb - 1) / wpb), wpb * 32>>>(A.m, A.rowptr, A.colidx, A.vals, X, ldx, S, alpha, beta, Y0, ldy0, Y, ldy);
    return cudaGetLastError();
}
static dim3 grid2(int64_t rows, int64_t S) { return dim3((unsigned)((rows + 255) / 256), (unsigned)std::min<int64_t>(S, 65535)); }

}  // namespace

#define RCK(call)                                                                                   \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) return ctqr_internal_set_error(CTQR_ERR_CUDA, #call, cudaGetErrorString(e_)); \
    } while (0)
#define RCI(call) do { int r_ = (call); if (r_ != 0) return r_; } while (0)

extern "C" int ctqr_internal_set_error(int code, const char* what, const char* detail);   // ctqr.cu: sets the thread-local message

template <typename T>
static int refined_typed(ctqr_handle_t h, int64_t m, int64_t n, const DevCsr* A, const DevCsr* At, const double* Ad, int64_t lda,
                         const double* B, int64_t ldb, int64_t S, double* X, int64_t ldx, int max_iters, double tol,
                         ctqr_refine_info_t* info, Bufs& bufs) {
    const ctqr_dtype_t code = sizeof(T) == 8 ? CTQR_F64 : CTQR_F32;
    (void)code;
    double *Bd, *Xd, *r, *g, *dcorr, *red;
    T *Bw, *Xw, *gw, *yw;
    const int64_t ldm = (m + 1) & ~(int64_t)1, ldn = (n + 1) & ~(int64_t)1;     // 16-byte aligned columns
    RCK(bufs.get(&Bd, (size_t)ldm * S * 8)); RCK(bufs.get(&r, (size_t)ldm * S * 8));
    RCK(bufs.get(&Xd, (size_t)ldn * S * 8)); RCK(bufs.get(&g, (size_t)ldn * S * 8)); RCK(bufs.get(&dcorr, (size_t)ldn * S * 8));
    RCK(bufs.get(&red, (size_t)3 * S * 8));
    const int64_t ldmw = (m + 3) & ~(int64_t)3, ldnw = (n + 3) & ~(int64_t)3;
    RCK(bufs.get(&Bw, (size_t)ldmw * S * sizeof(T)));
    RCK(bufs.get(&Xw, (size_t)ldnw * S * sizeof(T))); RCK(bufs.get(&gw, (size_t)ldnw * S * sizeof(T))); RCK(bufs.get(&yw, (size_t)ldnw * S * sizeof(T)));
    cudaEvent_t ev[4];
    for (auto& e : ev) RCK(cudaEventCreate(&e));
    struct EvGuard { cudaEvent_t* e; ~EvGuard() { for (int i = 0; i < 4; ++i) cudaEventDestroy(e[i]); } } evg{ev};
    float ms = 0;
    RCK(cudaEventRecord(ev[0], 0));
    RCK(cudaMemcpy2D(Bd, ldm * 8, B, ldb * 8, m * 8, S, on_device(B) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice));
    // ---- x_0 in the working precision (Eq. 3) ----
    cast_down_kernel<T><<<grid2(m, S), 256>>>(Bd, ldm, m, S, nullptr, Bw, ldmw);
    RCK(cudaGetLastError());
    RCK(cudaDeviceSynchronize());
    RCI(ct_qr_solve(h, Bw, ldmw, S, Xw, ldnw));
    add_up_kernel<T><<<grid2(n, S), 256>>>(Xw, ldnw, n, S, nullptr, 0, Xd, ldn, nullptr, 0);
    RCK(cudaGetLastError());
    RCK(cudaEventRecord(ev[1], 0));
    RCK(cudaEventSynchronize(ev[1]));
    RCK(cudaEventElapsedTime(&ms, ev[0], ev[1]));
    info->ms_initial_solve = ms;
    std::vector<double> hred((size_t)3 * S);
    double t_res = 0, t_cor = 0;
    info->iters_done = 0; info->converged = 0;
    for (int it = 0; it < max_iters; ++it) {
        // ---- r = b - A x,  g = A^T r  (fp64) ----
        RCK(cudaEventRecord(ev[1], 0));
        if (A) {
            RCK(spmm(*A, Xd, ldn, S, -1.0, 1.0, Bd, ldm, r, ldm));
            RCK(spmm(*At, r, ldm, S, 1.0, 0.0, nullptr, 0, g, ldn));
        } else {
            RCK(cudaMemcpy2DAsync(r, ldm * 8, Bd, ldm * 8, m * 8, S, cudaMemcpyDeviceToDevice, 0));
            RCI(ct_qr_gemm(0, m, S, n, -1.0, Ad, lda, Xd, ldn, 1.0, r, ldm, CTQR_F64, 0));
            RCI(ct_qr_gemm(1, n, S, m, 1.0, Ad, lda, r, ldm, 0.0, g, ldn, CTQR_F64, 0));
        }
        colreduce_kernel<0><<<(unsigned)S, 256>>>(g, ldn, n, red);               // scale: max |g| per slice
        colreduce_kernel<1><<<(unsigned)S, 256>>>(g, ldn, n, red + 2 * S);       // ||g||^2 per slice (reported)
        cast_down_kernel<T><<<grid2(n, S), 256>>>(g, ldn, n, S, red, gw, ldnw);
        RCK(cudaGetLastError());
        RCK(cudaEventRecord(ev[2], 0));
        RCK(cudaDeviceSynchronize());
        // ---- d = R^{-1} R^{-T} g  (working precision) ----
        RCI(ct_qr_trsm_t(h, gw, ldnw, S, yw, ldnw));
        RCI(ct_qr_trsm(h, yw, ldnw, S, gw, ldnw));
        add_up_kernel<T><<<grid2(n, S), 256>>>(gw, ldnw, n, S, red, 1, Xd, ldn, dcorr, ldn);
        colreduce_kernel<1><<<(unsigned)S, 256>>>(dcorr, ldn, n, red + S);       // ||d||^2 per slice
        colreduce_kernel<1><<<(unsigned)S, 256>>>(Xd, ldn, n, red);             // ||x||^2 per slice (scale no longer needed)
        RCK(cudaGetLastError());
        RCK(cudaEventRecord(ev[3], 0));
        RCK(cudaMemcpy(hred.data(), red, (size_t)3 * S * 8, cudaMemcpyDeviceToHost));
        RCK(cudaEventElapsedTime(&ms, ev[1], ev[2])); t_res += ms;
        RCK(cudaEventElapsedTime(&ms, ev[2], ev[3])); t_cor += ms;
        double worst = 0, gmax = 0;
        for (int64_t s = 0; s < S; ++s) {
            const double xn = sqrt(hred[s]), dn = sqrt(hred[S + s]);
            worst = std::max(worst, xn > 0 ? dn / xn : dn);
            gmax = std::max(gmax, sqrt(hred[2 * S + s]));
        }
        if (it < CTQR_REFINE_MAX_ITERS) { info->correction[it] = worst; info->gradient[it] = gmax; }
        info->iters_done = it + 1;
        if (!(worst == worst)) return ctqr_internal_set_error(CTQR_ERR_STATE, "refinement produced NaN", "");
        if (tol > 0 && worst <= tol) { info->converged = 1; break; }
    }
    info->ms_residual = t_res; info->ms_correction = t_cor;
    RCK(cudaMemcpy2D(X, ldx * 8, Xd, ldn * 8, n * 8, S, on_device(X) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    RCK(cudaEventRecord(ev[3], 0));
    RCK(cudaEventSynchronize(ev[3]));
    RCK(cudaEventElapsedTime(&ms, ev[0], ev[3]));
    info->ms_total = ms;
    return 0;
}

extern "C" int ct_qr_solve_refined(ctqr_handle_t h, const ctqr_csr_t* A, const ctqr_csr_t* At, const void* A_dense, int64_t lda,
                                   const double* B, int64_t ldb, int64_t S, double* X, int64_t ldx,
                                   int32_t max_iters, double tol, ctqr_refine_info_t* info) {
    ctqr_stats_t st;
    if (!h) return ctqr_internal_set_error(-1, "handle is NULL", "");
    RCI(ct_qr_get_stats(h, &st));
    const int64_t m = st.m, n = st.n;
    const bool sparse = A != nullptr || At != nullptr;
    if (sparse) {
        if (!A || A->m != m || A->n != n || A->nnz < 0 || !A->rowptr || (A->nnz > 0 && (!A->colidx || !A->vals)))
            return ctqr_internal_set_error(-2, "A must be an m x n CSR matrix matching the factor", "");
        if (!At || At->m != n || At->n != m || At->nnz != A->nnz || !At->rowptr || (At->nnz > 0 && (!At->colidx || !At->vals)))
            return ctqr_internal_set_error(-3, "At must be the n x m CSR transpose of A", "");
        if (A_dense) return ctqr_internal_set_error(-4, "give either the CSR pair or the dense matrix, not both", "");
        if (m > INT32_MAX) return ctqr_internal_set_error(-3, "CSR column indices are 32-bit: m too large for At", "");
    } else {
        if (!A_dense) return ctqr_internal_set_error(-4, "no operator: A / At (CSR) or A_dense (fp64, device) is required", "");
        if (lda < m) return ctqr_internal_set_error(-5, "lda < m", "");
        if (!on_device(A_dense)) return ctqr_internal_set_error(-4, "A_dense must be a device pointer", "");
    }
    if (!B) return ctqr_internal_set_error(-6, "B is NULL", "");
    if (ldb < m) return ctqr_internal_set_error(-7, "ldb < m", "");
    if (S < 0) return ctqr_internal_set_error(-8, "S < 0", "");
    if (!X) return ctqr_internal_set_error(-9, "X is NULL", "");
    if (ldx < n) return ctqr_internal_set_error(-10, "ldx < n", "");
    if (max_iters < 0) return ctqr_internal_set_error(-11, "max_iters < 0", "");
    if (!info) return ctqr_internal_set_error(-13, "info is NULL", "");
    memset(info, 0, sizeof *info);
    if (S == 0) return 0;
    if (st.out_of_core) return ctqr_internal_set_error(CTQR_ERR_STATE, "the refined solve needs an in-core factor", "");
    Bufs bufs;
    DevCsr dA{}, dAt{};
    if (sparse) {
        dA.m = m; dA.n = n; dAt.m = n; dAt.n = m;
        RCK(device_view(bufs, A->rowptr, (size_t)m + 1, &dA.rowptr));
        RCK(device_view(bufs, A->colidx, (size_t)A->nnz, &dA.colidx));
        RCK(device_view(bufs, A->vals, (size_t)A->nnz, &dA.vals));
        RCK(device_view(bufs, At->rowptr, (size_t)n + 1, &dAt.rowptr));
        RCK(device_view(bufs, At->colidx, (size_t)At->nnz, &dAt.colidx));
        RCK(device_view(bufs, At->vals, (size_t)At->nnz, &dAt.vals));
    }
    const int dt = ct_qr_dtype(h);
    return dt == CTQR_F64
        ? refined_typed<double>(h, m, n, sparse ? &dA : nullptr, sparse ? &dAt : nullptr, (const double*)A_dense, lda, B, ldb, S, X, ldx, max_iters, tol, info, bufs)
        : refined_typed<float>(h, m, n, sparse ? &dA : nullptr, sparse ? &dAt : nullptr, (const double*)A_dense, lda, B, ldb, S, X, ldx, max_iters, tol, info, bufs);
}
