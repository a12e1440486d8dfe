// small.cuh -- the small, latency-bound kernels around the contractions:
//   larft_kernel     SURVEY.md 8a row a2: T from the Gram matrix V^T V and tau (column recurrence
//                    T[0:j,j] = -tau_j T[0:j,0:j] (V[:,0:j]^T v_j), T[j][j] = tau_j)
//   ttw_kernel       W <- T^T * (sum of split-K partials of V^T C)   (middle step of larfb, a3/a6)
//   trsm_diag_kernel X_i = R_ii^{-1} C_i by back-substitution on one diagonal block (a7; the
//                    "R22 X2 = C2" task of PAPER.md:L62-73)
#pragma once
#include "common.cuh"
#include <algorithm>

namespace ctqr {

// ---- larft from Gram partials ------------------------------------------------------------
// G partials: nsplit buffers of nbw x nbw (ld = ldg, stride gstride) holding alpha*V^T V slices.
// One CTA of 1024 threads: 8 threads per row of T cooperate on each dot product.
template <typename T>
__global__ void __launch_bounds__(1024, 1)
larft_kernel(const T* __restrict__ Gp, int nsplit, int64_t gstride, int ldg, const T* __restrict__ tau,
             int nbw, T* __restrict__ Tout, int ldt) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // One (nbw x (nbw+1)) array: column j holds G[:,j] until step j, then T[:,j] (in place).
    T* Ms = reinterpret_cast<T*>(smem_raw);
    const int tid = threadIdx.x;
    const int ld = nbw + 1;
    for (int i = tid; i < nbw * nbw; i += blockDim.x) {
        int a = i % nbw, j = i / nbw;
        T s = T(0);
        for (int sp = 0; sp < nsplit; ++sp) s += Gp[(size_t)sp * gstride + a + (size_t)j * ldg];
        Ms[a * ld + j] = s;
    }
    __syncthreads();
    const int a = tid >> 3, sub = tid & 7;           // row a (< 128), 8 threads per row
    for (int j = 0; j < nbw; ++j) {
        const T tj = tau[j];
        T sum = T(0);
        if (a < j) {
            for (int b = a + sub; b < j; b += 8) sum = fma(Ms[a * ld + b], Ms[b * ld + j], sum);
        }
        sum += shfl_xor(sum, 4);
        sum += shfl_xor(sum, 2);
        sum += shfl_xor(sum, 1);
        __syncthreads();
        if (sub == 0 && a < nbw) {
            if (a < j) Ms[a * ld + j] = -tj * sum;
            else if (a == j) Ms[a * ld + j] = tj;
        }
        __syncthreads();
    }
    for (int i = tid; i < nbw * nbw; i += blockDim.x) {
        int r = i % nbw, c = i / nbw;
        Tout[r + (size_t)c * ldt] = (r <= c) ? Ms[r * ld + c] : T(0);
    }
}

// ---- W <- T^T * sum_s Wp[s] ---------------------------------------------------------------
// Wp: nsplit partial buffers (kw x N, ld = ldw, stride wstride).  T: kw x kw upper (ld = ldt).
// Output W (kw x N, ld = ldo).  Each CTA handles CW columns.
template <typename T, int CW>
__global__ void __launch_bounds__(256)
ttw_kernel(const T* __restrict__ Wp, int nsplit, int64_t wstride, int64_t ldw, const T* __restrict__ Tm, int ldt,
           int kw, int64_t N, T* __restrict__ Wout, int64_t ldo) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Tt = reinterpret_cast<T*>(smem_raw);          // [kw][kw+1]  Tt[i][k] = T[k][i]
    T* Ws = Tt + (size_t)kw * (kw + 1);              // [CW][kw]
    const int tid = threadIdx.x;
    const int64_t c0 = (int64_t)blockIdx.x * CW;
    for (int i = tid; i < kw * kw; i += 256) {
        int k = i % kw, col = i / kw;                // T[k][col], contiguous in k
        Tt[col * (kw + 1) + k] = Tm[k + (size_t)col * ldt];
    }
    for (int i = tid; i < kw * CW; i += 256) {
        int k = i % kw, c = i / kw;
        T s = T(0);
        if (c0 + c < N)
            for (int sp = 0; sp < nsplit; ++sp) s += Wp[(size_t)sp * wstride + k + (c0 + c) * ldw];
        Ws[c * kw + k] = s;
    }
    __syncthreads();
    for (int i = tid; i < kw * CW; i += 256) {
        int r = i % kw, c = i / kw;
        if (c0 + c >= N) continue;
        T acc = T(0);
        const T* tr = Tt + r * (kw + 1);
        const T* wc = Ws + c * kw;
        for (int k = 0; k <= r; ++k) acc = fma(tr[k], wc[k], acc);
        Wout[r + (c0 + c) * ldo] = acc;
    }
}

// ---- diagonal-block triangular solve -------------------------------------------------------
// R: kw x kw upper triangular (ld = ldr, explicit storage); C: kw x S in (ld = ldc); X out (ld = ldx).
// Thread layout: 16 threads per right-hand side (a half-warp), each owning rows r = sub + 16 q in
// registers; back-substitution row by row, x_i broadcast inside the half-warp by shuffle.
// Same operation order as scalar back-substitution restricted to the block.
template <typename T, int KW>
__global__ void __launch_bounds__(256)
trsm_diag_kernel(const T* __restrict__ R, int ldr, int kw, const T* __restrict__ C, int64_t ldc, int64_t S,
                 T* __restrict__ X, int64_t ldx) {
    constexpr int Q = KW / 16;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Rs = reinterpret_cast<T*>(smem_raw);          // [KW][KW+1]: Rs[i*(KW+1) + r] = R[r][i] (column i contiguous)
    const int tid = threadIdx.x, sub = tid & 15;
    const int64_t col = (int64_t)blockIdx.x * 16 + (tid >> 4);
    for (int i = tid; i < KW * KW; i += 256) {
        int r = i % KW, c = i / KW;
        Rs[c * (KW + 1) + r] = (r < kw && c < kw) ? R[r + (size_t)c * ldr] : (r == c ? T(1) : T(0));
    }
    T x[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        int r = sub + 16 * q;
        x[q] = (col < S && r < kw) ? C[r + col * ldc] : T(0);
    }
    __syncthreads();
#pragma unroll
    for (int qi = Q - 1; qi >= 0; --qi) {
        for (int si = 15; si >= 0; --si) {
            const int i = qi * 16 + si;
            const T* rc = Rs + i * (KW + 1);
            T xi = T(0);
            if (sub == si) { xi = Num<T>::div(x[qi], rc[i]); x[qi] = xi; }
            xi = __shfl_sync(0xffffffffu, xi, si, 16);
#pragma unroll
            for (int q = 0; q < Q; ++q) {
                if (q > qi) continue;
                const int r = sub + 16 * q;
                if (r < i) x[q] = fma(-rc[r], xi, x[q]);
            }
        }
    }
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        int r = sub + 16 * q;
        if (col < S && r < kw) X[r + col * ldx] = x[q];
    }
}

// ---- utility kernels -----------------------------------------------------------------------
template <typename T>
__global__ void copy2d_kernel(const T* __restrict__ src, int64_t lds, T* __restrict__ dst, int64_t ldd,
                              int64_t rows, int64_t cols) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (int64_t c = blockIdx.y; c < cols; c += gridDim.y)
        if (r < rows) dst[r + c * ldd] = src[r + c * lds];
}

// R accessor: assemble dense upper-triangular R from the in-matrix off-diagonal blocks and Rd.
template <typename T>
__global__ void gather_R_kernel(const T* __restrict__ A, int64_t lda, const T* __restrict__ Rd, int nb,
                                int64_t n, T* __restrict__ R, int64_t ldr) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    for (int64_t c = blockIdx.y; c < n; c += gridDim.y) {
        int64_t pc = c / nb, pr = r / nb;
        T v = T(0);
        if (pr < pc) v = A[r + c * lda];
        else if (pr == pc) v = Rd[(size_t)pc * nb * nb + (r - pc * nb) + (c - pc * nb) * (int64_t)nb];
        R[r + c * ldr] = v;
    }
}

// first index with a zero on the diagonal of R (from the Rd blocks); result[0] = min index or n
template <typename T>
__global__ void find_zero_diag_kernel(const T* __restrict__ Rd, int nb, int64_t n, int* result) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    int64_t pj = j / nb, o = j - pj * nb;
    if (Rd[(size_t)pj * nb * nb + o + o * (int64_t)nb] == T(0)) atomicMin(result, (int)j);
}

}  // namespace ctqr
