// small.cuh -- the small, latency-bound kernels around the contractions:
//   larft_kernel     SURVEY.md 8a row a2: T from the Gram matrix V^T V and tau (column recurrence
//                    T[0:j,j] = -tau_j T[0:j,0:j] (V[:,0:j]^T v_j), T[j][j] = tau_j)
//   ttw_kernel       W <- T^T * (sum of split-K partials of V^T C)   (middle step of larfb, a3/a6)
//   trsm_diag_kernel X_i = R_ii^{-1} C_i by back-substitution on one diagonal block (a7; the
//                    "R22 X2 = C2" task of PAPER.md:L62-73)
#pragma once
#include "common.cuh"
#include "kernels.h"
#include "gemm_mma.cuh"
#include <algorithm>

namespace ctqr {

// ---- larft from Gram partials, block by block ------------------------------------------------
// The panel kernel has already written the ib x ib inner T factors into the diagonal blocks of
// T_k.  For two reflector blocks H1 = I - V1 T1 V1^T, H2 = I - V2 T2 V2^T:
//   H1 H2 = I - [V1 V2] [[T1, -T1 (V1^T V2) T2], [0, T2]] [V1 V2]^T,
// so block column b of T_k is  T[0:ob, blk] = -T[0:ob,0:ob] * G[0:ob, blk] * T_bb  with G = V^T V
// (same values as the column recurrence T[0:j,j] = -tau_j T[0:j,0:j] V[:,0:j]^T v_j, two small
// matrix products per inner block instead of one dependent step per column).
// G partials: nseg buffers of nbw x nbw (ld = ldg, stride gstride), see SegInfo.  One CTA.
template <typename T>
__global__ void __launch_bounds__(1024, 1)
larft_kernel(const T* __restrict__ Gp, SegInfo seg, int64_t gstride, int ldg, int nbw, int ib,
             T* __restrict__ Tk, int ldt) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Ts = reinterpret_cast<T*>(smem_raw);          // [nbw][nbw+1]  Ts[r*ld + c] = T[r][c]
    const int ld = nbw + 1;
    T* Zs = Ts + (size_t)nbw * ld;                   // [nbw][ib+1]
    const int ldz = ib + 1;
    T* Gs = Zs + (size_t)nbw * ldz;                  // [nbw][ib+1]
    const int tid = threadIdx.x;
    for (int i = tid; i < nbw * nbw; i += blockDim.x) {
        const int r = i % nbw, c = i / nbw;
        Ts[r * ld + c] = (r <= c && r / ib == c / ib) ? Tk[r + (size_t)c * ldt] : T(0);
    }
    __syncthreads();
    for (int ob = ib; ob < nbw; ob += ib) {
        const int ibw = min(ib, nbw - ob);
        // stage G[0:ob, blk] = sum of its partials (independent, coalesced loads)
        for (int e = tid; e < ob * ibw; e += blockDim.x) {
            const int a = e % ob, k = e / ob, col = ob + k;
            T gv = T(0);
            if (seg.L > 0) {            // compact stream-K partial tiles (128 x BN slots), see gemm_mma.cuh
                const int64_t t = col / seg.BN, slot = (int64_t)128 * seg.BN;
                const int nseg = sk_nseg(t, seg.KT, seg.L);
                const T* base = Gp + (t + sk_first_cta(t, seg.KT, seg.L)) * slot + a + (col % seg.BN) * 128;
                for (int sp = 0; sp < nseg; ++sp) gv += base[(int64_t)sp * slot];
            } else {
                for (int sp = 0; sp < seg.nsplit; ++sp) gv += Gp[(size_t)sp * gstride + a + (size_t)col * ldg];
            }
            Gs[a * ldz + k] = gv;
        }
        __syncthreads();
        // Z = G[0:ob, blk] * T_bb   (T_bb upper triangular: k <= c)
        for (int e = tid; e < ob * ibw; e += blockDim.x) {
            const int a = e % ob, c = e / ob;
            T z = T(0);
            for (int k = 0; k <= c; ++k) z = fma(Gs[a * ldz + k], Ts[(ob + k) * ld + ob + c], z);
            Zs[a * ldz + c] = z;
        }
        __syncthreads();
        // T[0:ob, blk] = -T[0:ob,0:ob] * Z   (upper triangular: k >= a)
        for (int e = tid; e < ob * ibw; e += blockDim.x) {
            const int a = e % ob, c = e / ob;
            T t = T(0);
            for (int k = a; k < ob; ++k) t = fma(Ts[a * ld + k], Zs[k * ldz + c], t);
            Ts[a * ld + ob + c] = -t;
        }
        __syncthreads();
    }
    for (int i = tid; i < nbw * nbw; i += blockDim.x) {
        const int r = i % nbw, c = i / nbw;
        Tk[r + (size_t)c * ldt] = (r <= c) ? Ts[r * ld + c] : T(0);
    }
}

// ---- W <- T^T * sum_s Wp[s] ---- (scalar kernel for the narrow in-panel blocks, kw <= 32) ------
// Wp: nsplit partial buffers (kw x N, ld = ldw, stride wstride).  T: kw x kw upper (ld = ldt).
// Each CTA handles cw columns with kw * cw <= 64 outputs; the (many) split-K partials of an
// output are summed by a group of tpe threads in a fixed order, then combined by shuffles.
template <typename T>
__global__ void __launch_bounds__(256)
ttw_kernel(const T* __restrict__ Wp, int nsplit, int64_t wstride, int64_t ldw, const T* __restrict__ Tm, int ldt,
           int kw, int64_t N, T* __restrict__ Wout, int64_t ldo, int cw, int tpe) {
    __shared__ T Tt[32][33];                         // Tt[i][k] = T[k][i]
    __shared__ T Ws[64];                             // [cw][kw]
    const int tid = threadIdx.x;
    const int64_t c0 = (int64_t)blockIdx.x * cw;
    for (int i = tid; i < kw * kw; i += 256) {
        const int k = i % kw, col = i / kw;
        Tt[col][k] = Tm[k + (size_t)col * ldt];
    }
    const int ne = kw * cw;
    {
        const int e = tid / tpe, sub = tid % tpe;
        T s = T(0);
        if (e < ne) {
            const int k = e % kw, c = e / kw;
            if (c0 + c < N)
                for (int sp = sub; sp < nsplit; sp += tpe) s += Wp[(size_t)sp * wstride + k + (c0 + c) * ldw];
        }
        for (int off = tpe >> 1; off >= 1; off >>= 1) s += shfl_xor(s, off);
        if (e < ne && sub == 0) Ws[e] = s;
    }
    __syncthreads();
    if (tid < ne) {
        const int r = tid % kw, c = tid / kw;
        if (c0 + c < N) {
            T acc = T(0);
            for (int k = 0; k <= r; ++k) acc = fma(Tt[r][k], Ws[c * kw + k], acc);
            Wout[r + (c0 + c) * ldo] = acc;
        }
    }
}

// ---- W <- T^T * sum_s Wp[s] on the tensor cores (kw up to 128) -------------------------------
// One CTA per 64-column tile (the tile of the stream-K product that wrote the partials), 8 warps of
// 32 x 32.  T (upper triangular, explicit zeros below) sits in shared memory K-contiguous:
// Ts[m][k] = T[k][m]; the summed partial tile Ws[n][k] likewise.  Rows of T^T below the warp's
// m-range are zero, so the k-loop stops at the warp's last row.
template <typename T>
__global__ void __launch_bounds__(256, 1)
ttw_mma_kernel(const T* __restrict__ Wp, SegInfo seg, int64_t wstride, int64_t ldw, const T* __restrict__ Tm, int ldt,
               int kw, int64_t N, T* __restrict__ Wout, int64_t ldo) {
    using P = MmaPolicy<T>;
    constexpr int BN = 64, KMAX = 128, LD = KMAX + 4, MT = 32 / P::MFRAG, NTL = 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Ts = reinterpret_cast<T*>(smem_raw);          // [KMAX][LD]
    T* Ws = Ts + KMAX * LD;                          // [BN][LD]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp & 3, wn = warp >> 2;
    const int grp = lane >> 2, tig = lane & 3;
    const int64_t c0 = (int64_t)blockIdx.x * BN;
    const int kpad = (kw + P::KSTEP - 1) / P::KSTEP * P::KSTEP;
    const int nseg = seg.L > 0 ? sk_nseg(((int64_t)blockIdx.x * BN) / seg.BN, seg.KT, seg.L) : seg.nsplit;
    for (int i = tid; i < KMAX * kpad; i += 256) {
        const int k = i % kpad, mm = i / kpad;
        Ts[mm * LD + k] = (k < kw && mm < kw) ? Tm[k + (size_t)mm * ldt] : T(0);
    }
    for (int i = tid; i < BN * kpad; i += 256) {
        const int k = i % kpad, c = i / kpad;
        T s = T(0);
        if (k < kw && c0 + c < N) {
            if (seg.L > 0) {            // compact stream-K partial tiles (128 x 64 slots)
                const int64_t t = c0 / seg.BN, slot = (int64_t)128 * seg.BN;
                const T* base = Wp + (t + sk_first_cta(t, seg.KT, seg.L)) * slot + k + (int64_t)(c0 % seg.BN + c) * 128;
                for (int sp = 0; sp < nseg; ++sp) s += base[(int64_t)sp * slot];
            } else {
                for (int sp = 0; sp < nseg; ++sp) s += Wp[(size_t)sp * wstride + k + (c0 + c) * ldw];
            }
        }
        Ws[c * LD + k] = s;
    }
    __syncthreads();
    if (wm * 32 >= kw) return;
    T acc[MT][NTL][P::ACC];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NTL; ++j)
#pragma unroll
            for (int q = 0; q < P::ACC; ++q) acc[i][j][q] = T(0);
    const int kend = min(kpad, wm * 32 + 32);
    for (int kk = 0; kk < kend; kk += P::KSTEP)
        P::template kstep<true, MT, NTL, LD, LD>(Ts, Ws, kk, wm * 32, wn * 32, grp, tig, acc);
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NTL; ++j)
#pragma unroll
            for (int q = 0; q < P::ACC; ++q) {
                const int r = wm * 32 + i * P::MFRAG + P::frag_row(q, grp);
                const int64_t c = c0 + wn * 32 + j * 8 + P::frag_col(q, tig);
                if (r < kw && c < N) Wout[r + c * ldo] = acc[i][j][q];
            }
}

// ---- sum of the compact stream-K partial tiles of a (kw <= 128) x N product -> dense W (ld = ldo) ----
template <typename T>
__global__ void __launch_bounds__(256)
partial_sum_kernel(const T* __restrict__ Wp, SegInfo seg, int kw, int64_t N, T* __restrict__ Wout, int64_t ldo) {
    const int64_t c = (int64_t)blockIdx.x * 2 + (threadIdx.x >> 7);
    const int k = threadIdx.x & 127;
    if (c >= N || k >= kw) return;
    const int64_t t = c / seg.BN, slot = (int64_t)128 * seg.BN;
    const int nseg = sk_nseg(t, seg.KT, seg.L);
    const T* base = Wp + (t + sk_first_cta(t, seg.KT, seg.L)) * slot + k + (c % seg.BN) * 128;
    T s = T(0);
    for (int sp = 0; sp < nseg; ++sp) s += base[(int64_t)sp * slot];
    Wout[k + c * ldo] = s;
}

// ---- out = op(M) * in for a 128 x 128 triangular M and a narrow right-hand side ----------------
// The small products of the solve (and of the look-ahead block): W <- T_k^T (sum of the stream-K
// partial tiles) [TRANS, PARTIAL] and X_i <- R_ii^{-1} C_i [in place, !TRANS].  A tensor-core
// contraction launch costs ~16 us for these 128 x S x 128 products (4 CTAs busy) plus ~12 us for
// the partial sum; here one CTA takes 8 columns: M is staged once in shared memory (cp.async in
// fp64), the 128 x 8 slab of the input is summed / loaded by all 512 threads (segments dealt to 4
// thread groups, combined in a fixed order: deterministic), fp64 runs on DMMA.8x8x4 with the
// triangular k-range, fp32 on FFMA.  M upper triangular with explicit zeros below the diagonal.
constexpr int kMm128Threads = 512;
constexpr int kMm128Cols = 8;
template <typename T> struct Mm128Ld { static constexpr int M = 129, X = kMm128Cols; };
template <> struct Mm128Ld<double> { static constexpr int M = 132, X = 12; };

template <typename T, bool TRANS, bool PARTIAL>
__global__ void __launch_bounds__(kMm128Threads, 1)
mm128_kernel(const T* __restrict__ Mg, int ldm, const T* In, int64_t ldin, SegInfo seg, int64_t N, T* Out, int64_t ldo) {
    constexpr int NB = 128, NC = kMm128Cols, NT = kMm128Threads, NG = NT / NB, LDM = Mm128Ld<T>::M, LDX = Mm128Ld<T>::X;
    constexpr bool F64 = sizeof(T) == 8;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Ms = reinterpret_cast<T*>(smem_raw);          // [NB][LDM]: Ms[c * LDM + r] = M[r][c]
    T* Xs = Ms + NB * LDM;                           // [NB][LDX]: the input slab
    T* Ps = Xs + NB * LDX;                           // [NG][NB][NC + 1]: per-group partial sums
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t c0 = (int64_t)blockIdx.x * NC;
    if constexpr (F64) {
        for (int e = 2 * tid; e < NB * NB; e += 2 * NT) cp_async16(Ms + (e >> 7) * LDM + (e & (NB - 1)), Mg + (e & (NB - 1)) + (size_t)(e >> 7) * ldm, 16);
        cp_async_commit();
    } else {
        for (int e = tid; e < NB * NB; e += NT) Ms[(e >> 7) * LDM + (e & (NB - 1))] = Mg[(e & (NB - 1)) + (size_t)(e >> 7) * ldm];
    }
    {
        const int k = tid & (NB - 1), grp = tid >> 7;
        if constexpr (PARTIAL) {
            // segments sp = grp (mod NG) of the tile the columns belong to (NC divides the tile width)
            const int64_t t = c0 / seg.BN, slot = (int64_t)NB * seg.BN;
            const int nseg = sk_nseg(t, seg.KT, seg.L);
            const T* base = In + (t + sk_first_cta(t, seg.KT, seg.L)) * slot + k + (c0 % seg.BN) * NB;
            T acc[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[c] = T(0);
#pragma unroll 2
            for (int sp = grp; sp < nseg; sp += NG) {
                const T* b = base + (int64_t)sp * slot;
#pragma unroll
                for (int c = 0; c < NC; ++c) acc[c] += (c0 + c < N) ? b[c * NB] : T(0);
            }
#pragma unroll
            for (int c = 0; c < NC; ++c) Ps[(grp * NB + k) * (NC + 1) + c] = acc[c];
            __syncthreads();
            for (int e = tid; e < NB * NC; e += NT) {
                const int kk = e / NC, c = e - kk * NC;
                T v = T(0);
#pragma unroll
                for (int q = 0; q < NG; ++q) v += Ps[(q * NB + kk) * (NC + 1) + c];
                Xs[kk * LDX + c] = v;
            }
        } else {
            for (int c = grp; c < NC; c += NG) Xs[k * LDX + c] = (c0 + c < N) ? In[k + (c0 + c) * ldin] : T(0);
        }
    }
    if constexpr (F64) cp_async_wait<0>();
    __syncthreads();
    if constexpr (F64) {
        // warp w: rows 8w .. 8w+7 (16 warps x 8 rows), k in steps of 4 over the non-zero range of op(M)
        const int r = warp * 8 + (lane >> 2);
        const int tb = TRANS ? 0 : 2 * warp, te = TRANS ? 2 * warp + 2 : NB / 4;
        double d0[2] = {0.0, 0.0}, d1[2] = {0.0, 0.0};
        const T* xq = Xs + (lane & 3) * LDX + (lane >> 2);
#pragma unroll 4
        for (int t = tb; t < te; t += 2) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int k = 4 * (t + h) + (lane & 3);
                const double a = TRANS ? Ms[r * LDM + k] : Ms[k * LDM + r];
                dmma884(d0[h], d1[h], a, xq[4 * (t + h) * LDX]);
            }
        }
        const int64_t c = c0 + 2 * (lane & 3);
        if (c < N) Out[r + c * ldo] = d0[0] + d0[1];
        if (c + 1 < N) Out[r + (c + 1) * ldo] = d1[0] + d1[1];
    } else {
        const int r = tid & (NB - 1), ch = (tid >> 7) * (NC / NG);
        T acc[NC / NG];
#pragma unroll
        for (int c = 0; c < NC / NG; ++c) acc[c] = T(0);
        const int kb = TRANS ? 0 : r, ke = TRANS ? r + 1 : NB;
#pragma unroll 4
        for (int k = kb; k < ke; ++k) {
            const T a = TRANS ? Ms[r * LDM + k] : Ms[k * LDM + r];
#pragma unroll
            for (int c = 0; c < NC / NG; ++c) acc[c] = fma(a, Xs[k * LDX + ch + c], acc[c]);
        }
#pragma unroll
        for (int c = 0; c < NC / NG; ++c)
            if (c0 + ch + c < N) Out[r + (c0 + ch + c) * ldo] = acc[c];
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

// ---- inverse of the diagonal blocks of R (one CTA per block, thread j computes column j) ----------
// X = R_ii^{-1} by back-substitution on the identity, in the working precision.  Used by the blocked
// TRSM so that the diagonal task "R_ii X_i = C_i" becomes a tensor-core product
// X_i = R_ii^{-1} C_i instead of 128 dependent steps per right-hand side.
template <typename T>
__global__ void __launch_bounds__(128)
trinv_kernel(const T* __restrict__ Rd, int nb, int64_t n, T* __restrict__ Rinv, unsigned* __restrict__ cond_bits) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Ms = reinterpret_cast<T*>(smem_raw);          // [nb][nb+1]: R on entry, R^{-1} on exit (in place, column by column)
    const int ld = nb + 1;
    const int64_t i0 = (int64_t)blockIdx.x * nb;
    const int kw = (int)min((int64_t)nb, n - i0);
    const T* R = Rd + (size_t)blockIdx.x * nb * nb;
    for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) {
        const int i = e % nb, k = e / nb;
        Ms[i * ld + k] = (i < kw && k < kw && i <= k) ? R[i + (size_t)k * nb] : T(0);
    }
    __syncthreads();
    const int i = threadIdx.x;
    for (int j = 0; j < kw; ++j) {
        // X[0:j, j] = -X[0:j,0:j] * R[0:j, j] / R[j][j]   (the leading block is already inverted)
        const T xjj = Num<T>::div(T(1), Ms[j * ld + j]);
        T t = T(0);
        if (i < j)
            for (int k = i; k < j; ++k) t = fma(Ms[i * ld + k], Ms[k * ld + j], t);
        __syncthreads();
        if (i < j) Ms[i * ld + j] = -t * xjj;
        else if (i == j) Ms[j * ld + j] = xjj;
        __syncthreads();
    }
    T* out = Rinv + (size_t)blockIdx.x * nb * nb;
    for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) {
        const int r = e % nb, c = e / nb;
        out[r + (size_t)c * nb] = Ms[r * ld + c];
    }
    // conditioning guard: max|R_jj| / min|R_jj| = max|X_jj| / min|X_jj| of this block (a lower bound of cond(R_ii)),
    // max over the blocks through an atomicMax on the float's bit pattern (ratios are >= 1, so the order is the same)
    if (cond_bits && threadIdx.x < 32) {
        float lo = 3.0e38f, hi = 0.f;
        for (int j = threadIdx.x; j < kw; j += 32) {
            const float a = fabsf((float)Ms[j * ld + j]);
            lo = fminf(lo, a); hi = fmaxf(hi, a);
        }
        for (int off = 16; off >= 1; off >>= 1) {
            lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, off));
            hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, off));
        }
        if (threadIdx.x == 0) {
            const float ratio = (lo > 0.f && isfinite(hi)) ? hi / lo : __int_as_float(0x7f800000);
            atomicMax(cond_bits, __float_as_uint(ratio));
        }
    }
}

// Y = R^{-T} C in place on one diagonal block (the transposed solve of ct_qr_trsm_t when the inverted blocks are
// not used): forward substitution y_j = (c_j - sum_{k<j} R[k][j] y_k) / R[j][j], one thread per right-hand side,
// R staged in shared memory, the solution kept in shared memory (column per thread).
constexpr int kTrsmTThreads = 64;
template <typename T>
__global__ void __launch_bounds__(kTrsmTThreads)
trsm_diag_t_kernel(const T* __restrict__ R, int ldr, int kw, T* __restrict__ X, int64_t ldx, int64_t S) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NT = kTrsmTThreads;
    T* Rs = reinterpret_cast<T*>(smem_raw);          // [kw][kw + 1]: Rs[j * ld + k] = R[k][j] (column j contiguous)
    const int ld = kw + 1;
    T* Ys = Rs + (size_t)kw * ld;                    // [kw][NT]
    const int tid = threadIdx.x;
    const int64_t col = (int64_t)blockIdx.x * NT + tid;
    for (int e = tid; e < kw * kw; e += NT) {
        const int k = e % kw, j = e / kw;
        Rs[j * ld + k] = R[k + (size_t)j * ldr];
    }
    __syncthreads();
    if (col >= S) return;
    T* x = X + col * ldx;
    for (int j = 0; j < kw; ++j) {
        T acc = x[j];
        const T* rj = Rs + j * ld;
        for (int k = 0; k < j; ++k) acc = fma(-rj[k], Ys[k * NT + tid], acc);
        Ys[j * NT + tid] = Num<T>::div(acc, rj[j]);
    }
    for (int j = 0; j < kw; ++j) x[j] = Ys[j * NT + tid];
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
