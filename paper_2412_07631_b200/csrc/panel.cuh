// panel.cuh -- SURVEY.md 8a row a1: unblocked Householder factorisation of an IB-wide inner
// panel, the latency-bound heart of a blocked dgeqrf (Eq. 2).
//
// Design (differs from a LAPACK geqr2 loop, same arithmetic): the m_k x IB inner panel is
// spread over G co-resident CTAs (cooperative launch); every thread keeps RPT rows x IB
// columns in REGISTERS for the whole kernel.  Column j needs sigma^2 = sum x_i^2 and
// w_c = v^T a_c; both follow from s_c = sum_{i>j} x_i a_c[i] (c = 0..IB-1, one pass, before
// beta is known):  sigma^2 = s_j,  w_c = a_c[j] + s_c/(alpha-beta).  The same pass also yields
// V[:,0:j]^T v_j, so the inner T factor comes for free.  Hence ONE grid-wide reduction per
// column: warp-shuffle transpose-reduce -> shared memory -> per-CTA partial in global ->
// software grid barrier (release/acquire counter) -> every CTA sums the G partials in the
// same fixed order (bit-identical scalars everywhere, deterministic run to run).
// The update by reflector j and the dot products for column j+1 are fused into one register pass.
#pragma once
#include "common.cuh"
#include "kernels.h"

namespace ctqr {

// Sum IB per-thread values across the 32 lanes of a warp.  On return lane l holds in v[0] the
// warp total of column (l * IB) / 32 (IB = 32: column l; IB = 16: l>>1; IB = 8: l>>2).
template <typename T, int IB>
__device__ __forceinline__ void warp_transpose_reduce(T (&v)[IB], int lane) {
    int k = IB / 2;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        if (k >= 1) {
            const bool upper = (lane & off) != 0;
#pragma unroll
            for (int i = 0; i < IB / 2; ++i) {
                if (i < k) {
                    T send = upper ? v[i] : v[i + k];
                    T keep = upper ? v[i + k] : v[i];
                    v[i] = keep + shfl_xor(send, off);
                }
            }
            k >>= 1;
        } else {
            v[0] = v[0] + shfl_xor(v[0], off);
        }
    }
}

template <typename T, int IB, int RPT, int NT>
__global__ void __launch_bounds__(NT, 1) panel_geqr2_kernel(PanelArgs<T> p) {
    static_assert(IB == 8 || IB == 16 || IB == 32, "IB");
    constexpr int NW = NT / 32;
    constexpr int NG = NT / IB;                 // reducer groups for the cross-CTA sum
    constexpr int LPC = 32 / IB;                // lanes per column after the warp reduce
    __shared__ T sh_warp[NW][IB];
    __shared__ T sh_red[NG][IB];
    __shared__ T sh_tw[IB];                     // c > j: tau*w_c
    __shared__ T sh_scal[4];                    // denom, beta, tau, flag(sigma2 != 0)
    __shared__ T sh_T[IB][IB + 1];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x, G = gridDim.x;
    const int ibw = p.ibw;
    T* __restrict__ A = p.A;

    int64_t row[RPT];
    T a[RPT][IB];
#pragma unroll
    for (int q = 0; q < RPT; ++q) {
        row[q] = p.jb + ((int64_t)q * G + cta) * NT + tid;
#pragma unroll
        for (int c = 0; c < IB; ++c)
            a[q][c] = (row[q] < p.m && c < ibw) ? A[row[q] + (p.jb + c) * p.lda] : T(0);
    }
    if (cta == 0)
        for (int i = tid; i < IB * (IB + 1); i += NT) (&sh_T[0][0])[i] = T(0);

    unsigned bar_target = p.bar_base;

    // Reduce acc[] over the whole grid; afterwards warp 0 lane c (< IB) holds s_c and rj_c.
    auto grid_reduce = [&](T (&acc)[IB], int step, T& s_out, T& rj_out) {
        const int par = step & 1;
        warp_transpose_reduce<T, IB>(acc, lane);
        if ((lane % LPC) == 0) sh_warp[warp][lane / LPC] = acc[0];
        __syncthreads();
        if (tid < IB) {
            T t = sh_warp[0][tid];
#pragma unroll
            for (int w = 1; w < NW; ++w) t += sh_warp[w][tid];
            __stcg(&p.part[((size_t)par * G + cta) * IB + tid], t);
        }
        __syncthreads();
        bar_target += (unsigned)G;
        if (tid == 0) {
            __threadfence();
            red_release_add_u32(p.bar, 1u);
            while ((int)(ld_acquire_u32(p.bar) - bar_target) < 0) { }
            __threadfence();
        }
        __syncthreads();
        {
            // fixed summation order (same in every CTA); loads batched 4 deep to overlap L2 latency
            const int c = tid % IB, grp = tid / IB;
            const T* pp = p.part + (size_t)par * G * IB + c;
            T t = T(0);
            for (int b = grp; b < G; b += 4 * NG) {
                T v0 = __ldcg(pp + (size_t)b * IB);
                T v1 = (b + NG < G) ? __ldcg(pp + (size_t)(b + NG) * IB) : T(0);
                T v2 = (b + 2 * NG < G) ? __ldcg(pp + (size_t)(b + 2 * NG) * IB) : T(0);
                T v3 = (b + 3 * NG < G) ? __ldcg(pp + (size_t)(b + 3 * NG) * IB) : T(0);
                t += v0; t += v1; t += v2; t += v3;
            }
            sh_red[grp][c] = t;
        }
        __syncthreads();
        if (tid < IB) {
            T t = sh_red[0][tid];
#pragma unroll
            for (int gI = 1; gI < NG; ++gI) t += sh_red[gI][tid];
            s_out = t;
            rj_out = __ldcg(&p.rowbuf[par * IB + tid]);
        }
    };

    // dots for column jn: acc[c] = sum over own rows strictly below the pivot row jb+jn
    // (jn is a compile-time constant at every call site after unrolling)
    T s_c = T(0), rj_c = T(0);

#pragma unroll
    for (int j = 0; j < IB; ++j) {
        if (j >= ibw) break;
        // ---- (1) dots for column j (fused with the previous update at the end of the loop body
        //          for j > 0; computed here for j == 0) ----
        if (j == 0) {
            T acc[IB];
#pragma unroll
            for (int c = 0; c < IB; ++c) acc[c] = T(0);
#pragma unroll
            for (int q = 0; q < RPT; ++q) {
                const bool below = row[q] > p.jb;
                const T x = below ? a[q][0] : T(0);
#pragma unroll
                for (int c = 0; c < IB; ++c) acc[c] = fma(x, a[q][c], acc[c]);
            }
            if (cta == 0 && tid == 0) {
#pragma unroll
                for (int c = 0; c < IB; ++c) __stcg(&p.rowbuf[0 * IB + c], a[0][c]);
            }
            grid_reduce(acc, 0, s_c, rj_c);
        }
        // ---- (2) scalars of reflector j (warp 0, lanes < IB; identical in every CTA) ----
        if (warp == 0) {
            const T alpha = __shfl_sync(0xffffffffu, rj_c, j);
            const T sigma2 = __shfl_sync(0xffffffffu, s_c, j);
            T beta = alpha, tauj = T(0), denom = T(1);
            const bool nz = sigma2 != T(0);
            if (nz) {
                T nrm = Num<T>::sqrt(fma(alpha, alpha, sigma2));
                beta = (alpha >= T(0)) ? -nrm : nrm;
                tauj = Num<T>::div(beta - alpha, beta);
                denom = alpha - beta;
            }
            // g_c = row-j entry + s_c/denom : c > j gives w_c, c < j gives (V^T v_j)_c
            const T gc = nz ? rj_c + Num<T>::div(s_c, denom) : T(0);
            if (lane < IB) sh_tw[lane] = tauj * gc;
            if (lane == 0) { sh_scal[0] = denom; sh_scal[1] = beta; sh_scal[2] = tauj; sh_scal[3] = nz ? T(1) : T(0); }
            if (cta == 0) {
                // inner T: T[0:j, j] = -tau_j * T[0:j,0:j] * g[0:j],  T[j][j] = tau_j
                T sum = T(0);
                for (int b = 0; b < j; ++b) {
                    const T gb = __shfl_sync(0xffffffffu, gc, b);
                    if (lane < j && b >= lane) sum = fma(sh_T[lane][b], gb, sum);
                }
                __syncwarp();
                if (lane < j) sh_T[lane][j] = -tauj * sum;
                if (lane == j) sh_T[j][j] = tauj;
                if (lane == 0) p.tau[p.jb + j] = tauj;
            }
        }
        __syncthreads();
        const T denom = sh_scal[0], beta = sh_scal[1];
        const bool nz = sh_scal[3] != T(0);
        T tw[IB];
#pragma unroll
        for (int c = 0; c < IB; ++c) tw[c] = (c > j) ? sh_tw[c] : T(0);
        // ---- (3) apply reflector j to own rows, fused with the dots for column j+1 ----
        T acc[IB];
#pragma unroll
        for (int c = 0; c < IB; ++c) acc[c] = T(0);
#pragma unroll
        for (int q = 0; q < RPT; ++q) {
            const int64_t piv = p.jb + j;
            if (nz) {
                if (row[q] > piv) {
                    const T v = Num<T>::div(a[q][j], denom);
                    a[q][j] = v;
#pragma unroll
                    for (int c = j + 1; c < IB; ++c) a[q][c] = fma(-tw[c], v, a[q][c]);
                } else if (row[q] == piv) {
                    a[q][j] = beta;
#pragma unroll
                    for (int c = j + 1; c < IB; ++c) a[q][c] -= tw[c];
                }
            }
            if (j + 1 < IB) {
                const bool below = row[q] > piv + 1;
                const T x = below ? a[q][(j + 1) % IB] : T(0);
#pragma unroll
                for (int c = 0; c < IB; ++c) acc[c] = fma(x, a[q][c], acc[c]);
            }
        }
        if (j + 1 < ibw) {
            if (cta == 0 && tid == j + 1) {
#pragma unroll
                for (int c = 0; c < IB; ++c) __stcg(&p.rowbuf[((j + 1) & 1) * IB + c], a[0][c]);
            }
            grid_reduce(acc, j + 1, s_c, rj_c);
        }
    }

    // ---- write back: V below the diagonal, explicit 0/1 on and above it; R to Rd ----
    const int64_t off = p.jb - p.j0;    // position of this inner block inside the panel
#pragma unroll
    for (int q = 0; q < RPT; ++q) {
        if (row[q] >= p.m) continue;
        const bool diagblk = (cta == 0 && q == 0 && tid < IB);
#pragma unroll
        for (int c = 0; c < IB; ++c) {
            if (c >= ibw) continue;
            T val = a[q][c];
            if (diagblk && c >= tid) {
                p.Rd[(off + tid) + (off + c) * (int64_t)p.ldrd] = val;
                val = (c == tid) ? T(1) : T(0);
            }
            A[row[q] + (p.jb + c) * p.lda] = val;
        }
    }
    // rows j0 .. jb-1 of these columns are finished R entries of the panel's diagonal block
    if (cta == G - 1) {
        const int nr = (int)off;
        for (int i = tid; i < nr * ibw; i += NT) {
            int r = i % nr, c = i / nr;
            T* src = &A[(p.j0 + r) + (p.jb + c) * p.lda];
            p.Rd[r + (off + c) * (int64_t)p.ldrd] = *src;
            *src = T(0);
        }
    }
    if (cta == 0) {
        __syncthreads();
        for (int i = tid; i < IB * IB; i += NT) p.Tin[i] = sh_T[i % IB][i / IB];
    }
}

}  // namespace ctqr
