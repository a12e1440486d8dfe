// solve_small.cuh -- fused small-S path of the solve (SURVEY.md 8a row a6 for S <= 8, the
// memory-bound regime of PAPER.md Fig. 1 / Eq. 3: every element of V is read once per batch and
// used for only 4S flop).  The generic path launches 5 kernels per panel; at S = 1..8 that is
// launch-latency-bound (the factor was read at 2 % of the HBM copy bandwidth).  Here ONE
// cooperative kernel applies all P panels:
//   * the rows of B are dealt to the CTAs once (fixed contiguous chunks) and live in shared memory
//     for the whole kernel;
//   * per panel: every CTA forms its partial W = V_k^T B over its own rows, the partials are
//     summed across the grid in a fixed order with two flag-in-data ("LL") exchanges (publish
//     partials -> element owners reduce -> everyone gathers the sums): no atomics, deterministic;
//   * every CTA then forms T_k^T W redundantly and updates its own rows B -= V_k (T_k^T W),
//     re-reading its slice of V_k from L2.
#pragma once
#include "common.cuh"
#include "kernels.h"
#include "panel.cuh"      // ll_store / ll_load / ll_value (flag-in-data slots)

namespace ctqr {

constexpr int kSmallS = 8;          // most right-hand sides the fused path handles
constexpr int kSmallThreads = 256;

template <typename T>
struct SmallQtArgs {
    const T* A; int64_t lda; int64_t m, n; int nb, P;
    const T* Tm;                    // P blocks of nb x nb (ld nb)
    T* B; int64_t ldb; int S;
    uint4* part;                    // [2][G][nb * kSmallS] LL slots: per-CTA partial W
    uint4* sums;                    // [2][nb * kSmallS] LL slots: reduced W
    unsigned seq_base;              // step numbers seq_base + 1 .. seq_base + P are used by this launch
    int rpc;                        // rows per CTA (multiple of 32)
};

template <typename T>
__global__ void __launch_bounds__(kSmallThreads, 1) apply_qt_small_kernel(SmallQtArgs<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NB = 128, SM = kSmallS, NT = kSmallThreads, NW = NT / 32;
    T* Bs = reinterpret_cast<T*>(smem_raw);                 // [SM][rpc]   own rows of B, transposed
    T* Wp = Bs + (size_t)SM * p.rpc;                         // [NB][SM]    partial, then summed W
    T* W2 = Wp + NB * SM;                                   // [NB][SM]    T^T W
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = blockIdx.x, G = gridDim.x, S = p.S;
    const int64_t r0 = (int64_t)g * p.rpc, r1 = min(p.m, r0 + p.rpc);
    const int nrows = (int)max((int64_t)0, r1 - r0);

    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, r = i - s * p.rpc;
        Bs[i] = (s < S && r < nrows) ? p.B[r0 + r + (int64_t)s * p.ldb] : T(0);
    }
    __syncthreads();

    for (int k = 0; k < p.P; ++k) {
        const int64_t j0 = (int64_t)k * NB;
        const int kw = (int)min((int64_t)NB, p.n - j0);
        const unsigned seq = p.seq_base + (unsigned)k + 1u;
        const int par = k & 1;
        const T* V = p.A + j0 * p.lda;                       // column c of the panel at V + c * lda, rows absolute
        const int ra = (int)max((int64_t)0, j0 - r0);        // first own row (local) that takes part
        // ---- partial W[c][s] = sum over own rows of V[r, c] * B[r, s] ----
        // (four columns per pass so that 4 x rows/32 independent loads are in flight per lane)
        for (int cb = warp; cb < NB; cb += 4 * NW) {
            T acc[4][SM];
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int s = 0; s < SM; ++s) acc[u][s] = T(0);
            const T* vc = V + r0;
#pragma unroll 2
            for (int r = ra + lane; r < nrows; r += 32) {
                T v[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int c = cb + u * NW;
                    v[u] = (c < kw) ? __ldg(vc + (int64_t)c * p.lda + r) : T(0);
                }
#pragma unroll
                for (int s = 0; s < SM; ++s) {
                    const T b = Bs[s * p.rpc + r];
#pragma unroll
                    for (int u = 0; u < 4; ++u) acc[u][s] = fma(v[u], b, acc[u][s]);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int s = 0; s < SM; ++s) {
                    T t = acc[u][s];
#pragma unroll
                    for (int off = 16; off >= 1; off >>= 1) t += shfl_xor(t, off);
                    if (lane == 0) Wp[(cb + u * NW) * SM + s] = t;
                }
        }
        __syncthreads();
        // ---- publish the CTA's partial (LL slots) ----
        uint4* mine = p.part + ((size_t)par * G + g) * (NB * SM);
        for (int e = tid; e < NB * SM; e += NT) ll_store(mine + e, Wp[e], seq);
        // ---- element owners reduce over the CTAs in a fixed order: element e belongs to CTA e % G ----
        {
            const uint4* all = p.part + (size_t)par * G * (NB * SM);
            for (int e = g + warp * G; e < NB * SM; e += NW * G) {
                T t = T(0);
                for (int b = lane; b < G; b += 32) {
                    const uint4* slot = all + (size_t)b * (NB * SM) + e;
                    uint4 r = ll_load(slot);
                    while (r.y != seq || r.w != seq) r = ll_load(slot);
                    t += ll_value<T>(r);
                }
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) t += shfl_xor(t, off);
                if (lane == 0) ll_store(p.sums + (size_t)par * (NB * SM) + e, t, seq);
            }
        }
        // ---- everyone gathers the sums ----
        for (int e = tid; e < NB * SM; e += NT) {
            const uint4* slot = p.sums + (size_t)par * (NB * SM) + e;
            uint4 r = ll_load(slot);
            while (r.y != seq || r.w != seq) r = ll_load(slot);
            Wp[e] = ll_value<T>(r);
        }
        __syncthreads();
        // ---- W2 = T_k^T W  (T upper triangular: W2[r][s] = sum_{k <= r} T[k][r] W[k][s]) ----
        {
            const T* Tk = p.Tm + (size_t)k * NB * NB;
            const int r = tid & (NB - 1), sh = (tid >> 7) * (SM / 2);
            T acc[SM / 2];
#pragma unroll
            for (int s = 0; s < SM / 2; ++s) acc[s] = T(0);
            if (r < kw)
#pragma unroll 4
                for (int q = 0; q <= r; ++q) {
                    const T t = __ldg(Tk + q + (size_t)r * NB);
#pragma unroll
                    for (int s = 0; s < SM / 2; ++s) acc[s] = fma(t, Wp[q * SM + sh + s], acc[s]);
                }
#pragma unroll
            for (int s = 0; s < SM / 2; ++s) W2[r * SM + sh + s] = acc[s];
        }
        __syncthreads();
        // ---- own rows: B[r, :] -= V[r, 0:kw] * W2 ----
        for (int r = ra + tid; r < nrows; r += NT) {
            T d[SM];
#pragma unroll
            for (int s = 0; s < SM; ++s) d[s] = T(0);
            const T* vr = V + r0 + r;
#pragma unroll 8
            for (int c = 0; c < kw; ++c) {
                const T v = __ldg(vr + (int64_t)c * p.lda);
#pragma unroll
                for (int s = 0; s < SM; ++s) d[s] = fma(v, W2[c * SM + s], d[s]);
            }
#pragma unroll
            for (int s = 0; s < SM; ++s) Bs[s * p.rpc + r] -= d[s];
        }
        __syncthreads();
    }
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, r = i - s * p.rpc;
        if (s < S && r < nrows) p.B[r0 + r + (int64_t)s * p.ldb] = Bs[i];
    }
}

}  // namespace ctqr
