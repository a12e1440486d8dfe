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
constexpr int kSmallThreads = 512;
constexpr int kSmallChunk = 16;     // rows are dealt to the CTAs in chunks of this many, round-robin
// padded leading dimensions in shared memory: T_k is read as DMMA fragments in fp64 (ld == 4 mod 16 doubles is
// conflict-free) and row-per-thread in fp32 (odd ld); W / T^T W as DMMA B fragments in fp64 (ld 12), plain in fp32
template <typename T> struct SmallLd { static constexpr int T_ = 129, W = kSmallS; };
template <> struct SmallLd<double> { static constexpr int T_ = 132, W = 12; };

__device__ __forceinline__ void cp_async_elem(double* smem, const double* g) { cp_async8(smem, g, 8); }
__device__ __forceinline__ void cp_async_elem(float* smem, const float* g) { cp_async4(smem, g, 4); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

// Per-phase timers of CTA 0 (builds with -DCTQR_SMALL_PROFILE only): nanoseconds summed over the panels.
#ifdef CTQR_SMALL_PROFILE
__device__ unsigned long long g_small_prof[16];
#define CTQR_PH(i)                                                                       \
    if (tid == 0 && g == 0) {                                                            \
        unsigned long long t1_;                                                          \
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1_));                          \
        if (ph_t0) g_small_prof[i] += t1_ - ph_t0;                                       \
        ph_t0 = t1_;                                                                     \
    }
#else
#define CTQR_PH(i)
#endif

template <typename T>
struct SmallQtArgs {
    const T* A; int64_t lda; int64_t m, n; int nb, P;
    const T* Tm;                    // P blocks of nb x nb (ld nb)
    T* B; int64_t ldb; int S;
    uint4* part;                    // [2][G][nb * kSmallS] LL slots: per-CTA partial W
    uint4* sums;                    // [2][nb * kSmallS] LL slots: reduced W
    unsigned seq_base;              // step numbers seq_base + 1 .. seq_base + P are used by this launch
    int rpc;                        // local rows per CTA (multiple of kSmallChunk)
    int64_t kl;                     // 0 = dense; > 0: V(i, j) == 0 for i - j > kl (opt->lower_bandwidth), rows below are skipped
};

template <typename T>
__global__ void __launch_bounds__(kSmallThreads, 1) apply_qt_small_kernel(SmallQtArgs<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NB = 128, SM = kSmallS, NT = kSmallThreads, NW = NT / 32, CH = kSmallChunk, LDT = SmallLd<T>::T_, LDW = SmallLd<T>::W;
    constexpr int NQ = NT / NB, SQ = SM / NQ;
    constexpr bool F64 = sizeof(T) == 8;                   // fp64: the three products run on DMMA.8x8x4
    T* Ts = reinterpret_cast<T*>(smem_raw);                 // [NB][LDT]   T_k (column r at Ts + r * LDT)
    T* Ds = Ts;                                             // partial updates of the column groups; T_k is dead by then
    T* Wp = Ts + NB * LDT;                                  // [NB][LDW]   partial, then summed W
    T* W2 = Wp + NB * LDW;                                  // [NB][LDW]   T^T W
    T* Bs = W2 + NB * LDW;                                   // [SM][ldbs]  own rows of B, transposed
    const int ldbs = p.rpc + 4;                             // == 4 (mod 16): conflict-free DMMA fragment loads
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = blockIdx.x, G = gridDim.x, S = p.S;
    auto row_of = [&](int lr) -> int64_t { return ((int64_t)(lr / CH) * G + g) * CH + (lr % CH); };
    auto stage_t = [&](int k) {
        const T* Tk = p.Tm + (size_t)k * NB * NB;
        if constexpr (F64) {                                 // 16-byte copies: ld 132 keeps every column 16-byte aligned
            for (int e = 2 * tid; e < NB * NB; e += 2 * NT) cp_async16(Ts + (e >> 7) * LDT + (e & (NB - 1)), Tk + e, 16);
        } else {
            for (int e = tid; e < NB * NB; e += NT) cp_async_elem(Ts + (e >> 7) * LDT + (e & (NB - 1)), Tk + e);
        }
        cp_async_commit();
    };
    // local rows [la, nl) take part in panel k: la = first local row at or below row j0 (j0 is a multiple of CH)
    auto first_local = [&](int64_t j0) -> int {
        const int64_t q0 = j0 / CH;
        return q0 > g ? (int)((q0 - g + G - 1) / G) * CH : 0;
    };
    const int nl = first_local(round_up(p.m, (int64_t)CH));  // local rows that exist (the last chunk may be ragged)
    stage_t(0);
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        Bs[s * ldbs + lr] = (s < S && lr < nl && row < p.m) ? p.B[row + (int64_t)s * p.ldb] : T(0);
    }
    __syncthreads();

    for (int k = 0; k < p.P; ++k) {
        const int64_t j0 = (int64_t)k * NB;
        const int kw = (int)min((int64_t)NB, p.n - j0);
        const unsigned seq = p.seq_base + (unsigned)k + 1u;
        const int par = k & 1;
        const T* V = p.A + j0 * p.lda;                       // column c of the panel at V + c * lda, rows absolute
        const int la = first_local(j0);
        // band promise (p.kl > 0): V_k is zero below row kl + j0 + kw, so the panel stops at local row le
        const int le = p.kl > 0 ? min(nl, first_local(round_up(min(p.m, p.kl + j0 + kw), (int64_t)CH))) : nl;
        const int na = le - la;
        unsigned long long ph_t0 = 0; (void)ph_t0;
        CTQR_PH(0)
        // ---- partial W[c][s] = sum over own rows of V[r, c] * B[r, s] ----
        if constexpr (F64) {
            // warp w: columns 8w .. 8w+7 (M), right-hand sides (N), 4 consecutive local rows per k-step
            const int c = warp * 8 + (lane >> 2);
            const T* vc = V + (int64_t)c * p.lda;
            const T* bs = Bs + (lane >> 2) * ldbs + (lane & 3);
            const bool okc = c < kw;
            double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};   // four independent DMMA chains
#pragma unroll 8
            for (int t = 0; t < na / 4; t += 4) {            // na is a multiple of 16: a multiple of 4 steps
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int64_t row = row_of(la + 4 * (t + h) + (lane & 3));
                    const double a = (okc && row < p.m) ? __ldg(vc + row) : 0.0;
                    dmma884(c0[h], c1[h], a, bs[la + 4 * (t + h)]);
                }
            }
            Wp[c * LDW + 2 * (lane & 3)] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
            Wp[c * LDW + 2 * (lane & 3) + 1] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
        } else {
            // a warp takes 4 columns per pass, lanes over rows: 4 independent loads per lane and row step
            for (int cb = warp; cb < NB; cb += 4 * NW) {
                T acc[4 * SM];
#pragma unroll
                for (int u = 0; u < 4 * SM; ++u) acc[u] = T(0);
#pragma unroll 2
                for (int lr = la + lane; lr < le; lr += 32) {
                    const int64_t row = row_of(lr);
                    T v[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int c = cb + u * NW;
                        v[u] = (c < kw && row < p.m) ? __ldg(V + (int64_t)c * p.lda + row) : T(0);
                    }
#pragma unroll
                    for (int s = 0; s < SM; ++s) {
                        const T b = Bs[s * ldbs + lr];
#pragma unroll
                        for (int u = 0; u < 4; ++u) acc[u * SM + s] = fma(v[u], b, acc[u * SM + s]);
                    }
                }
                warp_transpose_reduce<T, 4 * SM>(acc, lane);  // lane l: total of acc[l] = (column cb + (l / SM) * NW, rhs l % SM)
                Wp[(cb + (lane / SM) * NW) * LDW + (lane % SM)] = acc[0];
            }
        }
        __syncthreads();
        CTQR_PH(1)
        // ---- publish the CTA's partial (LL slots) ----
        uint4* mine = p.part + ((size_t)par * G + g) * (NB * SM);
        for (int e = tid; e < NB * SM; e += NT) ll_store(mine + e, Wp[(e / SM) * LDW + (e % SM)], seq);
        CTQR_PH(2)
        // ---- pull this CTA's slice of the next panel towards L2 while the exchange is in flight ----
        if (k + 1 < p.P) {
            const int la1 = first_local(j0 + NB);
            const int le1 = p.kl > 0 ? min(nl, first_local(round_up(min(p.m, p.kl + j0 + 2 * NB), (int64_t)CH))) : nl;
            const T* vc = V + (int64_t)(NB + (tid & (NB - 1))) * p.lda;
            for (int lr = la1 + (tid >> 7) * CH; lr < le1; lr += NQ * CH) {
                const int64_t row = row_of(lr);
                prefetch_l2(vc + row);
                if (F64 && row + 8 < p.m) prefetch_l2(vc + row + 8);
            }
        }
        CTQR_PH(3)
        // ---- element owners reduce over the CTAs in a fixed order: element e belongs to CTA e % G ----
        {
            const uint4* all = p.part + (size_t)par * G * (NB * SM);
            constexpr int MAXB = 5;                          // loads of a lane issued before the first flag is examined
            for (int e = g + warp * G; e < NB * SM; e += NW * G) {
                T t = T(0);
                for (int b0 = lane; b0 < G; b0 += 32 * MAXB) {
                    uint4 r[MAXB];
#pragma unroll
                    for (int u = 0; u < MAXB; ++u) {
                        const int b = b0 + u * 32;
                        if (b < G) r[u] = ll_load(all + (size_t)b * (NB * SM) + e);
                    }
#pragma unroll
                    for (int u = 0; u < MAXB; ++u) {
                        const int b = b0 + u * 32;
                        if (b < G) {
                            while (r[u].y != seq || r[u].w != seq) r[u] = ll_load(all + (size_t)b * (NB * SM) + e);
                            t += ll_value<T>(r[u]);
                        }
                    }
                }
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) t += shfl_xor(t, off);
                if (lane == 0) ll_store(p.sums + (size_t)par * (NB * SM) + e, t, seq);
            }
        }
        CTQR_PH(4)
        // ---- everyone gathers the sums (both slots of a thread in flight) ----
        {
            const uint4* sl = p.sums + (size_t)par * (NB * SM);
            uint4 r[NB * SM / NT];
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) r[u] = ll_load(sl + tid + u * NT);
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) {
                const int e = tid + u * NT;
                while (r[u].y != seq || r[u].w != seq) r[u] = ll_load(sl + e);
                Wp[(e / SM) * LDW + (e % SM)] = ll_value<T>(r[u]);
            }
        }
        CTQR_PH(5)
        cp_async_wait<0>();
        __syncthreads();
        CTQR_PH(6)
        // ---- W2 = T_k^T W  (T upper triangular: W2[r][s] = sum_{q <= r} T[q][r] W[q][s]) ----
        if constexpr (F64) {
            // warp w: rows 8w .. 8w+7 of W2 (M), right-hand sides (N), q in steps of 4 up to the diagonal
            const int r = warp * 8 + (lane >> 2);
            const T* tr = Ts + r * LDT + (lane & 3);
            const T* wq = Wp + (lane & 3) * LDW + (lane >> 2);
            double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 2
            for (int t = 0; t < 2 * warp + 2; t += 4) {      // the last group may run past the diagonal: masked by q <= r
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int q = 4 * (t + h) + (lane & 3);
                    const double a = (q <= r && r < kw) ? tr[4 * (t + h)] : 0.0;
                    dmma884(c0[h], c1[h], a, wq[4 * (t + h) * LDW]);
                }
            }
            W2[r * LDW + 2 * (lane & 3)] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
            W2[r * LDW + 2 * (lane & 3) + 1] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
        } else {
            const int r = tid & (NB - 1), sh = (tid >> 7) * SQ;
            T acc[SQ];
#pragma unroll
            for (int s = 0; s < SQ; ++s) acc[s] = T(0);
            if (r < kw)
#pragma unroll 4
                for (int q = 0; q <= r; ++q) {
                    const T t = Ts[r * LDT + q];
#pragma unroll
                    for (int s = 0; s < SQ; ++s) acc[s] = fma(t, Wp[q * LDW + sh + s], acc[s]);
                }
#pragma unroll
            for (int s = 0; s < SQ; ++s) W2[r * LDW + sh + s] = acc[s];
        }
        __syncthreads();
        CTQR_PH(7)
        // ---- own rows: B[r, :] -= V[r, 0:kw] * W2, the columns split over CS groups ----
        if constexpr (F64) {
            // unit = (8 local rows, one of CS column ranges); a warp walks its units, 4 columns per k-step
            const int mt = na / 8;
            int CS = 1;
            while (CS < 8 && mt * CS < NW && 2 * CS * na * SM <= NB * LDT) CS *= 2;   // at least one unit per warp
            const int steps = NB / 4 / CS;
            for (int u = warp; u < mt * CS; u += NW) {
                const int cs = u / mt, l0 = (u - cs * mt) * 8;
                const int64_t row = row_of(la + l0 + (lane >> 2));
                const bool okr = row < p.m;
                const int cbeg = cs * steps * 4 + (lane & 3);
                const T* vr = V + (int64_t)cbeg * p.lda + row;
                const T* wb = W2 + cbeg * LDW + (lane >> 2);
                double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 8
                for (int t = 0; t < steps; t += 4) {           // steps = 32 / CS: a multiple of 4
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const double a = (okr && cbeg + 4 * (t + h) < kw) ? __ldg(vr + (int64_t)(4 * (t + h)) * p.lda) : 0.0;
                        dmma884(c0[h], c1[h], a, wb[4 * (t + h) * LDW]);
                    }
                }
                c0[0] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
                c1[0] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
                const int l = l0 + (lane >> 2), s0 = 2 * (lane & 3);
                if (CS == 1) {
                    Bs[s0 * ldbs + la + l] -= c0[0];
                    Bs[(s0 + 1) * ldbs + la + l] -= c1[0];
                } else {
                    Ds[(cs * SM + s0) * na + l] = c0[0];
                    Ds[(cs * SM + s0 + 1) * na + l] = c1[0];
                }
            }
            __syncthreads();
            if (CS > 1) {
                for (int idx = tid; idx < na * SM; idx += NT) {
                    const int s = idx / na, l = idx - s * na;
                    T t = T(0);
                    for (int cs = 0; cs < CS; ++cs) t += Ds[(cs * SM + s) * na + l];
                    Bs[s * ldbs + la + l] -= t;
                }
                __syncthreads();
            }
        } else {
            int CS = 1;
            while (CS < 8 && 2 * CS * na <= NT) CS *= 2;
            const int cpc = (kw + CS - 1) / CS;
            for (int idx = tid; idx < na * CS; idx += NT) {
                const int cs = idx / na, lr = la + idx - cs * na;
                const int64_t row = row_of(lr);
                T d[SM];
#pragma unroll
                for (int s = 0; s < SM; ++s) d[s] = T(0);
                if (row < p.m) {
                    const int c0 = cs * cpc, c1 = min(kw, c0 + cpc);
                    const T* vr = V + row;
#pragma unroll 16
                    for (int c = c0; c < c1; ++c) {
                        const T v = __ldg(vr + (int64_t)c * p.lda);
#pragma unroll
                        for (int s = 0; s < SM; ++s) d[s] = fma(v, W2[c * LDW + s], d[s]);
                    }
                }
                if (CS == 1) {
#pragma unroll
                    for (int s = 0; s < SM; ++s) Bs[s * ldbs + lr] -= d[s];
                } else {
#pragma unroll
                    for (int s = 0; s < SM; ++s) Ds[(cs * SM + s) * na + idx - cs * na] = d[s];
                }
            }
            __syncthreads();
            if (CS > 1) {
                for (int idx = tid; idx < na * SM; idx += NT) {
                    const int s = idx / na, l = idx - s * na;
                    T t = T(0);
                    for (int cs = 0; cs < CS; ++cs) t += Ds[(cs * SM + s) * na + l];
                    Bs[s * ldbs + la + l] -= t;
                }
                __syncthreads();
            }
        }
        CTQR_PH(8)
        if (k + 1 < p.P) stage_t(k + 1);                     // lands during the next panel's partial products and exchange
    }
    cp_async_wait<0>();
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        if (s < S && lr < nl && row < p.m) p.B[row + (int64_t)s * p.ldb] = Bs[s * ldbs + lr];
    }
}

// -------------------------------------------------------------------------------------------
// Fused blocked TRSM for S <= 8 (task list PAPER.md L62-73): bottom-up over the
// diagonal blocks, X_i = R_ii^{-1} C_i (inverted diagonal blocks, see trinv_kernel), then
// C_j <- C_j - R_ji X_i for all rows above.  One cooperative kernel:
//   * the rows of C are dealt to the CTAs in chunks of kTrsmChunk rows, round-robin, and stay in
//     shared memory: every block's rows are spread over several CTAs (short critical path) and
//     every CTA has rows throughout the matrix (balanced until the very top);
//   * per block the owners of its rows publish them through flag-in-data slots (one set of slots
//     per block: only the owners write, so no slot is reused inside a launch), every CTA gathers
//     them and forms X_i redundantly from R_ii^{-1}, which was prefetched into shared memory with
//     cp.async during the previous block;
//   * every CTA updates its own rows, streaming its part of the block column of R exactly once,
//     the 128 columns split over up to 8 thread groups so that enough loads are in flight.
// -------------------------------------------------------------------------------------------
constexpr int kTrsmThreads = 512;
constexpr int kTrsmChunk = 16;

template <typename T>
struct SmallTrsmArgs {
    const T* A; int64_t lda; int64_t n; int nb, P;
    const T* Rinv;                  // P blocks of nb x nb (ld nb)
    T* X; int64_t ldx; int S;       // in: C[0:n, :], out: X
    uint4* slots;                   // [P][nb * kSmallS] LL slots
    unsigned seq;                   // step number of this launch (unique per handle)
    int rpc;                        // local rows per CTA (multiple of kTrsmChunk)
};

template <typename T>
__global__ void __launch_bounds__(kTrsmThreads, 1) trsm_small_kernel(SmallTrsmArgs<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NB = 128, SM = kSmallS, NT = kTrsmThreads, CH = kTrsmChunk, NQ = NT / NB, SQ = SM / NQ;
    constexpr int VEC = 16 / (int)sizeof(T);
    T* Rs = reinterpret_cast<T*>(smem_raw);                 // [NB][NB]   R_ii^{-1}
    T* Ci = Rs + NB * NB;                                   // [NB][SM]   gathered C_i
    T* Xi = Ci + NB * SM;                                   // [NB][SM]   X_i
    T* Ds = Xi + NB * SM;                                   // [<=8][SM][lim] partial updates (groups * lim <= NT)
    T* Cs = Ds + SM * NT;                                   // [SM][rpc]  own rows, transposed
    const int tid = threadIdx.x;
    const int g = blockIdx.x, G = gridDim.x, S = p.S;
    auto row_of = [&](int lr) -> int64_t { return ((int64_t)(lr / CH) * G + g) * CH + (lr % CH); };
    auto stage_rinv = [&](int i) {
        const T* Ri = p.Rinv + (size_t)i * NB * NB;
        for (int e = tid * VEC; e < NB * NB; e += NT * VEC) cp_async16(Rs + e, Ri + e, 16);
        cp_async_commit();
    };
    stage_rinv(p.P - 1);
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        Cs[i] = (s < S && row < p.n) ? p.X[row + (int64_t)s * p.ldx] : T(0);
    }
    __syncthreads();
    for (int i = p.P - 1; i >= 0; --i) {
        const int64_t i0 = (int64_t)i * NB;
        const int kw = (int)min((int64_t)NB, p.n - i0);
        if ((int64_t)g * CH >= i0 + kw) break;                // no rows in or above this block: all own rows are final
        uint4* slots = p.slots + (size_t)i * (NB * SM);
        // ---- owners publish their rows of C_i ----
        for (int e = tid; e < NB * SM; e += NT) {
            const int rr = e / SM, s = e - rr * SM;
            const int64_t q = (i0 + rr) / CH;
            if (rr < kw && (int)(q % G) == g) ll_store(slots + e, Cs[s * p.rpc + (int)(q / G) * CH + (int)((i0 + rr) % CH)], p.seq);
        }
        // ---- gather C_i (NB * SM / NT = 2 slots per thread, both loads in flight) ----
        {
            uint4 r[NB * SM / NT];
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) {
                const int e = tid + u * NT;
                r[u] = (e / SM < kw) ? ll_load(slots + e) : make_uint4(0u, p.seq, 0u, p.seq);
            }
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) {
                const int e = tid + u * NT;
                while (r[u].y != p.seq || r[u].w != p.seq) r[u] = ll_load(slots + e);
                Ci[e] = (e / SM < kw) ? ll_value<T>(r[u]) : T(0);
            }
        }
        cp_async_wait<0>();
        __syncthreads();
        // ---- X_i = R_ii^{-1} C_i  (zero below the diagonal and in the padding) ----
        {
            const int r = tid & (NB - 1), sh = (tid >> 7) * SQ;
            T acc[SQ];
#pragma unroll
            for (int s = 0; s < SQ; ++s) acc[s] = T(0);
#pragma unroll 8
            for (int k = 0; k < NB; ++k) {
                const T t = Rs[r + k * NB];
#pragma unroll
                for (int s = 0; s < SQ; ++s) acc[s] = fma(t, Ci[k * SM + sh + s], acc[s]);
            }
#pragma unroll
            for (int s = 0; s < SQ; ++s) Xi[r * SM + sh + s] = acc[s];
        }
        __syncthreads();
        if (i > 0) stage_rinv(i - 1);
        // ---- own rows above the block: C[r, :] -= R[r, i0:i0+kw] X_i ; own rows inside it: C[r, :] = X_i ----
        const int64_t qlim = (i0 + kw + CH - 1) / CH;          // chunks that start below i0 + kw
        const int lim = (int)((qlim - g + G - 1) / G) * CH;     // local rows in those chunks (>= CH here)
        int CS = 1;
        while (CS < 8 && 2 * CS * lim <= NT) CS *= 2;
        const int cpc = (kw + CS - 1) / CS;
        for (int idx = tid; idx < lim * CS; idx += NT) {
            const int cs = idx / lim, lr = idx - cs * lim;
            const int64_t row = row_of(lr);
            T d[SM];
#pragma unroll
            for (int s = 0; s < SM; ++s) d[s] = T(0);
            if (row < i0) {
                const int c0 = cs * cpc, c1 = min(kw, c0 + cpc);
                const T* rr = p.A + row + i0 * p.lda;
#pragma unroll 16
                for (int c = c0; c < c1; ++c) {
                    const T v = __ldg(rr + (int64_t)c * p.lda);
#pragma unroll
                    for (int s = 0; s < SM; ++s) d[s] = fma(v, Xi[c * SM + s], d[s]);
                }
            } else if (row < i0 + kw && cs == 0) {
#pragma unroll
                for (int s = 0; s < SM; ++s) Cs[s * p.rpc + lr] = Xi[(int)(row - i0) * SM + s];
            }
            if (CS == 1) {
                if (row < i0)
#pragma unroll
                    for (int s = 0; s < SM; ++s) Cs[s * p.rpc + lr] -= d[s];
            } else {
#pragma unroll
                for (int s = 0; s < SM; ++s) Ds[(cs * SM + s) * lim + lr] = d[s];
            }
        }
        __syncthreads();
        if (CS > 1) {
            for (int idx = tid; idx < lim * SM; idx += NT) {
                const int s = idx / lim, lr = idx - s * lim;
                if (row_of(lr) < i0) {
                    T t = T(0);
                    for (int cs = 0; cs < CS; ++cs) t += Ds[(cs * SM + s) * lim + lr];
                    Cs[s * p.rpc + lr] -= t;
                }
            }
            __syncthreads();
        }
    }
    cp_async_wait<0>();
    __syncthreads();
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        if (s < S && row < p.n) p.X[row + (int64_t)s * p.ldx] = Cs[i];
    }
}

}  // namespace ctqr
