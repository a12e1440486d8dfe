// gemm.cuh -- the dense contractions of the hot path:
//   C <- alpha * op(A) * B + beta * C,  column-major,  op(A) = A^T (A is K x M) or A (M x K),
//   B is K x N.  Optional split-K: gridDim.z slices of K, slice z writes its partial product
//   (alpha applied, beta ignored) to C + z * split_stride.
//
// Two kernel families:
//   gemm_dmma  fp64 on the tensor cores: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, the only
//              native FP64 tensor instruction on sm_100a; tcgen05 has no f64 kind), operands
//              staged global->shared by a multi-stage cp.async (LDGSTS) pipeline into padded,
//              bank-conflict-free tiles, accumulators in registers.
//   gemm_simt  fp32 (FFMA) and fp64 (DFMA) register-tiled kernels: the fp32 product path and
//              the cross-check for the DMMA kernel.
// This is what larfb (Eq. 2 inside a blocked dgeqrf, L52), dormqr (Eq. 3)
// and the GEMM tasks of the blocked TRSM (L66-73) reduce to.
#pragma once
#include "common.cuh"
#include "kernels.h"

namespace ctqr {

// =========================================================================================
// fp64 tensor-core kernel
// =========================================================================================
template <bool TA, int BM, int BN, int WM, int WN, int BK, int STAGES>
struct DmmaCfg {
    static constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN;
    static constexpr int NT = WARPS_M * WARPS_N * 32;
    static constexpr int MT = WM / 8, NTL = WN / 8;
    // K-contiguous tile: [rows][BK + 4]; M-contiguous tile: [BK][BM + 4]  (ld == 4 mod 16 doubles
    // makes the m8n8k4 fragment loads hit 16 distinct 8-byte banks per half-warp)
    static constexpr int LDK = BK + 4;
    static constexpr int LDM = BM + 4;
    static constexpr int A_ELEMS = TA ? BM * LDK : BK * LDM;
    static constexpr int B_ELEMS = BN * LDK;
    static constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_ELEMS * sizeof(double);
};

template <bool TA, int BM, int BN, int WM, int WN, int BK, int STAGES, int MINB>
__global__ void __launch_bounds__(DmmaCfg<TA, BM, BN, WM, WN, BK, STAGES>::NT, MINB)
gemm_dmma_kernel(GemmArgs<double> g) {
    using Cfg = DmmaCfg<TA, BM, BN, WM, WN, BK, STAGES>;
    constexpr int NT = Cfg::NT, MT = Cfg::MT, NTL = Cfg::NTL, LDK = Cfg::LDK, LDM = Cfg::LDM;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* smem = reinterpret_cast<double*>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp % Cfg::WARPS_M, wn = warp / Cfg::WARPS_M;
    const int grp = lane >> 2, tig = lane & 3;
    const int64_t m0 = (int64_t)blockIdx.x * BM, n0 = (int64_t)blockIdx.y * BN;
    const int64_t kbeg = (int64_t)blockIdx.z * g.k_chunk;
    const int64_t kend = min(g.K, kbeg + g.k_chunk);
    const int KT = (int)ceil_div(max((int64_t)0, kend - kbeg), BK);
    double* Cout = g.C + (int64_t)blockIdx.z * g.split_stride;
    const bool split = gridDim.z > 1;

    double acc[MT][NTL][2];
    // accumulators start at (beta/alpha) * C so that the result alpha*acc is exact for |alpha| = 1
    const double cscale = (split || g.beta == 0.0) ? 0.0 : g.beta / g.alpha;
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NTL; ++j) {
            acc[i][j][0] = 0.0; acc[i][j][1] = 0.0;
            if (cscale != 0.0) {
                int64_t m = m0 + wm * WM + i * 8 + grp;
                int64_t n = n0 + wn * WN + j * 8 + 2 * tig;
                if (m < g.M) {
                    if (n < g.N) acc[i][j][0] = cscale * __ldcg(&g.C[m + n * g.ldc]);
                    if (n + 1 < g.N) acc[i][j][1] = cscale * __ldcg(&g.C[m + (n + 1) * g.ldc]);
                }
            }
        }

    auto load_stage = [&](int stage, int kt) {
        double* As = smem + (size_t)stage * Cfg::STAGE_ELEMS;
        double* Bs = As + Cfg::A_ELEMS;
        const int64_t k0 = kbeg + (int64_t)kt * BK;
        // ---- K-contiguous tiles: rows x BK, 2 doubles per 16-byte chunk ----
        auto load_kc = [&](double* S, const double* G, int64_t ld, int64_t r0, int64_t rmax, int rows, int vec_ok) {
            constexpr int CPR = BK / 2;                    // chunks per row
            for (int c = tid; c < rows * CPR; c += NT) {
                int r = c / CPR, ck = (c % CPR) * 2;
                int64_t gr = r0 + r, gk = k0 + ck;
                double* dst = S + r * LDK + ck;
                const double* src = G + gr * ld + gk;
                int valid = (gr < rmax) ? (int)max((int64_t)0, min((int64_t)2, kend - gk)) : 0;
                if (vec_ok) {
                    cp_async16(dst, valid ? src : G, valid * 8);
                } else {
                    cp_async8(dst, valid > 0 ? src : G, valid > 0 ? 8 : 0);
                    cp_async8(dst + 1, valid > 1 ? src + 1 : G, valid > 1 ? 8 : 0);
                }
            }
        };
        if (TA) {
            load_kc(As, g.A, g.lda, m0, g.M, BM, g.a_vec_ok);
        } else {
            // ---- M-contiguous tile: BK x BM ----
            constexpr int CPR = BM / 2;
            for (int c = tid; c < BK * CPR; c += NT) {
                int kk = c / CPR, cm = (c % CPR) * 2;
                int64_t gk = k0 + kk, gm = m0 + cm;
                double* dst = As + kk * LDM + cm;
                const double* src = g.A + gm + gk * g.lda;
                int valid = (gk < kend) ? (int)max((int64_t)0, min((int64_t)2, g.M - gm)) : 0;
                if (g.a_vec_ok) {
                    cp_async16(dst, valid ? src : g.A, valid * 8);
                } else {
                    cp_async8(dst, valid > 0 ? src : g.A, valid > 0 ? 8 : 0);
                    cp_async8(dst + 1, valid > 1 ? src + 1 : g.A, valid > 1 ? 8 : 0);
                }
            }
        }
        load_kc(Bs, g.B, g.ldb, n0, g.N, BN, g.b_vec_ok);
    };

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < KT) load_stage(s, s);
        cp_async_commit();
    }

    for (int kt = 0; kt < KT; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int nk = kt + STAGES - 1;
            if (nk < KT) load_stage(nk % STAGES, nk);
            cp_async_commit();
        }
        const double* As = smem + (size_t)(kt % STAGES) * Cfg::STAGE_ELEMS;
        const double* Bs = As + Cfg::A_ELEMS;
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[MT], b[NTL];
#pragma unroll
            for (int i = 0; i < MT; ++i) {
                int mrow = wm * WM + i * 8 + grp;
                a[i] = TA ? As[mrow * LDK + kk + tig] : As[(kk + tig) * LDM + mrow];
            }
#pragma unroll
            for (int j = 0; j < NTL; ++j) b[j] = Bs[(wn * WN + j * 8 + grp) * LDK + kk + tig];
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NTL; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();

#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NTL; ++j) {
            int64_t m = m0 + wm * WM + i * 8 + grp;
            int64_t n = n0 + wn * WN + j * 8 + 2 * tig;
            if (m < g.M) {
                if (n < g.N) Cout[m + n * g.ldc] = g.alpha * acc[i][j][0];
                if (n + 1 < g.N) Cout[m + (n + 1) * g.ldc] = g.alpha * acc[i][j][1];
            }
        }
}

// =========================================================================================
// SIMT register-tiled kernel (fp32 FFMA product path; fp64 DFMA cross-check)
// =========================================================================================
template <typename T, bool TA, int BM, int BN, int BK>
struct SimtCfg {
    static constexpr int TM = 8, TN = 8;
    static constexpr int TX = BM / TM, TY = BN / TN, NT = TX * TY;
    static constexpr int VEC = 16 / (int)sizeof(T);          // elements per 16-byte vector
    static constexpr int GM = TM / VEC, GN = TN / VEC;       // vector groups per thread
    static constexpr int LDA_S = BM + 4, LDB_S = BN + 4;
    static constexpr int A_ELEMS = BK * LDA_S, B_ELEMS = BK * LDB_S;
    static constexpr size_t SMEM = (size_t)2 * (A_ELEMS + B_ELEMS) * sizeof(T);
};

template <typename T, bool TA, int BM, int BN, int BK>
__global__ void __launch_bounds__(SimtCfg<T, TA, BM, BN, BK>::NT)
gemm_simt_kernel(GemmArgs<T> g) {
    using Cfg = SimtCfg<T, TA, BM, BN, BK>;
    constexpr int NT = Cfg::NT, VEC = Cfg::VEC, GM = Cfg::GM, GN = Cfg::GN;
    constexpr int LDA_S = Cfg::LDA_S, LDB_S = Cfg::LDB_S;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* smem = reinterpret_cast<T*>(smem_raw);
    T* As[2] = {smem, smem + Cfg::A_ELEMS + Cfg::B_ELEMS};
    T* Bs[2] = {As[0] + Cfg::A_ELEMS, As[1] + Cfg::A_ELEMS};

    const int tid = threadIdx.x, tx = tid % Cfg::TX, ty = tid / Cfg::TX;
    const int64_t m0 = (int64_t)blockIdx.x * BM, n0 = (int64_t)blockIdx.y * BN;
    const int64_t kbeg = (int64_t)blockIdx.z * g.k_chunk;
    const int64_t kend = min(g.K, kbeg + g.k_chunk);
    const int KT = (int)ceil_div(max((int64_t)0, kend - kbeg), BK);
    T* Cout = g.C + (int64_t)blockIdx.z * g.split_stride;
    const bool split = gridDim.z > 1;

    // element e (0..7) of the thread's m-range lives at tile row  (e/VEC)*(BM/GM) + tx*VEC + e%VEC
    auto m_of = [&](int e) { return (e / VEC) * (BM / GM) + tx * VEC + (e % VEC); };
    auto n_of = [&](int e) { return (e / VEC) * (BN / GN) + ty * VEC + (e % VEC); };

    T acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = T(0);

    // ---- global -> register staging ----
    // outer-contiguous tile (A when !TA): BK x BM, vectors along m
    constexpr int A_VECS = BM * BK / VEC, A_PER = (A_VECS + NT - 1) / NT;
    constexpr int B_VECS = BN * BK / VEC, B_PER = (B_VECS + NT - 1) / NT;
    T ra[A_PER][VEC], rb[B_PER][VEC];

    auto gload = [&](int kt) {
        const int64_t k0 = kbeg + (int64_t)kt * BK;
#pragma unroll
        for (int p = 0; p < A_PER; ++p) {
            int v = tid + p * NT;
#pragma unroll
            for (int e = 0; e < VEC; ++e) ra[p][e] = T(0);
            if (v < A_VECS) {
                if (TA) {   // K-contiguous: tile rows = m, vectors along k
                    int r = v / (BK / VEC), ck = (v % (BK / VEC)) * VEC;
                    int64_t gm = m0 + r, gk = k0 + ck;
                    if (gm < g.M) {
                        const T* src = g.A + gm * g.lda + gk;
                        if (g.a_vec_ok && gk + VEC <= kend) {
                            float4 t = __ldg(reinterpret_cast<const float4*>(src));
                            *reinterpret_cast<float4*>(&ra[p][0]) = t;
                        } else {
#pragma unroll
                            for (int e = 0; e < VEC; ++e) if (gk + e < kend) ra[p][e] = __ldg(src + e);
                        }
                    }
                } else {    // M-contiguous: tile rows = k, vectors along m
                    int kk = v / (BM / VEC), cm = (v % (BM / VEC)) * VEC;
                    int64_t gk = k0 + kk, gm = m0 + cm;
                    if (gk < kend) {
                        const T* src = g.A + gm + gk * g.lda;
                        if (g.a_vec_ok && gm + VEC <= g.M) {
                            float4 t = __ldg(reinterpret_cast<const float4*>(src));
                            *reinterpret_cast<float4*>(&ra[p][0]) = t;
                        } else {
#pragma unroll
                            for (int e = 0; e < VEC; ++e) if (gm + e < g.M) ra[p][e] = __ldg(src + e);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int p = 0; p < B_PER; ++p) {
            int v = tid + p * NT;
#pragma unroll
            for (int e = 0; e < VEC; ++e) rb[p][e] = T(0);
            if (v < B_VECS) {
                int r = v / (BK / VEC), ck = (v % (BK / VEC)) * VEC;
                int64_t gn = n0 + r, gk = k0 + ck;
                if (gn < g.N) {
                    const T* src = g.B + gn * g.ldb + gk;
                    if (g.b_vec_ok && gk + VEC <= kend) {
                        float4 t = __ldg(reinterpret_cast<const float4*>(src));
                        *reinterpret_cast<float4*>(&rb[p][0]) = t;
                    } else {
#pragma unroll
                        for (int e = 0; e < VEC; ++e) if (gk + e < kend) rb[p][e] = __ldg(src + e);
                    }
                }
            }
        }
    };
    auto sstore = [&](int buf) {
#pragma unroll
        for (int p = 0; p < A_PER; ++p) {
            int v = tid + p * NT;
            if (v < A_VECS) {
                if (TA) {
                    int r = v / (BK / VEC), ck = (v % (BK / VEC)) * VEC;
#pragma unroll
                    for (int e = 0; e < VEC; ++e) As[buf][(ck + e) * LDA_S + r] = ra[p][e];
                } else {
                    int kk = v / (BM / VEC), cm = (v % (BM / VEC)) * VEC;
                    *reinterpret_cast<float4*>(&As[buf][kk * LDA_S + cm]) = *reinterpret_cast<float4*>(&ra[p][0]);
                }
            }
        }
#pragma unroll
        for (int p = 0; p < B_PER; ++p) {
            int v = tid + p * NT;
            if (v < B_VECS) {
                int r = v / (BK / VEC), ck = (v % (BK / VEC)) * VEC;
#pragma unroll
                for (int e = 0; e < VEC; ++e) Bs[buf][(ck + e) * LDB_S + r] = rb[p][e];
            }
        }
    };

    if (KT > 0) { gload(0); sstore(0); }
    __syncthreads();
    for (int kt = 0; kt < KT; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < KT) gload(kt + 1);
#pragma unroll
        for (int kk = 0; kk < BK; ++kk) {
            T a[8], b[8];
#pragma unroll
            for (int gi = 0; gi < GM; ++gi)
                *reinterpret_cast<float4*>(&a[gi * VEC]) =
                    *reinterpret_cast<const float4*>(&As[buf][kk * LDA_S + gi * (BM / GM) + tx * VEC]);
#pragma unroll
            for (int gj = 0; gj < GN; ++gj)
                *reinterpret_cast<float4*>(&b[gj * VEC]) =
                    *reinterpret_cast<const float4*>(&Bs[buf][kk * LDB_S + gj * (BN / GN) + ty * VEC]);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
        if (kt + 1 < KT) sstore(buf ^ 1);
        __syncthreads();
    }

    const T beta = split ? T(0) : g.beta;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        int64_t n = n0 + n_of(j);
        if (n >= g.N) continue;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int64_t m = m0 + m_of(i);
            if (m < g.M) {
                T* p = Cout + m + n * g.ldc;
                T v = g.alpha * acc[i][j];
                if (beta != T(0)) v = fma(beta, *p, v);
                *p = v;
            }
        }
    }
}

// =========================================================================================
// host-side launchers
// =========================================================================================
template <typename K>
inline cudaError_t set_smem(K kernel, size_t bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

inline bool aligned16(const void* p, int64_t ld, size_t w) {
    return (((uintptr_t)p) % 16 == 0) && ((ld * (int64_t)w) % 16 == 0);
}

// Number of K splits for a skinny-output product: fill the SMs when the output tile grid is small.
inline int pick_splits(int64_t tiles, int64_t K, int bk, int sms, int ctas_per_sm, int64_t min_chunk) {
    int64_t slots = (int64_t)sms * ctas_per_sm;
    if (tiles >= slots) return 1;
    int64_t s = slots / tiles;
    int64_t maxs = K / min_chunk; if (maxs < 1) maxs = 1;
    if (s > maxs) s = maxs;
    if (s < 1) s = 1;
    (void)bk;
    return (int)s;
}

template <bool TA, int BM, int BN, int WM, int WN, int BK, int STAGES, int MINB>
inline cudaError_t launch_dmma(GemmArgs<double> g, int splits, cudaStream_t st) {
    using Cfg = DmmaCfg<TA, BM, BN, WM, WN, BK, STAGES>;
    auto kern = gemm_dmma_kernel<TA, BM, BN, WM, WN, BK, STAGES, MINB>;
    static SmemAttr attr;
    { cudaError_t e = ensure_dyn_smem(kern, Cfg::SMEM, attr); if (e != cudaSuccess) return e; }
    g.k_chunk = round_up(ceil_div(g.K, splits), BK);
    if (g.k_chunk <= 0) g.k_chunk = BK;
    dim3 grid((unsigned)ceil_div(g.M, BM), (unsigned)ceil_div(g.N, BN), (unsigned)splits);
    kern<<<grid, Cfg::NT, Cfg::SMEM, st>>>(g);
    return cudaGetLastError();
}

template <typename T, bool TA, int BM, int BN, int BK>
inline cudaError_t launch_simt(GemmArgs<T> g, int splits, cudaStream_t st) {
    using Cfg = SimtCfg<T, TA, BM, BN, BK>;
    auto kern = gemm_simt_kernel<T, TA, BM, BN, BK>;
    static SmemAttr attr;
    { cudaError_t e = ensure_dyn_smem(kern, Cfg::SMEM, attr); if (e != cudaSuccess) return e; }
    g.k_chunk = round_up(ceil_div(g.K, splits), BK);
    if (g.k_chunk <= 0) g.k_chunk = BK;
    dim3 grid((unsigned)ceil_div(g.M, BM), (unsigned)ceil_div(g.N, BN), (unsigned)splits);
    kern<<<grid, Cfg::NT, Cfg::SMEM, st>>>(g);
    return cudaGetLastError();
}

}  // namespace ctqr
