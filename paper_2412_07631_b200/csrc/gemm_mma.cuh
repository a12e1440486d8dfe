// gemm_mma.cuh -- persistent, stream-K, warp-level tensor-core contraction (SURVEY.md 8a rows
// a3 / a6 / a7: the larfb products W = V^T C and C <- C - V W, the Gram matrix of larft and the
// GEMM tasks of the blocked TRSM).
//
//   C <- alpha * op(A) * B + beta * C,  column-major, op(A) = A^T (A is K x M) or A (M x K), B is K x N.
//
// Why this shape (ncu, profiles/r1a_launches_c3_f64.md): the first kernels were latency-bound by
// occupancy (1-2 warps per SM sub-partition) and by wave quantisation (152 CTAs on 296 slots),
// not by DRAM or by the tensor pipe.  So:
//   * 8 warps per CTA with 32x32 warp tiles (<= 128 registers) -> 2 CTAs = 16 warps per SM;
//   * the grid is one wave of co-resident CTAs (a multiple of the SM count); the flattened
//     sequence of (output tile, k-tile) units is cut into equal contiguous ranges, one per CTA
//     ("stream-K"), so every CTA does the same work whatever the tile count;
//   * the cp.async pipeline runs over the FLAT unit sequence, i.e. it keeps prefetching across
//     tile boundaries: no prologue bubble per tile (matters for C <- C - V W where K is only nb);
//   * a tile whose k-range is cut writes per-segment partial tiles; the consumer kernel
//     (T^T W, larft) sums them in a fixed order -> deterministic, no atomics.
// Precision policies:
//   double: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) -- the only native FP64 tensor instruction
//           of sm_100a (tcgen05 has no f64 kind).
//   float : 3xTF32 split on mma.sync.m16n8k8.tf32 (SASS HMMA.1688.F32.TF32): x = hi + lo with
//           hi = tf32(x), lo = tf32(x - hi); a*b ~= hi_a*hi_b + hi_a*lo_b + lo_a*hi_b accumulated
//           in fp32.  Measured 278 TFLOP/s for the plain instruction on B200, i.e. <= 93 TFLOP/s of
//           fp32-equivalent work against 74 TFLOP/s of FFMA.  north_star allows it "only if it
//           meets the fp32 tolerance": the parity tests run on it.  The big products go to the
//           tcgen05 kernel of gemm_umma.cuh instead (4x the MMA rate); this one serves the rest.
#pragma once
#include <algorithm>
#include "common.cuh"
#include "kernels.h"

namespace ctqr {

// -------------------------------------------------------------------------------------------
// precision policies: fragment loads + MMA for one k-step of a (WM x WN) warp tile
// -------------------------------------------------------------------------------------------
template <typename T> struct MmaPolicy;

template <> struct MmaPolicy<double> {
    static constexpr int BK = 16;        // k-tile: 16 doubles = 128 bytes per row
    static constexpr int KSTEP = 4;      // k per MMA
    static constexpr int MFRAG = 8;      // rows per A fragment
    static constexpr int PAD_K = 4;      // K-contiguous tiles: ld = BK + 4  (== 4 mod 16 doubles)
    static constexpr int PAD_M = 4;      // M-contiguous tiles: ld = BM + 4
    static constexpr int ACC = 2;        // accumulator registers per (m-frag, n-frag)
    template <bool TA, int MT, int NTL, int LDK, int LDM>
    static __device__ __forceinline__ void kstep(const double* As, const double* Bs, int kk, int mrow0, int ncol0,
                                                 int grp, int tig, double (&acc)[MT][NTL][2]) {
        double a[MT], b[NTL];
#pragma unroll
        for (int i = 0; i < MT; ++i) {
            const int mrow = mrow0 + i * 8 + grp;
            a[i] = TA ? As[mrow * LDK + kk + tig] : As[(kk + tig) * LDM + mrow];
        }
#pragma unroll
        for (int j = 0; j < NTL; ++j) b[j] = Bs[(ncol0 + j * 8 + grp) * LDK + kk + tig];
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NTL; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
    // element (r, c) of accumulator register q inside an (8 x 8) fragment
    static __device__ __forceinline__ int frag_row(int q, int grp) { (void)q; return grp; }
    static __device__ __forceinline__ int frag_col(int q, int tig) { return 2 * tig + q; }
};

// x = hi + lo with hi, lo on the TF32 grid (10-bit mantissa).  cvt.rna.tf32.f32 is not a single
// instruction on sm_100a (it expands to ~8 integer ops per value and made the ALU pipe the
// co-bottleneck), so round to nearest on the bit pattern instead: add half a TF32 ulp, and mask
// where the exact value is needed.  The tensor core ignores the low 13 mantissa bits of a .tf32
// operand, so lo needs no mask.  (Values within 2^-11 of FLT_MAX would round to inf; not handled.)
__device__ __forceinline__ void split_tf32(float x, unsigned& hi, unsigned& lo) {
    hi = (__float_as_uint(x) + 0x1000u) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi)) + 0x1000u;
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const unsigned (&a)[4], const unsigned (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// d = a * b (zero accumulator input)
__device__ __forceinline__ void mma_tf32_zero(float (&d)[4], const unsigned (&a)[4], const unsigned (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};\n"
                 : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "f"(0.0f));
}

template <> struct MmaPolicy<float> {
    static constexpr int BK = 32;        // 32 floats = 128 bytes per row
    static constexpr int KSTEP = 8;
    static constexpr int MFRAG = 16;
    static constexpr int PAD_K = 4;      // ld = 36 == 4 mod 32 words: rows grp*4 + tig hit 32 distinct banks
    static constexpr int PAD_M = 8;      // ld = BM + 8 == 8 mod 32: tig*8 + grp distinct
    static constexpr int ACC = 4;
    template <bool TA, int MT, int NTL, int LDK, int LDM>
    static __device__ __forceinline__ void kstep(const float* As, const float* Bs, int kk, int mrow0, int ncol0,
                                                 int grp, int tig, float (&acc)[MT][NTL][4]) {
        // The tensor core adds into its fp32 accumulator with truncation: accumulating a long K
        // inside the MMA gives an error that grows linearly with K (measured 1.1e-5 at K = 1024,
        // 3.3e-4 at K = 32768 against 3e-6 for FFMA).  So every k-step's three products go into a
        // fresh accumulator (zero C input) and are added to the running sum with an ordinary
        // round-to-nearest FADD: the truncation then acts on one k-step's worth of magnitude only.
        unsigned ah[MT][4], al[MT][4];
#pragma unroll
        for (int i = 0; i < MT; ++i) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int mrow = mrow0 + i * 16 + grp + (q & 1) * 8;
                const int k = kk + tig + (q >> 1) * 4;
                const float x = TA ? As[mrow * LDK + k] : As[k * LDM + mrow];
                split_tf32(x, ah[i][q], al[i][q]);
            }
        }
#pragma unroll
        for (int j = 0; j < NTL; ++j) {
            unsigned bh[2], bl[2];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const float x = Bs[(ncol0 + j * 8 + grp) * LDK + kk + tig + q * 4];
                split_tf32(x, bh[q], bl[q]);
            }
#pragma unroll
            for (int i = 0; i < MT; ++i) {
                float t[4];
                mma_tf32_zero(t, al[i], bh);      // small terms first, the dominant hi*hi product last
                mma_tf32(t, ah[i], bl);
                mma_tf32(t, ah[i], bh);
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[i][j][q] += t[q];
            }
        }
    }
    static __device__ __forceinline__ int frag_row(int q, int grp) { return grp + (q >> 1) * 8; }
    static __device__ __forceinline__ int frag_col(int q, int tig) { return 2 * tig + (q & 1); }
};

// -------------------------------------------------------------------------------------------
// stream-K partition of the flattened (tile, k-tile) unit sequence
// -------------------------------------------------------------------------------------------
struct StreamK {
    int64_t tilesM, tilesN;   // output tiles; tile t = tn * tilesM + tm (m fastest)
    int KT;                   // k-tiles per output tile
    int64_t U;                // tilesM * tilesN * KT
    int64_t L;                // units per CTA (a multiple of KT in direct mode)
    int partial;              // 1: every segment writes alpha*acc to its compact partial slot; 0: direct
    // direct mode, Gm > 0: the tiles are numbered band by band (Gm tile rows per band; inside a band column block by column
    // block, tile rows fastest) and dealt round-robin (worker w takes the numbers w, w + G, w + 2G, ...), so that the G tiles
    // in flight are a compact Gm x (G / Gm) patch sharing Gm tiles of A and G / Gm tiles of B in L2.  With contiguous
    // per-worker ranges (Gm = 0) the workers sit at unrelated tile rows and cycle through all of A; at m = 1e5 the 223 MB
    // reflector pair no longer fits the L2 (ncu, profiles/r2_c4_f64.md: 349 GB of DRAM reads for 57 GB of C).
    int G, Gm;
    // SM confinement (see GemmLaunch::reserve): worker indices are drawn from tickets[1] by the CTAs that do
    // not retire on a reserved SM; `workers` = the planned grid
    unsigned* tickets; int reserve; int workers;
};
// first CTA that touches tile t, and how many CTAs (= partial slots) it has
__host__ __device__ inline int64_t sk_first_cta(int64_t t, int KT, int64_t L) { return (t * KT) / L; }
__host__ __device__ inline int sk_nseg(int64_t t, int KT, int64_t L) {
    return (int)((((t + 1) * KT - 1) / L) - ((t * KT) / L) + 1);
}

template <typename T, bool TA, int BM, int BN, int WM, int WN, int STAGES>
struct MmaCfg {
    using P = MmaPolicy<T>;
    static constexpr int BK = P::BK;
    static constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN;
    static constexpr int NT = WARPS_M * WARPS_N * 32;
    static constexpr int MT = WM / P::MFRAG, NTL = WN / 8;
    static constexpr int LDK = BK + P::PAD_K;
    static constexpr int LDM = BM + P::PAD_M;
    static constexpr int A_ELEMS = TA ? BM * LDK : BK * LDM;
    static constexpr int B_ELEMS = BN * LDK;
    static constexpr int STAGE_ELEMS = A_ELEMS + B_ELEMS;
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_ELEMS * sizeof(T);
    static constexpr int VEC = 16 / (int)sizeof(T);
};

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

// Requires 16-byte aligned operands (a_vec_ok && b_vec_ok); the host falls back to the classic
// kernels of gemm.cuh otherwise.
template <typename T, bool TA, int BM, int BN, int WM, int WN, int STAGES, int MINB, bool CONFINED = false>
__global__ void __launch_bounds__(MmaCfg<T, TA, BM, BN, WM, WN, STAGES>::NT, MINB)
gemm_mma_kernel(GemmArgs<T> g, StreamK sk) {
    using Cfg = MmaCfg<T, TA, BM, BN, WM, WN, STAGES>;
    using P = MmaPolicy<T>;
    constexpr int NT = Cfg::NT, MT = Cfg::MT, NTL = Cfg::NTL, LDK = Cfg::LDK, LDM = Cfg::LDM, BK = Cfg::BK;
    constexpr int VEC = Cfg::VEC, ACC = P::ACC, W = (int)sizeof(T);
    constexpr int CPR = BK / VEC;                         // 16-byte chunks per K-contiguous row
    constexpr int CPM = BM / VEC;                         // chunks per M-contiguous row (!TA)
    constexpr int PA = (TA ? BM * CPR : BK * CPM) / NT;   // chunks per thread per k-tile
    constexpr int PB = BN * CPR / NT;
    static_assert((TA ? BM * CPR : BK * CPM) % NT == 0 && (BN * CPR) % NT == 0, "tile/thread mismatch");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* smem = reinterpret_cast<T*>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // fp64: the stages are handed over through mbarriers instead of one __syncthreads per k-tile: full[s] completes when
    // the cp.async copies of all NT threads for that stage have landed (cp.async.mbarrier.arrive), empty[s] when all
    // warps have consumed it; a warp waits only for data, never for the slowest warp of the previous k-tile, and a stage
    // is refilled one k-tile after it was consumed (when every warp has normally long left it).  Measured at configs[3]:
    // C <- C - V W 27.0 -> 29.5 TFLOP/s, W = V^T C 31.0 -> 33.5 (a two-stage ring with a k-tile of 32 and __syncthreads
    // had given 32.7 for the latter), factorisation 28.3 -> 30.7 TFLOP/s.
    constexpr bool MBAR = sizeof(T) == 8 && STAGES >= 3;   // (a two-stage ring has no room for the refill-after-consume order)
    __shared__ __align__(8) unsigned long long s_bars[2 * STAGES];
    const unsigned bar0 = (unsigned)__cvta_generic_to_shared(s_bars);
    if constexpr (MBAR) {
        if (tid == 0) {
            for (int s = 0; s < STAGES; ++s) {
                asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar0 + 8u * s), "r"(NT));
                asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar0 + 8u * (STAGES + s)), "r"(NT / 32));
            }
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        }
        __syncthreads();
    }
    auto bar_wait = [&](unsigned bar, unsigned parity) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "MW: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
            "@p bra MD;\n\tbra MW;\n\tMD:\n\t}\n" ::"r"(bar), "r"(parity) : "memory");
    };
    const int wm = warp % Cfg::WARPS_M, wn = warp / Cfg::WARPS_M;
    const int grp = lane >> 2, tig = lane & 3;
    // worker index: blockIdx.x, or (CONFINED instantiation) a ticket when the launch is kept off some SMs
    // (StreamK::tickets); held in shared memory there: the kernel sits at its register cap
    __shared__ int s_worker_confined;
    if constexpr (CONFINED) {
        if (tid == 0) {
            unsigned smid, nsm;
            asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            asm volatile("mov.u32 %0, %%nsmid;" : "=r"(nsm));
            const bool retire = smid + (unsigned)sk.reserve >= nsm &&
                                atomicAdd(sk.tickets, 1u) < (unsigned)((int)gridDim.x - sk.workers);
            int id = -1;
            if (!retire) {
                id = (int)atomicAdd(sk.tickets + 1, 1u);
                if (id >= sk.workers) id = -1;
            }
            s_worker_confined = id;
        }
        __syncthreads();
        if (s_worker_confined < 0) return;
    }
#define s_worker (CONFINED ? s_worker_confined : (int)blockIdx.x)
    const int64_t u0 = (int64_t)s_worker * sk.L;
    const bool rr = !sk.partial && sk.Gm > 0;
    const int64_t u1 = !rr ? min(sk.U, u0 + sk.L)
                           : u0 + ((sk.tilesM * sk.tilesN - (int64_t)s_worker + sk.G - 1) / sk.G) * sk.KT;
    if (u0 >= u1) return;
    // flat tile index (contiguous per CTA) -> tile coordinates
    auto decode = [&](int64_t t, int64_t& tm, int64_t& tn) {
        if (!rr) { tn = t / sk.tilesM; tm = t - tn * sk.tilesM; return; }
        const int64_t rank = (t - u0 / sk.KT) * sk.G + (int64_t)s_worker;
        const int64_t per_band = (int64_t)sk.Gm * sk.tilesN;
        const int64_t band = rank / per_band, r = rank - band * per_band;
        const int64_t hb = min((int64_t)sk.Gm, sk.tilesM - band * sk.Gm);
        tn = r / hb; tm = band * sk.Gm + (r - tn * hb);
    };

    // L2 residency: the reflector block V (operand A) is re-read by every CTA -> keep it; the big
    // matrix C streams through once per launch -> let it go first.  In W = V^T C the streamed
    // matrix is operand B; in C <- C - V W operand B is the small W (keep) and C itself is
    // read/written by the accumulator path with streaming loads/stores.
    const uint64_t pol_a = l2_policy_evict_last();
    const uint64_t pol_b = TA ? l2_policy_evict_first() : l2_policy_evict_last();

    // ---- producer state: runs STAGES-1 units ahead of the consumer, advanced incrementally ----
    const T* pa[PA]; const T* pb[PB];
    uint64_t abytes = 0, bbytes = 0;      // 5 bits per chunk: valid bytes of the chunk's row/vector (0..16)
    int64_t ltile = u0 / sk.KT;
    int lkt = (int)(u0 - ltile * sk.KT);
    int64_t ltn, ltm;
    decode(ltile, ltm, ltn);
    auto set_tile = [&]() {
        const int64_t m0 = ltm * BM, n0 = ltn * BN;
        abytes = 0; bbytes = 0;
#pragma unroll
        for (int p = 0; p < PA; ++p) {
            const int c = tid + p * NT;
            if (TA) {
                const int r = c / CPR, ck = (c % CPR) * VEC;
                const int64_t gr = m0 + r;
                const bool ok = gr < g.M;
                pa[p] = g.A + (ok ? gr : 0) * g.lda + ck;
                abytes |= (uint64_t)(ok ? 16u : 0u) << (5 * p);
            } else {
                const int kk = c / CPM, cm = (c % CPM) * VEC;
                const int64_t gm = m0 + cm;
                const int nv = (int)max((int64_t)0, min((int64_t)VEC, g.M - gm));
                pa[p] = g.A + (nv ? gm : 0) + (int64_t)kk * g.lda;
                abytes |= (uint64_t)(nv * W) << (5 * p);
            }
        }
#pragma unroll
        for (int p = 0; p < PB; ++p) {
            const int c = tid + p * NT;
            const int r = c / CPR, ck = (c % CPR) * VEC;
            const int64_t gr = n0 + r;
            const bool ok = gr < g.N;
            pb[p] = g.B + (ok ? gr : 0) * g.ldb + ck;
            bbytes |= (uint64_t)(ok ? 16u : 0u) << (5 * p);
        }
    };
    auto issue = [&](int stage) {
        T* As = smem + (size_t)stage * Cfg::STAGE_ELEMS;
        T* Bs = As + Cfg::A_ELEMS;
        const int64_t k0 = (int64_t)lkt * BK;
        const bool tail = k0 + BK > g.K;
        const int64_t aoff = TA ? k0 : k0 * g.lda;
#pragma unroll
        for (int p = 0; p < PA; ++p) {
            const int c = tid + p * NT;
            int bytes = (int)((abytes >> (5 * p)) & 31u);
            if (TA) {
                const int r = c / CPR, ck = (c % CPR) * VEC;
                if (tail) bytes = min(bytes, max(0, (int)(g.K - k0 - ck) * W));
                cp_async16_hint(As + r * LDK + ck, pa[p] + aoff, bytes, pol_a);
            } else {
                const int kk = c / CPM, cm = (c % CPM) * VEC;
                if (tail && k0 + kk >= g.K) bytes = 0;
                cp_async16_hint(As + kk * LDM + cm, pa[p] + aoff, bytes, pol_a);
            }
        }
#pragma unroll
        for (int p = 0; p < PB; ++p) {
            const int c = tid + p * NT;
            const int r = c / CPR, ck = (c % CPR) * VEC;
            int bytes = (int)((bbytes >> (5 * p)) & 31u);
            if (tail) bytes = min(bytes, max(0, (int)(g.K - k0 - ck) * W));
            cp_async16_hint(Bs + r * LDK + ck, pb[p] + k0, bytes, pol_b);
        }
        // advance to the next unit
        if (++lkt == sk.KT) {
            lkt = 0;
            ++ltile;
            decode(ltile, ltm, ltn);
            set_tile();
        }
    };

    set_tile();
    int64_t lu = u0;                      // next unit the producer will issue
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (lu < u1) {
            issue(s); ++lu;
            if constexpr (MBAR) asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar0 + 8u * s) : "memory");
        }
        cp_async_commit();
    }
    unsigned fills = 0;                   // (MBAR) ring turns: units consumed so far / STAGES, tracked with cstage

    const T cscale = (sk.partial || g.beta == T(0)) ? T(0) : g.beta / g.alpha;
    int64_t t = u0 / sk.KT;
    int64_t tn, tm;
    decode(t, tm, tn);
    int64_t u = u0;
    int cstage = 0, pstage = STAGES - 1;  // consumer / producer ring positions
    while (u < u1) {
        const int64_t seg_end = min(u1, (t + 1) * sk.KT);
        const int64_t m0 = tm * BM, n0 = tn * BN;
        const bool interior = (m0 + BM <= g.M) && (n0 + BN <= g.N);
        T acc[MT][NTL][ACC];
        if (cscale != T(0)) {
            // all loads of the C tile are issued before the first use (one memory round trip per tile)
            const T* Cb = g.C + (m0 + wm * WM) + (n0 + wn * WN) * g.ldc;
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NTL; ++j)
#pragma unroll
                    for (int q = 0; q < ACC; ++q) {
                        const int r = i * P::MFRAG + P::frag_row(q, grp), c = j * 8 + P::frag_col(q, tig);
                        const bool ok = interior || (m0 + wm * WM + r < g.M && n0 + wn * WN + c < g.N);
                        acc[i][j][q] = ok ? __ldcs(Cb + r + c * g.ldc) : T(0);
                    }
            // scaled in a second loop on purpose: written as `cscale * load` the compiler pairs every load with its
            // multiply (32 serial memory round trips per tile; measured -22 % on the whole kernel at configs[3])
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NTL; ++j)
#pragma unroll
                    for (int q = 0; q < ACC; ++q) acc[i][j][q] *= cscale;
        } else {
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NTL; ++j)
#pragma unroll
                    for (int q = 0; q < ACC; ++q) acc[i][j][q] = T(0);
        }
        for (; u < seg_end; ++u) {
            if constexpr (MBAR) {
                // unit j = u - u0 sits in stage j % STAGES (= cstage), ring turn j / STAGES (= fills)
                bar_wait(bar0 + 8u * cstage, fills & 1u);
                const T* As = smem + (size_t)cstage * Cfg::STAGE_ELEMS;
                const T* Bs = As + Cfg::A_ELEMS;
#pragma unroll
                for (int kk = 0; kk < BK; kk += P::KSTEP)
                    P::template kstep<TA, MT, NTL, LDK, LDM>(As, Bs, kk, wm * WM, wn * WN, grp, tig, acc);
                __syncwarp();
                if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar0 + 8u * (STAGES + cstage)) : "memory");
                // refill the stage consumed one k-tile ago (pstage) with unit j + STAGES - 1: it was last used by unit
                // j - 1 (ring turn of that unit), which every warp has normally long finished
                if (lu < u1) {
                    const int64_t jn = lu - u0;           // unit index of the refill
                    if (jn >= STAGES) bar_wait(bar0 + 8u * (STAGES + pstage), (unsigned)((jn / STAGES) - 1) & 1u);
                    issue(pstage); ++lu;
                    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar0 + 8u * pstage) : "memory");
                }
                pstage = (pstage + 1 == STAGES) ? 0 : pstage + 1;
                if (++cstage == STAGES) { cstage = 0; ++fills; }
                continue;
            }
            cp_async_wait<STAGES - 2>();
            __syncthreads();
            if (lu < u1) { issue(pstage); ++lu; }
            cp_async_commit();
            pstage = (pstage + 1 == STAGES) ? 0 : pstage + 1;
            const T* As = smem + (size_t)cstage * Cfg::STAGE_ELEMS;
            const T* Bs = As + Cfg::A_ELEMS;
            cstage = (cstage + 1 == STAGES) ? 0 : cstage + 1;
#pragma unroll
            for (int kk = 0; kk < BK; kk += P::KSTEP)
                P::template kstep<TA, MT, NTL, LDK, LDM>(As, Bs, kk, wm * WM, wn * WN, grp, tig, acc);
        }
        // ---- epilogue of this segment ----
        if (sk.partial) {
            // compact partial tiles: the (CTA, tile) pairs of a stream-K schedule form a staircase
            // on which tile + CTA is strictly increasing, so that sum indexes a dense BM x BN slot
            T* Pt = g.C + (t + (int64_t)s_worker) * (int64_t)(BM * BN);
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NTL; ++j)
#pragma unroll
                    for (int q = 0; q < ACC; ++q) {
                        const int r = wm * WM + i * P::MFRAG + P::frag_row(q, grp);
                        const int c = wn * WN + j * 8 + P::frag_col(q, tig);
                        Pt[r + c * BM] = g.alpha * acc[i][j][q];
                    }
        } else {
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NTL; ++j)
#pragma unroll
                    for (int q = 0; q < ACC; ++q) {
                        const int64_t m = m0 + wm * WM + i * P::MFRAG + P::frag_row(q, grp);
                        const int64_t n = n0 + wn * WN + j * 8 + P::frag_col(q, tig);
                        if (interior || (m < g.M && n < g.N)) {
                            __stcs(&g.C[m + n * g.ldc], g.alpha * acc[i][j][q]);
                        }
                    }
        }
        ++t;
        decode(t, tm, tn);
    }
    cp_async_wait<0>();
}

// -------------------------------------------------------------------------------------------
// host side: plan + launch
// -------------------------------------------------------------------------------------------
#undef s_worker

struct MmaPlan {
    StreamK sk;
    int grid;        // CTAs
    int maxseg;      // most segments any tile has (partial mode)
    int64_t partial_elems;   // elements of the compact partial buffer: (tiles + grid) * BM * BN
};

// slots = co-resident CTAs (SMs * CTAs per SM).  Direct mode keeps whole tiles per CTA.
inline MmaPlan mma_plan(int64_t M, int64_t N, int64_t K, int BM, int BN, int BK, int slots, bool partial) {
    MmaPlan p{};
    p.sk.tilesM = ceil_div(M, BM); p.sk.tilesN = ceil_div(N, BN);
    p.sk.KT = (int)std::max<int64_t>(1, ceil_div(K, BK));
    const int64_t tiles = p.sk.tilesM * p.sk.tilesN;
    p.sk.U = tiles * p.sk.KT;
    p.sk.partial = partial ? 1 : 0;
    if (partial) {
        // no CTA shorter than ~1024 rows of K: a small product split over every SM costs more in the
        // consumer (which sums one partial tile per segment) than it gains in the contraction.  With
        // only a few output tiles (the look-ahead column block, the solve's 128 x S products) that
        // rule leaves most SMs idle, so the floor drops to 512 rows (<= 2 tiles) / 256 rows (<= 8):
        // measured at configs[2], solve S = 256 Q^T B 26.4 -> 23.4 ms, factor 644 -> 636 ms (fp64).
        const int rows = tiles > 8 ? 1024 : tiles > 2 ? 256 : 512;
        const int64_t min_units = std::max<int64_t>(8, rows / BK);
        int64_t G = std::min<int64_t>(slots, std::max<int64_t>(1, p.sk.U / min_units));
        p.sk.L = ceil_div(p.sk.U, G);
        p.grid = (int)ceil_div(p.sk.U, p.sk.L);
        p.maxseg = (int)std::min<int64_t>(ceil_div(p.sk.KT, p.sk.L) + 1, p.grid);
        if (p.sk.L >= p.sk.KT && p.sk.L % p.sk.KT == 0) p.maxseg = 1;
        p.partial_elems = (tiles + p.grid) * (int64_t)BM * BN;
    } else {
        const int64_t tpc = ceil_div(tiles, (int64_t)slots);
        p.sk.L = tpc * p.sk.KT;
        p.grid = (int)ceil_div(tiles, tpc);
        p.maxseg = 1;
        // banded round-robin tile order once A (M x K) is too large to stay in L2 beside the streamed C
        p.sk.G = p.grid;
        p.sk.Gm = (M * K * 8 > ((int64_t)24 << 20) && p.sk.tilesM >= 32) ? 16 : 0;
#ifdef CTQR_NO_BAND
        p.sk.Gm = 0;
#endif
    }
    return p;
}

template <typename T, bool TA, int BM, int BN, int WM, int WN, int STAGES, int MINB>
inline cudaError_t launch_mma(GemmArgs<T> g, const MmaPlan& p, cudaStream_t st) {
    using Cfg = MmaCfg<T, TA, BM, BN, WM, WN, STAGES>;
    if (p.sk.tickets) {
        if constexpr (sizeof(T) == 8 && MINB == 2) {
            auto kc = gemm_mma_kernel<T, TA, BM, BN, WM, WN, STAGES, MINB, true>;
            static SmemAttr attr_c;
            { cudaError_t e = ensure_dyn_smem(kc, Cfg::SMEM, attr_c); if (e != cudaSuccess) return e; }
            StreamK skc = p.sk;
            skc.workers = p.grid;
            kc<<<p.grid + MINB * skc.reserve, Cfg::NT, Cfg::SMEM, st>>>(g, skc);
            return cudaGetLastError();
        } else {
            return cudaErrorInvalidValue;
        }
    }
    auto kern = gemm_mma_kernel<T, TA, BM, BN, WM, WN, STAGES, MINB>;
    static SmemAttr attr;
    { cudaError_t e = ensure_dyn_smem(kern, Cfg::SMEM, attr); if (e != cudaSuccess) return e; }
    kern<<<p.grid, Cfg::NT, Cfg::SMEM, st>>>(g, p.sk);
    return cudaGetLastError();
}

}  // namespace ctqr
