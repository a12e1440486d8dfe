// solve_small2.cuh -- the memory-bound small-S Q^T B (SURVEY.md 8a row a6, S <= 8; Fig. 1 / Eq. 3), second
// generation, fp64: software-pipelined so that no CTA ever waits for a grid exchange, and fed by TMA.
//
// solve_small.cuh applies the panels strictly one after the other: partial W = V_k^T B -> grid exchange -> T^T W ->
// update -> next panel; ncu (profiles/r1_solve_c3.md) showed 9 of the 20.5 us per panel spent in the exchange and the
// HBM pipe idle meanwhile (19 % of the copy bandwidth).  Here the exchange is taken off the critical path:
//
//   * Y_j := V_j^T B_(j-2), the partial products of panel j, are formed from the rows as they are TWO panels earlier
//     (B_i = B after panels 0..i), published, and reduced over the grid while panels j-2 and j-1 are being applied.
//     The true W_j = V_j^T B_(j-1) differs by the update of panel j-1 alone (panel j-2's is already in B_(j-2)... see
//     below): B_(j-1) = B_(j-2) - V_(j-1) W2_(j-1), hence  W_j = Y_j - (V_j^T V_(j-1)) W2_(j-1).
//     With W2_(j-1) = T_(j-1)^T W_(j-1) this is W_j = Y_j - M_j W_(j-1), M_j = (V_j^T V_(j-1)) T_(j-1)^T (128 x 128, stored
//     transposed as "Mt" = T_(j-1) (V_(j-1)^T V_j), computed once per handle): the element owners of the reduction
//     subtract their row of M_j times the W_(j-1) they have just gathered, so the serial chain through the grid is one
//     hop per panel (owners publish W_j -> everybody gathers it) and T^T W, the update and the next partial products
//     all run while that hop is in flight.  128 KB of M per panel for the whole grid.
//     (Order inside iteration k: the rows are first updated with panel k, then Y_(k+2) is accumulated from them, so Y_(k+2)
//     sees B_k and only panel k+1 is missing.)
//   * The stream of V from HBM is issued by ONE thread as TMA box loads (16 rows x 128 columns, SWIZZLE_128B) into a
//     ring of shared-memory stages, as far ahead as the ring allows -- across panel boundaries too, V is read-only -- and
//     consumed by DMMA.8x8x4 straight from shared memory: the memory pipe never waits for the arithmetic or the exchange.
//   * T_k is read as DMMA fragments straight from L2 (it no longer fits beside the ring), the update pass re-reads the
//     CTA's slice of V_k from L2 with the whole row of 128 columns in flight.
// Deterministic: fixed reduction orders, flag-in-data exchanges (panel.cuh), no atomics.
#pragma once
#include "common.cuh"
#include "kernels.h"
#include "panel.cuh"
#include "solve_small.cuh"
#include "tma.cuh"

namespace ctqr {

template <typename T> struct Qt2Chunk { static constexpr int value = 128 / (int)sizeof(T); };   // rows per TMA box: 128 bytes, the swizzle span
constexpr int kQt2StageBytes = 128 * 128;        // one box: (16 fp64 | 32 fp32) rows x 128 columns
constexpr int kQt2Warps = 16;                    // compute warps; one more warp issues the TMA loads
constexpr int kQt2Threads = (kQt2Warps + 1) * 32;

template <typename T>
struct SmallQt2Args {
    const T* A; int64_t lda; int64_t m, n; int P;
    const T* Tm;                    // P blocks of 128 x 128 (ld 128)
    const T* Mt;               // P blocks of 128 x 128 (ld 128): Mt[j] = T_(j-1) (V_(j-1)^T V_j), j >= 1:
                                    // W_j[c, s] = Y_j[c, s] - sum_q Mt[j][q + c * 128] W_(j-1)[q, s]
    T* B; int64_t ldb; int S;
    uint4* part;                    // [2][G][128 * kSmallS] LL slots: per-CTA partial Y
    uint4* sums;                    // [2][128 * kSmallS] LL slots: reduced, corrected W
    unsigned seq_base;              // step numbers seq_base + 1 .. seq_base + P are used by this launch
    int rpc;                        // local rows per CTA (multiple of the box height)
    int64_t kl;                     // band promise (0 = dense)
    int nstage;                     // TMA ring stages
};

template <typename T>
inline size_t qt2_smem_bytes(int rpc, int nstage) {
    return 1024 + (size_t)nstage * kQt2StageBytes + 16 * (size_t)nstage + 64 +
           ((size_t)3 * 128 * SmallLd<T>::W + (size_t)kSmallS * (rpc + 4)) * sizeof(T);
}

// The ring carries ONE sequence of boxes, identical for the producer and for every consumer:
//   A(0), A(1), then for k = 0 .. P-1:  U(k), A(k+2)        (A(j) / U(j) = the CTA's row chunks of panel j, top down)
// A boxes feed the partial products Y_j (every compute warp reads every box: warp w owns columns 8w .. 8w+7);
// U boxes feed the row update of panel j (box i of the segment belongs to compute warp i mod 16 alone).
template <typename T>
__global__ void __launch_bounds__(kQt2Threads, 1)
apply_qt_small2_kernel(const __grid_constant__ CUtensorMap mapV, SmallQt2Args<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NB = 128, SM = kSmallS, NW = kQt2Warps, NT = NW * 32, CH = Qt2Chunk<T>::value, LDW = SmallLd<T>::W;
    constexpr bool F64 = sizeof(T) == 8;                    // fp64: DMMA.8x8x4 from the swizzled boxes; fp32: FFMA
    const unsigned sbase = (tma::smem_addr(smem_raw) + 1023u) & ~1023u;
    unsigned char* ring = smem_raw + (sbase - tma::smem_addr(smem_raw));
    const int NS = p.nstage;
    const unsigned bars = sbase + (unsigned)NS * kQt2StageBytes;            // full[NS], empty[NS]
    T* Wg = reinterpret_cast<T*>(ring + (size_t)NS * kQt2StageBytes + 16 * (size_t)NS + 64);   // gathered W_k
    T* Yp = Wg + NB * LDW;                                  // this CTA's partial Y
    T* W2 = Yp + NB * LDW;                                  // T_k^T W_k
    T* Bs = W2 + NB * LDW;                                  // [SM][ldbs] own rows of B, transposed
    const int ldbs = p.rpc + 4;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = blockIdx.x, G = gridDim.x, S = p.S;
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (NS + s); };
    auto row_of = [&](int lr) -> int64_t { return ((int64_t)(lr / CH) * G + g) * CH + (lr % CH); };
    auto first_local = [&](int64_t j0) -> int {             // first local row at or below row j0 (j0 a multiple of CH)
        const int64_t q0 = j0 / CH;
        return q0 > g ? (int)((q0 - g + G - 1) / G) * CH : 0;
    };
    const int nl = first_local(round_up(p.m, (int64_t)CH));
    auto range_of = [&](int j, int& la, int& le) {          // local rows [la, le) take part in panel j
        const int64_t j0 = (int64_t)j * NB;
        const int kw = (int)min((int64_t)NB, p.n - j0);
        la = first_local(j0);
        le = p.kl > 0 ? min(nl, first_local(round_up(min(p.m, p.kl + j0 + kw), (int64_t)CH))) : nl;
        if (le < la) le = la;
    };

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { tma::mbar_init(full(s), 1); tma::mbar_init(empty(s), NW); }
        tma::mbar_init_fence();
        tma::prefetch_map(&mapV);
    }
    for (int i = tid; i < SM * p.rpc; i += kQt2Threads) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        Bs[s * ldbs + lr] = (s < S && lr < nl && row < p.m) ? p.B[row + (int64_t)s * p.ldb] : T(0);
    }
    __syncthreads();

    if (warp == NW) {
        // ================= TMA producer: the whole box sequence, as far ahead as the ring allows =================
        if (lane == 0) {
            unsigned icount = 0;
            // the first read of a box (A segment) asks the L2 to keep the lines, the second (U segment, two panels
            // later) to drop them first: three panels of V must survive in the L2 between the two reads
            const uint64_t keep = l2_policy_evict_last(), drop = l2_policy_evict_first();
            auto segment = [&](int j, uint64_t pol) {
                int la, le; range_of(j, la, le);
                for (int lr = la; lr < le; lr += CH, ++icount) {
                    const int st = (int)(icount % (unsigned)NS);
                    tma::mbar_wait(empty(st), ((icount / (unsigned)NS) & 1u) ^ 1u);
                    tma::mbar_expect_tx(full(st), (unsigned)kQt2StageBytes);
                    tma::load_2d_hint(sbase + (unsigned)st * kQt2StageBytes, &mapV, (int)row_of(lr), j * NB, full(st), pol);
                }
            };
            segment(0, keep);
            if (p.P > 1) segment(1, keep);
            for (int k = 0; k < p.P; ++k) {
                segment(k, drop);
                if (k + 2 < p.P) segment(k + 2, keep);
            }
        }
        return;                                             // the compute warps synchronise among themselves (named barrier 1)
    }
    auto sync_compute = [&]() { asm volatile("bar.sync 1, %0;\n" ::"n"(NT) : "memory"); };
    unsigned ccount = 0;                                    // boxes of the sequence passed so far (every compute thread)

    // partial Y_j over the own rows from the ring: warp w owns columns 8w .. 8w+7; result to Yp, then published
    auto pass_a = [&](int j) {
        int la, le; range_of(j, la, le);
        if constexpr (F64) {
            const int c = warp * 8 + (lane >> 2);
            const double* bs = Bs + (lane >> 2) * ldbs + (lane & 3);
            double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
            for (int lr = la; lr < le; lr += CH, ++ccount) {
                const int st = (int)(ccount % (unsigned)NS);
                tma::mbar_wait(full(st), (ccount / (unsigned)NS) & 1u);
                const unsigned char* vs = ring + (size_t)st * kQt2StageBytes + c * 128;
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int r = 4 * h + (lane & 3);
                    const double a = *reinterpret_cast<const double*>(vs + ((((r >> 1) ^ (c & 7)) << 4) | ((r & 1) << 3)));
                    dmma884(c0[h], c1[h], a, bs[lr + 4 * h]);
                }
                __syncwarp();
                if (lane == 0) tma::mbar_arrive(empty(st));
            }
            sync_compute();                                 // the previous publication has finished reading Yp
            Yp[c * LDW + 2 * (lane & 3)] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
            Yp[c * LDW + 2 * (lane & 3) + 1] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
        } else {
            // fp32: lane = row of the box (32 rows), the warp's 8 columns x 8 right-hand sides in registers; the sums over the
            // rows are formed once per panel by two transpose-reductions (32 values each)
            float acc[2][4 * SM];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int u = 0; u < 4 * SM; ++u) acc[h][u] = 0.f;
            for (int lr = la; lr < le; lr += CH, ++ccount) {
                const int st = (int)(ccount % (unsigned)NS);
                tma::mbar_wait(full(st), (ccount / (unsigned)NS) & 1u);
                const unsigned char* vs = ring + (size_t)st * kQt2StageBytes;
                float b[SM];
#pragma unroll
                for (int q = 0; q < SM; ++q) b[q] = Bs[q * ldbs + lr + lane];
#pragma unroll
                for (int cc = 0; cc < 8; ++cc) {
                    const int c = warp * 8 + cc;
                    const float v = *reinterpret_cast<const float*>(vs + c * 128 + ((((lane >> 2) ^ (c & 7)) << 4) | ((lane & 3) << 2)));
#pragma unroll
                    for (int q = 0; q < SM; ++q) acc[cc >> 2][(cc & 3) * SM + q] = fmaf(v, b[q], acc[cc >> 2][(cc & 3) * SM + q]);
                }
                __syncwarp();
                if (lane == 0) tma::mbar_arrive(empty(st));
            }
            warp_transpose_reduce<float, 4 * SM>(acc[0], lane);   // lane l: total of value l = (column l / SM, rhs l % SM)
            warp_transpose_reduce<float, 4 * SM>(acc[1], lane);
            sync_compute();
            Yp[(warp * 8 + lane / SM) * LDW + (lane % SM)] = acc[0][0];
            Yp[(warp * 8 + 4 + lane / SM) * LDW + (lane % SM)] = acc[1][0];
        }
        sync_compute();
        const unsigned seq = p.seq_base + (unsigned)j + 1u;
        uint4* mine = p.part + ((size_t)(j & 1) * G + g) * (NB * SM);
        for (int e = tid; e < NB * SM; e += NT) ll_store(mine + e, Yp[(e / SM) * LDW + (e % SM)], seq);
    };
    // own rows: B[r, :] -= V_j[r, :] W2 from the ring; box i of the segment is shared by the two warps 2 (i mod 8) and
    // 2 (i mod 8) + 1, one 8-row group each (a stage is then held for 32 DMMAs instead of 64: the ring turns over faster)
    auto pass_u = [&](int j) {
        int la, le; range_of(j, la, le);
        int i = 0;
        for (int lr = la; lr < le; lr += CH, ++ccount, ++i) {
            if ((i % (NW / 2)) != (warp >> 1)) continue;
            const int st = (int)(ccount % (unsigned)NS);
            tma::mbar_wait(full(st), (ccount / (unsigned)NS) & 1u);
            const unsigned char* vs = ring + (size_t)st * kQt2StageBytes;
            if constexpr (F64) {
                const double* wb = W2 + (lane & 3) * LDW + (lane >> 2);
                const int r = 8 * (warp & 1) + (lane >> 2);
                double d0[4] = {0.0, 0.0, 0.0, 0.0}, d1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 8
                for (int t = 0; t < NB / 4; ++t) {
                    const int col = 4 * t + (lane & 3);
                    const double a = *reinterpret_cast<const double*>(vs + col * 128 + ((((r >> 1) ^ (col & 7)) << 4) | ((r & 1) << 3)));
                    dmma884(d0[t & 3], d1[t & 3], a, wb[4 * t * LDW]);
                }
                const int s0 = 2 * (lane & 3), l = lr + r;
                Bs[s0 * ldbs + l] -= (d0[0] + d0[1]) + (d0[2] + d0[3]);
                Bs[(s0 + 1) * ldbs + l] -= (d1[0] + d1[1]) + (d1[2] + d1[3]);
            } else {
                // fp32: the warp takes 16 of the 32 rows; lane = (row, column half), the halves combined by one shuffle
                const int r = 16 * (warp & 1) + (lane & 15), ch = lane >> 4;
                float d[SM];
#pragma unroll
                for (int q = 0; q < SM; ++q) d[q] = 0.f;
#pragma unroll 8
                for (int cc = 0; cc < NB / 2; ++cc) {
                    const int col = ch * (NB / 2) + ((cc + 4 * ch) & (NB / 2 - 1));   // (the halves hit disjoint banks)
                    const float v = *reinterpret_cast<const float*>(vs + col * 128 + ((((r >> 2) ^ (col & 7)) << 4) | ((r & 3) << 2)));
                    const float4 w0 = *reinterpret_cast<const float4*>(W2 + col * LDW), w1 = *reinterpret_cast<const float4*>(W2 + col * LDW + 4);
                    d[0] = fmaf(v, w0.x, d[0]); d[1] = fmaf(v, w0.y, d[1]); d[2] = fmaf(v, w0.z, d[2]); d[3] = fmaf(v, w0.w, d[3]);
                    d[4] = fmaf(v, w1.x, d[4]); d[5] = fmaf(v, w1.y, d[5]); d[6] = fmaf(v, w1.z, d[6]); d[7] = fmaf(v, w1.w, d[7]);
                }
#pragma unroll
                for (int q = 0; q < SM; ++q) d[q] += shfl_xor(d[q], 16);
                if (ch == 0)
#pragma unroll
                    for (int q = 0; q < SM; ++q) Bs[q * ldbs + lr + r] -= d[q];
            }
            __syncwarp();
            if (lane == 0) tma::mbar_arrive_n(empty(st), (unsigned)(NW / 2));
        }
    };
    // element owners: sum the partials of Y_j over the CTAs in a fixed order, subtract M_j W_(j-1) (Wg in shared memory
    // holds the gathered W_(j-1) when this runs), publish W_j.  One element per warp (128 * 8 elements over G CTAs x 16 warps);
    // the loads are issued by reduce_issue and consumed by reduce_finish so that the row update runs in between.
    constexpr int MAXB = 5;                                 // partial slots per lane: G <= 160 CTAs
    auto reduce_issue_e = [&](int j, int e, T (&gv)[4], uint4 (&r)[MAXB]) {
        const uint4* all = p.part + (size_t)(j & 1) * G * (NB * SM);
        const T* gt = p.Mt + (size_t)j * NB * NB + (size_t)(e / SM) * NB;
#pragma unroll
        for (int u = 0; u < 4; ++u) gv[u] = j >= 1 ? __ldg(gt + lane + 32 * u) : T(0);
#pragma unroll
        for (int u = 0; u < MAXB; ++u) {
            const int b = lane + u * 32;
            if (b < G) r[u] = ll_load(all + (size_t)b * (NB * SM) + e);
        }
    };
    auto reduce_finish_e = [&](int j, int e, const T (&gv)[4], uint4 (&r)[MAXB]) {
        const unsigned seq = p.seq_base + (unsigned)j + 1u;
        const uint4* all = p.part + (size_t)(j & 1) * G * (NB * SM);
        const int s = e % SM;
        T t = T(0);
#pragma unroll
        for (int u = 0; u < MAXB; ++u) {
            const int b = lane + u * 32;
            if (b < G) {
                while (r[u].y != seq || r[u].w != seq) r[u] = ll_load(all + (size_t)b * (NB * SM) + e);
                t += ll_value<T>(r[u]);
            }
        }
        T corr = T(0);
        if (j >= 1) {                                       // (Wg is not yet written when W_0 is formed)
#pragma unroll
            for (int u = 0; u < 4; ++u) corr = fma(gv[u], Wg[(lane + 32 * u) * LDW + s], corr);
        }
        t -= corr;
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) t += shfl_xor(t, off);
        if (lane == 0) ll_store(p.sums + (size_t)(j & 1) * (NB * SM) + e, t, seq);
    };
    // the first element of a warp is split into issue / finish (the gather runs in between); a grid of fewer than 64 CTAs
    // leaves more than one element per warp, the others follow back to back
    auto reduce_issue = [&](int j, T (&gv)[4], uint4 (&r)[MAXB]) {
        const int e = g + warp * G;
        if (e < NB * SM) reduce_issue_e(j, e, gv, r);
    };
    auto reduce_finish = [&](int j, T (&gv)[4], uint4 (&r)[MAXB]) {
        int e = g + warp * G;
        if (e >= NB * SM) return;
        reduce_finish_e(j, e, gv, r);
        for (e += NW * G; e < NB * SM; e += NW * G) {
            reduce_issue_e(j, e, gv, r);
            reduce_finish_e(j, e, gv, r);
        }
    };

    // ---- prologue: Y_0 and Y_1 from the rows as given; W_0 needs no correction ----
    pass_a(0);
    if (p.P > 1) pass_a(1);
    {
        T gv[4]; uint4 rr[MAXB];
        reduce_issue(0, gv, rr);
        reduce_finish(0, gv, rr);
    }

    for (int k = 0; k < p.P; ++k) {
        const int64_t j0 = (int64_t)k * NB;
        const int kw = (int)min((int64_t)NB, p.n - j0);
        const unsigned seq = p.seq_base + (unsigned)k + 1u;
        unsigned long long ph_t0 = 0; (void)ph_t0;
        CTQR_PH(0)
        // ---- element owners of W_(k+1): the loads of the partials (published one iteration ago) and of their row of
        //      M_(k+1) are issued before the gather spins, and consumed right after it ----
        T gv[4]; uint4 rr[MAXB];
        if (k + 1 < p.P) reduce_issue(k + 1, gv, rr);
        // ---- gather W_k (reduced and corrected by its element owners during the previous iteration) ----
        {
            const uint4* sl = p.sums + (size_t)(k & 1) * (NB * SM);
            uint4 r[NB * SM / NT];
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) r[u] = ll_load(sl + tid + u * NT);
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) {
                const int e = tid + u * NT;
                while (r[u].y != seq || r[u].w != seq) r[u] = ll_load(sl + e);
                Wg[(e / SM) * LDW + (e % SM)] = ll_value<T>(r[u]);
            }
        }
        sync_compute();
        CTQR_PH(1)
        // ---- W_(k+1) = sum of the partials - M_(k+1) W_k, published: the only step on the chain through the grid ----
        if (k + 1 < p.P) reduce_finish(k + 1, gv, rr);
        CTQR_PH(2)
        // ---- W2 = T_k^T W_k, T_k straight from L2 (upper triangular: q <= r) ----
        if constexpr (F64) {
            // DMMA fragments, every load of the warp in flight at once
            const int tr_row = warp * 8 + (lane >> 2);
            const double* tr = p.Tm + (size_t)k * NB * NB + (size_t)tr_row * NB + (lane & 3);
            double ta[NB / 4];
#pragma unroll
            for (int t = 0; t < NB / 4; ++t) {
                const int q = 4 * t + (lane & 3);
                ta[t] = (t < 2 * warp + 2 && q <= tr_row && tr_row < kw) ? __ldg(tr + 4 * t) : 0.0;
            }
            const double* wq = Wg + (lane & 3) * LDW + (lane >> 2);
            double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int t = 0; t < NB / 4; ++t)
                if (t < 2 * warp + 2) dmma884(c0[t & 3], c1[t & 3], ta[t], wq[4 * t * LDW]);
            W2[tr_row * LDW + 2 * (lane & 3)] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
            W2[tr_row * LDW + 2 * (lane & 3) + 1] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
        } else {
            // fp32: warp w forms rows 8w .. 8w+7 of W2; lanes over q (coalesced reads of column r of T), the sums over q by
            // two transpose-reductions
            const float* tk = p.Tm + (size_t)k * NB * NB;
            float tv[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int r = warp * 8 + i;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int q = lane + 32 * u;
                    tv[i][u] = (q <= r && r < kw) ? __ldg(tk + q + (size_t)r * NB) : 0.f;
                }
            }
            float acc[2][4 * SM];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int x = 0; x < 4 * SM; ++x) acc[h][x] = 0.f;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int q = lane + 32 * u;
                const float4 w0 = *reinterpret_cast<const float4*>(Wg + q * LDW), w1 = *reinterpret_cast<const float4*>(Wg + q * LDW + 4);
                const float wv[SM] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int q2 = 0; q2 < SM; ++q2) acc[i >> 2][(i & 3) * SM + q2] = fmaf(tv[i][u], wv[q2], acc[i >> 2][(i & 3) * SM + q2]);
            }
            warp_transpose_reduce<float, 4 * SM>(acc[0], lane);
            warp_transpose_reduce<float, 4 * SM>(acc[1], lane);
            W2[(warp * 8 + lane / SM) * LDW + (lane % SM)] = acc[0][0];
            W2[(warp * 8 + 4 + lane / SM) * LDW + (lane % SM)] = acc[1][0];
        }
        sync_compute();
        CTQR_PH(3)
        // ---- own rows updated with panel k ----
        pass_u(k);
        sync_compute();
        CTQR_PH(4)
        // ---- Y_(k+2) from the updated rows, published for the reduction ----
        if (k + 2 < p.P) pass_a(k + 2);
        CTQR_PH(5)
    }
    sync_compute();
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        if (s < S && lr < nl && row < p.m) p.B[row + (int64_t)s * p.ldb] = Bs[s * ldbs + lr];
    }
}


// -------------------------------------------------------------------------------------------------------------------
// Pipelined small-S blocked TRSM (task list PAPER.md:L62-73), both precisions.
//
// trsm_small_kernel (solve_small.cuh) has TWO grid hops on the critical path of every diagonal block: the row owners
// publish C_i -> everybody gathers it and forms X_i redundantly -> everybody updates -> the owners of the next block
// publish.  Here the chain through the grid is ONE hop per block:
//   * the rows of block i are published "stale", as they are after the updates of the blocks >= i+2 (Cst_i), while the
//     previous block is still being solved; the missing update is applied algebraically,
//         X_i = R_ii^{-1} (Cst_i - R_{i,i+1} X_{i+1}) = R_ii^{-1} Cst_i - N_i X_{i+1},   N_i = R_ii^{-1} R_{i,i+1}
//     (N_i: 128 x 128 per block, built once per handle next to the inverted diagonal blocks);
//   * X_i is formed element by element by element owners (one warp per element, element e belongs to CTA e mod G), each
//     reading one row of R_ii^{-1} and of N_i, and published; the bulk update of the rows above with X_{i+1} -- the pass
//     that streams R from HBM -- runs while that publication is in flight, starting with the rows of block i-1 so that
//     their owners can publish Cst_{i-1} early.
// Same row distribution as trsm_small_kernel (chunks of 16 rows dealt round-robin), deterministic.
// -------------------------------------------------------------------------------------------------------------------
template <typename T>
struct SmallTrsm2Args {
    const T* A; int64_t lda; int64_t n; int P;
    const T* Rinv;                  // P blocks of 128 x 128 (ld 128), zero-padded last block
    const T* Nm;                    // P blocks of 128 x 128 (ld 128): Nm[i] = Rinv_i R[i-th row block, (i+1)-th column block]
    T* X; int64_t ldx; int S;       // in: C[0:n, :], out: X
    uint4* cslots;                  // [2][128 * kSmallS] LL slots: stale rows of a block
    uint4* xslots;                  // [2][128 * kSmallS] LL slots: X of a block
    unsigned seq_base;              // step numbers seq_base + 1 .. seq_base + P are used by this launch
    int rpc;                        // local rows per CTA (multiple of kTrsmChunk)
};

template <typename T>
__global__ void __launch_bounds__(kTrsmThreads, 1) trsm_small2_kernel(SmallTrsm2Args<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NB = 128, SM = kSmallS, NT = kTrsmThreads, NW = NT / 32, CH = kTrsmChunk;
    T* Xs = reinterpret_cast<T*>(smem_raw);                 // [NB][SM]   X of the block solved last
    T* Ds = Xs + NB * SM;                                   // [<=8][SM][lim] partial updates (groups * lim <= NT)
    T* Cs = Ds + SM * NT;                                   // [SM][rpc]  own rows, transposed
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = blockIdx.x, G = gridDim.x, S = p.S;
    auto row_of = [&](int lr) -> int64_t { return ((int64_t)(lr / CH) * G + g) * CH + (lr % CH); };
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        Cs[i] = (s < S && row < p.n) ? p.X[row + (int64_t)s * p.ldx] : T(0);
    }
    __syncthreads();
    // the owners of the rows of block b publish them as they are now
    auto publish_rows = [&](int b) {
        const int64_t b0 = (int64_t)b * NB;
        const int kwb = (int)min((int64_t)NB, p.n - b0);
        const unsigned seq = p.seq_base + (unsigned)(p.P - 1 - b) + 1u;
        uint4* slots = p.cslots + (size_t)(b & 1) * (NB * SM);
        for (int e = tid; e < NB * SM; e += NT) {
            const int rr = e / SM, s = e - rr * SM;
            const int64_t q = (b0 + rr) / CH;
            if (rr < kwb && (int)(q % G) == g) ll_store(slots + e, Cs[s * p.rpc + (int)(q / G) * CH + (int)((b0 + rr) % CH)], seq);
        }
    };
    // own rows [lr0, lr1) (local indices; all above block b): C[r, :] -= R[r, block b] Xs, the 128 columns split over CS
    // thread groups so that enough loads are in flight
    auto update_rows = [&](int b, int lr0, int lr1) {
        const int64_t b0 = (int64_t)b * NB;
        const int kwb = (int)min((int64_t)NB, p.n - b0);
        const int cnt = lr1 - lr0;
        if (cnt <= 0) return;                                // (uniform over the CTA)
        int CS = 1;
        while (CS < 8 && 2 * CS * cnt <= NT) CS *= 2;
        const int cpc = (kwb + CS - 1) / CS;
        for (int base = 0; base < cnt; base += NT / CS) {    // NT / CS rows per sweep
            const int rows = min(cnt - base, NT / CS);
            const int cs = tid / rows, li = tid - cs * rows;
            T d[SM];
#pragma unroll
            for (int s = 0; s < SM; ++s) d[s] = T(0);
            const bool act = cs < CS;
            const int lr = lr0 + base + li;
            if (act) {
                const int64_t row = row_of(lr);
                const int c0 = cs * cpc, c1 = min(kwb, c0 + cpc);
                const T* rr = p.A + row + b0 * p.lda;
#pragma unroll 16
                for (int c = c0; c < c1; ++c) {
                    const T v = __ldg(rr + (int64_t)c * p.lda);
#pragma unroll
                    for (int s = 0; s < SM; ++s) d[s] = fma(v, Xs[c * SM + s], d[s]);
                }
            }
            if (CS == 1) {
                if (act)
#pragma unroll
                    for (int s = 0; s < SM; ++s) Cs[s * p.rpc + lr] -= d[s];
            } else {
                if (act)
#pragma unroll
                    for (int s = 0; s < SM; ++s) Ds[(cs * SM + s) * rows + li] = d[s];
                __syncthreads();
                for (int idx = tid; idx < rows * SM; idx += NT) {
                    const int s = idx / rows, l = idx - s * rows;
                    T t = T(0);
                    for (int c2 = 0; c2 < CS; ++c2) t += Ds[(c2 * SM + s) * rows + l];
                    Cs[s * p.rpc + lr0 + base + l] -= t;
                }
            }
            __syncthreads();
        }
    };
    // local row range [lo, hi) of the global rows [r0, r1) (both multiples of CH or the matrix end)
    auto local_of = [&](int64_t r) -> int {                 // number of own rows below global row r (r a multiple of CH)
        const int64_t q = r / CH;
        return q > g ? (int)((q - g + G - 1) / G) * CH : 0;
    };

    publish_rows(p.P - 1);
    for (int i = p.P - 1; i >= 0; --i) {
        const int64_t i0 = (int64_t)i * NB;
        const int kw = (int)min((int64_t)NB, p.n - i0);
        const unsigned seq = p.seq_base + (unsigned)(p.P - 1 - i) + 1u;
        // ---- 1. element owners: X_i[r, s] = sum_q Rinv_i[r, q] Cst_i[q, s] - sum_q N_i[r, q] X_(i+1)[q, s], published ----
        {
            const uint4* cst = p.cslots + (size_t)(i & 1) * (NB * SM);
            const T* ri = p.Rinv + (size_t)i * NB * NB;
            const T* ni = p.Nm + (size_t)i * NB * NB;
            for (int e = g + warp * G; e < NB * SM; e += NW * G) {
                const int r = e / SM, s = e - r * SM;
                T a[4], b[4];
                uint4 c[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int q = lane + 32 * u;
                    a[u] = __ldg(ri + r + (size_t)q * NB);
                    b[u] = (i + 1 < p.P) ? __ldg(ni + r + (size_t)q * NB) : T(0);
                    c[u] = q < kw ? ll_load(cst + q * SM + s) : make_uint4(0u, seq, 0u, seq);
                }
                T t = T(0);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int q = lane + 32 * u;
                    while (c[u].y != seq || c[u].w != seq) c[u] = ll_load(cst + q * SM + s);
                    t = fma(a[u], q < kw ? ll_value<T>(c[u]) : T(0), t);
                    if (i + 1 < p.P) t = fma(-b[u], Xs[q * SM + s], t);
                }
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) t += shfl_xor(t, off);
                if (lane == 0) ll_store(p.xslots + (size_t)(i & 1) * (NB * SM) + e, t, seq);
            }
        }
        // ---- 2. bulk update with X_(i+1) (still in Xs) of the own rows above block i, the rows of block i-1 first; their
        //         owners then publish them for the next block ----
        const int l_im1 = local_of(i0 > NB ? i0 - NB : 0), l_i = local_of(i0);      // own rows below (i-1) * NB, below i * NB
        if (i + 1 < p.P) update_rows(i + 1, l_im1, l_i);
        else __syncthreads();
        if (i >= 1) publish_rows(i - 1);
        if (i + 1 < p.P) update_rows(i + 1, 0, l_im1);
        // ---- 3. gather X_i; the owners of the rows of block i store it as their final rows ----
        __syncthreads();
        {
            const uint4* xs = p.xslots + (size_t)(i & 1) * (NB * SM);
            uint4 r[NB * SM / NT];
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) r[u] = ll_load(xs + tid + u * NT);
#pragma unroll
            for (int u = 0; u < NB * SM / NT; ++u) {
                const int e = tid + u * NT;
                while (r[u].y != seq || r[u].w != seq) r[u] = ll_load(xs + e);
                Xs[e] = ll_value<T>(r[u]);
            }
        }
        __syncthreads();
        for (int e = tid; e < NB * SM; e += NT) {
            const int rr = e / SM, s = e - rr * SM;
            const int64_t q = (i0 + rr) / CH;
            if (rr < kw && (int)(q % G) == g) Cs[s * p.rpc + (int)(q / G) * CH + (int)((i0 + rr) % CH)] = Xs[e];
        }
    }
    __syncthreads();
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        if (s < S && row < p.n) p.X[row + (int64_t)s * p.ldx] = Cs[i];
    }
}

}  // namespace ctqr
