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
//     G_j = V_(j-1)^T V_j (128 x 128, "Gt" below) is computed once per handle; the element owners of the reduction
//     subtract their rows of G_j^T W2_(j-1) before they publish the sums -- 128 KB of G per panel for the whole grid.
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

constexpr int kQt2Chunk = 16;                    // fp64 rows per TMA box: 128 bytes, the swizzle span
constexpr int kQt2StageBytes = kQt2Chunk * 128 * 8;
constexpr int kQt2DsElems = 2048;                // scratch of the column-split update (doubles)

struct SmallQt2Args {
    const double* A; int64_t lda; int64_t m, n; int P;
    const double* Tm;               // P blocks of 128 x 128 (ld 128)
    const double* Gt;               // P blocks of 128 x 128 (ld 128): Gt[j][q + c * 128] = (V_(j-1)^T V_j)[q][c], j >= 1
    double* B; int64_t ldb; int S;
    uint4* part;                    // [2][G][128 * kSmallS] LL slots: per-CTA partial Y
    uint4* sums;                    // [2][128 * kSmallS] LL slots: reduced, corrected W
    unsigned seq_base;              // step numbers seq_base + 1 .. seq_base + P are used by this launch
    int rpc;                        // local rows per CTA (multiple of kQt2Chunk)
    int64_t kl;                     // band promise (0 = dense)
    int nstage;                     // TMA ring stages
};

inline size_t qt2_smem_bytes(int rpc, int nstage) {
    return 1024 + (size_t)nstage * kQt2StageBytes + 16 * (size_t)nstage + 64 +
           ((size_t)3 * 128 * SmallLd<double>::W + kQt2DsElems + (size_t)kSmallS * (rpc + 4)) * sizeof(double);
}

__global__ void __launch_bounds__(kSmallThreads, 1)
apply_qt_small2_kernel(const __grid_constant__ CUtensorMap mapV, SmallQt2Args p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NB = 128, SM = kSmallS, NT = kSmallThreads, NW = NT / 32, CH = kQt2Chunk, LDW = SmallLd<double>::W;
    const unsigned sbase = (tma::smem_addr(smem_raw) + 1023u) & ~1023u;
    unsigned char* ring = smem_raw + (sbase - tma::smem_addr(smem_raw));
    const int NS = p.nstage;
    const unsigned bars = sbase + (unsigned)NS * kQt2StageBytes;            // full[NS], empty[NS]
    double* Wg = reinterpret_cast<double*>(ring + (size_t)NS * kQt2StageBytes + 16 * (size_t)NS + 64);   // gathered W_k
    double* Yp = Wg + NB * LDW;                             // this CTA's partial Y
    double* W2 = Yp + NB * LDW;                             // T_k^T W_k
    double* Ds = W2 + NB * LDW;                             // column-split partial updates
    double* Bs = Ds + kQt2DsElems;                          // [SM][ldbs] own rows of B, transposed
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
    // ---- issuer state (thread 0 only): next box = (panel ij, local row il) ----
    int ij = 0, il = 0, ile = 0;
    unsigned icount = 0;
    if (tid == 0) { range_of(0, il, ile); while (ij < p.P && il >= ile) { if (++ij < p.P) range_of(ij, il, ile); } }
    auto issue_next = [&]() {                               // thread 0: one more box, if any is left
        if (ij >= p.P) return;
        const int st = (int)(icount % (unsigned)NS);
        tma::mbar_wait(empty(st), ((icount / (unsigned)NS) & 1u) ^ 1u);
        tma::mbar_expect_tx(full(st), (unsigned)kQt2StageBytes);
        tma::load_2d(sbase + (unsigned)st * kQt2StageBytes, &mapV, (int)row_of(il), ij * NB, full(st));
        ++icount;
        il += CH;
        while (ij < p.P && il >= ile) { if (++ij < p.P) range_of(ij, il, ile); }
    };
    unsigned ccount = 0;                                    // boxes consumed so far (same order, every thread)

    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        Bs[s * ldbs + lr] = (s < S && lr < nl && row < p.m) ? p.B[row + (int64_t)s * p.ldb] : 0.0;
    }
    __syncthreads();
    if (tid == 0) for (int s = 0; s < NS; ++s) issue_next();

    // partial Y_j over the own rows from the TMA ring: warp w owns columns 8w .. 8w+7; result to Yp, then published
    auto pass_a = [&](int j) {
        int la, le; range_of(j, la, le);
        const int c = warp * 8 + (lane >> 2);
        const double* bs = Bs + (lane >> 2) * ldbs + (lane & 3);
        double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
        for (int lr = la; lr < le; lr += CH) {
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
            ++ccount;
            if (tid == 0) issue_next();
        }
        Yp[c * LDW + 2 * (lane & 3)] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
        Yp[c * LDW + 2 * (lane & 3) + 1] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
        __syncthreads();
        const unsigned seq = p.seq_base + (unsigned)j + 1u;
        uint4* mine = p.part + ((size_t)(j & 1) * G + g) * (NB * SM);
        for (int e = tid; e < NB * SM; e += NT) ll_store(mine + e, Yp[(e / SM) * LDW + (e % SM)], seq);
    };
    // element owners: sum the partials of Y_j over the CTAs in a fixed order, subtract (V_j^T V_(j-1)) W2_(j-1) (W2 in shared
    // memory holds W2_(j-1) when this runs), publish W_j
    auto reduce_j = [&](int j) {
        const unsigned seq = p.seq_base + (unsigned)j + 1u;
        const uint4* all = p.part + (size_t)(j & 1) * G * (NB * SM);
        const double* gt = p.Gt + (size_t)j * NB * NB;
        constexpr int MAXB = 5;
        for (int e = g + warp * G; e < NB * SM; e += NW * G) {
            const int c = e / SM, s = e - c * SM;
            double corr = 0.0;
            if (j >= 1) {
                double gv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) gv[u] = __ldg(gt + c * NB + lane + 32 * u);
#pragma unroll
                for (int u = 0; u < 4; ++u) corr = fma(gv[u], W2[(lane + 32 * u) * LDW + s], corr);
            }
            double t = 0.0;
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
                        t += ll_value<double>(r[u]);
                    }
                }
            }
            t -= corr;
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) t += shfl_xor(t, off);
            if (lane == 0) ll_store(p.sums + (size_t)(j & 1) * (NB * SM) + e, t, seq);
        }
    };

    // ---- prologue: Y_0 and Y_1 from the rows as given; W_0 needs no correction ----
    pass_a(0);
    if (p.P > 1) pass_a(1);
    reduce_j(0);

    for (int k = 0; k < p.P; ++k) {
        const int64_t j0 = (int64_t)k * NB;
        const int kw = (int)min((int64_t)NB, p.n - j0);
        const unsigned seq = p.seq_base + (unsigned)k + 1u;
        const double* V = p.A + j0 * p.lda;
        int la, le; range_of(k, la, le);
        const int na = le - la;
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
                Wg[(e / SM) * LDW + (e % SM)] = ll_value<double>(r[u]);
            }
        }
        __syncthreads();
        // ---- W2 = T_k^T W_k, T_k as DMMA fragments straight from L2 (upper triangular: q <= r) ----
        {
            const int r = warp * 8 + (lane >> 2);
            const double* tr = p.Tm + (size_t)k * NB * NB + (size_t)r * NB + (lane & 3);
            const double* wq = Wg + (lane & 3) * LDW + (lane >> 2);
            double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 4
            for (int t = 0; t < 2 * warp + 2; t += 4) {
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int q = 4 * (t + h) + (lane & 3);
                    const double a = (q <= r && r < kw) ? __ldg(tr + 4 * (t + h)) : 0.0;
                    dmma884(c0[h], c1[h], a, wq[4 * (t + h) * LDW]);
                }
            }
            W2[r * LDW + 2 * (lane & 3)] = (c0[0] + c0[1]) + (c0[2] + c0[3]);
            W2[r * LDW + 2 * (lane & 3) + 1] = (c1[0] + c1[1]) + (c1[2] + c1[3]);
        }
        __syncthreads();
        // ---- element owners: W_(k+1) from the partials published one iteration ago, corrected with W2_k ----
        if (k + 1 < p.P) reduce_j(k + 1);
        // ---- own rows: B[r, :] -= V_k[r, 0:kw] W2_k  (V_k from L2; a unit = 8 rows x one of CS column ranges) ----
        {
            const int mt = na / 8;
            int CS = 1;
            while (CS < 8 && mt * CS < NW && 2 * CS * na * SM <= kQt2DsElems) CS *= 2;
            const int steps = NB / 4 / CS;
            for (int u = warp; u < mt * CS; u += NW) {
                const int cs = u / mt, l0 = (u - cs * mt) * 8;
                const int64_t row = row_of(la + l0 + (lane >> 2));
                const bool okr = row < p.m;
                const int cbeg = cs * steps * 4 + (lane & 3);
                const double* vr = V + (int64_t)cbeg * p.lda + row;
                const double* wb = W2 + cbeg * LDW + (lane >> 2);
                double c0[4] = {0.0, 0.0, 0.0, 0.0}, c1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 8
                for (int t = 0; t < steps; t += 4) {
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
                    double t = 0.0;
                    for (int cs = 0; cs < CS; ++cs) t += Ds[(cs * SM + s) * na + l];
                    Bs[s * ldbs + la + l] -= t;
                }
                __syncthreads();
            }
        }
        // ---- Y_(k+2) from the updated rows (the boxes are already in the ring), published for the reduction ----
        if (k + 2 < p.P) pass_a(k + 2);
    }
    for (int i = tid; i < SM * p.rpc; i += NT) {
        const int s = i / p.rpc, lr = i - s * p.rpc;
        const int64_t row = row_of(lr);
        if (s < S && lr < nl && row < p.m) p.B[row + (int64_t)s * p.ldb] = Bs[s * ldbs + lr];
    }
}

}  // namespace ctqr
