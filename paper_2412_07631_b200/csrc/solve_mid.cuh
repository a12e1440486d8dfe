// solve_mid.cuh -- Q^T B for a medium number of right-hand sides (8 < S <= 32 per launch, fp64): the pipelined, TMA-fed
// cooperative kernel of solve_small2.cuh with the right-hand sides in NG groups of eight (PAPER.md
// Fig. 1 / Eq. 3: throughput against the number of slices solved at once).
//
// The per-panel path spends three launches per panel on this regime (W = V_k^T B as split-K partial tiles, T_k^T W, the
// update): at S = 64 the products have ONE 128 x 64 output tile, so the split can use only as many SMs as the consumer of
// the partial tiles can afford to sum -- 62 CTAs, 51 + 11 + 31 us per panel at configs[2] -- and the chain of 3 P launches
// is 11 ms long where the arithmetic needs 3.7 ms and the memory traffic 0.7 ms.  Here the whole application is one launch:
// everything solve_small2.cuh says about the order of the passes, the stale products Y_j = V_j^T B_(j-2), the correction
// W_j = Y_j - M_j W_(j-1) by the element owners, the one-hop chain and the TMA ring holds unchanged; what changes is that a
// V fragment read from a box feeds NG DMMAs (one per group of eight right-hand sides) instead of one, so the kernel moves
// from the memory-latency bound towards the DMMA pipe as S grows.  Shared memory bounds S: the CTA's rows of B, two
// 128 x S blocks (gathered W; T^T W, reused for the partial Y) and the ring must fit in 225 KB (the host picks NG and the stage count;
// S beyond one launch is applied in column chunks).  Deterministic, like the small-S kernel.
#pragma once
#include "solve_small2.cuh"

namespace ctqr {

template <int NG> struct MidCfg {
    static constexpr int SM = 8 * NG;          // right-hand sides per launch
    static constexpr int LDW = SM + 4;         // row length of the 128 x SM blocks: fragment reads hit 32 distinct banks
    static constexpr int KC = NG >= 4 ? 1 : 4 / NG;   // independent accumulator chains per group (DMMA latency)
};

template <int NG> constexpr int qt_mid_min_stages() { return (kQt2Warps / (2 * NG)) > 3 ? (kQt2Warps / (2 * NG)) : 3; }

template <int NG>
inline size_t qt_mid_smem_bytes(int rpc, int nstage) {
    return 1024 + (size_t)nstage * kQt2StageBytes + 16 * (size_t)nstage + 64 +
           ((size_t)2 * 128 * MidCfg<NG>::LDW + (size_t)MidCfg<NG>::SM * (rpc + 4)) * sizeof(double);
}

// Arguments: SmallQt2Args<double> with part = [2][G][128 * SM] and sums = [2][128 * SM] LL slots.
template <int NG>
__global__ void __launch_bounds__(kQt2Threads, 1)
apply_qt_mid_kernel(const __grid_constant__ CUtensorMap mapV, SmallQt2Args<double> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using T = double;
    constexpr int NB = 128, SM = MidCfg<NG>::SM, NW = kQt2Warps, NT = NW * 32, CH = Qt2Chunk<T>::value, LDW = MidCfg<NG>::LDW,
                  KC = MidCfg<NG>::KC;
    const unsigned sbase = (tma::smem_addr(smem_raw) + 1023u) & ~1023u;
    unsigned char* ring = smem_raw + (sbase - tma::smem_addr(smem_raw));
    const int NS = p.nstage;
    const unsigned bars = sbase + (unsigned)NS * kQt2StageBytes;            // full[NS], empty[NS]
    T* Wg = reinterpret_cast<T*>(ring + (size_t)NS * kQt2StageBytes + 16 * (size_t)NS + 64);   // gathered W_k
    T* W2 = Wg + NB * LDW;                                  // T_k^T W_k: dead once the update pass has its fragments in registers
    T* Yp = W2;                                             // this CTA's partial Y (written after the update pass, published
                                                            // before the next T^T W): shares the block with W2
    T* Bs = W2 + NB * LDW;                                  // [SM][ldbs] own rows of B, transposed
    const int ldbs = p.rpc + 4;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, grp = lane >> 2, tig = lane & 3;
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
        // ================= TMA producer: the box sequence A(0), A(1), { U(k), A(k+2) }, as far ahead as the ring allows ====
        if (lane == 0) {
            unsigned icount = 0;
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

    // partial Y_j over the own rows from the ring: warp w owns columns 8w .. 8w+7 of the panel, all SM right-hand sides
    auto pass_a = [&](int j) {
        int la, le; range_of(j, la, le);
        const int c = warp * 8 + grp;
        const double* bs = Bs + grp * ldbs + tig;
        double c0[NG][KC], c1[NG][KC];
#pragma unroll
        for (int gi = 0; gi < NG; ++gi)
#pragma unroll
            for (int q = 0; q < KC; ++q) { c0[gi][q] = 0.0; c1[gi][q] = 0.0; }
        for (int lr = la; lr < le; lr += CH, ++ccount) {
            const int st = (int)(ccount % (unsigned)NS);
            tma::mbar_wait(full(st), (ccount / (unsigned)NS) & 1u);
            const unsigned char* vs = ring + (size_t)st * kQt2StageBytes + c * 128;
            double a[4];
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const int r = 4 * h + tig;
                a[h] = *reinterpret_cast<const double*>(vs + ((((r >> 1) ^ (c & 7)) << 4) | ((r & 1) << 3)));
            }
#pragma unroll
            for (int h = 0; h < 4; ++h)
#pragma unroll
                for (int gi = 0; gi < NG; ++gi) dmma884(c0[gi][h % KC], c1[gi][h % KC], a[h], bs[(size_t)(8 * gi) * ldbs + lr + 4 * h]);
            __syncwarp();
            if (lane == 0) tma::mbar_arrive(empty(st));
        }
        sync_compute();                                     // the previous publication has finished reading Yp
#pragma unroll
        for (int gi = 0; gi < NG; ++gi) {
            double s0 = c0[gi][0], s1 = c1[gi][0];
#pragma unroll
            for (int q = 1; q < KC; ++q) { s0 += c0[gi][q]; s1 += c1[gi][q]; }
            Yp[c * LDW + 8 * gi + 2 * tig] = s0;
            Yp[c * LDW + 8 * gi + 2 * tig + 1] = s1;
        }
        sync_compute();
        const unsigned seq = p.seq_base + (unsigned)j + 1u;
        uint4* mine = p.part + ((size_t)(j & 1) * G + g) * (NB * SM);
        for (int e = tid; e < NB * SM; e += NT) ll_store(mine + e, Yp[(e / SM) * LDW + (e % SM)], seq);
    };
    // own rows: B[r, :] -= V_j[r, :] W2 from the ring.  A box (16 rows) is shared by 2 NG warps: (8-row group) x (group of
    // eight right-hand sides), so NW / (2 NG) boxes are in work at a time and every warp keeps the 32 W2 fragments of its
    // group in registers for the whole pass.  (A warp waits for a box up to NBX - 1 boxes ahead of the oldest one still in
    // work: the ring must have at least NBX stages, or the parity test of the mbarrier would see a phase two behind.)
    auto pass_u = [&](int j) {
        int la, le; range_of(j, la, le);
        constexpr int WPB = 2 * NG, NBX = NW / WPB;
        const int set = warp / WPB, wi = warp % WPB, rg = wi & 1, gi = wi >> 1;
        const int r = 8 * rg + grp;
        double wf[NB / 4];
        {
            const double* wb = W2 + tig * LDW + 8 * gi + grp;
#pragma unroll
            for (int t = 0; t < NB / 4; ++t) wf[t] = wb[4 * t * LDW];
        }
        int i = 0;
        for (int lr = la; lr < le; lr += CH, ++ccount, ++i) {
            if ((i % NBX) != set) continue;
            const int st = (int)(ccount % (unsigned)NS);
            tma::mbar_wait(full(st), (ccount / (unsigned)NS) & 1u);
            const unsigned char* vs = ring + (size_t)st * kQt2StageBytes;
            double d0[4] = {0.0, 0.0, 0.0, 0.0}, d1[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int t = 0; t < NB / 4; ++t) {
                const int col = 4 * t + tig;
                const double a = *reinterpret_cast<const double*>(vs + col * 128 + ((((r >> 1) ^ (col & 7)) << 4) | ((r & 1) << 3)));
                dmma884(d0[t & 3], d1[t & 3], a, wf[t]);
            }
            const int l = lr + r;
            Bs[(8 * gi + 2 * tig) * ldbs + l] -= (d0[0] + d0[1]) + (d0[2] + d0[3]);
            Bs[(8 * gi + 2 * tig + 1) * ldbs + l] -= (d1[0] + d1[1]) + (d1[2] + d1[3]);
            __syncwarp();
            if (lane == 0) tma::mbar_arrive_n(empty(st), (unsigned)NBX);
        }
    };
    // element owners: element e of W_j (e = column c * SM + right-hand side s) belongs to warp (e / G) mod 16 of CTA e mod G:
    // sum the partials of the CTAs in a fixed order, subtract row c of M_j times W_(j-1) (in Wg), publish
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
        // ---- element owners of W_(k+1): loads issued before the gather spins, consumed right after it ----
        T gv[4]; uint4 rr[MAXB];
        if (k + 1 < p.P) reduce_issue(k + 1, gv, rr);
        // ---- gather W_k (reduced and corrected by its element owners during the previous iteration) ----
        {
            const uint4* sl = p.sums + (size_t)(k & 1) * (NB * SM);
            constexpr int PER = 4;                          // loads in flight per thread
#pragma unroll 1
            for (int base = 0; base < NB * SM; base += PER * NT) {
                uint4 r[PER];
#pragma unroll
                for (int u = 0; u < PER; ++u) r[u] = ll_load(sl + base + tid + u * NT);
#pragma unroll
                for (int u = 0; u < PER; ++u) {
                    const int e = base + tid + u * NT;
                    while (r[u].y != seq || r[u].w != seq) r[u] = ll_load(sl + e);
                    Wg[(e / SM) * LDW + (e % SM)] = ll_value<T>(r[u]);
                }
            }
        }
        sync_compute();
        CTQR_PH(1)
        // ---- W_(k+1) = sum of the partials - M_(k+1) W_k, published: the only step on the chain through the grid ----
        if (k + 1 < p.P) reduce_finish(k + 1, gv, rr);
        CTQR_PH(2)
        // ---- W2 = T_k^T W_k, T_k as DMMA fragments straight from L2 (upper triangular: q <= r) ----
        {
            const int tr_row = warp * 8 + grp;
            const double* tr = p.Tm + (size_t)k * NB * NB + (size_t)tr_row * NB + tig;
            double ta[NB / 4];
#pragma unroll
            for (int t = 0; t < NB / 4; ++t) {
                const int q = 4 * t + tig;
                ta[t] = (t < 2 * warp + 2 && q <= tr_row && tr_row < kw) ? __ldg(tr + 4 * t) : 0.0;
            }
            const double* wq = Wg + tig * LDW + grp;
            double c0[NG][KC], c1[NG][KC];
#pragma unroll
            for (int gi = 0; gi < NG; ++gi)
#pragma unroll
                for (int q = 0; q < KC; ++q) { c0[gi][q] = 0.0; c1[gi][q] = 0.0; }
#pragma unroll
            for (int t = 0; t < NB / 4; ++t)
                if (t < 2 * warp + 2) {
#pragma unroll
                    for (int gi = 0; gi < NG; ++gi) dmma884(c0[gi][t % KC], c1[gi][t % KC], ta[t], wq[4 * t * LDW + 8 * gi]);
                }
#pragma unroll
            for (int gi = 0; gi < NG; ++gi) {
                double s0 = c0[gi][0], s1 = c1[gi][0];
#pragma unroll
                for (int q = 1; q < KC; ++q) { s0 += c0[gi][q]; s1 += c1[gi][q]; }
                W2[tr_row * LDW + 8 * gi + 2 * tig] = s0;
                W2[tr_row * LDW + 8 * gi + 2 * tig + 1] = s1;
            }
        }
        sync_compute();
        CTQR_PH(3)
        // ---- own rows updated with panel k, then Y_(k+2) from the updated rows, published for the reduction ----
        pass_u(k);
        sync_compute();
        CTQR_PH(4)
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

}  // namespace ctqr
