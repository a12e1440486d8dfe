// gemm_f64.cu -- fp64 instantiations of the contraction kernels: persistent stream-K DMMA kernel
// (gemm_mma.cuh) for the big products, the classic DMMA grid kernel for skinny in-panel shapes,
// SIMT DFMA as cross-check (impl 1).
#include <algorithm>
#include "gemm.cuh"
#include "gemm_mma.cuh"

namespace ctqr {

static GemmLaunch classic_plan(int64_t M, int64_t N, int64_t K, int bm, int bn, int sms, int64_t min_chunk,
                               bool partial, int64_t max_elems, int64_t sstride, int cfg) {
    const int64_t max_slots = sstride > 0 ? max_elems / sstride : 1;
    GemmLaunch L{};
    L.kind = 0; L.cfg = cfg; L.partial = partial ? 1 : 0;
    int s = 1;
    if (partial) {
        s = pick_splits(ceil_div(M, bm) * ceil_div(N, bn), K, 16, sms, 2, min_chunk);
        if (s > max_slots) s = (int)std::max<int64_t>(1, max_slots);
    }
    L.splits = s; L.slots = s;
    L.seg = SegInfo{s, 0, 0, bn};
    return L;
}

static GemmLaunch streamk_plan(int64_t M, int64_t N, int64_t K, int bm, int bn, int bk, int sms, bool partial,
                               int64_t max_elems, int64_t sstride, int cfg, int ctas_per_sm = 2) {
    (void)sstride;
    int slots = sms * ctas_per_sm;
    MmaPlan p = mma_plan(M, N, K, bm, bn, bk, slots, partial);
    while (partial && p.partial_elems > max_elems && slots > 1) { slots /= 2; p = mma_plan(M, N, K, bm, bn, bk, slots, partial); }
    GemmLaunch L{};
    L.kind = 1; L.cfg = cfg; L.grid = p.grid; L.tilesM = p.sk.tilesM; L.tilesN = p.sk.tilesN; L.U = p.sk.U;
    L.L = p.sk.L; L.KT = p.sk.KT; L.partial = p.sk.partial; L.slots = p.maxseg; L.splits = 1;
    L.G = p.sk.G; L.Gm = p.sk.Gm;
    L.seg = SegInfo{1, p.sk.KT, p.sk.L, bn};
    return L;
}

GemmLaunch gemm_plan_f64(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems,
                         int64_t sstride, bool aligned) {
    if (impl == 1) return classic_plan(M, N, K, 64, 64, sms, 256, partial, max_elems, sstride, 9);
    if (ta) {
        if (M <= 32) return classic_plan(M, N, K, 32, 128, sms, 256, partial, max_elems, sstride, 0);
        if (!aligned) return classic_plan(M, N, K, 128, 64, sms, 512, partial, max_elems, sstride, 6);
        return streamk_plan(M, N, K, 128, 64, MmaPolicy<double>::BK, sms, partial, max_elems, sstride, 1);
    }
    if (N <= 32) return classic_plan(M, N, K, 128, 32, sms, 256, partial, max_elems, sstride, 2);
    if (!aligned) return classic_plan(M, N, K, 128, 64, sms, 512, partial, max_elems, sstride, 7);
    return streamk_plan(M, N, K, 128, 64, MmaPolicy<double>::BK, sms, partial, max_elems, sstride, 3);
}

static MmaPlan to_plan(const GemmLaunch& L) {
    MmaPlan p{};
    p.sk.tilesM = L.tilesM; p.sk.tilesN = L.tilesN; p.sk.KT = L.KT; p.sk.U = L.U; p.sk.L = L.L; p.sk.partial = L.partial;
    p.grid = L.grid; p.maxseg = L.slots; p.sk.G = L.G; p.sk.Gm = L.Gm;
    p.sk.tickets = L.tickets; p.sk.reserve = L.reserve;
    return p;
}

cudaError_t gemm_run_f64(bool ta, GemmArgs<double> g, const GemmLaunch& L, int impl, cudaStream_t st) {
    if (g.M <= 0 || g.N <= 0) return cudaSuccess;
    g.a_vec_ok = aligned16(g.A, g.lda, 8);
    g.b_vec_ok = aligned16(g.B, g.ldb, 8);
    (void)impl;
    switch (L.cfg) {
        case 9: return ta ? launch_simt<double, true, 64, 64, 8>(g, L.splits, st)
                          : launch_simt<double, false, 64, 64, 8>(g, L.splits, st);
        case 0: return launch_dmma<true, 32, 128, 32, 32, 16, 4, 2>(g, L.splits, st);
        case 1: return launch_mma<double, true, 128, 64, 32, 32, 3, 2>(g, to_plan(L), st);
        case 2: return launch_dmma<false, 128, 32, 32, 32, 16, 3, 2>(g, L.splits, st);
        case 6: return launch_dmma<true, 128, 64, 64, 32, 16, 3, 2>(g, L.splits, st);
        case 7: return launch_dmma<false, 128, 64, 64, 32, 16, 3, 2>(g, L.splits, st);
        case 3: return launch_mma<double, false, 128, 64, 32, 32, 3, 2>(g, to_plan(L), st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace ctqr
