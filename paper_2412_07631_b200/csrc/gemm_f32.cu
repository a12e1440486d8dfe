// gemm_f32.cu -- fp32 instantiations of the contraction kernels: persistent stream-K 3xTF32
// tensor-core kernel (gemm_mma.cuh) for the big products, SIMT FFMA for skinny in-panel shapes
// and as the impl = 1 cross-check.
#include <algorithm>
#include "gemm.cuh"
#include "gemm_mma.cuh"
#include "gemm_umma.cuh"
#include "gemm_umma_tma.cuh"

namespace ctqr {

static GemmLaunch classic_plan(int64_t M, int64_t N, int64_t K, int bm, int bn, int sms, int64_t min_chunk,
                               bool partial, int64_t max_elems, int64_t sstride, int cfg) {
    const int64_t max_slots = sstride > 0 ? max_elems / sstride : 1;
    GemmLaunch L{};
    L.kind = 0; L.cfg = cfg; L.partial = partial ? 1 : 0;
    int s = 1;
    if (partial) {
        s = pick_splits(ceil_div(M, bm) * ceil_div(N, bn), K, 8, sms, 2, min_chunk);
        if (s > max_slots) s = (int)std::max<int64_t>(1, max_slots);
    }
    L.splits = s; L.slots = s;
    L.seg = SegInfo{s, 0, 0, bn};
    return L;
}

static GemmLaunch streamk_plan(int64_t M, int64_t N, int64_t K, int bm, int bn, int bk, int sms, bool partial,
                               int64_t max_elems, int64_t sstride, int cfg) {
    (void)sstride;
    int slots = sms * 2;
    MmaPlan p = mma_plan(M, N, K, bm, bn, bk, slots, partial);
    while (partial && p.partial_elems > max_elems && slots > 1) { slots /= 2; p = mma_plan(M, N, K, bm, bn, bk, slots, partial); }
    GemmLaunch L{};
    L.kind = 1; L.cfg = cfg; L.grid = p.grid; L.tilesM = p.sk.tilesM; L.tilesN = p.sk.tilesN; L.U = p.sk.U;
    L.L = p.sk.L; L.KT = p.sk.KT; L.partial = p.sk.partial; L.slots = p.maxseg; L.splits = 1;
    L.G = p.sk.G; L.Gm = p.sk.Gm;
    L.seg = SegInfo{1, p.sk.KT, p.sk.L, bn};
    return L;
}

// tcgen05 (UMMA) plan: 128 x 128 tiles, one CTA per SM
static GemmLaunch umma_plan_f32(int64_t M, int64_t N, int64_t K, int bn, int sms, bool partial, int64_t max_elems, int cfg) {
    int slots = sms;
    MmaPlan p = umma::umma_plan(M, N, K, bn, slots, partial);
    while (partial && p.partial_elems > max_elems && slots > 1) { slots /= 2; p = umma::umma_plan(M, N, K, bn, slots, partial); }
    GemmLaunch L{};
    L.kind = 1; L.cfg = cfg; L.grid = p.grid; L.tilesM = p.sk.tilesM; L.tilesN = p.sk.tilesN; L.U = p.sk.U;
    L.L = p.sk.L; L.KT = p.sk.KT; L.partial = p.sk.partial; L.slots = p.maxseg; L.splits = 1;
    L.G = p.sk.G; L.Gm = p.sk.Gm;
    L.seg = SegInfo{1, p.sk.KT, p.sk.L, bn};
    return L;
}

GemmLaunch gemm_plan_f32(bool ta, int64_t M, int64_t N, int64_t K, int impl, int sms, bool partial, int64_t max_elems,
                         int64_t sstride, bool aligned) {
    if (impl == 1 || !aligned) {
        if (ta) return M <= 32 ? classic_plan(M, N, K, 32, 128, sms, 256, partial, max_elems, sstride, 0)
                               : classic_plan(M, N, K, 128, 128, sms, 512, partial, max_elems, sstride, 4);
        return N <= 32 ? classic_plan(M, N, K, 128, 32, sms, 256, partial, max_elems, sstride, 2)
                       : classic_plan(M, N, K, 128, 128, sms, 512, partial, max_elems, sstride, 5);
    }
    // the big products go to the tcgen05 kernel (float4 chunks: K, and M when A is m-contiguous, multiples of 4)
    const bool umma_ok = N >= 128 && K % 4 == 0;
    if (ta) {
        if (M <= 32) return classic_plan(M, N, K, 32, 128, sms, 256, partial, max_elems, sstride, 0);
        if (umma_ok && M <= 128) return umma_plan_f32(M, N, K, 128, sms, partial, max_elems, 21);
        return streamk_plan(M, N, K, 128, 64, 32, sms, partial, max_elems, sstride, 1);
    }
    if (N <= 32) return classic_plan(M, N, K, 128, 32, sms, 256, partial, max_elems, sstride, 2);
    if (umma_ok && M % 4 == 0) return umma_plan_f32(M, N, K, partial ? 128 : 64, sms, partial, max_elems, partial ? 24 : 23);
    return streamk_plan(M, N, K, 128, 64, 32, sms, partial, max_elems, sstride, 3);
}

cudaError_t split_tf32_launch(const float* src, int64_t ld, int64_t rows, int64_t cols, float* hi, float* lo, int64_t ld_out, cudaStream_t st) {
    return split_tf32_launch_impl(src, ld, rows, cols, hi, lo, ld_out, st);
}
cudaError_t upd_presplit_launch(int64_t M, int64_t N, int64_t K, float alpha, const float* Ahi, const float* Alo, int64_t lda,
                                const float* Bhi, const float* Blo, int64_t ldb, float beta, float* C, int64_t ldc, int ctas, cudaStream_t st) {
    return upd_presplit_launch_impl(M, N, K, alpha, Ahi, Alo, lda, Bhi, Blo, ldb, beta, C, ldc, ctas, st);
}

static MmaPlan to_plan(const GemmLaunch& L) {
    MmaPlan p{};
    p.sk.tilesM = L.tilesM; p.sk.tilesN = L.tilesN; p.sk.KT = L.KT; p.sk.U = L.U; p.sk.L = L.L; p.sk.partial = L.partial;
    p.grid = L.grid; p.maxseg = L.slots; p.sk.G = L.G; p.sk.Gm = L.Gm;
    return p;
}

cudaError_t vtc_presplit_launch(const GemmArgs<float>& g, const float* Ahi, const float* Alo, int64_t lda, const GemmLaunch& L, cudaStream_t st) {
    if (L.kind != 1 || L.cfg != 21 || !L.partial) return cudaErrorNotSupported;
    return vtc_presplit_launch_impl(g, Ahi, Alo, lda, to_plan(L), st);
}

cudaError_t gemm_run_f32(bool ta, GemmArgs<float> g, const GemmLaunch& L, int impl, cudaStream_t st) {
    if (g.M <= 0 || g.N <= 0) return cudaSuccess;
    g.a_vec_ok = aligned16(g.A, g.lda, 4);
    g.b_vec_ok = aligned16(g.B, g.ldb, 4);
    (void)impl;
    switch (L.cfg) {
        case 0: return launch_simt<float, true, 32, 128, 8>(g, L.splits, st);
        case 4: return launch_simt<float, true, 128, 128, 8>(g, L.splits, st);
        case 2: return launch_simt<float, false, 128, 32, 8>(g, L.splits, st);
        case 5: return launch_simt<float, false, 128, 128, 8>(g, L.splits, st);
        case 1: return launch_mma<float, true, 128, 64, 32, 32, 3, 2>(g, to_plan(L), st);
        case 3: return launch_mma<float, false, 128, 64, 32, 32, 3, 2>(g, to_plan(L), st);
        case 21: return umma::launch_umma<true, 128>(g, to_plan(L), st);
        case 23: return umma::launch_umma_ws<false, 64>(g, to_plan(L), st);
        case 24: return umma::launch_umma<false, 128>(g, to_plan(L), st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace ctqr
