// gemm_f64.cu -- fp64 instantiations of the contraction kernels (DMMA tensor-core path + SIMT check).
#include "gemm.cuh"

namespace ctqr {

void gemm_tile_f64(bool ta, int64_t M, int64_t N, int impl, int* bm, int* bn) {
    if (impl == 1) { *bm = 64; *bn = 64; return; }
    if (ta) { if (M <= 32) { *bm = 32; *bn = 128; } else { *bm = 128; *bn = 64; } }
    else    { if (N <= 32) { *bm = 128; *bn = 32; } else { *bm = 128; *bn = 64; } }
}

cudaError_t gemm_f64(bool ta, GemmArgs<double> g, int splits, int impl, cudaStream_t st) {
    if (g.M <= 0 || g.N <= 0) return cudaSuccess;
    g.a_vec_ok = aligned16(g.A, g.lda, 8);
    g.b_vec_ok = aligned16(g.B, g.ldb, 8);
    if (impl == 1) {
        return ta ? launch_simt<double, true, 64, 64, 8>(g, splits, st)
                  : launch_simt<double, false, 64, 64, 8>(g, splits, st);
    }
    if (ta) {
        if (g.M <= 32) return launch_dmma<true, 32, 128, 32, 32, 16, 4, 2>(g, splits, st);
        return launch_dmma<true, 128, 64, 64, 32, 16, 3, 2>(g, splits, st);
    }
    if (g.N <= 32) return launch_dmma<false, 128, 32, 32, 32, 16, 3, 2>(g, splits, st);
    return launch_dmma<false, 128, 64, 64, 32, 16, 3, 2>(g, splits, st);
}

}  // namespace ctqr
