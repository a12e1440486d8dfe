// gemm_f32.cu -- fp32 instantiations of the contraction kernels (FFMA register-tiled path).
#include "gemm.cuh"

namespace ctqr {

void gemm_tile_f32(bool ta, int64_t M, int64_t N, int impl, int* bm, int* bn) {
    (void)impl;
    if (ta) { if (M <= 32) { *bm = 32; *bn = 128; } else { *bm = 128; *bn = 128; } }
    else    { if (N <= 32) { *bm = 128; *bn = 32; } else { *bm = 128; *bn = 128; } }
}

cudaError_t gemm_f32(bool ta, GemmArgs<float> g, int splits, int impl, cudaStream_t st) {
    if (g.M <= 0 || g.N <= 0) return cudaSuccess;
    g.a_vec_ok = aligned16(g.A, g.lda, 4);
    g.b_vec_ok = aligned16(g.B, g.ldb, 4);
    (void)impl;
    if (ta) {
        if (g.M <= 32) return launch_simt<float, true, 32, 128, 8>(g, splits, st);
        return launch_simt<float, true, 128, 128, 8>(g, splits, st);
    }
    if (g.N <= 32) return launch_simt<float, false, 128, 32, 8>(g, splits, st);
    return launch_simt<float, false, 128, 128, 8>(g, splits, st);
}

}  // namespace ctqr
