// gemm_umma_tma.cuh -- C <- alpha * A * B + beta * C in fp32 as a 3xTF32 split on tcgen05 with PRE-SPLIT operands fed by
// TMA (the larfb product C <- C - V W, the dominant kernel of the fp32 factorisation).
//
// gemm_umma.cuh splits every operand tile into hi + lo again for every output tile (the producer warps took 60 % of the
// issue slots, ncu profiles/r1_final_c3.md) and drains the TMEM accumulator after every 32 of K.  Here
//   * A (= the reflector block V, M x K, m-contiguous) and B (= W, K x N, k-contiguous) are split ONCE per panel pair into
//     hi / lo arrays of TF32 bit patterns by split_tf32_kernel -- both are small and re-read by every tile;
//   * one thread issues cp.async.bulk.tensor (TMA) loads of the four operand tiles of a k-block straight into the UMMA
//     canonical shared-memory layouts (K-major SWIZZLE_128B for B, MN-major SWIZZLE_128B with 32-byte atoms for A: the
//     hardware swizzles, nothing is transposed), completing on the stage's `full` mbarrier; there are no producer warps;
//   * one thread issues the tcgen05.mma kind::tf32 instructions (128 x 128 x 8, three per k-step: lo*hi, hi*lo, hi*hi);
//   * the accumulator stays in TMEM for kDrain k-blocks (128 of K) before the drainer warps add it to the running sum in
//     registers with round-to-nearest FADDs (the tensor core's own accumulation truncates: an error growing linearly in
//     the number of accumulated terms, 1e-5 at K = 1024; 128 terms keep it at FFMA level);
//   * 128 x 128 output tiles: a 128 x 64 tile needs 6 KB of shared-memory operand reads per 35-clock MMA, more than the
//     128 B/clk the SM delivers; 128 x 128 needs 8 KB per 69 clocks.
// Warp roles: warp 0 TMA producer, warp 1 MMA issuer (owns the TMEM allocation), warps 2-9 drainers / epilogue.
#pragma once
#include "common.cuh"
#include "gemm_umma.cuh"
#include "tma.cuh"

namespace ctqr {
namespace umma {

constexpr int kTBN = 128, kTStages = 3, kDrain = 4;
constexpr int kTTile = 128 * BK * 4;                       // one operand tile: 128 rows x 32 floats = 16 KB
constexpr int kTStage = 4 * kTTile;                        // A_hi, A_lo, B_hi, B_lo
constexpr int kTSmem = kTStages * kTStage + 1024 + 256;
constexpr int kTDrainThreads = 256, kTThreads = 64 + kTDrainThreads;

struct UpdTmaArgs {
    int64_t M, N, K;
    float* C; int64_t ldc;
    float alpha, beta;
    int64_t tilesM, tilesN;
    int KT;                           // k-blocks of 32
    int Gm;                           // tile rows per band of the tile order (see tile_of)
};

// Tile order with L2 locality.  Tiles are numbered band by band (Gm tile rows per band), inside a band column block by
// column block, tile rows fastest, and dealt round-robin: CTA g takes the numbers g, g + G, g + 2G, ...  The G tiles in
// flight at any time are then consecutive numbers, i.e. a compact Gm x (G / Gm) patch that shares Gm tiles of A and G / Gm
// tiles of B.  (With contiguous per-CTA ranges the CTAs sit at unrelated tile rows and cycle through ALL of the pre-split
// A -- 221 MB at m = 1e5 -- which no longer fits the L2: ncu showed 109 GB of DRAM reads for 14 GB of C, L2 hit rate 29 %.)
__device__ __forceinline__ void tile_of(const UpdTmaArgs& g, int64_t q, int64_t& tm, int64_t& tn) {
    const int64_t per_band = (int64_t)g.Gm * g.tilesN;
    const int64_t band = q / per_band, r = q - band * per_band;
    const int64_t hb = min((int64_t)g.Gm, g.tilesM - band * g.Gm);
    tn = r / hb; tm = band * g.Gm + (r - tn * hb);
}

// hi / lo TF32 bit patterns of a column-major block (ld_out >= rows; the padding rows are written as zeros)
__global__ void split_tf32_kernel(const float* __restrict__ src, int64_t ld, int64_t rows, int64_t cols,
                                  float* __restrict__ hi, float* __restrict__ lo, int64_t ld_out) {
    const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (r >= ld_out) return;
    for (int64_t c = blockIdx.y; c < cols; c += gridDim.y) {
        float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
        const float* s = src + r + c * ld;
        if (r + 3 < rows && ((uintptr_t)s & 15) == 0) x = __ldg(reinterpret_cast<const float4*>(s));
        else {
            if (r < rows) x.x = s[0];
            if (r + 1 < rows) x.y = s[1];
            if (r + 2 < rows) x.z = s[2];
            if (r + 3 < rows) x.w = s[3];
        }
        uint4 h, l;
        split4(x, h, l);
        *reinterpret_cast<uint4*>(hi + r + c * ld_out) = h;
        *reinterpret_cast<uint4*>(lo + r + c * ld_out) = l;
    }
}

__global__ void __launch_bounds__(kTThreads, 1)
upd_tma_kernel(const __grid_constant__ CUtensorMap mAh, const __grid_constant__ CUtensorMap mAl,
               const __grid_constant__ CUtensorMap mBh, const __grid_constant__ CUtensorMap mBl, UpdTmaArgs g) {
    extern __shared__ unsigned char smem_raw[];
    const unsigned sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const unsigned bars = sbase + kTStages * kTStage;
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (kTStages + s); };
    auto tfull = [&](int b) { return bars + 8u * (2 * kTStages + b); };
    auto tempty = [&](int b) { return bars + 8u * (2 * kTStages + 2 + b); };
    unsigned* tmem_slot = reinterpret_cast<unsigned*>(sgen + kTStages * kTStage + 8 * (2 * kTStages + 4));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t tiles = g.tilesM * g.tilesN;
    const int64_t t0 = (int64_t)blockIdx.x, t1 = tiles, tstep = (int64_t)gridDim.x;

    if (tid == 0) {
        for (int s = 0; s < kTStages; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull(b), 1); mbar_init(tempty(b), kTDrainThreads); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        tma::prefetch_map(&mAh); tma::prefetch_map(&mAl); tma::prefetch_map(&mBh); tma::prefetch_map(&mBl);
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)), "r"(256u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = *tmem_slot;

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            int s = 0; unsigned ph = 1;
            for (int64_t t = t0; t < t1; t += tstep) {
                int64_t tm, tn;
                tile_of(g, t, tm, tn);
                const int m0 = (int)(tm * BM), n0 = (int)(tn * kTBN);
                for (int kb = 0; kb < g.KT; ++kb) {
                    mbar_wait(empty(s), ph);
                    tma::mbar_expect_tx(full(s), (unsigned)kTStage);
                    const unsigned st = sbase + s * kTStage;
                    const int k0 = kb * BK;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {          // A: four boxes of 32 m x 32 k (4 KB each), m-groups 4 KB apart
                        tma::load_2d(st + i * 4096, &mAh, m0 + 32 * i, k0, full(s));
                        tma::load_2d(st + kTTile + i * 4096, &mAl, m0 + 32 * i, k0, full(s));
                    }
                    tma::load_2d(st + 2 * kTTile, &mBh, k0, n0, full(s));      // B: one box of 32 k x 128 n
                    tma::load_2d(st + 3 * kTTile, &mBl, k0, n0, full(s));
                    if (++s == kTStages) { s = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer =================
        const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | ((unsigned)(kTBN >> 3) << 17) | ((unsigned)(BM >> 4) << 24);
        int s = 0; unsigned fph = 0;
        int64_t d = 0;                                     // accumulator generations handed to the drainers so far
        for (int64_t t = t0; t < t1; t += tstep) {
            for (int kb = 0; kb < g.KT; ++kb) {
                const int b = (int)(d & 1);
                const bool first = (kb % kDrain) == 0, last = (kb % kDrain) == kDrain - 1 || kb == g.KT - 1;
                if (first) mbar_wait(tempty(b), (unsigned)(((d >> 1) & 1) ^ 1));
                mbar_wait(full(s), fph);
                tc_fence_after();
                if (lane == 0) {
                    const unsigned a_hi = sbase + s * kTStage, a_lo = a_hi + kTTile, b_hi = a_hi + 2 * kTTile, b_lo = a_hi + 3 * kTTile;
                    const unsigned dt = tmem + (unsigned)b * kTBN;
#pragma unroll
                    for (int ks = 0; ks < BK / 8; ++ks) {
                        // A, MN-major SWIZZLE_128B_BASE32B: atoms of 32 m x 4 k (512 B); m-groups 4 KB apart (LBO), k-groups of
                        // 4 are 512 B apart (SBO), one K = 8 instruction spans two of them.  B, K-major SWIZZLE_128B.
                        const uint64_t dah = make_desc(a_hi + ks * 1024, 4096, 512, 1), dal = make_desc(a_lo + ks * 1024, 4096, 512, 1);
                        const uint64_t dbh = make_desc(b_hi + ks * 32, 16, 1024), dbl = make_desc(b_lo + ks * 32, 16, 1024);
                        tc_mma_tf32(dt, dal, dbh, idesc, (first && ks == 0) ? 0u : 1u);     // small terms first
                        tc_mma_tf32(dt, dah, dbl, idesc, 1u);
                        tc_mma_tf32(dt, dah, dbh, idesc, 1u);
                    }
                    tc_commit(empty(s));
                    if (last) tc_commit(tfull(b));
                }
                __syncwarp();
                if (last) ++d;
                if (++s == kTStages) { s = 0; fph ^= 1u; }
            }
        }
    } else {
        // ================= drainers + epilogue =================
        const int dw = warp - 2;                          // 0..7
        const int rowq = (warp & 3) * 32 + lane;          // TMEM lanes a warp may read: 32 * (warp % 4) ..
        const int colh = (dw >> 2) * 64;
        constexpr int NC = 64;
        float acc[NC];
        const bool use_c = g.beta != 0.f;
        const float cs = use_c ? g.beta / g.alpha : 0.f;
        int64_t d = 0;
        const int ndrain = (g.KT + kDrain - 1) / kDrain;
        for (int64_t t = t0; t < t1; t += tstep) {
            int64_t tm, tn;
            tile_of(g, t, tm, tn);
            const int64_t m = tm * BM + rowq, n0 = tn * kTBN + colh;
            float* Cp = g.C + m + n0 * g.ldc;
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[c] = (use_c && m < g.M && n0 + c < g.N) ? __ldcs(Cp + c * g.ldc) : 0.f;
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[c] *= cs;
            for (int q = 0; q < ndrain; ++q, ++d) {
                const int b = (int)(d & 1);
                mbar_wait(tfull(b), (unsigned)((d >> 1) & 1));
                tc_fence_after();
                const unsigned taddr = tmem + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)(b * kTBN + colh);
#pragma unroll
                for (int c0 = 0; c0 < NC; c0 += 32) {
                    float v[32];
                    tmem_ld32(taddr + c0, v);
#pragma unroll
                    for (int c = 0; c < 32; ++c) acc[c0 + c] += v[c];
                }
                tc_fence_before();
                mbar_arrive(tempty(b));
            }
            if (m < g.M) {
#pragma unroll
                for (int c = 0; c < NC; ++c)
                    if (n0 + c < g.N) __stcs(Cp + c * g.ldc, g.alpha * acc[c]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(256u) : "memory");
}

}  // namespace umma

// ---- host side (declared in kernels.h) -------------------------------------------------------------
inline cudaError_t split_tf32_launch_impl(const float* src, int64_t ld, int64_t rows, int64_t cols, float* hi, float* lo,
                                          int64_t ld_out, cudaStream_t st) {
    if (rows <= 0 || cols <= 0) return cudaSuccess;
    dim3 grid((unsigned)ceil_div(ld_out, 4 * 256), (unsigned)std::min<int64_t>(cols, 65535));
    umma::split_tf32_kernel<<<grid, 256, 0, st>>>(src, ld, rows, cols, hi, lo, ld_out);
    return cudaGetLastError();
}

// C <- alpha (Ahi + Alo)(Bhi + Blo) + beta C on `ctas` CTAs (one per SM).  Ahi / Alo: M x K, m-contiguous, leading dimension
// lda (multiple of 4, 16-byte aligned base); Bhi / Blo: K x N, k-contiguous, leading dimension ldb (same constraints).
inline cudaError_t upd_presplit_launch_impl(int64_t M, int64_t N, int64_t K, float alpha, const float* Ahi, const float* Alo,
                                            int64_t lda, const float* Bhi, const float* Blo, int64_t ldb, float beta, float* C,
                                            int64_t ldc, int ctas, cudaStream_t st) {
    if (M <= 0 || N <= 0) return cudaSuccess;
    if (K <= 0 || alpha == 0.f || lda % 4 || ldb % 4 || ((uintptr_t)Ahi | (uintptr_t)Alo | (uintptr_t)Bhi | (uintptr_t)Blo) % 16)
        return cudaErrorInvalidValue;
    CUtensorMap mAh, mAl, mBh, mBl;
    cudaError_t e;
    if ((e = tma::map_2d(&mAh, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Ahi, M, K, lda, 32, 32, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B)) != cudaSuccess) return e;
    if ((e = tma::map_2d(&mAl, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Alo, M, K, lda, 32, 32, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B)) != cudaSuccess) return e;
    if ((e = tma::map_2d(&mBh, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Bhi, K, N, ldb, 32, 128, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    if ((e = tma::map_2d(&mBl, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Blo, K, N, ldb, 32, 128, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    umma::UpdTmaArgs g{};
    g.M = M; g.N = N; g.K = K; g.C = C; g.ldc = ldc; g.alpha = alpha; g.beta = beta;
    g.tilesM = ceil_div(M, umma::BM); g.tilesN = ceil_div(N, umma::kTBN);
    g.KT = (int)ceil_div(K, umma::BK);
    const int64_t tiles = g.tilesM * g.tilesN;
    g.Gm = (int)std::min<int64_t>(16, g.tilesM);
    const int grid = (int)std::min<int64_t>(tiles, std::max(1, ctas));
    static SmemAttr attr;
    if ((e = ensure_dyn_smem(umma::upd_tma_kernel, umma::kTSmem, attr)) != cudaSuccess) return e;
    umma::upd_tma_kernel<<<grid, umma::kTThreads, umma::kTSmem, st>>>(mAh, mAl, mBh, mBl, g);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------------
// W = A^T B as stream-K partial tiles (W = V^T C of larfb) with the small operand A = V pre-split and TMA-fed; the streamed
// operand B = C is read once per launch, so it is still split on the fly by the worker warps -- half the producer work of
// gemm_umma_kernel<true, 128> -- and the TMEM accumulator is drained once per kDrain k-blocks instead of every k-block.
// Same unit sequence, partial-tile slots and consumers (partial_sum / mm128 / T^T W) as gemm_umma.cuh.
//   warps 0-7  workers: C chunks global -> registers (one k-block ahead) -> hi / lo -> B_hi, B_lo of the stage; drain; epilogue
//   warp 8     TMA producer of A_hi, A_lo (K-major boxes of 32 k x 128 m, SWIZZLE_128B)
//   warp 9     MMA issuer (owns the TMEM allocation)
// ---------------------------------------------------------------------------------------------------------------------
namespace umma {

constexpr int kVWorkers = 256, kVThreads = kVWorkers + 64;

__global__ void __launch_bounds__(kVThreads, 1)
vtc_tma_kernel(const __grid_constant__ CUtensorMap mAh, const __grid_constant__ CUtensorMap mAl, GemmArgs<float> g, StreamK sk) {
    constexpr int BN = 128, NC = BN / 2, PBN = BN * 8 / kVWorkers;
    extern __shared__ unsigned char smem_raw[];
    const unsigned sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const unsigned bars = sbase + kTStages * kTStage;           // fullA[S], fullB[S], empty[S], tfull[2], tempty[2]
    auto fullA = [&](int s) { return bars + 8u * s; };
    auto fullB = [&](int s) { return bars + 8u * (kTStages + s); };
    auto empty = [&](int s) { return bars + 8u * (2 * kTStages + s); };
    auto tfull = [&](int b) { return bars + 8u * (3 * kTStages + b); };
    auto tempty = [&](int b) { return bars + 8u * (3 * kTStages + 2 + b); };
    unsigned* tmem_slot = reinterpret_cast<unsigned*>(sgen + kTStages * kTStage + 8 * (3 * kTStages + 4));
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t u0 = (int64_t)blockIdx.x * sk.L, u1 = min(sk.U, u0 + sk.L), nunits = u1 - u0;
    // An accumulator generation = up to kDrain consecutive units of one tile segment: it closes with its kDrain-th unit, with
    // the last k-block of the tile, or with the CTA's last unit.  Both the MMA issuer and the workers follow that rule with
    // incremental counters (no division on the per-k-block path).
    const int kt0 = (int)(u0 % sk.KT);
    if (tid == 0) {
        for (int s = 0; s < kTStages; ++s) { mbar_init(fullA(s), 1); mbar_init(fullB(s), kVWorkers); mbar_init(empty(s), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull(b), 1); mbar_init(tempty(b), kVWorkers); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        tma::prefetch_map(&mAh); tma::prefetch_map(&mAl);
    }
    if (warp == 9) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)), "r"(256u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = *tmem_slot;

    if (warp == 8) {
        // ================= TMA producer of A = V (M <= 128 columns of V, zero-filled beyond) =================
        if (lane == 0) {
            int s = 0; unsigned ph = 1;
            int kt = kt0;
            for (int64_t j = 0; j < nunits; ++j, kt = (kt + 1 == sk.KT) ? 0 : kt + 1) {
                mbar_wait(empty(s), ph);
                tma::mbar_expect_tx(fullA(s), 2u * kTTile);
                tma::load_2d(sbase + s * kTStage, &mAh, kt * BK, 0, fullA(s));
                tma::load_2d(sbase + s * kTStage + kTTile, &mAl, kt * BK, 0, fullA(s));
                if (++s == kTStages) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == 9) {
        // ================= MMA issuer =================
        const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(BN >> 3) << 17) | ((unsigned)(BM >> 4) << 24);
        int s = 0; unsigned fph = 0;
        int64_t d = 0;
        int kt = kt0, run = 0;
        for (int64_t j = 0; j < nunits; ++j) {
            const int b = (int)(d & 1);
            const bool first = run == 0, last = kt == sk.KT - 1 || j == nunits - 1 || run == kDrain - 1;
            run = last ? 0 : run + 1;
            kt = (kt + 1 == sk.KT) ? 0 : kt + 1;
            if (first) mbar_wait(tempty(b), (unsigned)(((d >> 1) & 1) ^ 1));
            mbar_wait(fullA(s), fph);
            mbar_wait(fullB(s), fph);
            tc_fence_after();
            if (lane == 0) {
                const unsigned a_hi = sbase + s * kTStage, a_lo = a_hi + kTTile, b_hi = a_hi + 2 * kTTile, b_lo = a_hi + 3 * kTTile;
                const unsigned dt = tmem + (unsigned)b * BN;
#pragma unroll
                for (int ks = 0; ks < BK / 8; ++ks) {
                    const uint64_t dah = make_desc(a_hi + ks * 32, 16, 1024), dal = make_desc(a_lo + ks * 32, 16, 1024);
                    const uint64_t dbh = make_desc(b_hi + ks * 32, 16, 1024), dbl = make_desc(b_lo + ks * 32, 16, 1024);
                    tc_mma_tf32(dt, dal, dbh, idesc, (first && ks == 0) ? 0u : 1u);
                    tc_mma_tf32(dt, dah, dbl, idesc, 1u);
                    tc_mma_tf32(dt, dah, dbh, idesc, 1u);
                }
                tc_commit(empty(s));
                if (last) tc_commit(tfull(b));
            }
            __syncwarp();
            if (last) ++d;
            if (++s == kTStages) { s = 0; fph ^= 1u; }
        }
    } else {
        // ================= workers: B = C producer + accumulator drain + partial-tile epilogue =================
        const int rowq = (warp & 3) * 32 + lane;          // TMEM lane = output row (a column of V)
        const int colh = (warp >> 2) * NC;
        float acc[NC];
        float4 rb[PBN];
        int64_t pt = u0 / sk.KT; int pkt = (int)(u0 - pt * sk.KT);
        auto load_regs = [&]() {
            const int64_t n0 = pt * BN, k0 = (int64_t)pkt * BK;     // tilesM == 1 in partial mode: tile index = column block
#pragma unroll
            for (int p = 0; p < PBN; ++p) {
                const int c = tid + p * kVWorkers;
                const int r = c >> 3, kc = (c & 7) * 4;
                rb[p] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (n0 + r < g.N && k0 + kc < g.K) rb[p] = __ldg(reinterpret_cast<const float4*>(g.B + (n0 + r) * g.ldb + k0 + kc));
            }
            if (++pkt == sk.KT) { pkt = 0; ++pt; }
        };
        auto store_stage = [&](int s) {
            unsigned char* st = sgen + (size_t)s * kTStage + 2 * kTTile;
#pragma unroll
            for (int p = 0; p < PBN; ++p) {
                const int c = tid + p * kVWorkers;
                const int r = c >> 3, kc = c & 7;
                const unsigned off = (r >> 3) * 1024 + (r & 7) * 128 + ((kc ^ (r & 7)) << 4);
                uint4 hi, lo;
                split4(rb[p], hi, lo);
                *reinterpret_cast<uint4*>(st + off) = hi;
                *reinterpret_cast<uint4*>(st + kTTile + off) = lo;
            }
        };
        int64_t ct = u0 / sk.KT;
        int64_t pi = 0, ci = 0, d = 0;                    // produced units, units whose accumulator has been drained, generations
        int ckt = kt0;                                    // k-block index (inside its tile) of unit ci
        int ps = 0; unsigned pph = 1;
        bool fresh = true;
        load_regs();
        while (ci < nunits) {
            if (pi < nunits) {
                mbar_wait(empty(ps), pph);
                store_stage(ps);
                fence_proxy_async();
                mbar_arrive(fullB(ps));
                if (++ps == kTStages) { ps = 0; pph ^= 1u; }
                ++pi;
                if (pi < nunits) load_regs();
            }
            // drain every generation that closed at least kTStages - 1 units behind the producer (or everything at the end)
            for (;;) {
                // the unit that closes the generation starting at ci
                const int64_t ce = ci + min((int64_t)min(kDrain - 1, sk.KT - 1 - ckt), nunits - 1 - ci);
                if (!(ce + (kTStages - 1) <= pi || pi == nunits)) break;
                if (fresh) {
#pragma unroll
                    for (int c = 0; c < NC; ++c) acc[c] = 0.f;
                    fresh = false;
                }
                const int b = (int)(d & 1);
                mbar_wait(tfull(b), (unsigned)((d >> 1) & 1));
                tc_fence_after();
                const unsigned taddr = tmem + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)(b * BN + colh);
#pragma unroll
                for (int c0 = 0; c0 < NC; c0 += 32) {
                    float v[32];
                    tmem_ld32(taddr + c0, v);
#pragma unroll
                    for (int c = 0; c < 32; ++c) acc[c0 + c] += v[c];
                }
                tc_fence_before();
                mbar_arrive(tempty(b));
                ++d;
                const int kte = ckt + (int)(ce - ci);     // k-block index of the closing unit
                ci = ce + 1;
                ckt = (kte + 1 == sk.KT) ? 0 : kte + 1;
                if (kte == sk.KT - 1 || ci == nunits) {
                    // segment of tile ct ends: compact partial tile (see gemm_mma.cuh)
                    float* Pt = g.C + (ct + (int64_t)blockIdx.x) * (int64_t)(BM * BN) + rowq + (int64_t)colh * BM;
#pragma unroll
                    for (int c = 0; c < NC; ++c) Pt[c * BM] = g.alpha * acc[c];
                    ++ct; fresh = true;
                }
                if (ci >= nunits) break;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 9)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(256u) : "memory");
}

}  // namespace umma

// stream-K partial tiles of A^T B with A = Ahi + Alo pre-split (K x M, k-contiguous, M <= 128, lda multiple of 4, 16-byte
// aligned) and B fp32 (K x N, k-contiguous, 16-byte aligned rows).  p: the umma_plan of (M, N, K) in partial mode.
inline cudaError_t vtc_presplit_launch_impl(GemmArgs<float> g, const float* Ahi, const float* Alo, int64_t lda, const MmaPlan& p, cudaStream_t st) {
    if (g.M <= 0 || g.N <= 0) return cudaSuccess;
    if (g.M > 128 || !p.sk.partial || p.sk.tilesM != 1 || lda % 4 || ((uintptr_t)Ahi | (uintptr_t)Alo) % 16) return cudaErrorInvalidValue;
    CUtensorMap mAh, mAl;
    cudaError_t e;
    if ((e = tma::map_2d(&mAh, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Ahi, g.K, g.M, lda, 32, 128, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    if ((e = tma::map_2d(&mAl, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Alo, g.K, g.M, lda, 32, 128, CU_TENSOR_MAP_SWIZZLE_128B)) != cudaSuccess) return e;
    static SmemAttr attr;
    if ((e = ensure_dyn_smem(umma::vtc_tma_kernel, umma::kTSmem, attr)) != cudaSuccess) return e;
    umma::vtc_tma_kernel<<<p.grid, umma::kVThreads, umma::kTSmem, st>>>(mAh, mAl, g, p.sk);
    return cudaGetLastError();
}

}  // namespace ctqr
