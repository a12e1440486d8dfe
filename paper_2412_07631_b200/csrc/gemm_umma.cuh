// gemm_umma.cuh -- fp32 contraction on the 5th-generation tensor cores (tcgen05.mma kind::tf32,
// accumulators in TMEM) as a 3xTF32 split: the Blackwell-native version of gemm_mma.cuh's float
// policy, for the two big larfb products (W = V^T C and C <- C - V W).
//
//   C <- alpha * op(A) * B + beta * C,  column-major fp32, op(A) = A^T (A is K x M, "TA") or A (M x K).
//
// Structure (one CTA per SM, 128 x BN output tile -- BN = 128 for W = V^T C, 64 for C <- C - V W so
// that the C tile fits in registers until the epilogue -- k-blocks of 32):
//   * warps 0-7 ("workers", 256 threads) load fp32 operand chunks global -> registers (one k-block
//     ahead), split every value into hi + lo on the TF32 grid and store the four tiles A_hi, A_lo,
//     B_hi, B_lo into shared memory in the UMMA canonical 128-byte-swizzled layouts (K-major for
//     k-contiguous operands, MN-major for the m-contiguous V of C <- C - V W: no transposes);
//   * warp 8 issues, per k-block, 4 k-steps x 3 products (lo*hi, hi*lo, hi*hi) of
//     tcgen05.mma.cta_group::1.kind::tf32 (M = 128, N = BN, K = 8) into one of two BN-column TMEM
//     accumulators, the first with accumulate = 0, and commits to mbarriers;
//   * the workers drain that TMEM accumulator (tcgen05.ld 32x32b, thread = row) and add it to the
//     running sum in registers with round-to-nearest FADDs.  The tensor core's own accumulation
//     truncates (gemm_mma.cuh measured an error growing linearly with K), so it is only trusted
//     with one k-block (12 MMAs) at a time.
//   * same flat stream-K unit sequence, compact partial tiles and epilogues as gemm_mma.cuh.
// Pipelines: full/empty mbarriers per shared-memory stage (workers <-> MMA), tfull/tempty per
// TMEM accumulator (MMA <-> workers).  Generic-proxy stores are made visible to the tensor core
// with fence.proxy.async before the arrive.
#pragma once
#include <algorithm>
#include "common.cuh"
#include "kernels.h"
#include "gemm_mma.cuh"

namespace ctqr {
namespace umma {

constexpr int BM = 128, BK = 32, STAGES = 3;   // BN: 128 for W = V^T C, 64 for C <- C - V W (template)
constexpr int WORKERS = 256, NT = WORKERS + 32;
constexpr int TILE_BYTES = 128 * BK * 4;                 // one operand tile: 16 KB
constexpr int STAGE_BYTES = 4 * TILE_BYTES;              // A_hi, A_lo, B_hi, B_lo (B tiles sized for BN = 128)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra D;\n\tbra W;\n\tD:\n\t}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_commit(unsigned bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc], kind::tf32, single-thread issue
__device__ __forceinline__ void tc_mma_tf32(unsigned d_tmem, uint64_t adesc, uint64_t bdesc, unsigned idesc, unsigned accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}\n" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(0u)
        : "memory");
}
// shared-memory matrix descriptor (cute::UMMA::SmemDescriptor): start>>4 [0,14), LBO>>4 [16,30),
// SBO>>4 [32,46), version = 1 [46,48), layout SWIZZLE_128B = 2 [61,64)
// layout: 2 = SWIZZLE_128B (K-major tiles), 1 = SWIZZLE_128B_BASE32B (the only layout for MN-major
// 32-bit operands: 128-byte rows along M, 4 rows along K per atom, 32-byte units XORed with row & 3)
__device__ __forceinline__ uint64_t make_desc(unsigned saddr, unsigned lbo_bytes, unsigned sbo_bytes, unsigned layout = 2) {
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46) | ((uint64_t)layout << 61);
}
// 32 consecutive TMEM columns of this thread's lane -> registers
__device__ __forceinline__ void tmem_ld32(unsigned taddr, float (&v)[32]) {
    unsigned r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}


// fp32 vector of 4 -> hi / lo TF32 bit patterns
__device__ __forceinline__ void split4(const float4& x, uint4& hi, uint4& lo) {
    split_tf32(x.x, hi.x, lo.x); split_tf32(x.y, hi.y, lo.y);
    split_tf32(x.z, hi.z, lo.z); split_tf32(x.w, hi.w, lo.w);
}

template <bool TA, int BN>
__global__ void __launch_bounds__(NT, 1) gemm_umma_kernel(GemmArgs<float> g, StreamK sk) {
    constexpr int NC = BN / 2;                 // output columns per worker thread
    constexpr int PBN = BN * 8 / WORKERS;      // B chunks per thread per k-block
    constexpr bool DEFER = (BN == 64);         // registers allow holding the C tile until the epilogue
    extern __shared__ unsigned char smem_raw[];
    const unsigned sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;          // SWIZZLE_128B atoms need 1 KB alignment
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const unsigned bars = sbase + STAGES * STAGE_BYTES;                   // full[S], empty[S], tfull[2], tempty[2]
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (STAGES + s); };
    auto tfull = [&](int b) { return bars + 8u * (2 * STAGES + b); };
    auto tempty = [&](int b) { return bars + 8u * (2 * STAGES + 2 + b); };
    unsigned* tmem_slot = reinterpret_cast<unsigned*>(sgen + STAGES * STAGE_BYTES + 8 * (2 * STAGES + 4));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t u0 = (int64_t)blockIdx.x * sk.L;
    const int64_t u1 = min(sk.U, u0 + sk.L);
    const int64_t nunits = u1 - u0;                                       // > 0 for every launched CTA

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), WORKERS); mbar_init(empty(s), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull(b), 1); mbar_init(tempty(b), WORKERS); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 8) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)), "r"(256u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = *tmem_slot;

    if (warp == 8) {
        // ================= MMA issuer =================
        // instruction descriptor (cute::UMMA::InstrDescriptor): D = F32, A = B = TF32, A major, N >> 3, M >> 4
        const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((TA ? 0u : 1u) << 15) | ((unsigned)(BN >> 3) << 17) |
                               ((unsigned)(BM >> 4) << 24);
        int s = 0; unsigned fph = 0;
        for (int64_t j = 0; j < nunits; ++j) {
            const int b = (int)(j & 1);
            mbar_wait(tempty(b), (unsigned)(((j >> 1) & 1) ^ 1));
            mbar_wait(full(s), fph);
            tc_fence_after();
            if (lane == 0) {
                const unsigned a_hi = sbase + s * STAGE_BYTES, a_lo = a_hi + TILE_BYTES;
                const unsigned b_hi = a_hi + 2 * TILE_BYTES, b_lo = a_hi + 3 * TILE_BYTES;
                const unsigned d = tmem + (unsigned)b * BN;
#pragma unroll
                for (int ks = 0; ks < BK / 8; ++ks) {
                    // K-major tile: 8-row groups 1 KB apart, k-step = 32 bytes inside the swizzled row.
                    // MN-major A (SWIZZLE_128B_BASE32B): atoms of 32 m x 4 k = 512 B; m-groups 512 B apart
                    // (LBO), k-groups of 4 are 2 KB apart (SBO); one K = 8 instruction spans two k-groups.
                    const unsigned aoff = TA ? ks * 32 : ks * 4096;
                    const uint64_t dah = TA ? make_desc(a_hi + aoff, 16, 1024) : make_desc(a_hi + aoff, 512, 2048, 1);
                    const uint64_t dal = TA ? make_desc(a_lo + aoff, 16, 1024) : make_desc(a_lo + aoff, 512, 2048, 1);
                    const uint64_t dbh = make_desc(b_hi + ks * 32, 16, 1024);
                    const uint64_t dbl = make_desc(b_lo + ks * 32, 16, 1024);
                    tc_mma_tf32(d, dal, dbh, idesc, ks > 0 ? 1u : 0u);     // small terms first
                    tc_mma_tf32(d, dah, dbl, idesc, 1u);
                    tc_mma_tf32(d, dah, dbh, idesc, 1u);
                }
                tc_commit(empty(s));       // shared-memory stage may be refilled once these MMAs have read it
                tc_commit(tfull(b));       // accumulator b is complete
            }
            __syncwarp();
            if (++s == STAGES) { s = 0; fph ^= 1u; }
        }
    } else {
        // ================= workers: producer + accumulator drain + epilogue =================
        const int rowq = (warp & 3) * 32 + lane;         // TMEM lane = output row inside the tile
        const int colh = (warp >> 2) * NC;               // this thread's NC output columns
        float acc[NC], cin[DEFER ? NC : 1];
        float4 ra[4], rb[PBN];                             // one k-block of operand chunks, in flight
        // ---- producer state ----
        int64_t pt = u0 / sk.KT; int pkt = (int)(u0 - pt * sk.KT);
        int64_t ptn = pt / sk.tilesM, ptm = pt - ptn * sk.tilesM;     // advanced incrementally (no division per k-block)
        auto load_regs = [&]() {
            const int64_t m0 = ptm * BM, n0 = ptn * BN, k0 = (int64_t)pkt * BK;
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int c = tid + p * WORKERS;
                ra[p] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (TA) {
                    const int r = c >> 3, kc = (c & 7) * 4;
                    if (m0 + r < g.M && k0 + kc < g.K)
                        ra[p] = __ldg(reinterpret_cast<const float4*>(g.A + (m0 + r) * g.lda + k0 + kc));
                } else {
                    const int kk = c >> 5, mc = (c & 31) * 4;
                    if (k0 + kk < g.K && m0 + mc < g.M)
                        ra[p] = __ldg(reinterpret_cast<const float4*>(g.A + (m0 + mc) + (k0 + kk) * g.lda));
                }
                if (p < PBN) {
                    const int r = c >> 3, kc = (c & 7) * 4;
                    rb[p < PBN ? p : 0] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (n0 + r < g.N && k0 + kc < g.K)
                        rb[p < PBN ? p : 0] = __ldg(reinterpret_cast<const float4*>(g.B + (n0 + r) * g.ldb + k0 + kc));
                }
            }
            if (++pkt == sk.KT) { pkt = 0; if (++ptm == sk.tilesM) { ptm = 0; ++ptn; } }
        };
        auto store_stage = [&](int s) {
            unsigned char* st = sgen + (size_t)s * STAGE_BYTES;
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int c = tid + p * WORKERS;
                uint4 hi, lo;
                unsigned off;
                if (TA) { const int r = c >> 3, kc = c & 7; off = (r >> 3) * 1024 + (r & 7) * 128 + ((kc ^ (r & 7)) << 4); }
                else    { const int kk = c >> 5, mc = c & 31, x = mc & 7;
                          off = (kk >> 2) * 2048 + (mc >> 3) * 512 + (kk & 3) * 128 + ((((x >> 1) ^ (kk & 3)) << 5) | ((x & 1) << 4)); }
                split4(ra[p], hi, lo);
                *reinterpret_cast<uint4*>(st + off) = hi;
                *reinterpret_cast<uint4*>(st + TILE_BYTES + off) = lo;
                if (p < PBN) {
                    const int r = c >> 3, kc = c & 7;
                    off = (r >> 3) * 1024 + (r & 7) * 128 + ((kc ^ (r & 7)) << 4);
                    split4(rb[p < PBN ? p : 0], hi, lo);
                    *reinterpret_cast<uint4*>(st + 2 * TILE_BYTES + off) = hi;
                    *reinterpret_cast<uint4*>(st + 3 * TILE_BYTES + off) = lo;
                }
            }
        };
        // ---- consumer state ----
        int64_t ct = u0 / sk.KT; int ckt = (int)(u0 - ct * sk.KT);
        int64_t ctn = ct / sk.tilesM, ctm = ct - ctn * sk.tilesM;
        bool fresh = true;                                // next drain starts a tile segment
        const float cscale = (sk.partial || g.beta == 0.f) ? 0.f : (DEFER ? 1.f : g.beta / g.alpha);

        int64_t pi = 0, ci = 0;
        int ps = 0; unsigned pph = 1;
        load_regs();
        while (ci < nunits) {
            if (pi < nunits) {
                mbar_wait(empty(ps), pph);
                store_stage(ps);
                fence_proxy_async();
                mbar_arrive(full(ps));
                if (++ps == STAGES) { ps = 0; pph ^= 1u; }
                ++pi;
                if (pi < nunits) load_regs();
            }
            if (pi - ci >= STAGES - 1 || pi == nunits) {
                const int b = (int)(ci & 1);
                const int64_t m0 = ctm * BM, n0 = ctn * BN;
                if (fresh) {
                    // direct mode: DEFER requests the C tile now and uses it only in the epilogue, so
                    // its memory latency hides behind this tile's drains (C <- C - V W has just 4
                    // k-blocks per tile); otherwise the running sum starts at (beta/alpha) * C
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        const int64_t m = m0 + rowq, n = n0 + colh + c;
                        float cv = 0.f;
                        if (cscale != 0.f && m < g.M && n < g.N) cv = __ldcs(&g.C[m + n * g.ldc]);
                        if (DEFER) { cin[c] = cv; acc[c] = 0.f; } else acc[c] = cscale * cv;
                    }
                    fresh = false;
                }
                mbar_wait(tfull(b), (unsigned)((ci >> 1) & 1));
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
                ++ci;
                if (++ckt == sk.KT || ci == nunits) {
                    // ---- epilogue of this tile segment ----
                    if (sk.partial) {
                        float* Pt = g.C + (ct + (int64_t)blockIdx.x) * (int64_t)(BM * BN) + rowq + (int64_t)colh * BM;
#pragma unroll
                        for (int c = 0; c < NC; ++c) Pt[c * BM] = g.alpha * acc[c];
                    } else {
#pragma unroll
                        for (int c = 0; c < NC; ++c) {
                            const int64_t m = m0 + rowq, n = n0 + colh + c;
                            if (m < g.M && n < g.N)
                                __stcs(&g.C[m + n * g.ldc], DEFER ? fmaf(g.alpha, acc[c], g.beta * cin[c < (DEFER ? NC : 1) ? c : 0]) : g.alpha * acc[c]);
                        }
                    }
                    ckt = 0; ++ct; fresh = true;
                    if (++ctm == sk.tilesM) { ctm = 0; ++ctn; }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(256u) : "memory");
}

// -------------------------------------------------------------------------------------------
// Fully warp-specialised variant (used for C <- C - V W, BN = 64): the combined worker of the
// kernel above stalls once per k-block on its own global loads (prefetch distance = one drain),
// which with only 4 k-blocks per tile left the tensor core idle most of the time.  Here
//   warps 0-3   producers: global -> registers TWO k-blocks ahead, split, store UMMA tiles
//   warps 4-11  drainers:  TMEM -> registers, running sum, C tile requested at tile start and
//                          consumed in the epilogue
//   warp 12     MMA issuer
// so global-load latency, tensor-core latency and C latency overlap instead of adding up.
// -------------------------------------------------------------------------------------------
constexpr int WS_PROD = 128, WS_DRAIN = 256, WS_NT = WS_PROD + WS_DRAIN + 32;
// memory-level parallelism: the operands of a k-block are fetched with cp.async into a staging ring
// WS_DEPTH k-blocks ahead (registers held only 2 k-blocks = 48 KB per SM in flight, which at ~1.5 us
// of loaded memory latency capped a tile at ~3 us; the tensor core needs < 1 us)
constexpr int WS_USTAGES = 2;
__host__ __device__ constexpr int ws_nstg(int bn) { return bn == 64 ? 5 : 3; }   // staging stages that fit beside the two UMMA stages
template <int BN> struct WsSmem {
    static constexpr int B_TILE = BN * BK * 4;
    static constexpr int USTAGE = 2 * TILE_BYTES + 2 * B_TILE;                 // A_hi, A_lo, B_hi, B_lo
    static constexpr int CHUNKS = (1024 + BN * 8) / WS_PROD;                   // 16-byte chunks per producer thread per k-block
    static constexpr int STG = CHUNKS * WS_PROD * 16;                          // one staging stage
    static constexpr int NSTG = ws_nstg(BN);
    static constexpr int BAR_OFF = WS_USTAGES * USTAGE + NSTG * STG;
    static constexpr int BYTES = BAR_OFF + 256 + 1024;
};

template <bool TA, int BN>
__global__ void __launch_bounds__(WS_NT, 1) gemm_umma_ws_kernel(GemmArgs<float> g, StreamK sk) {
    constexpr int NC = BN / 2;                 // output columns per drainer thread
    constexpr int PA = 1024 / WS_PROD;         // A chunks (float4) per producer thread per k-block
    constexpr int PB = BN * 8 / WS_PROD;       // B chunks
    constexpr int WS_NSTG = WsSmem<BN>::NSTG, WS_DEPTH = WS_NSTG - 1;
    constexpr bool DEFER = (BN == 64);         // drainer registers allow holding the C tile until the epilogue
    extern __shared__ unsigned char smem_raw[];
    const unsigned sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    using SM = WsSmem<BN>;
    constexpr int STAGES = WS_USTAGES;
    constexpr int STAGE_BYTES = SM::USTAGE;
    constexpr int B_TILE = SM::B_TILE;
    const unsigned bars = sbase + SM::BAR_OFF;
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (STAGES + s); };
    auto tfull = [&](int b) { return bars + 8u * (2 * STAGES + b); };
    auto tempty = [&](int b) { return bars + 8u * (2 * STAGES + 2 + b); };
    unsigned* tmem_slot = reinterpret_cast<unsigned*>(sgen + SM::BAR_OFF + 8 * (2 * STAGES + 4));
    unsigned char* stg = sgen + WS_USTAGES * SM::USTAGE;                       // staging ring

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int MMA_WARP = (WS_PROD + WS_DRAIN) / 32;
    const int64_t u0 = (int64_t)blockIdx.x * sk.L;
    const int64_t u1 = min(sk.U, u0 + sk.L);
    const int64_t nunits = u1 - u0;

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), WS_PROD); mbar_init(empty(s), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull(b), 1); mbar_init(tempty(b), WS_DRAIN); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == MMA_WARP) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)), "r"(256u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = *tmem_slot;

    if (warp == MMA_WARP) {
        const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((TA ? 0u : 1u) << 15) | ((unsigned)(BN >> 3) << 17) |
                               ((unsigned)(BM >> 4) << 24);
        int s = 0; unsigned fph = 0;
        for (int64_t j = 0; j < nunits; ++j) {
            const int b = (int)(j & 1);
            mbar_wait(tempty(b), (unsigned)(((j >> 1) & 1) ^ 1));
            mbar_wait(full(s), fph);
            tc_fence_after();
            if (lane == 0) {
                const unsigned a_hi = sbase + s * STAGE_BYTES, a_lo = a_hi + TILE_BYTES;
                const unsigned b_hi = a_hi + 2 * TILE_BYTES, b_lo = b_hi + B_TILE;
                const unsigned d = tmem + (unsigned)b * BN;
#pragma unroll
                for (int ks = 0; ks < BK / 8; ++ks) {
                    const unsigned aoff = TA ? ks * 32 : ks * 4096;
                    const uint64_t dah = TA ? make_desc(a_hi + aoff, 16, 1024) : make_desc(a_hi + aoff, 512, 2048, 1);
                    const uint64_t dal = TA ? make_desc(a_lo + aoff, 16, 1024) : make_desc(a_lo + aoff, 512, 2048, 1);
                    const uint64_t dbh = make_desc(b_hi + ks * 32, 16, 1024);
                    const uint64_t dbl = make_desc(b_lo + ks * 32, 16, 1024);
                    tc_mma_tf32(d, dal, dbh, idesc, ks > 0 ? 1u : 0u);
                    tc_mma_tf32(d, dah, dbl, idesc, 1u);
                    tc_mma_tf32(d, dah, dbh, idesc, 1u);
                }
                tc_commit(empty(s));
                tc_commit(tfull(b));
            }
            __syncwarp();
            if (++s == STAGES) { s = 0; fph ^= 1u; }
        }
    } else if (warp < WS_PROD / 32) {
        // ================= producers =================
        // tile coordinates advance incrementally: no 64-bit division on the per-k-block path
        int64_t pt = u0 / sk.KT; int pkt = (int)(u0 - pt * sk.KT);
        int64_t ptn = pt / sk.tilesM, ptm = pt - ptn * sk.tilesM;
        // cp.async of k-block (pt, pkt) into staging stage q: chunk p of this thread sits at
        // (p * WS_PROD + tid) * 16 -- every thread later reads back exactly the chunks it copied, so
        // cp.async.wait_group is the only synchronisation the staging ring needs
        auto issue_copy = [&](int q) {
            const int64_t m0 = ptm * BM, n0 = ptn * BN, k0 = (int64_t)pkt * BK;
            unsigned char* dst = stg + (size_t)q * SM::STG + tid * 16;
#pragma unroll
            for (int p = 0; p < PA; ++p) {
                const int c = tid + p * WS_PROD;
                const float* src = g.A; int bytes = 0;
                if (TA) {
                    const int r = c >> 3, kc = (c & 7) * 4;
                    if (m0 + r < g.M && k0 + kc < g.K) { src = g.A + (m0 + r) * g.lda + k0 + kc; bytes = 16; }
                } else {
                    const int kk = c >> 5, mc = (c & 31) * 4;
                    if (k0 + kk < g.K && m0 + mc < g.M) { src = g.A + (m0 + mc) + (k0 + kk) * g.lda; bytes = 16; }
                }
                cp_async16(dst + p * WS_PROD * 16, src, bytes);
            }
#pragma unroll
            for (int p = 0; p < PB; ++p) {
                const int c = tid + p * WS_PROD;
                const int r = c >> 3, kc = (c & 7) * 4;
                const float* src = g.B; int bytes = 0;
                if (n0 + r < g.N && k0 + kc < g.K) { src = g.B + (n0 + r) * g.ldb + k0 + kc; bytes = 16; }
                cp_async16(dst + (PA + p) * WS_PROD * 16, src, bytes);
            }
            if (++pkt == sk.KT) { pkt = 0; if (++ptm == sk.tilesM) { ptm = 0; ++ptn; } }
        };
        auto read_stage = [&](int q, float4 (&ra)[PA], float4 (&rb)[PB]) {
            const unsigned char* srcp = stg + (size_t)q * SM::STG + tid * 16;
#pragma unroll
            for (int p = 0; p < PA; ++p) ra[p] = *reinterpret_cast<const float4*>(srcp + p * WS_PROD * 16);
#pragma unroll
            for (int p = 0; p < PB; ++p) rb[p] = *reinterpret_cast<const float4*>(srcp + (PA + p) * WS_PROD * 16);
        };
        auto store_stage = [&](int s, const float4 (&ra)[PA], const float4 (&rb)[PB]) {
            unsigned char* st = sgen + (size_t)s * STAGE_BYTES;
            uint4 hi, lo;
#pragma unroll
            for (int p = 0; p < PA; ++p) {
                const int c = tid + p * WS_PROD;
                unsigned off;
                if (TA) { const int r = c >> 3, kc = c & 7; off = (r >> 3) * 1024 + (r & 7) * 128 + ((kc ^ (r & 7)) << 4); }
                else    { const int kk = c >> 5, mc = c & 31, x = mc & 7;
                          off = (kk >> 2) * 2048 + (mc >> 3) * 512 + (kk & 3) * 128 + ((((x >> 1) ^ (kk & 3)) << 5) | ((x & 1) << 4)); }
                split4(ra[p], hi, lo);
                *reinterpret_cast<uint4*>(st + off) = hi;
                *reinterpret_cast<uint4*>(st + TILE_BYTES + off) = lo;
            }
#pragma unroll
            for (int p = 0; p < PB; ++p) {
                const int c = tid + p * WS_PROD;
                const int r = c >> 3, kc = c & 7;
                const unsigned off = (r >> 3) * 1024 + (r & 7) * 128 + ((kc ^ (r & 7)) << 4);
                split4(rb[p], hi, lo);
                *reinterpret_cast<uint4*>(st + 2 * TILE_BYTES + off) = hi;
                *reinterpret_cast<uint4*>(st + 2 * TILE_BYTES + B_TILE + off) = lo;
            }
        };
        int ps = 0; unsigned pph = 1;                       // UMMA stage ring position / empty-barrier parity
        auto publish = [&](const float4 (&ra)[PA], const float4 (&rb)[PB]) {
            mbar_wait(empty(ps), pph);
            store_stage(ps, ra, rb);
            fence_proxy_async();
            mbar_arrive(full(ps));
            if (++ps == STAGES) { ps = 0; pph ^= 1u; }
        };
        float4 ra[PA], rb[PB];
        int64_t issued = 0;
        int qi = 0, qr = 0;                                 // staging ring: next stage to fill / to read
        for (int i = 0; i < WS_DEPTH; ++i) {
            if (issued < nunits) { issue_copy(qi); ++issued; if (++qi == WS_NSTG) qi = 0; }
            cp_async_commit();
        }
        for (int64_t pi = 0; pi < nunits; ++pi) {
            cp_async_wait<WS_DEPTH - 1>();                 // this thread's copies of k-block pi have landed
            read_stage(qr, ra, rb);
            if (++qr == WS_NSTG) qr = 0;
            if (issued < nunits) { issue_copy(qi); ++issued; if (++qi == WS_NSTG) qi = 0; }
            cp_async_commit();
            publish(ra, rb);
        }
        cp_async_wait<0>();
    } else {
        // ================= drainers + epilogue =================
        const int dw = warp - WS_PROD / 32;              // 0..7
        const int rowq = (dw & 3) * 32 + lane;           // TMEM lane = output row (warp % 4 selects the lane quarter)
        const int colh = (dw >> 2) * NC;
        float acc[NC], cin[DEFER ? NC : 1];
        int64_t ct = u0 / sk.KT; int ckt = (int)(u0 - ct * sk.KT);
        int64_t ctn = ct / sk.tilesM, ctm = ct - ctn * sk.tilesM;
        int64_t m0 = 0, n0 = 0;
        bool fresh = true;
        const bool use_c = !sk.partial && g.beta != 0.f;
        for (int64_t ci = 0; ci < nunits; ++ci) {
            const int b = (int)(ci & 1);
            if (fresh) {
                m0 = ctm * BM; n0 = ctn * BN;
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const int64_t m = m0 + rowq, n = n0 + colh + c;
                    const float cv = (use_c && m < g.M && n < g.N) ? __ldcs(&g.C[m + n * g.ldc]) : 0.f;
                    if (DEFER) { cin[c] = cv; acc[c] = 0.f; } else acc[c] = cv * (g.beta / g.alpha);
                }
                fresh = false;
            }
            mbar_wait(tfull(b), (unsigned)((ci >> 1) & 1));
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
            if (++ckt == sk.KT || ci + 1 == nunits) {
                if (sk.partial) {
                    float* Pt = g.C + (ct + (int64_t)blockIdx.x) * (int64_t)(BM * BN) + rowq + (int64_t)colh * BM;
#pragma unroll
                    for (int c = 0; c < NC; ++c) Pt[c * BM] = g.alpha * acc[c];
                } else {
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        const int64_t m = m0 + rowq, n = n0 + colh + c;
                        if (m < g.M && n < g.N)
                            __stcs(&g.C[m + n * g.ldc], DEFER ? fmaf(g.alpha, acc[c], g.beta * cin[DEFER ? c : 0]) : g.alpha * acc[c]);
                    }
                }
                ckt = 0; ++ct; fresh = true;
                if (++ctm == sk.tilesM) { ctm = 0; ++ctn; }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == MMA_WARP)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(256u) : "memory");
}

template <bool TA, int BN>
inline cudaError_t launch_umma_ws(GemmArgs<float> g, const MmaPlan& p, cudaStream_t st) {
    auto kern = gemm_umma_ws_kernel<TA, BN>;
    static SmemAttr attr;
    { cudaError_t e = ensure_dyn_smem(kern, WsSmem<BN>::BYTES, attr); if (e != cudaSuccess) return e; }
    kern<<<p.grid, WS_NT, WsSmem<BN>::BYTES, st>>>(g, p.sk);
    return cudaGetLastError();
}

// plan: same stream-K partition as gemm_mma.cuh with 128 x 128 tiles, one CTA per SM
inline MmaPlan umma_plan(int64_t M, int64_t N, int64_t K, int bn, int sms, bool partial) {
    return mma_plan(M, N, K, BM, bn, BK, sms, partial);
}

template <bool TA, int BN>
inline cudaError_t launch_umma(GemmArgs<float> g, const MmaPlan& p, cudaStream_t st) {
    auto kern = gemm_umma_kernel<TA, BN>;
    static SmemAttr attr;
    { cudaError_t e = ensure_dyn_smem(kern, SMEM_BYTES, attr); if (e != cudaSuccess) return e; }
    kern<<<p.grid, NT, SMEM_BYTES, st>>>(g, p.sk);
    return cudaGetLastError();
}

}  // namespace umma
}  // namespace ctqr
