// tma.cuh -- Tensor Memory Accelerator plumbing (sm_100a): host-side tensor-map encoding through the driver entry
// point (no link against libcuda), device-side cp.async.bulk.tensor loads that complete on an mbarrier.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctqr {
namespace tma {

// cuTensorMapEncodeTiled, resolved once per process through the runtime (the library links only libcudart)
inline CUresult encode_tiled(CUtensorMap* map, CUtensorMapDataType dt, cuuint32_t rank, void* base, const cuuint64_t* dims,
                             const cuuint64_t* strides, const cuuint32_t* box, const cuuint32_t* estrides,
                             CUtensorMapSwizzle swz) {
    typedef CUresult (*Fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                           const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                           CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static Fn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return (Fn)p;
    }();
    if (!fn) return CUDA_ERROR_NOT_SUPPORTED;
    return fn(map, dt, rank, base, dims, strides, box, estrides, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

// 2-D map over a column-major matrix: element (i0, i1) at base + (i0 + i1 * ld) * elem_bytes; dim0 is contiguous.
// Boxes of box0 x box1 elements; out-of-range elements of a box are delivered as zeros.
inline cudaError_t map_2d(CUtensorMap* map, CUtensorMapDataType dt, int elem_bytes, const void* base, int64_t dim0, int64_t dim1,
                          int64_t ld, int box0, int box1, CUtensorMapSwizzle swz) {
    cuuint64_t dims[2] = {(cuuint64_t)dim0, (cuuint64_t)dim1};
    cuuint64_t strides[1] = {(cuuint64_t)ld * (cuuint64_t)elem_bytes};
    cuuint32_t box[2] = {(cuuint32_t)box0, (cuuint32_t)box1};
    cuuint32_t es[2] = {1, 1};
    return encode_tiled(map, dt, 2, const_cast<void*>(base), dims, strides, box, es, swz) == CUDA_SUCCESS ? cudaSuccess
                                                                                                          : cudaErrorInvalidValue;
}

#ifdef __CUDACC__
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_n(unsigned bar, unsigned n) {      // n arrivals at once
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(n) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "TW: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra TD;\n\tbra TW;\n\tTD:\n\t}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
// box at element coordinates (c0, c1) -> shared memory at `dst`; completes `bytes of the box` on mbarrier `bar`
__device__ __forceinline__ void load_2d(unsigned dst, const CUtensorMap* map, int c0, int c1, unsigned bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
                 ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar)
                 : "memory");
}
// same with an L2 eviction-priority hint (createpolicy value)
__device__ __forceinline__ void load_2d_hint(unsigned dst, const CUtensorMap* map, int c0, int c1, unsigned bar, uint64_t policy) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;\n"
                 ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar), "l"(policy)
                 : "memory");
}
__device__ __forceinline__ void prefetch_map(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(map) : "memory");
}
#endif

}  // namespace tma
}  // namespace ctqr
