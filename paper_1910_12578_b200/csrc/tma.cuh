// tma.cuh -- the sm_100a asynchronous-copy primitives the advance kernels use (inline PTX; no library):
//   * tensor-map (TMA) tile loads global -> shared that complete on an mbarrier (cp.async.bulk.tensor),
//   * bulk / tensor prefetches global -> L2 (cp.async.bulk.prefetch[.tensor]),
//   * mbarrier init / expect_tx / parity wait, and the proxy fences that order generic-proxy accesses of shared
//     memory against the async proxy that TMA writes through.
// Host side: tensor maps are encoded with the driver's cuTensorMapEncodeTiled, reached through
// cudaGetDriverEntryPoint (libcst.so does not link libcuda).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{   // make the initialised barriers visible to the async proxy
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{   // generic-proxy reads / writes of shared memory before this point are ordered before later async-proxy (TMA) writes
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) { }
}

// 3-D tile load: box of the tensor map at element coordinates (x, y, z) -> dense rows at dst (128-byte aligned)
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int x, int y, int z, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 :: "r"(smem_u32(dst)), "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap* map, int x, int y, int z)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];"
                 :: "l"(map), "r"(x), "r"(y), "r"(z) : "memory");
}
// contiguous bytes -> L2 (16-byte aligned address, size a multiple of 16)
__device__ __forceinline__ void bulk_prefetch_l2(const void* gptr, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(gptr), "r"(bytes) : "memory");
}
// contiguous bytes global -> shared, completing on an mbarrier (16-byte aligned, size a multiple of 16)
__device__ __forceinline__ void bulk_load(void* dst, const void* gptr, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(dst)), "l"(gptr), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---- host: fp64 rank-3 tensor map over a C-contiguous array [d2][d1][d0] (d0 fastest) with a box of (b0, b1, b2) elements.
// Returns false if the driver entry point is missing or the encode fails (callers then take their non-TMA path).
inline bool tma_encode_3d_f64(CUtensorMap* map, const void* base, unsigned long long d0, unsigned long long d1,
                              unsigned long long d2, unsigned b0, unsigned b1, unsigned b2)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn fn = nullptr;
    static bool looked = false;
    if (!looked) {
        looked = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (encode_fn)p;
        else
            (void)cudaGetLastError();
    }
    if (!fn) return false;
    const cuuint64_t dims[3] = { d0, d1, d2 };
    const cuuint64_t strides[2] = { d0 * 8ull, d0 * d1 * 8ull };          // bytes, dims 1 and 2
    const cuuint32_t box[3] = { b0, b1, b2 };
    const cuuint32_t estr[3] = { 1, 1, 1 };
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
