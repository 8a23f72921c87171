// tma.cuh -- sm_100a bulk-tensor copy (TMA) and mbarrier primitives used by the staged Dhop kernel.
//
// Device side: thin inline-PTX wrappers (mbarrier init / expect_tx / parity wait, 5-D tiled
// cp.async.bulk.tensor global -> shared).  Host side: tensor-map encoding through the driver
// entry point cuTensorMapEncodeTiled, fetched with cudaGetDriverEntryPoint so that libdwf does
// not link against libcuda.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace dwf {

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Arrive that is issued only after the shared-memory loads whose results are passed in have returned
// their data (the values are unused inputs of the asm statement, so the instruction depends on them).
// This is how a consumer hands a staged region back to the TMA producer right after READING it: a plain
// arrive placed behind the loads in program order may execute while they are still in flight (ptxas
// does not make SYNCS.ARRIVE wait for earlier LDS, and __syncwarp() compiles to nothing in converged
// code), and the refilling bulk copy -- async proxy -- then overwrites the data before it is read;
// observed on the fp64 kernel as stale last-issued loads.  One 32-bit word of every load instruction is
// enough: a warp-wide LDS releases its scoreboard when all lanes have their data.
__device__ __forceinline__ void mbar_arrive_after8(uint32_t bar, double a, double b, double c, double d, double e, double f,
                                                   double g, double h)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar), "d"(a), "d"(b), "d"(c), "d"(d), "d"(e), "d"(f), "d"(g),
                 "d"(h) : "memory");
}
// the same with one witness: a value that the arithmetic has derived from EVERY load of the region (the staged fp32
// kernel passes an accumulator component, which depends on a word of each of the twelve 128-bit loads of a leg pair)
__device__ __forceinline__ void mbar_arrive_after1(uint32_t bar, float witness)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar), "f"(witness) : "memory");
}
__device__ __forceinline__ void mbar_arrive_after12(uint32_t bar, float a, float b, float c, float d, float e, float f, float g,
                                                    float h, float i, float j, float k, float l)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar), "f"(a), "f"(b), "f"(c), "f"(d), "f"(e), "f"(f), "f"(g),
                 "f"(h), "f"(i), "f"(j), "f"(k), "f"(l) : "memory");
}
// blocks until the phase with the given parity has completed
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
// 5-D tiled tensor copy global -> shared, completion signalled on an mbarrier (SASS: UTMALDG)
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1,
                                            int c2, int c3, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2),
        "r"(c3), "r"(c4) : "memory");
}
// the same copy carrying an L2 eviction-priority policy (createpolicy) for the lines it touches
__device__ __forceinline__ void tma_load_5d_hint(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1,
                                                 int c2, int c3, int c4, uint64_t policy)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1, {%3, %4, %5, %6, %7}], [%2], %8;" ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2),
        "r"(c3), "r"(c4), "l"(policy) : "memory");
}
// L2 eviction-priority policies: 0 evict_normal, 1 evict_first, 2 evict_last
__device__ __forceinline__ uint64_t l2_policy(int kind)
{
    uint64_t p;
    if (kind == 1)      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else                asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// global load / store of one complex with an L2 policy, bypassing L1 (data touched once per CTA)
__device__ __forceinline__ float2 ldg_hint(const float2 *p, uint64_t policy)
{
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;"
                 : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(policy));
    return v;
}
__device__ __forceinline__ float4 ldg128_hint(const float4 *p, uint64_t policy)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(policy));
    return v;
}
__device__ __forceinline__ void stg128_hint(float4 *p, float4 v, uint64_t policy)
{
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x),
                 "f"(v.y), "f"(v.z), "f"(v.w), "l"(policy) : "memory");
}
__device__ __forceinline__ void stg_hint(float2 *p, float2 v, uint64_t policy)
{
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y),
                 "l"(policy) : "memory");
}
// orders this thread's earlier generic-proxy accesses before later async-proxy (TMA) ones
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// register reallocation between warpgroups (all four warps of a warpgroup must execute it)
template <int N> __device__ __forceinline__ void reg_alloc()
{
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N> __device__ __forceinline__ void reg_dealloc()
{
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// ---- host ------------------------------------------------------------------------------------
typedef CUresult (*PFN_tensorMapEncodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                             const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                             const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
PFN_tensorMapEncodeTiled get_tensor_map_encoder();   // nullptr if the driver does not provide it

}  // namespace dwf
