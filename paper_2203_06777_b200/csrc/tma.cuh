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
// Release of a staged region by a consumer: an arrive that CANNOT issue before the shared-memory loads of the region
// have delivered their data.  Program order is not enough: ptxas does not make SYNCS.ARRIVE wait for earlier LDS,
// __syncwarp() compiles to nothing in converged code, and an asm statement that merely lists the loaded values as unused
// operands keeps them alive for the C++ front end only (the PTX text of the arrive does not mention them).  With a bare
// arrive the fp64 kernel read data of the NEXT fill in the last-issued load of a leg (r02: found with a field whose value
// encodes its slice).  Here the barrier ADDRESS is computed from witness values that derive from every load of the region:
// addr = bar + (bits(w) & zero), where `zero` is a kernel argument that is 0 at run time, so ptxas cannot fold the term
// away and the arrive depends on the data.  A warp-wide LDS releases its scoreboard when all lanes have their data, so
// lane 0's witness covers the warp; __syncwarp() in front of it states the same for the memory model.
// The float form has no "memory" clobber: the loads of the region are tied to the arrive by the data dependence, and
// the loads of other regions (the next legs) stay free to move across it.
__device__ __forceinline__ void mbar_arrive_dep(uint32_t bar, uint32_t zero, float w)
{
    asm volatile(
        "{\n\t.reg .b32 t;\n\t"
        "mov.b32 t, %2;\n\tand.b32 t, t, %1;\n\tadd.u32 t, t, %0;\n\t"
        "mbarrier.arrive.shared::cta.b64 _, [t];\n\t}"
        ::"r"(bar), "r"(zero), "f"(w));
}
__device__ __forceinline__ void mbar_arrive_dep(uint32_t bar, uint32_t zero, double a, double b)
{
    asm volatile(
        "{\n\t.reg .b32 la, lb, hh, t;\n\t"
        "mov.b64 {la, hh}, %2;\n\tmov.b64 {lb, hh}, %3;\n\tor.b32 t, la, lb;\n\tand.b32 t, t, %1;\n\tadd.u32 t, t, %0;\n\t"
        "mbarrier.arrive.shared::cta.b64 _, [t];\n\t}"
        ::"r"(bar), "r"(zero), "d"(a), "d"(b) : "memory");
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
__device__ __forceinline__ void stg64_hint(uint2 *p, uint2 v, uint64_t policy)
{
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v2.b32 [%0], {%1, %2}, %3;" ::"l"(p), "r"(v.x), "r"(v.y),
                 "l"(policy) : "memory");
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
