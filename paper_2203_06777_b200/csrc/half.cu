// half.cu -- fp16 STORAGE of spinor fields with fp32 arithmetic (third variant; not in PAPER.md: the
// traffic model of DESIGN.md 6.8).  A field in fp16 storage is the fp32 device layout (pack.cu) element by element, two
// bytes per real: the same permutation, half the bytes.  The links stay fp32.
//   dwf_to_f16 / dwf_from_f16   conversion of a device field (round to nearest even / exact)
//   dwf_dhop_oe_f16 / _eo_f16   the staged fp32 kernel in its HALF instantiation (dhop_staged.cu MODE 7): TMA moves fp16
//                               rows, a consumer widens them to fp32 right after the shared-memory load, accumulates in
//                               fp32 and rounds once, in the store
#include <cuda_fp16.h>

#include "dwf_internal.cuh"

namespace dwf {

__global__ void __launch_bounds__(256) to_f16_kernel(const float4 *__restrict__ in, uint2 *__restrict__ out, size_t nvec)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        const float4 v = __ldcs(in + i);
        const __half2 lo = __floats2half2_rn(v.x, v.y), hi = __floats2half2_rn(v.z, v.w);
        out[i] = make_uint2(*reinterpret_cast<const uint32_t *>(&lo), *reinterpret_cast<const uint32_t *>(&hi));
    }
}

__global__ void __launch_bounds__(256) from_f16_kernel(const uint2 *__restrict__ in, float4 *__restrict__ out, size_t nvec)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        const uint2 v = __ldcs(in + i);
        const float2 lo = __half22float2(*reinterpret_cast<const __half2 *>(&v.x)), hi = __half22float2(*reinterpret_cast<const __half2 *>(&v.y));
        out[i] = make_float4(lo.x, lo.y, hi.x, hi.y);
    }
}

static int convert(const dwf_geometry *g, const void *in, void *out, int parity, bool to_half, void *stream, const char *who)
{
    if (!g || !in || !out || !parity_ok(parity)) { set_error("%s: bad argument", who); return DWF_ERR_INVALID_ARG; }
    if (g->prec != DWF_F32) { set_error("%s: fp16 storage goes with fp32 geometries", who); return DWF_ERR_UNSUPPORTED; }
    if (!aligned16(in) || !aligned16(out)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t nvec = dwf_field_bytes(g, parity) / 16;           // four reals per thread and pass
    const size_t cap = (size_t)g->sm_count * 16;
    const unsigned grid = (unsigned)((nvec + 255) / 256 < cap ? (nvec + 255) / 256 : cap);
    wait_for_exports(g, st, out, dwf_field_bytes(g, parity));
    if (to_half) to_f16_kernel<<<grid, 256, 0, st>>>(static_cast<const float4 *>(in), static_cast<uint2 *>(out), nvec);
    else         from_f16_kernel<<<grid, 256, 0, st>>>(static_cast<const uint2 *>(in), static_cast<float4 *>(out), nvec);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

static int dhop_f16(const dwf_geometry *g, const void *in, void *out, int parity_out, void *stream, const char *who)
{
    if (!g || !in || !out) { set_error("%s: NULL argument", who); return DWF_ERR_INVALID_ARG; }
    if (in == out) { set_error("%s: in-place application is not defined (in == out)", who); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(out)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("%s: call dwf_load_gauge first", who); return DWF_ERR_NO_GAUGE; }
    if (g->prec != DWF_F32 || !staged_supports_half(g)) {
        set_error("%s: fp16 storage needs an fp32 geometry with a staged variant and L0 a multiple of 16", who);
        return DWF_ERR_UNSUPPORTED;
    }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    wait_for_exports(g, st, out, dwf_field_bytes(g, parity_out) / 2);
    return launch_dhop_staged(g, in, out, parity_out, st, nullptr, nullptr, false, nullptr, 0.f, 0.f, 1, false, false, true);
}

}  // namespace dwf

using namespace dwf;

extern "C" {

int dwf_to_f16(const dwf_geometry *g, const void *field_f32, int parity, void *field_f16, void *stream)
{
    return convert(g, field_f32, field_f16, parity, true, stream, "dwf_to_f16");
}
int dwf_from_f16(const dwf_geometry *g, const void *field_f16, int parity, void *field_f32, void *stream)
{
    return convert(g, field_f16, field_f32, parity, false, stream, "dwf_from_f16");
}
int dwf_dhop_oe_f16(const dwf_geometry *g, const void *in_even_f16, void *out_odd_f16, void *stream)
{
    return dhop_f16(g, in_even_f16, out_odd_f16, DWF_ODD, stream, "dwf_dhop_oe_f16");
}
int dwf_dhop_eo_f16(const dwf_geometry *g, const void *in_odd_f16, void *out_even_f16, void *stream)
{
    return dhop_f16(g, in_odd_f16, out_even_f16, DWF_EVEN, stream, "dwf_dhop_eo_f16");
}

}  // extern "C"
