// norm2_static.cu -- dwf_norm2_static: the norm2 reduction (hot path row a7 of SURVEY.md section 8; the paper's
// accelerator_sum primitive, section 2.1) for callers that must not allocate: code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc.  dwf_norm2 (reduce.cu) keeps its per-CTA
// partial sums in scratch memory that dwf_create_geometry allocates; this variant needs no geometry and keeps them
// in a file-scope __device__ array of fixed size, which every GPU that loads the library holds until the process
// exits (512.25 KB).  The entry point calls no cudaMalloc, cudaFree or allocating library routine.
//
// One launch, deterministic: CTA b sums the 2048 128-bit vectors [2048 b, 2048 b + 2048) of the buffer in fp64 in a
// fixed order and writes partial b; the CTA that arrives last at a counter adds the partials in a fixed order and
// writes the result.  The counter must start at zero: it is cleared on the stream before every launch (and by the
// last CTA), the partials need no clearing (a launch reads only what it wrote).  ALL calls on a device share the
// array: calls that overlap on the GPU (different streams, or graph branches) race on it -- the caller serialises.
#include <mutex>

#include "dwf_internal.cuh"
#include "reduce.cuh"

namespace dwf {

constexpr int NS_THREADS = 256, NS_UNROLL = 8;
constexpr size_t NS_VEC_PER_CTA = (size_t)NS_THREADS * NS_UNROLL;          // 2048 vectors = 32 KB per CTA
constexpr size_t NS_MAX_CTAS = 65536;
constexpr size_t NS_MAX_BYTES = NS_MAX_CTAS * NS_VEC_PER_CTA * 16;         // 2 GiB per call (DWF_NORM2_STATIC_MAX_BYTES)
constexpr int NS_HEAD = 32;                                                // doubles in front of the partials (256 B): word 0 = counter
static_assert(NS_MAX_BYTES == DWF_NORM2_STATIC_MAX_BYTES, "dwf.h states the limit");

// the scratch: [0] arrival counter (as unsigned int), [NS_HEAD + b] partial of CTA b.  In HOST code this name is only a
// handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) double norm2_static_scratch[NS_HEAD + NS_MAX_CTAS];

template <typename T>
__global__ void __launch_bounds__(NS_THREADS)
norm2_static_kernel(const T *__restrict__ x, size_t nreal, double *scratch, double *__restrict__ result)
{
    __shared__ double smem[32];
    __shared__ bool is_last;
    constexpr int W = 16 / sizeof(T);                       // reals per 128-bit vector
    using V = typename std::conditional<sizeof(T) == 4, float4, double2>::type;
    const size_t nvec = nreal / W;
    auto sq = [](V q) -> double {
        if constexpr (sizeof(T) == 4) return ((double)q.x * q.x + (double)q.y * q.y) + ((double)q.z * q.z + (double)q.w * q.w);
        else return q.x * q.x + q.y * q.y;
    };
    const size_t base = blockIdx.x * NS_VEC_PER_CTA + threadIdx.x;
    double a[NS_UNROLL];
    if (base + (NS_UNROLL - 1) * NS_THREADS < nvec) {       // whole chunk: eight independent loads in flight
        V q[NS_UNROLL];
#pragma unroll
        for (int u = 0; u < NS_UNROLL; u++) q[u] = __ldcs(reinterpret_cast<const V *>(x) + base + u * NS_THREADS);
#pragma unroll
        for (int u = 0; u < NS_UNROLL; u++) a[u] = sq(q[u]);
    } else {
#pragma unroll
        for (int u = 0; u < NS_UNROLL; u++) {
            const size_t i = base + u * NS_THREADS;
            a[u] = i < nvec ? sq(__ldcs(reinterpret_cast<const V *>(x) + i)) : 0.0;
        }
    }
    double acc[1] = {((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]))};
    if (blockIdx.x == 0 && threadIdx.x == 0)                // reals behind the last whole vector
        for (size_t i = nvec * W; i < nreal; i++) acc[0] += (double)x[i] * (double)x[i];
    block_sum<1>(acc, smem);
    unsigned int *counter = reinterpret_cast<unsigned int *>(scratch);
    if (threadIdx.x == 0) {
        scratch[NS_HEAD + blockIdx.x] = acc[0];
        __threadfence();                                    // the partial is visible before the arrival
        is_last = atomicAdd(counter, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();                                        // every other CTA's partial is visible to this one
    double t[1] = {0.0};
    for (unsigned int b = threadIdx.x; b < gridDim.x; b += NS_THREADS) t[0] += __ldcg(scratch + NS_HEAD + b);
    block_sum<1>(t, smem);
    if (threadIdx.x == 0) {
        *result = t[0];
        *counter = 0u;
    }
}

// device address of the scratch, looked up once per device with that device current
static double *scratch_address(int device)
{
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static double *addr[MAXDEV] = {};
    if (device < 0 || device >= MAXDEV) { set_error("dwf_norm2_static: device ordinal %d out of range", device); return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        double *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), norm2_static_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            set_error("dwf_norm2_static: cudaGetSymbolAddress failed on device %d: %s", device, cudaGetErrorString(e));
            return nullptr;
        }
        addr[device] = p;
    }
    return addr[device];
}

}  // namespace dwf

using namespace dwf;

extern "C" int dwf_norm2_static(const void *x_dev, size_t n_reals, int precision, int cuda_device, double *result_dev, void *stream)
{
    if (!x_dev || !result_dev) { set_error("dwf_norm2_static: NULL argument"); return DWF_ERR_INVALID_ARG; }
    if (precision != DWF_F32 && precision != DWF_F64) { set_error("dwf_norm2_static: precision must be DWF_F32 or DWF_F64"); return DWF_ERR_UNSUPPORTED; }
    if (!aligned16(x_dev) || (reinterpret_cast<uintptr_t>(result_dev) & 7)) {
        set_error("dwf_norm2_static: x_dev must be 16-byte aligned, result_dev 8-byte aligned");
        return DWF_ERR_INVALID_ARG;
    }
    if (n_reals > NS_MAX_BYTES / (size_t)precision) {
        set_error("dwf_norm2_static: %zu reals of %d bytes exceed the %zu bytes (DWF_NORM2_STATIC_MAX_BYTES) that the static scratch covers; "
                  "use dwf_norm2 or split the buffer", n_reals, precision, NS_MAX_BYTES);
        return DWF_ERR_INVALID_ARG;
    }
    DeviceGuard guard(cuda_device);
    if (!guard.ok) { set_error("dwf_norm2_static: cannot select device %d", cuda_device); return DWF_ERR_CUDA; }
    double *scratch = scratch_address(cuda_device);
    if (!scratch) return DWF_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t nvec = n_reals / (16 / (size_t)precision);
    const unsigned int grid = nvec ? (unsigned int)((nvec + NS_VEC_PER_CTA - 1) / NS_VEC_PER_CTA) : 1u;
    DWF_CUDA_CHECK(cudaMemsetAsync(scratch, 0, NS_HEAD * sizeof(double), st));       // the counter starts at zero
    if (precision == DWF_F32)
        norm2_static_kernel<float><<<grid, NS_THREADS, 0, st>>>(static_cast<const float *>(x_dev), n_reals, scratch, result_dev);
    else
        norm2_static_kernel<double><<<grid, NS_THREADS, 0, st>>>(static_cast<const double *>(x_dev), n_reals, scratch, result_dev);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}
