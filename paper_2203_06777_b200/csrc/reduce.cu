// reduce.cu -- norm2 and inner product (hot path row a7 of SURVEY.md section 8; the paper's
// accelerator_sum primitive, section 2.1).
//
// Two passes, both deterministic: (1) a fixed-size grid strides over the field with 128-bit
// loads, accumulates in fp64 per thread, reduces with warp shuffles and one shared-memory step
// to one partial per CTA; (2) a single CTA adds the partials in a fixed order.  The device
// layout is a permutation of the canonical one, so the sum runs over the raw buffer.
#include "dwf_internal.cuh"
#include "reduce.cuh"

namespace dwf {

template <typename T>
__global__ void __launch_bounds__(256)
norm2_partial_kernel(const T *__restrict__ x, size_t nreal, double *__restrict__ partials)
{
    __shared__ double smem[32];
    constexpr int W = 16 / sizeof(T);                       // reals per 128-bit vector
    using V = typename std::conditional<sizeof(T) == 4, float4, double2>::type;
    const size_t nvec = nreal / W;
    // four independent 128-bit loads in flight per thread, one fp64 accumulator each (added in a
    // fixed order afterwards, so the result does not depend on timing)
    constexpr int UN = 4;
    double a4[UN] = {0.0, 0.0, 0.0, 0.0};
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    auto sq = [](V q) -> double {
        if constexpr (sizeof(T) == 4) return ((double)q.x * q.x + (double)q.y * q.y) + ((double)q.z * q.z + (double)q.w * q.w);
        else return q.x * q.x + q.y * q.y;
    };
    for (; i + (UN - 1) * stride < nvec; i += UN * stride) {
        V q[UN];
#pragma unroll
        for (int u = 0; u < UN; u++) q[u] = __ldcs(reinterpret_cast<const V *>(x) + i + u * stride);
#pragma unroll
        for (int u = 0; u < UN; u++) a4[u] += sq(q[u]);
    }
    for (; i < nvec; i += stride) a4[0] += sq(__ldcs(reinterpret_cast<const V *>(x) + i));
    double acc[1] = {(a4[0] + a4[1]) + (a4[2] + a4[3])};
    // tail (nreal is a multiple of 24, so this never runs for fp32/fp64 fields; kept for safety)
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (size_t i = nvec * W; i < nreal; i++) acc[0] += (double)x[i] * (double)x[i];
    block_sum<1>(acc, smem);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc[0];
}

template <typename T>
__global__ void __launch_bounds__(256)
inner_partial_kernel(const T *__restrict__ a, const T *__restrict__ b, size_t ncomplex, double *__restrict__ partials)
{
    __shared__ double smem[64];
    using V = typename std::conditional<sizeof(T) == 4, float4, double2>::type;
    constexpr int CW = 8 / sizeof(T);                       // complex numbers per 128-bit vector
    const size_t nvec = ncomplex / CW;
    double acc[2] = {0.0, 0.0};
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        V p = __ldcs(reinterpret_cast<const V *>(a) + i);
        V q = __ldcs(reinterpret_cast<const V *>(b) + i);
        // conj(a) * b = (ar br + ai bi) + i (ar bi - ai br)
        if constexpr (sizeof(T) == 4) {
            // fp32 vector = (re, re', im, im') of two spin components (pack.cu)
            acc[0] += ((double)p.x * q.x + (double)p.z * q.z) + ((double)p.y * q.y + (double)p.w * q.w);
            acc[1] += ((double)p.x * q.z - (double)p.z * q.x) + ((double)p.y * q.w - (double)p.w * q.y);
        } else {
            acc[0] += (double)p.x * q.x + (double)p.y * q.y;
            acc[1] += (double)p.x * q.y - (double)p.y * q.x;
        }
    }
    // no tail: a field holds 12 complex per site, a multiple of the CW complex of a vector
    block_sum<2>(acc, smem);
    if (threadIdx.x == 0) {
        partials[2 * blockIdx.x] = acc[0];
        partials[2 * blockIdx.x + 1] = acc[1];
    }
}

// one CTA: result[i] = sum over blocks of partials[NV*block + i], fixed order.  The result also goes
// straight into the geometry's mapped host mailbox (values, then a sequence number behind a
// system-scope fence), so that the host can pick it up without a copy and a stream synchronise.
template <int NV>
__global__ void __launch_bounds__(256)
final_sum_kernel(const double *__restrict__ partials, int nblocks, double *__restrict__ result,
                 double *mailbox, unsigned long long seq)
{
    __shared__ double smem[NV * 32];
    double acc[NV];
#pragma unroll
    for (int i = 0; i < NV; i++) acc[i] = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
#pragma unroll
        for (int i = 0; i < NV; i++) acc[i] += partials[NV * b + i];
    block_sum<NV>(acc, smem);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NV; i++) { result[i] = acc[i]; mailbox[i] = acc[i]; }
        __threadfence_system();
        *reinterpret_cast<volatile unsigned long long *>(mailbox + 2) = seq;
    }
}

// sequence number of the next reduction of this geometry (reductions of one geometry are serialised
// by contract: they share the partials and the mailbox)
static unsigned long long next_seq(const dwf_geometry *g)
{
    return ++const_cast<dwf_geometry *>(g)->mailbox_seq;
}
// the mailbox is a ring of MAILBOX_SLOTS slots of four words: reduction number q writes slot q % MAILBOX_SLOTS, so that a
// caller may leave up to MAILBOX_SLOTS - 1 results unread while it enqueues more work (dwf_dhop_*_norm2_async)
static double *mailbox_slot(const dwf_geometry *g, unsigned long long seq)
{
    return g->mailbox_dev + 4 * (seq % MAILBOX_SLOTS);
}

int launch_norm2(const dwf_geometry *g, const void *field, size_t nreal, cudaStream_t st)
{
    const int nb = g->reduce_blocks;
    if (g->prec == DWF_F32)
        norm2_partial_kernel<float><<<nb, 256, 0, st>>>(static_cast<const float *>(field), nreal, g->partials);
    else
        norm2_partial_kernel<double><<<nb, 256, 0, st>>>(static_cast<const double *>(field), nreal, g->partials);
    { const unsigned long long q = next_seq(g); final_sum_kernel<1><<<1, 256, 0, st>>>(g->partials, nb, g->result_dev, mailbox_slot(g, q), q); }
    count_launch(2);
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

int launch_final_sum(const dwf_geometry *g, int nblocks, cudaStream_t st)
{
    { const unsigned long long q = next_seq(g); final_sum_kernel<1><<<1, 256, 0, st>>>(g->partials, nblocks, g->result_dev, mailbox_slot(g, q), q); }
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

int launch_inner(const dwf_geometry *g, const void *a, const void *b, size_t ncomplex, cudaStream_t st)
{
    const int nb = g->reduce_blocks;
    if (g->prec == DWF_F32)
        inner_partial_kernel<float><<<nb, 256, 0, st>>>(static_cast<const float *>(a), static_cast<const float *>(b), ncomplex, g->partials);
    else
        inner_partial_kernel<double><<<nb, 256, 0, st>>>(static_cast<const double *>(a), static_cast<const double *>(b), ncomplex, g->partials);
    { const unsigned long long q = next_seq(g); final_sum_kernel<2><<<1, 256, 0, st>>>(g->partials, nb, g->result_dev, mailbox_slot(g, q), q); }
    count_launch(2);
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

}  // namespace dwf
