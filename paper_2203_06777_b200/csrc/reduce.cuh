// reduce.cuh -- warp / block sums in a fixed order (deterministic), shared by the reduction kernels.
#pragma once
#include <cuda_runtime.h>

namespace dwf {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// block-wide sum of NV values per thread; result valid in thread 0
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double *smem /* [NV][32] */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int i = 0; i < NV; i++) {
        v[i] = warp_sum(v[i]);
        if (lane == 0) smem[i * 32 + warp] = v[i];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int i = 0; i < NV; i++) {
            double t = (lane < nwarp) ? smem[i * 32 + lane] : 0.0;
            v[i] = warp_sum(t);
        }
    }
}

}  // namespace dwf
