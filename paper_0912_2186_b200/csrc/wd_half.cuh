// wd_half.cuh -- binary16 <-> float32 helpers shared by the half-precision storage kernels (wd_half.cu, wd_half_stage.cu).
// Reading RH: 16-byte vectors of 8 halves; spinors carry a float32 scale per site.
#pragma once
#include <cuda_fp16.h>

namespace wd {

__device__ __forceinline__ void unpack8(const uint4 &v, float *r)
{
    const __half2 *h = reinterpret_cast<const __half2 *>(&v);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float2 f = __half22float2(h[i]);
        r[2 * i] = f.x;
        r[2 * i + 1] = f.y;
    }
}

__device__ __forceinline__ uint4 pack8(const float *r)
{
    uint4 v;
    __half2 *h = reinterpret_cast<__half2 *>(&v);
#pragma unroll
    for (int i = 0; i < 4; ++i) h[i] = __halves2half2(__float2half_rn(r[2 * i]), __float2half_rn(r[2 * i + 1]));
    return v;
}

} // namespace wd
