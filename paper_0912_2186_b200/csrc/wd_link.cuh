// wd_link.cuh -- load one SU(3) link from the native link field into registers (device only).
// Native link layout: wd_layout.cuh.  For RECON == 12 the third row is rebuilt as
// conj(row0 x row1).
#pragma once
#include "wd_layout.cuh"
#include "wd_math.cuh"

namespace wd {

template <typename T, int RECON>
__device__ __forceinline__ void load_link(const T *__restrict__ links, long long V, int mu, long long site, T (&u)[18])
{
    using L = LinkLayout<T, RECON>;
    const typename L::Vec *q = reinterpret_cast<const typename L::Vec *>(links) + (long long)mu * L::NCH * V + site;
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) {
        const typename L::Vec v = __ldg(q + (long long)c * V);
        unpack(v, &u[c * L::CR]);
    }
    if (RECON == 12) reconstruct_row2(u);
}

} // namespace wd
