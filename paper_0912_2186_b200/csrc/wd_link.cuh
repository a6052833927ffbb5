// wd_link.cuh -- load one SU(3) link from the native link field into registers (device only).
// Native link layout: wd_layout.cuh ([block][vector][lane], the four links of a site together).
// For RECON == 12 the third row is rebuilt as conj(row0 x row1) (
// PAPER.md:167).
#pragma once
#include "wd_layout.cuh"
#include "wd_math.cuh"

namespace wd {

// address of vector 0 of the links of `site`; vector j is at + j*BLK
template <typename T, int RECON>
__device__ __forceinline__ const typename LinkLayout<T, RECON>::Vec *link_ptr(const T *__restrict__ links, long long site)
{
    using L = LinkLayout<T, RECON>;
    return reinterpret_cast<const typename L::Vec *>(links) + (site >> 5) * (L::NVEC * BLK) + (site & (BLK - 1));
}

// U_MU(site) -> u[18].  Link MU occupies reals [MU*RECON, (MU+1)*RECON) of the site's link record;
// for fp32 recon 18 an odd MU starts in the middle of a 16-byte vector, so 5 vectors are fetched
// and 18 of their 20 reals are kept (indices resolved at compile time).
template <int MU, typename T, int RECON>
__device__ __forceinline__ void load_link(const T *__restrict__ links, long long site, T (&u)[18])
{
    using L = LinkLayout<T, RECON>;
    constexpr int first = (MU * RECON) / L::CR, last = (MU * RECON + RECON - 1) / L::CR;
    constexpr int skip = MU * RECON - first * L::CR;
    const typename L::Vec *q = link_ptr<T, RECON>(links, site);
    T tmp[(last - first + 1) * L::CR];
#pragma unroll
    for (int j = first; j <= last; ++j) {
        const typename L::Vec v = __ldg(q + j * BLK);
        unpack(v, &tmp[(j - first) * L::CR]);
    }
#pragma unroll
    for (int i = 0; i < RECON; ++i) u[i] = tmp[skip + i];
    if (RECON == 12) reconstruct_row2(u);
    if (RECON == 8) reconstruct_from8(u);
}

} // namespace wd
