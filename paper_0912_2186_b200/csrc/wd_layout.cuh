// wd_layout.cuh -- NATIVE (HBM) field layouts and their register load/store helpers.
//
// SURVEY.md section 8(a) step a0 (site ordering and field layout; the build's own choice).
//
// Site index: site = x + Lx*(y + Ly*(z + Lz*t)), x fastest (same order as the canonical layout).
// Sites are grouped in BLOCKS of 32 consecutive site indices; inside a block the data is a
// structure of arrays of 16-byte vectors:
//
//   spinor, native:  [rhs][block b][vector c][lane l]   site = 32*b + l
//       fp32: vector = float4  = reals 4c..4c+3 of the 24 reals [spin][colour][re,im];  6 vectors
//       fp64: vector = double2 = reals 2c..2c+1;                                       12 vectors
//   links, native:   [block b][vector j][lane l]        all FOUR links of a site together:
//       the site's 4*RECON reals [mu][row][col][re,im] (rows 0,1 only for RECON 12) cut into
//       16-byte vectors: fp32 r18 18, fp32 r12 12, fp32 r8 8, fp64 r18 36, fp64 r12 24, fp64 r8 16 vectors per site
//       (RECON 8: the parametrisation of wd_math.cuh:reconstruct_from8).
//
// Why blocks: (1) a warp reading vector c of 32 consecutive sites issues ONE contiguous 512-byte
// request (128 bits per lane, fully coalesced); (2) the distance between two vectors of a site is
// the compile-time constant 512 B, so all loads of a site share one base register and use
// immediate offsets (the [vector][site] layout of round 1 spent ~20 % of its instructions on
// 64-bit address arithmetic); (3) a block's data is one contiguous 3 KB (spinor) / 9 KB (links)
// piece of HBM instead of 6 + 36 streams V apart (DRAM page locality).
// The volume is padded to a multiple of 32 sites (padded_volume); pad sites are never read.
#pragma once
#include <cuda_runtime.h>

namespace wd {

constexpr int BLK = 32; // sites per layout block

__host__ __device__ inline long long padded_volume(long long V) { return (V + (BLK - 1)) & ~(long long)(BLK - 1); }

template <typename T> struct SpinorLayout;
template <> struct SpinorLayout<float> {
    using Vec = float4;
    static constexpr int CR = 4;   // reals per vector
    static constexpr int NCH = 6;  // vectors per spinor
};
template <> struct SpinorLayout<double> {
    using Vec = double2;
    static constexpr int CR = 2;
    static constexpr int NCH = 12;
};

// all four links of a site: NVEC vectors of CR reals; link mu = reals [mu*RECON, (mu+1)*RECON)
template <typename T, int RECON> struct LinkLayout;
template <> struct LinkLayout<float, 18> { using Vec = float4; static constexpr int CR = 4, NVEC = 18; };
template <> struct LinkLayout<float, 12> { using Vec = float4; static constexpr int CR = 4, NVEC = 12; };
template <> struct LinkLayout<double, 18> { using Vec = double2; static constexpr int CR = 2, NVEC = 36; };
template <> struct LinkLayout<double, 12> { using Vec = double2; static constexpr int CR = 2, NVEC = 24; };
template <> struct LinkLayout<float, 8> { using Vec = float4; static constexpr int CR = 4, NVEC = 8; };
template <> struct LinkLayout<double, 8> { using Vec = double2; static constexpr int CR = 2, NVEC = 16; };

__device__ __forceinline__ void unpack(const float4 &v, float *r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void unpack(const double2 &v, double *r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void pack(float4 &v, const float *r) { v = make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ void pack(double2 &v, const double *r) { v = make_double2(r[0], r[1]); }

// address of vector 0 of `site` in ONE right-hand side's field; vector c is at + c*BLK
template <typename T>
__device__ __forceinline__ const typename SpinorLayout<T>::Vec *spinor_ptr(const T *__restrict__ field, long long site)
{
    using L = SpinorLayout<T>;
    return reinterpret_cast<const typename L::Vec *>(field) + (site >> 5) * (L::NCH * BLK) + (site & (BLK - 1));
}

// field: base of ONE right-hand side (padded_volume(V)*24 reals)
template <typename T>
__device__ __forceinline__ void load_spinor(const T *__restrict__ field, long long site, T (&p)[24])
{
    using L = SpinorLayout<T>;
    const typename L::Vec *q = spinor_ptr(field, site);
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) {
        const typename L::Vec v = __ldg(q + c * BLK);
        unpack(v, &p[c * L::CR]);
    }
}

// same, through ordinary coherent loads: for fields the SAME launch also writes (ld.global.nc / __ldg is only valid
// for data that stays read-only for the whole kernel)
template <typename T>
__device__ __forceinline__ void load_spinor_rw(const T *field, long long site, T (&p)[24])
{
    using L = SpinorLayout<T>;
    const typename L::Vec *q = reinterpret_cast<const typename L::Vec *>(field) + (site >> 5) * (L::NCH * BLK) + (site & (BLK - 1));
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) {
        const typename L::Vec v = q[c * BLK];
        unpack(v, &p[c * L::CR]);
    }
}

template <typename T>
__device__ __forceinline__ void store_spinor(T *__restrict__ field, long long site, const T (&p)[24])
{
    using L = SpinorLayout<T>;
    typename L::Vec *q = reinterpret_cast<typename L::Vec *>(field) + (site >> 5) * (L::NCH * BLK) + (site & (BLK - 1));
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) {
        typename L::Vec v;
        pack(v, &p[c * L::CR]);
        q[c * BLK] = v;
    }
}

} // namespace wd
