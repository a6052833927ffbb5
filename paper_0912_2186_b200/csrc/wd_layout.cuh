// wd_layout.cuh -- NATIVE (HBM) field layouts and their register load/store helpers.
//
// SURVEY.md section 8(a) step a0 (site ordering and field layout; the build's own choice).
//
// Site index: site = x + Lx*(y + Ly*(z + Lz*t)), x fastest (same order as the canonical layout),
// so that the 32 threads of a warp walk along x and every per-component access below is one
// contiguous, 16-byte-per-lane (128-bit) request.
//
// Spinor, native:  [rhs][chunk c][site] of 16-byte chunks.
//     fp32: chunk = float4  = reals 4c..4c+3 of the 24 reals [spin][colour][re,im];  6 chunks
//     fp64: chunk = double2 = reals 2c..2c+1;                                        12 chunks
// Links, native:   [mu][chunk c][site]
//     fp32 recon 18: chunk = float2  (9 chunks: one complex matrix element each, row major)
//     fp32 recon 12: chunk = float4  (3 chunks: rows 0,1)
//     fp64 recon 18: chunk = double2 (9 chunks)       fp64 recon 12: double2 (6 chunks)
#pragma once
#include <cuda_runtime.h>

namespace wd {

template <typename T> struct SpinorLayout;
template <> struct SpinorLayout<float> {
    using Vec = float4;
    static constexpr int CR = 4;   // reals per chunk
    static constexpr int NCH = 6;  // chunks per spinor
};
template <> struct SpinorLayout<double> {
    using Vec = double2;
    static constexpr int CR = 2;
    static constexpr int NCH = 12;
};

template <typename T, int RECON> struct LinkLayout;
template <> struct LinkLayout<float, 18> { using Vec = float2; static constexpr int CR = 2, NCH = 9; };
template <> struct LinkLayout<float, 12> { using Vec = float4; static constexpr int CR = 4, NCH = 3; };
template <> struct LinkLayout<double, 18> { using Vec = double2; static constexpr int CR = 2, NCH = 9; };
template <> struct LinkLayout<double, 12> { using Vec = double2; static constexpr int CR = 2, NCH = 6; };

__device__ __forceinline__ void unpack(const float4 &v, float *r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void unpack(const float2 &v, float *r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void unpack(const double2 &v, double *r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void pack(float4 &v, const float *r) { v = make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ void pack(float2 &v, const float *r) { v = make_float2(r[0], r[1]); }
__device__ __forceinline__ void pack(double2 &v, const double *r) { v = make_double2(r[0], r[1]); }

// field: base of ONE right-hand side (NCH*V chunks)
template <typename T>
__device__ __forceinline__ void load_spinor(const T *__restrict__ field, long long V, long long site, T (&p)[24])
{
    using L = SpinorLayout<T>;
    const typename L::Vec *q = reinterpret_cast<const typename L::Vec *>(field) + site;
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) {
        const typename L::Vec v = __ldg(q + (long long)c * V);
        unpack(v, &p[c * L::CR]);
    }
}

template <typename T>
__device__ __forceinline__ void store_spinor(T *__restrict__ field, long long V, long long site, const T (&p)[24])
{
    using L = SpinorLayout<T>;
    typename L::Vec *q = reinterpret_cast<typename L::Vec *>(field) + site;
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) {
        typename L::Vec v;
        pack(v, &p[c * L::CR]);
        q[(long long)c * V] = v;
    }
}

} // namespace wd
