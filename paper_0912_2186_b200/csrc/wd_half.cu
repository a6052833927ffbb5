// wd_half.cu -- half-precision STORAGE of links and spinors, fp32 arithmetic (PAPER.md:159-167,
// Table 2 row "Half": the paper's fastest kernel row stores its fields in 16 bits).  Reading RH:
//
//   links    every stored real (18, 12 or 8 per link; all |.| <= 1, the two phases of the 8-real format being in units of pi)
//            as IEEE binary16
//   spinors  per site a float32 scale s = max |component| over the site's 24 reals and the 24 ratios component / s
//            (float32 IEEE division) as binary16; a site with s = 0 stores zeros.  value = s * q.
//
// Native layouts (16-byte vectors of 8 halves; same block-of-32-sites structure as wd_layout.cuh):
//   spinor  [rhs][block][vector c = 0..2][lane]  (reals 8c .. 8c+7 of [spin][colour][re,im]), then after ALL right-hand
//           sides the scales  float[rhs][padded site]                       -> 52 bytes per site and right-hand side
//   links   [block][vector j][lane], the four links of a site together, 4*RECON halves = RECON/2 vectors per site
//
// Kernel: one thread per site (the general path of wd_dslash_site.cu with half loads and a requantising store), any
// extents >= 1, projector sign as a template parameter (D and D^dagger), right-hand sides along gridDim.y.  Per site it
// moves 2 * 52 + 8 * RECON bytes (200 B with 12-real links against 384 B in fp32): the same arithmetic at about half the
// traffic.  The canonical side of wd_pack_spinor / wd_unpack_spinor / wd_load_gauge is float32 for this precision.
#include <cuda_fp16.h>
#include "wd_half.cuh"
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_math.cuh"

namespace wd {

namespace {

constexpr int HT = 128; // threads per CTA


// half spinor of `site` of one right-hand side -> 24 floats (value = scale * ratio)
__device__ __forceinline__ void load_spinor_h(const uint4 *__restrict__ field, const float *__restrict__ scale, long long site,
                                              float (&p)[24])
{
    const uint4 *q = field + (site >> 5) * (3 * BLK) + (site & (BLK - 1));
    const float s = __ldg(scale + site);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const uint4 v = __ldg(q + c * BLK);
        unpack8(v, &p[8 * c]);
    }
#pragma unroll
    for (int i = 0; i < 24; ++i) p[i] *= s;
}

// 24 floats -> scale + ratios (reading RH).  EXACT: the ratios are IEEE divisions, the same arithmetic as
// oracle/wd_storage.py:quantise_half_spinor (wd_pack_spinor: what is stored is bit for bit what the oracle holds);
// otherwise (kernel epilogues) one reciprocal and 24 products, which may differ by one float ulp before the binary16 rounding.
template <bool EXACT>
__device__ __forceinline__ void store_spinor_h(uint4 *__restrict__ field, float *__restrict__ scale, long long site, const float (&p)[24])
{
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 24; ++i) s = fmaxf(s, fabsf(p[i]));
    float r[24];
    const float rs = s > 0.f ? __frcp_rn(s) : 0.f;
#pragma unroll
    for (int i = 0; i < 24; ++i) r[i] = EXACT ? (s > 0.f ? __fdiv_rn(p[i], s) : 0.f) : p[i] * rs;
    uint4 *q = field + (site >> 5) * (3 * BLK) + (site & (BLK - 1));
#pragma unroll
    for (int c = 0; c < 3; ++c) q[c * BLK] = pack8(&r[8 * c]);
    scale[site] = s;
}

template <int MU, int RECON> __device__ __forceinline__ void load_link_h(const uint4 *__restrict__ links, long long site, float (&u)[18])
{
    constexpr int NVEC = RECON / 2; // 4 * RECON halves / 8
    constexpr int first = (MU * RECON) / 8, last = (MU * RECON + RECON - 1) / 8, skip = MU * RECON - first * 8;
    const uint4 *q = links + (site >> 5) * (NVEC * BLK) + (site & (BLK - 1));
    float tmp[(last - first + 1) * 8];
#pragma unroll
    for (int j = first; j <= last; ++j) {
        const uint4 v = __ldg(q + j * BLK);
        unpack8(v, &tmp[(j - first) * 8]);
    }
#pragma unroll
    for (int i = 0; i < RECON; ++i) u[i] = tmp[skip + i];
    if (RECON == 12) reconstruct_row2(u);
    if (RECON == 8) reconstruct_from8(u);
}

template <int MU, int SGN, int RECON>
__device__ __forceinline__ void hop_pair_h(float (&acc)[24], const uint4 *in, const float *scale, const uint4 *links, long long site,
                                           long long sf, long long sb)
{
    float u[18], p[24];
    load_link_h<MU, RECON>(links, site, u);
    load_spinor_h(in, scale, sf, p);
    hop_forward_s<MU, SGN>(acc, u, p);
    load_link_h<MU, RECON>(links, sb, u);
    load_spinor_h(in, scale, sb, p);
    hop_backward_s<MU, SGN>(acc, u, p);
}

template <int RECON, int SGN>
__global__ void __launch_bounds__(HT)
dslash_half_kernel(uint4 *__restrict__ out, float *__restrict__ out_scale, const uint4 *__restrict__ in,
                   const float *__restrict__ in_scale, const uint4 *__restrict__ links, int Lx, int Ly, int Lz, int Lt, long long V,
                   float cdiag)
{
    const long long site = (long long)blockIdx.x * HT + threadIdx.x;
    if (site >= V) return;
    const long long Vp = padded_volume(V);
    const long long rhs = blockIdx.y;
    in += rhs * Vp * 3;
    out += rhs * Vp * 3;
    in_scale += rhs * Vp;
    out_scale += rhs * Vp;
    long long rem = site;
    const int x = (int)(rem % Lx); rem /= Lx;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const int t = (int)(rem / Lz);
    const long long sy = Lx, sz = (long long)Lx * Ly, st = (long long)Lx * Ly * Lz;
    const long long xf = site + (x + 1 == Lx ? -(Lx - 1) : 1), xb = site + (x == 0 ? (Lx - 1) : -1);
    const long long yf = site + (y + 1 == Ly ? -(Ly - 1) * sy : sy), yb = site + (y == 0 ? (Ly - 1) * sy : -sy);
    const long long zf = site + (z + 1 == Lz ? -(Lz - 1) * sz : sz), zb = site + (z == 0 ? (Lz - 1) * sz : -sz);
    const long long tf = site + (t + 1 == Lt ? -(Lt - 1) * st : st), tb = site + (t == 0 ? (Lt - 1) * st : -st);
    float acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0.f;
    hop_pair_h<0, SGN, RECON>(acc, in, in_scale, links, site, xf, xb);
    hop_pair_h<1, SGN, RECON>(acc, in, in_scale, links, site, yf, yb);
    hop_pair_h<2, SGN, RECON>(acc, in, in_scale, links, site, zf, zb);
    hop_pair_h<3, SGN, RECON>(acc, in, in_scale, links, site, tf, tb);
    float p[24];
    load_spinor_h(in, in_scale, site, p);
#pragma unroll
    for (int i = 0; i < 24; ++i) p[i] = fmaf(cdiag, p[i], -0.5f * acc[i]);
    store_spinor_h<false>(out, out_scale, site, p);
}

// canonical float32 [rhs][site][24] <-> native half
template <bool TO_NATIVE>
__global__ void spinor_half_kernel(uint4 *native, float *scale, float *canon, long long V)
{
    const long long site = (long long)blockIdx.x * HT + threadIdx.x;
    if (site >= V) return;
    const long long Vp = padded_volume(V), rhs = blockIdx.y;
    native += rhs * Vp * 3;
    scale += rhs * Vp;
    float *c = canon + (rhs * V + site) * 24;
    float p[24];
    if (TO_NATIVE) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const float4 v = reinterpret_cast<const float4 *>(c)[i];
            p[4 * i] = v.x; p[4 * i + 1] = v.y; p[4 * i + 2] = v.z; p[4 * i + 3] = v.w;
        }
        store_spinor_h<true>(native, scale, site, p);
    } else {
        load_spinor_h(native, scale, site, p);
#pragma unroll
        for (int i = 0; i < 6; ++i) reinterpret_cast<float4 *>(c)[i] = make_float4(p[4 * i], p[4 * i + 1], p[4 * i + 2], p[4 * i + 3]);
    }
}

// canonical float32 U[mu][site][18] -> native half links (recon 8: the parametrisation of wd_math.cuh, angles in double)
template <int RECON> __global__ void pack_links_half_kernel(uint4 *__restrict__ dst, const float *__restrict__ src, long long V, int *bad)
{
    const long long site = (long long)blockIdx.x * HT + threadIdx.x;
    if (site >= V) return;
    constexpr int NVEC = RECON / 2;
    float r[4 * RECON];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const float *p = src + ((long long)mu * V + site) * 18;
        if (RECON == 8) {
            r[mu * 8 + 0] = p[2]; r[mu * 8 + 1] = p[3]; r[mu * 8 + 2] = p[4]; r[mu * 8 + 3] = p[5];
            r[mu * 8 + 4] = p[6]; r[mu * 8 + 5] = p[7];
            r[mu * 8 + 6] = (float)(atan2((double)p[1], (double)p[0]) / 3.14159265358979323846);
            r[mu * 8 + 7] = (float)(atan2((double)p[13], (double)p[12]) / 3.14159265358979323846);
            if (p[2] == 0.f && p[3] == 0.f && p[4] == 0.f && p[5] == 0.f && bad) atomicOr(bad, 1);
        } else {
#pragma unroll
            for (int i = 0; i < RECON; ++i) r[mu * RECON + i] = p[i];
        }
    }
    uint4 *q = dst + (site >> 5) * (NVEC * BLK) + (site & (BLK - 1));
#pragma unroll
    for (int j = 0; j < NVEC; ++j) q[j * BLK] = pack8(&r[8 * j]);
}

template <int RECON> cudaError_t launch_half_r(const ApplyArgs &a)
{
    const long long Vp = padded_volume(a.V);
    const long long nb = (a.V + HT - 1) / HT;
    if (nb > 0x7fffffffLL || a.nrhs > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)nb, (unsigned)a.nrhs);
    uint4 *out = (uint4 *)a.out;
    const uint4 *in = (const uint4 *)a.in;
    float *out_scale = (float *)((char *)a.out + (size_t)a.nrhs * Vp * 48);
    const float *in_scale = (const float *)((const char *)a.in + (size_t)a.nrhs * Vp * 48);
    const float cdiag = (float)(4.0 + a.mass);
    if (a.dagger)
        dslash_half_kernel<RECON, +1><<<grid, HT, 0, a.stream>>>(out, out_scale, in, in_scale, (const uint4 *)a.links, a.dims[0],
                                                                  a.dims[1], a.dims[2], a.dims[3], a.V, cdiag);
    else
        dslash_half_kernel<RECON, -1><<<grid, HT, 0, a.stream>>>(out, out_scale, in, in_scale, (const uint4 *)a.links, a.dims[0],
                                                                  a.dims[1], a.dims[2], a.dims[3], a.V, cdiag);
    count_launch();
    return cudaGetLastError();
}

// ---- red/black (even-odd) blocks in half storage: the kernel of wd_dslash_eo.cu with half loads and a requantising
// store.  Half fields of one parity: the layout above over the checkerboard index cb = lex / 2 (Vh = V / 2 sites); links:
// the parity-ordered copy of the half link records (wd_gauge::links_eo).
//     out_p = alpha * x_p + beta * sum_mu [ (1-g_mu) U_mu(x) in_q(x+mu) + (1+g_mu) U_mu(x-mu)^dag in_q(x-mu) ]
constexpr int EH = 128;

template <int RECON, int SGN>
__global__ void __launch_bounds__(EH)
dslash_eo_half_kernel(uint4 *__restrict__ out, float *__restrict__ out_scale, const uint4 *__restrict__ in,
                      const float *__restrict__ in_scale, const uint4 *__restrict__ xin, const float *__restrict__ xin_scale,
                      const uint4 *__restrict__ links_p, const uint4 *__restrict__ links_q, int Lx, int Ly, int Lz, int Lt,
                      long long Vh, float alpha, float beta, int parity)
{
    const long long cb = (long long)blockIdx.x * EH + threadIdx.x;
    if (cb >= Vh) return;
    const long long Vhp = padded_volume(Vh), rhs = blockIdx.y;
    in += rhs * Vhp * 3;
    out += rhs * Vhp * 3;
    in_scale += rhs * Vhp;
    out_scale += rhs * Vhp;
    const int Lxh = Lx / 2;
    long long rem = cb;
    const int xh = (int)(rem % Lxh); rem /= Lxh;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const int t = (int)(rem / Lz);
    const int x = 2 * xh + ((y + z + t + parity) & 1);
    const long long sy = Lx, sz = (long long)Lx * Ly, st = (long long)Lx * Ly * Lz;
    const long long site = x + sy * y + sz * z + st * t;
    const long long xf = site + (x + 1 == Lx ? -(long long)(Lx - 1) : 1), xb = site + (x == 0 ? (long long)(Lx - 1) : -1);
    const long long yf = site + (y + 1 == Ly ? -(Ly - 1) * sy : sy), yb = site + (y == 0 ? (Ly - 1) * sy : -sy);
    const long long zf = site + (z + 1 == Lz ? -(Lz - 1) * sz : sz), zb = site + (z == 0 ? (Lz - 1) * sz : -sz);
    const long long tf = site + (t + 1 == Lt ? -(Lt - 1) * st : st), tb = site + (t == 0 ? (Lt - 1) * st : -st);
    float acc[24], u[18], p[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0.f;
    load_link_h<0, RECON>(links_p, cb, u);      load_spinor_h(in, in_scale, xf >> 1, p); hop_forward_s<0, SGN>(acc, u, p);
    load_link_h<0, RECON>(links_q, xb >> 1, u); load_spinor_h(in, in_scale, xb >> 1, p); hop_backward_s<0, SGN>(acc, u, p);
    load_link_h<1, RECON>(links_p, cb, u);      load_spinor_h(in, in_scale, yf >> 1, p); hop_forward_s<1, SGN>(acc, u, p);
    load_link_h<1, RECON>(links_q, yb >> 1, u); load_spinor_h(in, in_scale, yb >> 1, p); hop_backward_s<1, SGN>(acc, u, p);
    load_link_h<2, RECON>(links_p, cb, u);      load_spinor_h(in, in_scale, zf >> 1, p); hop_forward_s<2, SGN>(acc, u, p);
    load_link_h<2, RECON>(links_q, zb >> 1, u); load_spinor_h(in, in_scale, zb >> 1, p); hop_backward_s<2, SGN>(acc, u, p);
    load_link_h<3, RECON>(links_p, cb, u);      load_spinor_h(in, in_scale, tf >> 1, p); hop_forward_s<3, SGN>(acc, u, p);
    load_link_h<3, RECON>(links_q, tb >> 1, u); load_spinor_h(in, in_scale, tb >> 1, p); hop_backward_s<3, SGN>(acc, u, p);
    if (xin) {
        load_spinor_h(xin + rhs * Vhp * 3, xin_scale + rhs * Vhp, cb, p);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = fmaf(alpha, p[i], beta * acc[i]);
    } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = beta * acc[i];
    }
    store_spinor_h<false>(out, out_scale, cb, acc);
}

// canonical float32 full-lattice field <-> native half-storage field of one parity
template <bool TO_NATIVE>
__global__ void parity_half_kernel(uint4 *native, float *scale, float *canon, int Lx, int Ly, int Lz, long long V, int parity)
{
    const long long Vh = V / 2, Vhp = padded_volume(Vh), rhs = blockIdx.y;
    const long long cb = (long long)blockIdx.x * EH + threadIdx.x;
    if (cb >= Vh) return;
    const int Lxh = Lx / 2;
    long long rem = cb;
    const int xh = (int)(rem % Lxh); rem /= Lxh;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const long long t = rem / Lz;
    const int x = 2 * xh + (int)((y + z + t + parity) & 1);
    const long long site = x + (long long)Lx * (y + (long long)Ly * (z + (long long)Lz * t));
    native += rhs * Vhp * 3;
    scale += rhs * Vhp;
    float *c = canon + (rhs * V + site) * 24;
    float p[24];
    if (TO_NATIVE) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const float4 v = reinterpret_cast<const float4 *>(c)[i];
            p[4 * i] = v.x; p[4 * i + 1] = v.y; p[4 * i + 2] = v.z; p[4 * i + 3] = v.w;
        }
        store_spinor_h<true>(native, scale, cb, p);
    } else {
        load_spinor_h(native, scale, cb, p);
#pragma unroll
        for (int i = 0; i < 6; ++i) reinterpret_cast<float4 *>(c)[i] = make_float4(p[4 * i], p[4 * i + 1], p[4 * i + 2], p[4 * i + 3]);
    }
}

template <int RECON>
cudaError_t launch_eo_half_r(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger)
{
    const long long Vh = a.V / 2, Vhp = padded_volume(Vh);
    const long long nb = (Vh + EH - 1) / EH;
    if (nb > 0x7fffffffLL || a.nrhs > 65535) return cudaErrorInvalidConfiguration;
    if (!a.links_eo) return cudaErrorInvalidValue;
    dim3 grid((unsigned)nb, (unsigned)a.nrhs);
    const size_t sc_off = (size_t)a.nrhs * Vhp * 48; // the scales follow the vectors of all right-hand sides
    const char *le = (const char *)a.links_eo;
    const size_t half = eo_links_half_bytes(a.V, 16, a.recon);
    auto kern = dagger ? dslash_eo_half_kernel<RECON, +1> : dslash_eo_half_kernel<RECON, -1>;
    kern<<<grid, EH, 0, a.stream>>>((uint4 *)a.out, (float *)((char *)a.out + sc_off), (const uint4 *)a.in,
                                    (const float *)((const char *)a.in + sc_off), (const uint4 *)xin,
                                    xin ? (const float *)((const char *)xin + sc_off) : nullptr, (const uint4 *)(le + parity * half),
                                    (const uint4 *)(le + (1 - parity) * half), a.dims[0], a.dims[1], a.dims[2], a.dims[3], Vh,
                                    (float)alpha, (float)beta, parity);
    count_launch();
    return cudaGetLastError();
}

} // namespace

cudaError_t launch_eo_half(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger)
{
    return a.recon == 18 ? launch_eo_half_r<18>(a, xin, alpha, beta, parity, dagger)
           : a.recon == 12 ? launch_eo_half_r<12>(a, xin, alpha, beta, parity, dagger)
                           : launch_eo_half_r<8>(a, xin, alpha, beta, parity, dagger);
}

cudaError_t launch_parity_copy_half(void *native, void *canon, const int dims[4], long long V, int nrhs, int parity, bool to_native,
                                    cudaStream_t s)
{
    const long long Vh = V / 2;
    if (Vh <= 0 || nrhs <= 0) return cudaSuccess;
    if (nrhs > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)((Vh + EH - 1) / EH), (unsigned)nrhs);
    float *scale = (float *)((char *)native + (size_t)nrhs * padded_volume(Vh) * 48);
    if (to_native) parity_half_kernel<true><<<grid, EH, 0, s>>>((uint4 *)native, scale, (float *)canon, dims[0], dims[1], dims[2], V, parity);
    else parity_half_kernel<false><<<grid, EH, 0, s>>>((uint4 *)native, scale, (float *)canon, dims[0], dims[1], dims[2], V, parity);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_half(const ApplyArgs &a)
{
    return a.recon == 18 ? launch_half_r<18>(a) : a.recon == 12 ? launch_half_r<12>(a) : launch_half_r<8>(a);
}

cudaError_t launch_spinor_half(void *native, void *canonical, long long V, int nrhs, bool to_native, cudaStream_t s)
{
    if (V <= 0) return cudaSuccess;
    const long long nb = (V + HT - 1) / HT;
    if (nb > 0x7fffffffLL || nrhs > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)nb, (unsigned)nrhs);
    float *scale = (float *)((char *)native + (size_t)nrhs * padded_volume(V) * 48);
    if (to_native) {
        // pad sites of the last block: defined values (zeros), never read by the kernels
        spinor_half_kernel<true><<<grid, HT, 0, s>>>((uint4 *)native, scale, (float *)canonical, V);
    } else
        spinor_half_kernel<false><<<grid, HT, 0, s>>>((uint4 *)native, scale, (float *)canonical, V);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pack_links_half(void *native, const void *canonical, long long V, int recon, cudaStream_t s, int *bad_dev)
{
    if (V <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((V + HT - 1) / HT);
    if (recon == 18) pack_links_half_kernel<18><<<grid, HT, 0, s>>>((uint4 *)native, (const float *)canonical, V, bad_dev);
    else if (recon == 12) pack_links_half_kernel<12><<<grid, HT, 0, s>>>((uint4 *)native, (const float *)canonical, V, bad_dev);
    else pack_links_half_kernel<8><<<grid, HT, 0, s>>>((uint4 *)native, (const float *)canonical, V, bad_dev);
    count_launch();
    return cudaGetLastError();
}

} // namespace wd
