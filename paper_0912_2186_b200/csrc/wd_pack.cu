// wd_pack.cu -- canonical <-> native layout conversion (pure data movement, no arithmetic).
// SURVEY.md section 8(a) step a0; canonical layouts are DESIGN.md readings S5/S6.
#include "wd_internal.h"
#include "wd_layout.cuh"

namespace wd {

constexpr int PACK_SITES = 128; // sites per CTA; also the CTA size

// canonical [rhs][site][NCH vectors]  <->  native [rhs][block][vector][lane] (wd_layout.cuh);
// transposed through shared memory so that both the global reads and the global writes are
// contiguous 16-byte-per-lane.  Pad sites of the last native block are left untouched.
template <typename Vec, int NCH, bool TO_NATIVE>
__global__ void __launch_bounds__(PACK_SITES) spinor_transpose_kernel(Vec *__restrict__ dst, const Vec *__restrict__ src,
                                                                     long long V, long long first, long long end)
{
    __shared__ Vec tile[NCH][PACK_SITES + 1];
    const long long site0 = first + (long long)blockIdx.x * PACK_SITES; // first is a multiple of PACK_SITES
    const int rhs = blockIdx.y;
    const int tid = threadIdx.x;
    const long long nsite = min((long long)PACK_SITES, end - site0);
    const Vec *canon_src = src + ((long long)rhs * V + site0) * NCH;
    Vec *canon_dst = dst + ((long long)rhs * V + site0) * NCH;
    // native vector 0 of site site0 + tid (site0 is a multiple of 32)
    const long long nat = (long long)rhs * padded_volume(V) * NCH + ((site0 + tid) >> 5) * (NCH * BLK) + (tid & (BLK - 1));
    if (TO_NATIVE) {
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
            const int idx = i * PACK_SITES + tid;
            if (idx < nsite * NCH) tile[idx % NCH][idx / NCH] = canon_src[idx];
        }
        __syncthreads();
        if (tid < nsite) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) dst[nat + c * BLK] = tile[c][tid];
        }
    } else {
        if (tid < nsite) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) tile[c][tid] = src[nat + c * BLK];
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
            const int idx = i * PACK_SITES + tid;
            if (idx < nsite * NCH) canon_dst[idx] = tile[idx % NCH][idx / NCH];
        }
    }
}

template <bool TO_NATIVE>
static cudaError_t transpose_spinor(void *dst, const void *src, long long V, int nrhs, int precision, cudaStream_t s,
                                    long long site0, long long nsites)
{
    if (nsites < 0) nsites = V - site0;
    if (V <= 0 || nrhs <= 0 || nsites <= 0) return cudaSuccess;
    if (site0 % PACK_SITES || site0 + nsites > V) return cudaErrorInvalidValue;
    const long long end = site0 + nsites;
    dim3 grid((unsigned)((nsites + PACK_SITES - 1) / PACK_SITES), (unsigned)nrhs);
    if (precision == 32)
        spinor_transpose_kernel<float4, 6, TO_NATIVE><<<grid, PACK_SITES, 0, s>>>((float4 *)dst, (const float4 *)src, V, site0, end);
    else
        spinor_transpose_kernel<double2, 12, TO_NATIVE><<<grid, PACK_SITES, 0, s>>>((double2 *)dst, (const double2 *)src, V, site0, end);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pack_spinor(void *native, const void *canonical, long long V, int nrhs, int precision, cudaStream_t s,
                               long long site0, long long nsites)
{
    return transpose_spinor<true>(native, canonical, V, nrhs, precision, s, site0, nsites);
}

cudaError_t launch_unpack_spinor(void *canonical, const void *native, long long V, int nrhs, int precision,
                                 cudaStream_t s, long long site0, long long nsites)
{
    return transpose_spinor<false>(canonical, native, V, nrhs, precision, s, site0, nsites);
}

// canonical U[mu][site][a][b][re,im] -> native [block][vector][lane], the four links of a site
// together (wd_layout.cuh); recon 12 keeps rows a = 0,1 of every link.
// recon 8 stores (Re a2, Im a2, Re a3, Im a3, Re b1, Im b1, arg(a1)/pi, arg(c1)/pi) of the rows a, b, c (wd_math.cuh:
// reconstruct_from8), the two angles formed in double and rounded once; *bad is set if some link has a2 = a3 = 0
// (not representable).
template <typename T, int RECON>
__global__ void pack_links_kernel(T *__restrict__ dst, const T *__restrict__ src, long long V, int *bad)
{
    using L = LinkLayout<T, RECON>;
    const long long site = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= V) return;
    typename L::Vec *q = reinterpret_cast<typename L::Vec *>(dst) + (site >> 5) * (L::NVEC * BLK) + (site & (BLK - 1));
    T r[4 * RECON];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const T *p = src + ((long long)mu * V + site) * 18;
        if (RECON == 8) {
            r[mu * RECON + 0] = p[2]; r[mu * RECON + 1] = p[3]; // a2
            r[mu * RECON + 2] = p[4]; r[mu * RECON + 3] = p[5]; // a3
            r[mu * RECON + 4] = p[6]; r[mu * RECON + 5] = p[7]; // b1
            r[mu * RECON + 6] = (T)(atan2((double)p[1], (double)p[0]) / 3.14159265358979323846);   // arg(a1) / pi
            r[mu * RECON + 7] = (T)(atan2((double)p[13], (double)p[12]) / 3.14159265358979323846); // arg(c1) / pi
            if (p[2] == (T)0 && p[3] == (T)0 && p[4] == (T)0 && p[5] == (T)0 && bad) atomicOr(bad, 1);
        } else {
#pragma unroll
            for (int i = 0; i < RECON; ++i) r[mu * RECON + i] = p[i];
        }
    }
#pragma unroll
    for (int j = 0; j < L::NVEC; ++j) {
        typename L::Vec v;
        pack(v, &r[j * L::CR]);
        q[j * BLK] = v;
    }
}

size_t native_link_bytes(long long V, int precision, int recon)
{
    return (size_t)4 * (size_t)padded_volume(V) * (size_t)recon * (precision == 16 ? 2 : precision == 32 ? 4 : 8);
}

cudaError_t launch_pack_links(void *native, const void *canonical, long long V, int precision, int recon, cudaStream_t s,
                              int *bad_dev)
{
    if (V <= 0) return cudaSuccess;
    dim3 grid((unsigned)((V + 127) / 128));
    if (precision == 32 && recon == 18)
        pack_links_kernel<float, 18><<<grid, 128, 0, s>>>((float *)native, (const float *)canonical, V, bad_dev);
    else if (precision == 32 && recon == 12)
        pack_links_kernel<float, 12><<<grid, 128, 0, s>>>((float *)native, (const float *)canonical, V, bad_dev);
    else if (precision == 32)
        pack_links_kernel<float, 8><<<grid, 128, 0, s>>>((float *)native, (const float *)canonical, V, bad_dev);
    else if (recon == 18)
        pack_links_kernel<double, 18><<<grid, 128, 0, s>>>((double *)native, (const double *)canonical, V, bad_dev);
    else if (recon == 12)
        pack_links_kernel<double, 12><<<grid, 128, 0, s>>>((double *)native, (const double *)canonical, V, bad_dev);
    else
        pack_links_kernel<double, 8><<<grid, 128, 0, s>>>((double *)native, (const double *)canonical, V, bad_dev);
    count_launch();
    return cudaGetLastError();
}

// flag |= 1 if some U_t(x, t) with t < Lt-1 differs from the unit matrix by more than tol (native links)
template <typename T, int RECON>
__global__ void check_temporal_gauge_kernel(const T *__restrict__ links, long long S3, long long V, double tol, int *flag)
{
    using L = LinkLayout<T, RECON>;
    const long long site = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= V - S3) return; // the last slice may hold anything
    const typename L::Vec *q = reinterpret_cast<const typename L::Vec *>(links) + (site >> 5) * (L::NVEC * BLK) + (site & (BLK - 1));
    bool bad = false;
    for (int i = 0; i < RECON; ++i) { // reals of link 3: [3*RECON, 4*RECON)
        const int r = 3 * RECON + i;
        T v[L::CR];
        unpack(q[(r / L::CR) * BLK], v);
        const int elem = i / 2, a = elem / 3, b = elem % 3;
        const double want = (i % 2 == 0 && a == b) ? 1.0 : 0.0;
        if (!(fabs((double)v[r % L::CR] - want) <= tol)) bad = true; // (NaN fails too)
    }
    if (bad) atomicOr(flag, 1);
}

cudaError_t launch_check_temporal_gauge(const void *links, const int dims[4], long long V, int precision, int recon, int *flag_dev,
                                        cudaStream_t s)
{
    const long long S3 = (long long)dims[0] * dims[1] * dims[2];
    if (V <= S3) return cudaSuccess;
    const unsigned grid = (unsigned)((V - S3 + 127) / 128);
    const double tol = precision == 32 ? 1e-6 : 1e-12;
    if (precision == 32 && recon == 18) check_temporal_gauge_kernel<float, 18><<<grid, 128, 0, s>>>((const float *)links, S3, V, tol, flag_dev);
    else if (precision == 32) check_temporal_gauge_kernel<float, 12><<<grid, 128, 0, s>>>((const float *)links, S3, V, tol, flag_dev);
    else if (recon == 18) check_temporal_gauge_kernel<double, 18><<<grid, 128, 0, s>>>((const double *)links, S3, V, tol, flag_dev);
    else check_temporal_gauge_kernel<double, 12><<<grid, 128, 0, s>>>((const double *)links, S3, V, tol, flag_dev);
    count_launch();
    return cudaGetLastError();
}

} // namespace wd
