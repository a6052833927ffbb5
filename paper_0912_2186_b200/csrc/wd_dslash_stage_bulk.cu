// wd_dslash_stage_bulk.cu -- bulk-copy member of WD_KERNEL_STAGE for Lx = 32 (fp32 and fp64, D and D^dagger, 18/12/8-real links).
//
// Same decomposition, same arithmetic and the same staging schedule as dslash_stage_kernel (wd_dslash_stage.cu: a CTA owns a
// 32 x 2 x 2 tile of a time slice and marches along t; groups P = own spinor of slice t+1, A = links x,y + y face, B = links z,t
// + z face, each refilled for slice t+1 right after slice t consumed it), but the copies are not issued per thread.  With
// Lx = 32 a warp is one x-row of the tile = one 32-site block of the native layout, so everything a warp stages per slice is
// a handful of CONTIGUOUS pieces of global memory: its spinor row (NCH x 512 B), the two halves of its link record, the
// out-of-tile y and z neighbour rows and, for the rows with yy = 0 / zz = 0, the vectors of the neighbour row's link record that
// hold U_y / U_z.  Lane 0 of the warp copies each piece with ONE cp.async.bulk (SASS UBLKCP) into the warp's own part of
// shared memory and the warp waits for a group on an mbarrier: 7 bulk copies per warp and slice replace 40 LDGSTS.128 per
// thread and slice (36 % of the LSU data-pipe wavefronts of the per-thread kernel, which is its second limit under the power
// cap: DESIGN.md section 6.3) and their address arithmetic.
// Hazards: a refill (async proxy) of a piece the warp has just read (generic proxy) needs __syncwarp + fence.proxy.async first
// (measured in wd_dslash_rloop.cu: without the fence a refill can overtake the reads); the slice buffer is also read by the
// other warps of the CTA, whose reads all precede the CTA barrier (B) that ends the previous slice.
// Measured on 32^3 x 64, fp32, 18-real links, same box, 100-apply loop (profiles/r02_ncu.md section 11): per-thread cp.async
// 174-176 us, this member 181-185 us (with the hand-over written as an mbarrier arrive by every lane + wait by lane 0 instead
// of __syncwarp + proxy fence: 189 us); fp64 equal (410-412 us).  Bit-identical results.  NOT the default (stage_bulk = 1 selects it).
#include <cstdio>
#include <cstdlib>
#define WD_USE_F32X2 // packed FFMA2 SU(3) products (wd_math.cuh)
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_bulk.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

namespace {

template <int NV, typename Vec, typename T>
__device__ __forceinline__ void ldsv(const Vec *row, int lane, T *r) // NV vectors of a [vec][32 lanes] record
{
    constexpr int CR = 16 / sizeof(T);
#pragma unroll
    for (int c = 0; c < NV; ++c) unpack(row[c * 32 + lane], &r[c * CR]);
}

template <int MU, int RECON, typename T> struct LinkPiece { // vectors of a site's link record that hold link MU
    static constexpr int CR = 16 / sizeof(T);
    static constexpr int first = (MU * RECON) / CR, last = (MU * RECON + RECON - 1) / CR, n = last - first + 1;
    static constexpr int skip = MU * RECON - first * CR;
};

// link MU out of a staged [vec][32] record whose first staged vector is vector `first0` of the site's record
template <int MU, int RECON, typename Vec, typename T>
__device__ __forceinline__ void lds_link(const Vec *rec, int first0, int lane, T (&u)[18])
{
    using LP = LinkPiece<MU, RECON, T>;
    T tmp[LP::n * LP::CR];
    ldsv<LP::n>(rec + (LP::first - first0) * 32, lane, tmp);
#pragma unroll
    for (int i = 0; i < RECON; ++i) u[i] = tmp[LP::skip + i];
    if (RECON == 12) reconstruct_row2(u);
    if (RECON == 8) reconstruct_from8(u);
}

template <typename T>
__device__ __forceinline__ void shfl12(T (&dst)[12], const T (&src)[12], int src_lane)
{
#pragma unroll
    for (int i = 0; i < 12; ++i) dst[i] = __shfl_sync(0xffffffffu, src[i], src_lane);
}

} // namespace

// shared memory of one CTA: 16-byte vectors, then 4 warps x 3 mbarriers
template <typename T, int RECON> constexpr int stage_bulk_vecs()
{
    using SL = SpinorLayout<T>;
    return 128 * (2 * SL::NCH + 2 * (SL::NCH / 2) + LinkLayout<T, RECON>::NVEC + 2 * SL::NCH) +
           64 * (LinkPiece<1, RECON, T>::n + LinkPiece<2, RECON, T>::n);
}
template <typename T, int RECON> constexpr size_t stage_bulk_bytes() { return (size_t)stage_bulk_vecs<T, RECON>() * 16 + 12 * 8; }

// blockDim.x = 128 (tile 32 x 2 x 2); block order as in dslash_stage_kernel
template <typename T, int RECON, int SGN>
__global__ void __launch_bounds__(128, 1)
dslash_stage_bulk_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ links, int Ly, int Lz, int Lt,
                         long long V, T cdiag, int nrhs, int nchunk, int tgauge, int patch)
{
    constexpr int Lx = 32, ty = 2, tz = 2, nt = 128;
    constexpr int FS = SGN, BS = -SGN;
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH, CR = SL::CR, HCH = NCH / 2;
    constexpr int NVEC = LinkLayout<T, RECON>::NVEC;
    using FY = LinkPiece<1, RECON, T>;
    using FZ = LinkPiece<2, RECON, T>;
    constexpr int A_END = FY::last + 1; // links x,y = vectors [0, A_END), z,t = [A_END, NVEC)
    constexpr unsigned VB = 512;        // bytes of one vector of a 32-site row
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int yy = w & 1, zz = w >> 1; // warp-uniform
    Vec *const plane0 = reinterpret_cast<Vec *>(smem_raw); // two slice buffers [4 rows][NCH][32]
    constexpr int plane_sz = 4 * NCH * 32;
    Vec *const xchg_y = plane0 + 2 * plane_sz;              // [HCH][128]  U_y^dag P psi, for the site at y+1
    Vec *const xchg_z = xchg_y + HCH * nt;                  // [HCH][128]
    Vec *const lnk_w = xchg_z + HCH * nt + w * NVEC * 32;   // this row's link record [NVEC][32]
    Vec *const fy_w = xchg_z + HCH * nt + 4 * NVEC * 32 + w * NCH * 32; // out-of-tile y neighbour row
    Vec *const fz_w = fy_w + 4 * NCH * 32;                  // out-of-tile z neighbour row
    Vec *const fl0 = xchg_z + HCH * nt + 4 * NVEC * 32 + 8 * NCH * 32;
    Vec *const fly_w = fl0 + zz * FY::n * 32;               // U_y vectors of the row below (rows with yy == 0)
    Vec *const flz_w = fl0 + 2 * FY::n * 32 + yy * FZ::n * 32; // U_z vectors of the row below in z (rows with zz == 0)
    unsigned long long *const mb = reinterpret_cast<unsigned long long *>(fl0 + 2 * FY::n * 32 + 2 * FZ::n * 32) + w * 3;
    unsigned long long *const mbP = mb, *const mbA = mb + 1, *const mbB = mb + 2;

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    int col, rhs, k;
    if (patch > 0) {
        const int per_chunk = ncol * nrhs;
        k = blockIdx.x / per_chunk;
        const int r = blockIdx.x - k * per_chunk;
        const int per_patch = patch * patch * nrhs;
        const int p = r / per_patch, ww = r - p * per_patch;
        rhs = ww % nrhs;
        const int c = ww / nrhs;
        const int npy = ncy / patch;
        col = (p % npy) * patch + c % patch + ncy * ((p / npy) * patch + c / patch);
    } else {
        col = blockIdx.x % ncol;
        const int kg = blockIdx.x / ncol;
        rhs = kg % nrhs;
        k = kg / nrhs;
    }
    in += (long long)rhs * 24 * padded_volume(V);
    out += (long long)rhs * 24 * padded_volume(V);

    const int lane_r = (lane + 1) & 31, lane_l = (lane - 1) & 31;
    const int slot_yb = tid - 32, slot_zb = tid - 64; // exchange slots of the in-tile sites below (yy == 1 / zz == 1 rows)
    const long long S3 = (long long)Lx * Ly * Lz;
    const int t_begin = (int)((long long)Lt * k / nchunk), t_end = (int)((long long)Lt * (k + 1) / nchunk);
    const int cy = col % ncy, cz = col / ncy;
    const int y = cy * ty + yy, z = cz * tz + zz;
    const long long r3 = (long long)Lx * (y + (long long)Ly * z); // first site of this warp's row
    const long long r3_y = yy ? r3 + (y + 1 == Ly ? -(long long)(Ly - 1) * Lx : (long long)Lx)
                              : r3 + (y == 0 ? (long long)(Ly - 1) * Lx : -(long long)Lx);
    const long long r3_z = zz ? r3 + (z + 1 == Lz ? -(long long)(Lz - 1) * Lx * Ly : (long long)Lx * Ly)
                              : r3 + (z == 0 ? (long long)(Lz - 1) * Lx * Ly : -(long long)Lx * Ly);
    // rows as contiguous blocks of the native layout (row start = a multiple of 32 sites)
    const Vec *const row_own = spinor_ptr(static_cast<const T *>(in), r3), *const row_y = spinor_ptr(static_cast<const T *>(in), r3_y),
                     *const row_z = spinor_ptr(static_cast<const T *>(in), r3_z);
    const Vec *const lk_own = link_ptr<T, RECON>(links, r3), *const lk_y = link_ptr<T, RECON>(links, r3_y),
                     *const lk_z = link_ptr<T, RECON>(links, r3_z);
    Vec *const out_own = const_cast<Vec *>(spinor_ptr(static_cast<const T *>(out), r3)) + lane;

    if (t_begin >= t_end) return;
    if (lane == 0) {
        mbar_init(mbP, 1);
        mbar_init(mbA, 1);
        mbar_init(mbB, 1);
        fence_mbar_init();
    }
    __syncwarp();

    auto unit_t = [&](int t) { return tgauge && t != Lt - 1; };
    // ---- bulk copies, lane 0 only ----
    auto copy_P = [&](int buf, long long toff) {
        mbar_expect(mbP, NCH * VB);
        bulk_g2s(plane0 + buf * plane_sz + w * NCH * 32, row_own + toff * NCH, NCH * VB, mbP);
    };
    auto copy_A = [&](long long toff) { // links x,y of the row, the y neighbour row, U_y of the row below
        mbar_expect(mbA, (A_END + NCH + (yy ? 0 : FY::n)) * VB);
        bulk_g2s(lnk_w, lk_own + toff * NVEC, A_END * VB, mbA);
        bulk_g2s(fy_w, row_y + toff * NCH, NCH * VB, mbA);
        if (!yy) bulk_g2s(fly_w, lk_y + toff * NVEC + FY::first * 32, FY::n * VB, mbA);
    };
    auto copy_B = [&](long long toff, int t) { // links z,t (z only where U_t = 1), the z neighbour row, U_z of the row below
        const int jend = unit_t(t) ? FZ::last + 1 : NVEC;
        mbar_expect(mbB, (jend - A_END + NCH + (zz ? 0 : FZ::n)) * VB);
        bulk_g2s(lnk_w + A_END * 32, lk_own + toff * NVEC + A_END * 32, (jend - A_END) * VB, mbB);
        bulk_g2s(fz_w, row_z + toff * NCH, NCH * VB, mbB);
        if (!zz) bulk_g2s(flz_w, lk_z + toff * NVEC + FZ::first * 32, FZ::n * VB, mbB);
    };

    T chi_t[12]; // U_t(t-1)^dag P psi(t-1) of this site
    int cur = 0;
    unsigned phP = 0, phA = 0, phB = 0;
    { // ---- start the march at slice t_begin ----
        const long long toff = (long long)t_begin * S3;
        if (lane == 0) {
            copy_P(cur, toff);
            copy_A(toff);
            copy_B(toff, t_begin);
        }
        const int tb = t_begin == 0 ? Lt - 1 : t_begin - 1;
        const long long site_tb = r3 + lane + (long long)tb * S3;
        T u[18], p[24], h[12];
        load_spinor(static_cast<const T *>(in), site_tb, p);
        project<3, BS>(p, h);
        if (unit_t(tb)) {
#pragma unroll
            for (int i = 0; i < 12; ++i) chi_t[i] = h[i];
        } else {
            load_link<3, T, RECON>(links, site_tb, u);
            su3_dag_mul(u, h, chi_t);
        }
        mbar_wait(mbP, phP); // own row of slice t_begin
        phP ^= 1;
    }

    for (int t = t_begin; t < t_end; ++t) {
        const long long toff = (long long)t * S3;
        const int tn = t + 1 == Lt ? 0 : t + 1;
        const long long toff_n = (long long)tn * S3;
        const bool more = (t + 1 < t_end);
        // P: own row of slice t+1 -> the other slice buffer; every read of its old content (slice t-1, by any warp)
        // precedes barrier (B) of the previous slice
        if (lane == 0) {
            fence_proxy_async();
            copy_P(cur ^ 1, toff_n);
        }
        mbar_wait(mbA, phA); // group A of slice t
        phA ^= 1;
        __syncthreads(); // (A) every warp has seen its own row of slice t land

        const Vec *const pl = plane0 + cur * plane_sz;
        T acc[24], psi[24], u[18];
        ldsv<NCH>(pl + w * NCH * 32, lane, psi);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = (T)0;
        reconstruct_add<3, BS>(acc, chi_t);

        // ---- x: both hops through warp shuffles ----
        lds_link<0, RECON>(lnk_w, 0, lane, u);
        {
            T h[12], g[12], chi[12];
            project<0, FS>(psi, h);
            shfl12(g, h, lane_r);
            su3_mul(u, g, chi);
            reconstruct_add<0, FS>(acc, chi);
            project<0, BS>(psi, h);
            su3_dag_mul(u, h, chi);
            shfl12(g, chi, lane_l);
            reconstruct_add<0, BS>(acc, g);
        }
        // ---- y ----
        lds_link<1, RECON>(lnk_w, 0, lane, u);
        {
            T pn[24], h[12], chi[12];
            if (yy) ldsv<NCH>(fy_w, lane, pn);                   // the row above is outside the tile
            else ldsv<NCH>(pl + (w ^ 1) * NCH * 32, lane, pn);
            hop_forward_s<1, SGN>(acc, u, pn);
            project<1, BS>(psi, h);
            su3_dag_mul(u, h, chi);
#pragma unroll
            for (int c = 0; c < HCH; ++c) pack(xchg_y[c * nt + tid], &chi[c * CR]);
            if (!yy) { // the row below is outside the tile: do its backward hop here
                lds_link<1, RECON>(fly_w, FY::first, lane, u);
                ldsv<NCH>(fy_w, lane, pn);
                hop_backward_s<1, SGN>(acc, u, pn);
            }
        }
        __syncwarp();
        if (lane == 0 && more) { // the pieces of group A are free again
            fence_proxy_async();
            copy_A(toff_n);
        }
        mbar_wait(mbB, phB); // group B of slice t
        phB ^= 1;
        // ---- z ----
        lds_link<2, RECON>(lnk_w, 0, lane, u);
        {
            T pn[24], h[12], chi[12];
            if (zz) ldsv<NCH>(fz_w, lane, pn);
            else ldsv<NCH>(pl + (w ^ 2) * NCH * 32, lane, pn);
            hop_forward_s<2, SGN>(acc, u, pn);
            project<2, BS>(psi, h);
            su3_dag_mul(u, h, chi);
#pragma unroll
            for (int c = 0; c < HCH; ++c) pack(xchg_z[c * nt + tid], &chi[c * CR]);
            if (!zz) {
                lds_link<2, RECON>(flz_w, FZ::first, lane, u);
                ldsv<NCH>(fz_w, lane, pn);
                hop_backward_s<2, SGN>(acc, u, pn);
            }
        }
        // ---- t: forward hop now, backward product for the next slice ----
        const bool ut = unit_t(t);
        if (!ut) lds_link<3, RECON>(lnk_w, 0, lane, u);
        mbar_wait(mbP, phP); // own row of slice t+1
        phP ^= 1;
        {
            T pn[24], h[12];
            ldsv<NCH>(plane0 + (cur ^ 1) * plane_sz + w * NCH * 32, lane, pn);
            if (ut) {
                project<3, FS>(pn, h);
                reconstruct_add<3, FS>(acc, h);
                project<3, BS>(psi, chi_t);
            } else {
                hop_forward_s<3, SGN>(acc, u, pn);
                project<3, BS>(psi, h);
                su3_dag_mul(u, h, chi_t);
            }
        }
        __syncwarp();
        if (lane == 0 && more) { // the pieces of group B are free again
            fence_proxy_async();
            copy_B(toff_n, tn);
        }
        __syncthreads(); // (B) exchange buffers complete; nobody reads slice t-1's buffer or this slice's y/z neighbours any more
        if (yy) {
            T chi[12];
#pragma unroll
            for (int c = 0; c < HCH; ++c) unpack(xchg_y[c * nt + slot_yb], &chi[c * CR]);
            reconstruct_add<1, BS>(acc, chi);
        }
        if (zz) {
            T chi[12];
#pragma unroll
            for (int c = 0; c < HCH; ++c) unpack(xchg_z[c * nt + slot_zb], &chi[c * CR]);
            reconstruct_add<2, BS>(acc, chi);
        }
#pragma unroll
        for (int i = 0; i < 24; ++i) psi[i] = fma(cdiag, psi[i], (T)-0.5 * acc[i]);
        {
            Vec *q = out_own + toff * NCH;
#pragma unroll
            for (int c = 0; c < NCH; ++c) pack(q[c * BLK], &psi[c * CR]);
        }
        cur ^= 1;
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
namespace {

template <typename T, int RECON, int SGN> cudaError_t launch_bulk_s(const ApplyArgs &a)
{
    auto kern = dslash_stage_bulk_kernel<T, RECON, SGN>;
    const size_t smem = stage_bulk_bytes<T, RECON>();
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    const int tc = tn.tile_tc >= 1 ? tn.tile_tc : 16; // as dslash_stage_kernel
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (tn.tile_nchunk >= 1 && tn.tile_nchunk <= a.dims[3]) nchunk = tn.tile_nchunk;
    if (nchunk < 1) nchunk = 1;
    const int ncy = a.dims[1] / 2, ncz = a.dims[2] / 2;
    const long long ncol = (long long)ncy * ncz;
    if (ncol * nchunk * a.nrhs > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    int patch = 0;
    if (a.nrhs > 1) {
        patch = tn.mrhs_patch >= 0 ? tn.mrhs_patch : 4;
        while (patch > 1 && (ncy % patch || ncz % patch)) patch >>= 1;
        if (patch < 1 || ncy % patch || ncz % patch) patch = 0;
    }
    const T cdiag = (T)(4.0 + a.mass); // formed in double, rounded once (reading S8)
    kern<<<(unsigned)(ncol * nchunk * a.nrhs), 128, smem, a.stream>>>((T *)a.out, (const T *)a.in, (const T *)a.links, a.dims[1],
                                                                       a.dims[2], a.dims[3], a.V, cdiag, a.nrhs, nchunk, a.tgauge, patch);
    count_launch();
    return cudaGetLastError();
}

template <typename T, int RECON> cudaError_t launch_bulk_r(const ApplyArgs &a)
{
    return a.dagger ? launch_bulk_s<T, RECON, +1>(a) : launch_bulk_s<T, RECON, -1>(a);
}

} // namespace

// Lx = 32, tile 32 x 2 x 2 (the caller checks)
cudaError_t launch_stage_bulk(const ApplyArgs &a)
{
    if (a.precision == 32)
        return a.recon == 18 ? launch_bulk_r<float, 18>(a) : a.recon == 12 ? launch_bulk_r<float, 12>(a) : launch_bulk_r<float, 8>(a);
    return a.recon == 18 ? launch_bulk_r<double, 18>(a) : a.recon == 12 ? launch_bulk_r<double, 12>(a) : launch_bulk_r<double, 8>(a);
}

} // namespace wd
