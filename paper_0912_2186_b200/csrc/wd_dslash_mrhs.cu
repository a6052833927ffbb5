// wd_dslash_mrhs.cu -- the multi-right-hand-side member of WD_KERNEL_STAGE (fp32): D applied to the
// N_v test vectors of the adaptive set-up with ONE link load per site shared by the vectors
// (SURVEY.md 8(a) step a'; BASELINE.json:configs[4]).
//
// Same t-marching tile decomposition and cp.async staging as wd_dslash_stage.cu, with a
// right-hand-side dimension in the CTA: blockDim.x = (Lx*ty*tz sites) x (nrb right-hand sides).
//   * The links of the tile's sites (and the backward-face links) sit in shared memory ONCE and are
//     read by the nrb threads of a site; their cp.async copies are spread over those threads.
//     They are single buffered in two halves: links z,t of slice t are (re)filled right after the
//     barrier at the top of step t (the previous slice's z,t hops are over) and used half a step
//     later; links x,y of slice t+1 right after the mid-step barrier (this slice's x,y hops are
//     over) and used at the top of the next step.
//   * With the links of in-tile neighbours in shared memory, a backward hop in y or z is computed by
//     the receiving site itself (neighbour's link + neighbour's spinor from the slice buffer): no
//     exchange buffers, every thread does exactly eight hops.  x hops use warp shuffles, t hops
//     registers, as in the single-RHS kernels.
//   * Spinor data stay private per (site, rhs) thread: two slice buffers + two face slots = 384 B.
//   * Blocks are ordered (t-chunk, RHS group, tile column): all groups of a chunk run back to back, so
//     the chunk's links come from HBM once and from L2 for the other groups.
// cp.async groups per step t (commit order):  c1 = {links z,t + z-face link of t, own spinor of t+1}
// after barrier A;  c2 = {y-face spinor of t+1} after the y hops;  c3 = {links x,y + y-face link of
// t+1} after barrier M;  c4 = {z-face spinor of t+1} after the z hops.  Waits: wait_group 1 before A
// (c2, c3 of the previous step done) and wait_group 1 before M (c4 of the previous step, c1 done).
#include <cstdio>
#include <cstdlib>
#include <type_traits>
#define WD_USE_F32X2 // packed FFMA2 SU(3) products (wd_math.cuh)
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_async.cuh"
#include "wd_bulk.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

namespace {


// bulk-copy (cp.async.bulk + mbarrier) variant of the link staging: the A/B the round-1 review asked for; helpers in wd_bulk.cuh

template <int NV>
__device__ __forceinline__ void lds_vecs(const float4 *buf, int stride, int slot, float *r)
{
#pragma unroll
    for (int c = 0; c < NV; ++c) unpack(buf[c * stride + slot], &r[c * 4]);
}

template <int MU, int RECON> struct LinkVecs {
    static constexpr int first = (MU * RECON) / 4, last = (MU * RECON + RECON - 1) / 4, n = last - first + 1;
    static constexpr int skip = MU * RECON - first * 4;
};

// link MU of site slot `slot` out of a staged record [vec][stride]; `base` is vector `first0` of the record
template <int MU, int RECON>
__device__ __forceinline__ void lds_link(const float4 *base, int first0, int stride, int slot, float (&u)[18])
{
    using LV = LinkVecs<MU, RECON>;
    float tmp[LV::n * 4];
    lds_vecs<LV::n>(base + (LV::first - first0) * stride, stride, slot, tmp);
#pragma unroll
    for (int i = 0; i < RECON; ++i) u[i] = tmp[LV::skip + i];
    if (RECON == 12) reconstruct_row2(u);
    if (RECON == 8) reconstruct_from8(u);
}

// link MU of tile site slot s out of the staged links: [vector][slot] (default) or, for the bulk-copy variant,
// [row of 32 sites][vector][lane]
template <int MU, int RECON, bool BULK>
__device__ __forceinline__ void own_link_rd(const float4 *lnk, int nts, int s, float (&u)[18])
{
    constexpr int NVEC = LinkLayout<float, RECON>::NVEC;
    if (BULK) lds_link<MU, RECON>(lnk + (s >> 5) * (NVEC * 32), 0, 32, s & 31, u);
    else lds_link<MU, RECON>(lnk, 0, nts, s, u);
}

__device__ __forceinline__ void shfl12(float (&dst)[12], const float (&src)[12], int src_lane)
{
#pragma unroll
    for (int i = 0; i < 12; ++i) dst[i] = __shfl_sync(0xffffffffu, src[i], src_lane);
}

} // namespace

// shared-memory float4 vectors of one CTA
template <int RECON> constexpr int mrhs_smem_vecs(int nts, int nrb, int nyb, int nzb)
{
    return nts * nrb * (2 * 6 + 6 + 6) + nts * LinkLayout<float, RECON>::NVEC + nyb * LinkVecs<1, RECON>::n +
           nzb * LinkVecs<2, RECON>::n;
}

// Work items = (t-chunk, RHS group, tile column) in the order described below; block b < n_full runs item b over its
// whole t-chunk, the blocks after that run the LAST (partial) wave of items cut into ksplit shorter marches each, so
// that the tail of the launch keeps every SM busy (one CTA per SM: without the cut a launch of 3.46 waves costs 4).
// blockDim.x = nts * NRB, nts = Lx*ty*tz sites of the tile (a multiple of 32, at most 128).
// NTS: sites per tile known at compile time (128, the default tile) or 0 = blockDim.x / NRB
// XS: x hops by warp shuffles (Lx a power of two); otherwise (e.g. Lx = 24, the paper's 24^3 x 64 volume)
// x is handled like y and z: neighbour spinor from the slice buffer, neighbour link from the staged links, periodic
// wrap in the slot arithmetic (the tile always spans the whole x extent).
// BULK: the link halves are staged by cp.async.bulk (one 512-byte copy per (vector, 32-site row), each issued by one
// thread, completion through an mbarrier) instead of one 16-byte cp.async per thread and vector; Lx = 32 only (a row of
// the tile is one layout block).  Selected by the tuning variable mrhs_bulk; measured against the default in
// profiles/r02_ncu.md section 6.
template <int RECON, int NRB, int NTS, bool XS, bool BULK = false, int SGN = -1>
__global__ void __launch_bounds__(128 * NRB, 1)
dslash_mrhs_kernel(float *__restrict__ out, const float *__restrict__ in, const float *__restrict__ links, int Lx, int Ly,
                   int Lz, int Lt, int ty, int tz, long long V, float cdiag, int nrhs, int nchunk, int patch, int tgauge,
                   int n_full, int ksplit)
{
    constexpr int NVEC = LinkLayout<float, RECON>::NVEC;
    using FY = LinkVecs<1, RECON>;
    using FZ = LinkVecs<2, RECON>;
    constexpr int A_END = FY::last + 1; // links x,y = vectors [0, A_END), links z,t = [A_END, NVEC)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nts = NTS ? NTS : (int)blockDim.x / NRB, tid = threadIdx.x;
    const int nt = nts * NRB;
    const int st = tid % nts, rr = tid / nts; // site slot of the tile, right-hand side of the group
    const int nyb = Lx * tz, nzb = Lx * ty;
    float4 *plane0 = reinterpret_cast<float4 *>(smem_raw); // two slice buffers [6][nt], private slots
    const int plane_sz = 6 * nt;
    float4 *fy = plane0 + 2 * plane_sz; // [6][nt] out-of-tile y neighbour spinor (face threads)
    float4 *fz = fy + 6 * nt;           // [6][nt] out-of-tile z neighbour spinor
    float4 *lnk = fz + 6 * nt;          // [NVEC][nts] the four links of every tile site (shared by the RHS)
    float4 *fly = lnk + NVEC * nts;     // [FY::n][nyb] U_y of the -y neighbour of the yy == 0 sites
    float4 *flz = fly + FY::n * nyb;    // [FZ::n][nzb] U_z of the -z neighbour of the zz == 0 sites

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    const int ngroups = (nrhs + NRB - 1) / NRB;
    int col, g, k;
    int item = blockIdx.x, sub = 0;
    if ((int)blockIdx.x >= n_full) { // last wave: ksplit blocks share one item
        const int j = blockIdx.x - n_full;
        item = n_full + j / ksplit;
        sub = j - (j / ksplit) * ksplit;
    }
    if (patch > 0) {
        // (t-chunk, patch of patch x patch tile columns, column in patch, RHS group), group FASTEST: the
        // ~#SM resident CTAs are all RHS groups of one compact patch of columns marching through the
        // same slices, so a slice's links are read from HBM by one group and from L2 by the others,
        // and only faces on the patch boundary leave the patch.
        const int per_chunk = ncol * ngroups;
        k = item / per_chunk;
        const int r = item - k * per_chunk;
        const int per_patch = patch * patch * ngroups;
        const int p = r / per_patch, w = r - p * per_patch;
        g = w % ngroups;
        const int c = w / ngroups;                 // column within the patch
        const int npy = ncy / patch;               // patches along y
        const int cyy = (p % npy) * patch + c % patch, czz = (p / npy) * patch + c / patch;
        col = cyy + ncy * czz;
    } else { // (t-chunk, RHS group, tile column)
        col = item % ncol;
        const int kg = item / ncol;
        g = kg % ngroups;
        k = kg / ngroups;
    }
    const int rhs = g * NRB + rr;
    const bool live = rhs < nrhs; // a partial last group computes a duplicate and does not store it
    in += (long long)(live ? rhs : nrhs - 1) * 24 * padded_volume(V);
    out += (long long)(live ? rhs : nrhs - 1) * 24 * padded_volume(V);

    const int row = st / Lx;
    const int x = st - row * Lx;
    const int yy = row % ty, zz = row / ty;
    const int lane = tid & 31;
    const int lane_r = (lane & ~(Lx - 1)) | ((lane + 1) & (Lx - 1));
    const int lane_l = (lane & ~(Lx - 1)) | ((lane - 1) & (Lx - 1));
    const bool face_yb = (yy == 0), face_yf = (yy == ty - 1), face_zb = (zz == 0), face_zf = (zz == tz - 1);
    const int rank_y = zz * Lx + x, rank_z = yy * Lx + x;

    const long long S3 = (long long)Lx * Ly * Lz;
    int t_begin = (int)((long long)Lt * k / nchunk), t_end = (int)((long long)Lt * (k + 1) / nchunk);
    if ((int)blockIdx.x >= n_full) { // this block's share of the chunk
        const int len = t_end - t_begin;
        t_end = t_begin + (int)((long long)len * (sub + 1) / ksplit);
        t_begin += (int)((long long)len * sub / ksplit);
    }
    const int cy = col % ncy, cz = col / ncy;
    const int y = cy * ty + yy, z = cz * tz + zz;
    const long long s3 = x + (long long)Lx * (y + (long long)Ly * z);
    // out-of-tile neighbour of a face thread (at most one per direction since ty, tz >= 2)
    const long long s3_y = face_yf ? s3 + (y + 1 == Ly ? -(long long)(Ly - 1) * Lx : (long long)Lx)
                                   : s3 + (y == 0 ? (long long)(Ly - 1) * Lx : -(long long)Lx);
    const long long s3_z = face_zf ? s3 + (z + 1 == Lz ? -(long long)(Lz - 1) * Lx * Ly : (long long)Lx * Ly)
                                   : s3 + (z == 0 ? (long long)(Lz - 1) * Lx * Ly : -(long long)Lx * Ly);

    // Native addresses: Lx*Ly*Lz is a multiple of the 32-site layout block, so moving a site by `toff`
    // (a whole number of slices) moves its record by toff * (vectors per site): one base pointer per
    // stream, computed once, plus a per-slice offset.
    const float4 *sp_own = spinor_ptr(in, s3), *sp_y = spinor_ptr(in, s3_y), *sp_z = spinor_ptr(in, s3_z);
    const float4 *lk_own = link_ptr<float, RECON>(links, s3), *lk_y = link_ptr<float, RECON>(links, s3_y),
                 *lk_z = link_ptr<float, RECON>(links, s3_z);
    float4 *out_own = const_cast<float4 *>(spinor_ptr(out, s3));

    // ---- staging helpers ----
    auto stage_spinor = [&](float4 *dst, const float4 *base, long long toff) { // private slot
        const float4 *q = base + toff * 6;
#pragma unroll
        for (int c = 0; c < 6; ++c) cpa16(dst + c * nt + tid, q + c * BLK);
    };
    // link copies of a site are dealt out to its NRB threads: vector j goes to rr == j % NRB.  rr is
    // warp uniform; the dispatch below makes `j % NRB == RR` a compile-time test, so the cp.async
    // instructions sit in plain (unpredicated) branches.
    // (Tried and dropped: createpolicy evict_last hints on the link copies to keep a chunk's links in
    // L2 across RHS groups -- within noise on B200, and one launch shape faulted.)
    auto copy_links = [&](auto rr_tag, int j0, int j1, float4 *dst, int stride, int slot, const float4 *src, int src0) {
        constexpr int RR = decltype(rr_tag)::value;
#pragma unroll
        for (int j = 0; j < NVEC; ++j)
            if (j >= j0 && j < j1 && (j - j0) % NRB == RR) cpa16(dst + (j - j0) * stride + slot, src + (src0 + j - j0) * BLK);
    };
    auto deal_links = [&](int j0, int j1, float4 *dst, int stride, int slot, const float4 *src, int src0) {
        if (NRB == 1 || rr == 0) copy_links(std::integral_constant<int, 0>{}, j0, j1, dst, stride, slot, src, src0);
        else if (NRB == 2 || rr == 1) copy_links(std::integral_constant<int, 1 % NRB>{}, j0, j1, dst, stride, slot, src, src0);
        else copy_links(std::integral_constant<int, 2 % NRB>{}, j0, j1, dst, stride, slot, src, src0);
    };
    __shared__ unsigned long long mbar[2]; // BULK: completion of the x,y half / the z,t half
    unsigned ph_xy = 0, ph_zt = 0;
    if (BULK) {
        if (tid == 0) {
            mbar_init(&mbar[0], 1);
            mbar_init(&mbar[1], 1);
            fence_mbar_init();
        }
        __syncthreads();
    }
    // BULK: copy c of a half = (vector j, row r) of the tile's own links, then the face rows.  Row r of the tile
    // (yy = r % ty, zz = r / ty) is the 32-site layout block of site (0, y, z); its record is NVEC * 512 bytes.
    const int nrow = nts >> 5, nrow_y = nyb >> 5, nrow_z = nzb >> 5;
    auto row_block = [&](int yyy, int zzz) { // layout block of the row (y, z) of the lattice, wrapped
        const int Y = (yyy + Ly) % Ly, Z = (zzz + Lz) % Lz;
        return ((long long)Lx * (Y + (long long)Ly * Z)) >> 5;
    };
    // BULK shared-memory layout of the links: [row][vector][lane] (a row's record is contiguous, as in global memory),
    // so a half of a row is ONE copy of (j1 - j0) * 512 bytes; face rows likewise.
    auto bulk_half = [&](unsigned long long *bar, int j0, int j1, const float4 *base_t, int fn, int ffirst, float4 *fdst, int frow,
                         bool yface) {
        if (tid == 0) mbar_expect(bar, (unsigned)(nrow * (j1 - j0) + frow * fn) * 512u);
        if (tid < nrow + frow) {
            fence_proxy_async(); // earlier generic-proxy reads of these slots (before the barrier) precede the async writes
            if (tid < nrow) {
                const int r = tid;
                const long long blk = row_block(cy * ty + r % ty, cz * tz + r / ty);
                bulk_g2s(lnk + (r * NVEC + j0) * 32, base_t + (blk * NVEC + j0) * BLK, (unsigned)(j1 - j0) * 512u, bar);
            } else {
                const int r = tid - nrow; // face row r: yface: zz = r, yy = 0; zface: yy = r, zz = 0
                const long long blk = yface ? row_block(cy * ty - 1, cz * tz + r) : row_block(cy * ty + r, cz * tz - 1);
                bulk_g2s(fdst + r * fn * 32, base_t + (blk * NVEC + ffirst) * BLK, (unsigned)fn * 512u, bar);
            }
        }
    };
    auto stage_XY = [&](long long toff) { // links x,y of the site + the y-face link
        if (BULK) {
            bulk_half(&mbar[0], 0, A_END, reinterpret_cast<const float4 *>(links) + (toff >> 5) * (NVEC * BLK), FY::n, FY::first, fly,
                      nrow_y, true);
            return;
        }
        deal_links(0, A_END, lnk, nts, st, lk_own + toff * NVEC, 0);
        if (face_yb) deal_links(0, FY::n, fly, nyb, rank_y, lk_y + toff * NVEC, FY::first);
    };
    // temporal gauge (wd_set_temporal_gauge): U_t(x,t) = 1 for t < Lt-1 -- those links are neither copied nor read
    auto unit_t = [&](int t) { return tgauge && t != Lt - 1; };
    auto stage_ZT = [&](long long toff, int t) { // links z,t of the site + the z-face link
        if (BULK) {
            bulk_half(&mbar[1], A_END, unit_t(t) ? FZ::last + 1 : NVEC,
                      reinterpret_cast<const float4 *>(links) + (toff >> 5) * (NVEC * BLK), FZ::n, FZ::first, flz, nrow_z, false);
            return;
        }
        deal_links(A_END, unit_t(t) ? FZ::last + 1 : NVEC, lnk + A_END * nts, nts, st, lk_own + toff * NVEC, A_END);
        if (face_zb) deal_links(0, FZ::n, flz, nzb, rank_z, lk_z + toff * NVEC, FZ::first);
    };

    float chi_t[12]; // U_t(t-1)^dag P+_t psi(t-1) of this (site, rhs)
    int cur = 0;
    if (t_begin < t_end) { // ---- start the march at slice t_begin ----
        const long long toff = (long long)t_begin * S3;
        stage_spinor(plane0 + cur * plane_sz, sp_own, toff);
        cpa_commit(); // c0
        if (face_yf | face_yb) stage_spinor(fy, sp_y, toff);
        cpa_commit(); // c2'
        stage_XY(toff);
        cpa_commit(); // c3'
        if (face_zf | face_zb) stage_spinor(fz, sp_z, toff);
        cpa_commit(); // c4'
        const int tb = t_begin == 0 ? Lt - 1 : t_begin - 1;
        const long long site_tb = s3 + (long long)tb * S3;
        float u[18], p[24], h[12];
        load_spinor(in, site_tb, p);
        project<3, -SGN>(p, h);
        if (unit_t(tb)) {
#pragma unroll
            for (int i = 0; i < 12; ++i) chi_t[i] = h[i];
        } else {
            load_link<3, float, RECON>(links, site_tb, u);
            su3_dag_mul(u, h, chi_t);
        }
    }

    float psi[24]; // own spinor of the current slice: read from the slice buffer once (as the t+1 neighbour), then carried
    for (int t = t_begin; t < t_end; ++t) {
        const long long toff = (long long)t * S3;
        const long long toff_n = (long long)(t + 1 == Lt ? 0 : t + 1) * S3;
        const bool more = (t + 1 < t_end);
        cpa_wait<1>();   // links x,y and the y-face spinor of slice t have landed (own copies)
        if (BULK) {
            mbar_wait(&mbar[0], ph_xy);
            ph_xy ^= 1;
        }
        __syncthreads(); // (A) ... everybody's; the z,t hops of slice t-1 are over
        stage_ZT(toff, t);
        stage_spinor(plane0 + (cur ^ 1) * plane_sz, sp_own, toff_n);
        cpa_commit(); // c1

        const float4 *pl = plane0 + cur * plane_sz;
        float acc[24], u[18], pn[24], pnx[24];
        if (t == t_begin) lds_vecs<6>(pl, nt, tid, psi);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0.f;
        reconstruct_add<3, -SGN>(acc, chi_t); // backward t hop, product carried from the previous slice

        // ---- x: both hops through warp shuffles (XS), else like y and z ----
        own_link_rd<0, RECON, BULK>(lnk, nts, st, u);
        if (!XS) {
            const int dxf = (x + 1 == Lx ? 1 - Lx : 1), dxb = (x == 0 ? Lx - 1 : -1);
            lds_vecs<6>(pl, nt, tid + dxf, pn);
            hop_forward_s<0, SGN>(acc, u, pn);
            own_link_rd<0, RECON, BULK>(lnk, nts, st + dxb, u);
            lds_vecs<6>(pl, nt, tid + dxb, pn);
            hop_backward_s<0, SGN>(acc, u, pn);
        } else {
            float h[12], gg[12], chi[12];
            project<0, SGN>(psi, h);
            shfl12(gg, h, lane_r); // P-_x psi(x+1)
            su3_mul(u, gg, chi);
            reconstruct_add<0, SGN>(acc, chi);
            project<0, -SGN>(psi, h);
            su3_dag_mul(u, h, chi); // U_x(x)^dag P+_x psi(x): belongs to x+1
            shfl12(gg, chi, lane_l);
            reconstruct_add<0, -SGN>(acc, gg);
        }
        // ---- y: forward with the own link, backward with the link of the site below ----
        own_link_rd<1, RECON, BULK>(lnk, nts, st, u);
        if (face_yf) lds_vecs<6>(fy, nt, tid, pn);
        else lds_vecs<6>(pl, nt, tid + Lx, pn);
        hop_forward_s<1, SGN>(acc, u, pn);
        if (face_yb) {
            if (BULK) lds_link<1, RECON>(fly + (rank_y >> 5) * (FY::n * 32), FY::first, 32, rank_y & 31, u);
            else lds_link<1, RECON>(fly, FY::first, nyb, rank_y, u);
            lds_vecs<6>(fy, nt, tid, pn);
        } else {
            own_link_rd<1, RECON, BULK>(lnk, nts, st - Lx, u);
            lds_vecs<6>(pl, nt, tid - Lx, pn);
        }
        hop_backward_s<1, SGN>(acc, u, pn);
        if (more && (face_yf | face_yb)) stage_spinor(fy, sp_y, toff_n);
        cpa_commit(); // c2
        cpa_wait<1>();   // links z,t of slice t, own spinor of slice t+1, z-face spinor of slice t have landed
        if (BULK) {
            mbar_wait(&mbar[1], ph_zt);
            ph_zt ^= 1;
        }
        __syncthreads(); // (M) ... everybody's; the x,y hops of slice t are over
        if (more) stage_XY(toff_n);
        cpa_commit(); // c3
        // ---- z ----
        own_link_rd<2, RECON, BULK>(lnk, nts, st, u);
        if (face_zf) lds_vecs<6>(fz, nt, tid, pn);
        else lds_vecs<6>(pl, nt, tid + Lx * ty, pn);
        hop_forward_s<2, SGN>(acc, u, pn);
        if (face_zb) {
            if (BULK) lds_link<2, RECON>(flz + (rank_z >> 5) * (FZ::n * 32), FZ::first, 32, rank_z & 31, u);
            else lds_link<2, RECON>(flz, FZ::first, nzb, rank_z, u);
            lds_vecs<6>(fz, nt, tid, pn);
        } else {
            own_link_rd<2, RECON, BULK>(lnk, nts, st - Lx * ty, u);
            lds_vecs<6>(pl, nt, tid - Lx * ty, pn);
        }
        hop_backward_s<2, SGN>(acc, u, pn);
        if (more && (face_zf | face_zb)) stage_spinor(fz, sp_z, toff_n);
        cpa_commit(); // c4
        // ---- t: forward hop now, backward product for the next slice ----
        {
            float h[12];
            lds_vecs<6>(plane0 + (cur ^ 1) * plane_sz, nt, tid, pnx);
            if (unit_t(t)) { // U_t(x,t) = 1: projection and reconstruction only
                project<3, SGN>(pnx, h);
                reconstruct_add<3, SGN>(acc, h);
                project<3, -SGN>(psi, chi_t);
            } else {
                own_link_rd<3, RECON, BULK>(lnk, nts, st, u);
                hop_forward_s<3, SGN>(acc, u, pnx);
                project<3, -SGN>(psi, h);
                su3_dag_mul(u, h, chi_t);
            }
        }
        // fused diagonal (step a6) and store (a7)
#pragma unroll
        for (int i = 0; i < 24; ++i) psi[i] = fmaf(cdiag, psi[i], -0.5f * acc[i]);
        if (live) {
            float4 *q = out_own + toff * 6;
#pragma unroll
            for (int c = 0; c < 6; ++c) q[c * BLK] = make_float4(psi[4 * c], psi[4 * c + 1], psi[4 * c + 2], psi[4 * c + 3]);
        }
#pragma unroll
        for (int i = 0; i < 24; ++i) psi[i] = pnx[i]; // the spinor of slice t+1 is the next step's own spinor
        cur ^= 1;
    }
    cpa_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
namespace {

template <int RECON, int NRB, int NTS, bool XS, bool BULK = false, int SGN = -1>
cudaError_t launch_mrhs_n(const ApplyArgs &a, int ty, int tz)
{
    auto kern = dslash_mrhs_kernel<RECON, NRB, NTS, XS, BULK, SGN>;
    const int Lx = a.dims[0];
    const int nts = Lx * ty * tz;
    const size_t smem = (size_t)mrhs_smem_vecs<RECON>(nts, NRB, Lx * tz, Lx * ty) * sizeof(float4);
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    // slices per t-chunk (tile_tc / tile_nchunk override): with (columns x RHS groups) already many
    // times the SM count, long marches win (measured for 24 RHS on 32^3 x 64: 64 > 32 > 16 > 8)
    const int tc = tn.tile_tc >= 1 ? tn.tile_tc : 64;
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (tn.tile_nchunk >= 1 && tn.tile_nchunk <= a.dims[3]) nchunk = tn.tile_nchunk;
    if (nchunk < 1) nchunk = 1;
    const long long ncol = (long long)(a.dims[1] / ty) * (a.dims[2] / tz);
    const long long ngroups = (a.nrhs + NRB - 1) / NRB;
    const long long nitems = ncol * nchunk * ngroups;
    if (nitems > 0x3fffffffLL) return cudaErrorInvalidConfiguration;
    // block order: patches of 4 x 4 tile columns with the RHS group fastest when the column grid allows
    // it (mrhs_patch = 0 / n overrides), else (t-chunk, RHS group, column)
    int patch = tn.mrhs_patch >= 0 ? tn.mrhs_patch : 4;
    const int ncyh = a.dims[1] / ty, nczh = a.dims[2] / tz;
    if (patch < 1 || ncyh % patch || nczh % patch) patch = 0;
    // the last, partial wave: its items are cut into ksplit shorter marches (at least 8 slices each) so that it
    // fills the machine and ends after 1/ksplit of a wave.  CTAs resident per SM: by shared memory.
    const int per_sm = smem > 113 * 1024 ? 1 : 2;
    const long long slots = (long long)sm_count() * per_sm;
    long long n_full = nitems, ksplit = 1;
    const long long rem = nitems % slots;
    const int chunk_len = a.dims[3] / nchunk;
    if (rem > 0 && nitems > slots && tn.mrhs_no_tail <= 0) {
        ksplit = slots / rem;
        if (ksplit > chunk_len / 8) ksplit = chunk_len / 8;
        if (ksplit < 1) ksplit = 1;
        if (ksplit > 1) n_full = nitems - rem;
    }
    dim3 grid((unsigned)(n_full + (nitems - n_full) * ksplit));
    const float cdiag = (float)(4.0 + a.mass); // formed in double, rounded once (reading S8)
    kern<<<grid, nts * NRB, smem, a.stream>>>((float *)a.out, (const float *)a.in, (const float *)a.links, a.dims[0],
                                               a.dims[1], a.dims[2], a.dims[3], ty, tz, a.V, cdiag, a.nrhs, nchunk, patch, a.tgauge,
                                               (int)n_full, (int)ksplit);
    count_launch();
    return cudaGetLastError();
}

template <int RECON, int NRB>
cudaError_t launch_mrhs_t(const ApplyArgs &a, int ty, int tz)
{
    const int nts = a.dims[0] * ty * tz;
    if ((a.dims[0] & (a.dims[0] - 1)) && a.dagger) return cudaErrorInvalidConfiguration;
    if (a.dims[0] & (a.dims[0] - 1)) return nts == 96 ? launch_mrhs_n<RECON, NRB, 96, false>(a, ty, tz) : launch_mrhs_n<RECON, NRB, 0, false>(a, ty, tz);
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    if (nts == 128 && a.dims[0] == 32 && NRB == 3 && tn.mrhs_bulk > 0) return launch_mrhs_n<RECON, NRB, 128, true, true>(a, ty, tz);
    // D^dagger = gamma5 D gamma5 (projector signs swapped): the default tile of a power-of-two Lx
    if (a.dagger) return nts == 128 ? launch_mrhs_n<RECON, NRB, 128, true, false, +1>(a, ty, tz) : cudaErrorInvalidConfiguration;
    return nts == 128 ? launch_mrhs_n<RECON, NRB, 128, true>(a, ty, tz) : launch_mrhs_n<RECON, NRB, 0, true>(a, ty, tz);
}

template <int RECON>
cudaError_t launch_mrhs_r(const ApplyArgs &a, int ty, int tz)
{
    // right-hand sides per CTA: 3 (12 warps per SM; 24 = 8 x 3) unless tile_nrb says otherwise
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    int nrb = a.nrhs >= 3 ? 3 : a.nrhs;
    if (tn.tile_nrb >= 1 && tn.tile_nrb <= 3) nrb = tn.tile_nrb;
    if (nrb >= 3) {
        // A partial last group of three computes duplicates that are thrown away (4 right-hand sides cost what 6 do).
        // Measured on 32^3 x 64 (profiles/r02_ncu.md section 12): it pays to give the remainder its own launch when it is a
        // single right-hand side (the single-RHS staged kernel) or a pair behind at least two full groups (groups of two).
        const int rem = a.nrhs % 3;
        if (tn.tile_nrb < 0 && a.nrhs > 3 && (rem == 1 || (rem == 2 && a.nrhs >= 8))) {
            ApplyArgs m = a, r = a;
            m.nrhs = a.nrhs - rem;
            cudaError_t e = launch_mrhs_t<RECON, 3>(m, ty, tz);
            if (e != cudaSuccess) return e;
            const size_t field = (size_t)24 * padded_volume(a.V) * sizeof(float); // one right-hand side (fp32)
            r.in = (const char *)a.in + field * m.nrhs;
            r.out = (char *)a.out + field * m.nrhs;
            r.nrhs = rem;
            return rem == 1 ? launch_stage(r) : launch_mrhs_t<RECON, 2>(r, ty, tz);
        }
        return launch_mrhs_t<RECON, 3>(a, ty, tz);
    }
    if (nrb == 2) return launch_mrhs_t<RECON, 2>(a, ty, tz);
    return launch_mrhs_t<RECON, 1>(a, ty, tz);
}

} // namespace

// shape: chosen by the caller (wd_dslash_stage.cu: same rule as the single-RHS staged kernel)
cudaError_t launch_mrhs(const ApplyArgs &a, int ty, int tz)
{
    return a.recon == 18 ? launch_mrhs_r<18>(a, ty, tz) : launch_mrhs_r<12>(a, ty, tz);
}

} // namespace wd
