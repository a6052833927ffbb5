// wd_dslash_rloop.cu -- multi-right-hand-side member of WD_KERNEL_STAGE with the links in REGISTERS (fp32, Lx a power of two):
// D (or D^dagger) applied to the N_v test vectors of the adaptive set-up with ONE link load per site and time slice, shared by a
// group of right-hand sides (SURVEY.md 8(a) step a'; BASELINE.json:configs[4]).
//
// wd_dslash_mrhs.cu shares the links of a tile in shared memory: every (site, rhs) thread still reads them with its own LDS,
// and the shared-memory / LSU data pipe is that kernel's wall (65 LDS.128 + 26 LDGSTS.128 per (site, rhs) and slice;
// profiles/r02_ncu.md section 4).  Here a thread owns a SITE: it marches along t, and at every slice it loads the site's four
// links into registers ONCE and loops over the right-hand sides of its group.  What crosses threads is the projected half
// spinor (12 reals), never the full spinor (24) and never a link:
//   x   both hops by warp shuffles: the neighbour sends P psi (forward hop) or U_x^dag P psi (backward hop, multiplied at the
//       source site, which holds the link)                                                         24 SHFL
//   y,z inside the tile through a double-buffered exchange area in shared memory (3 STS.128 + 3 LDS.128 per hop, ONE barrier
//       per (slice, rhs)); across the tile boundary the neighbour's spinor comes straight from global memory (L2), and for a
//       backward face hop the neighbour's link too (the same five vectors for every right-hand side: L1)
//   t   forward: the spinor of slice t+1 from global memory (its first touch; it is this thread's own spinor one slice later,
//       then an L2 hit); backward: U_t^dag P psi computed one slice earlier and kept per right-hand side in a private
//       shared-memory slot (3 STS.128 + 3 LDS.128)
// Per (site, rhs) and slice: 24 LDG.128 + 6 STG.128 + 9 LDS.128 + 9 STS.128 (+ 5 L1-hit LDG for a backward face) + 24 SHFL
// against 65 LDS + 26 LDGSTS + 6 STG + 24 SHFL; the 12-real / 8-real rebuild is paid once per site and slice, not per
// right-hand side.  Registers, not shared memory, bound the CTA: 128 threads (one tile of Lx x ty x tz sites), two CTAs per SM.
// Blocks are ordered (t-chunk, patch of tile columns, column, RHS group) like wd_dslash_mrhs.cu, so that the groups of a
// patch march through the same slices together and the links reach the later groups from L2.
// The HBM streams (the spinor rows of the next slice, the link records of the next slice) are requested ahead of time by
// one lane per warp with cp.async.bulk.prefetch.L2, so that the loads that need them are L2 hits.
//
// Measured (24 right-hand sides on 32^3 x 64, fp32, 18-real links; profiles/r02_ncu.md section 10): the LSU work per (site, rhs)
// falls as planned (LSU pipe 68 % -> 50 % busy), but 206-236 registers per thread leave 8 warps per SM and the FMA pipe reaches
// 40 % (ring member) / 31 % (plain loads): 3.6 / 4.4 ms against 3.1 ms for the 12-warp shared-memory member.  Selected by the
// tuning variable mrhs_reg; the default route only for 8-real links with several right-hand sides on Lx = 32 (3.94 against
// 4.19 ms: the rebuild is paid once per group).
#include <cstdio>
#include <cstdlib>
#define WD_USE_F32X2 // packed FFMA2 SU(3) products (wd_math.cuh)
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"
#include "wd_bulk.cuh"

namespace wd {

namespace {

// (Measured: ld.global.nc.L1::no_allocate -- SASS LDG.E.NA -- is looked up in L2 as evict_first, and the re-reads this kernel
// relies on -- a slice's spinor one step after its first touch, the face spinors -- then miss: 17.1 GB of HBM reads instead
// of 5.4 GB.  Plain read-only loads.)
__device__ __forceinline__ float4 ldg_stream(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ void ld_spinor(const float4 *q, float (&p)[24])
{
#pragma unroll
    for (int c = 0; c < 6; ++c) unpack(ldg_stream(q + c * BLK), &p[4 * c]);
}
__device__ __forceinline__ void prefetch_l2(const void *p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(p), "r"(bytes) : "memory");
}
// half spinor <-> three 16-byte vectors of a [3][stride] shared-memory record
__device__ __forceinline__ void sts_half(float4 *rec, int stride, int slot, const float (&h)[12])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) rec[c * stride + slot] = make_float4(h[4 * c], h[4 * c + 1], h[4 * c + 2], h[4 * c + 3]);
}
__device__ __forceinline__ void lds_half(const float4 *rec, int stride, int slot, float (&h)[12])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) unpack(rec[c * stride + slot], &h[4 * c]);
}
__device__ __forceinline__ void shfl_half(float (&dst)[12], const float (&src)[12], int src_lane)
{
#pragma unroll
    for (int i = 0; i < 12; ++i) dst[i] = __shfl_sync(0xffffffffu, src[i], src_lane);
}

} // namespace

// shared memory of one CTA in 16-byte vectors: the exchange area (two buffers; per direction one [3][nts] record array when the
// tile extent is 2 -- a site then sends to exactly one in-tile neighbour -- else two) and rgrp carried t products [3][nts]
constexpr int rloop_exch_arrays(int ty, int tz) { return (ty == 2 ? 1 : 2) + (tz == 2 ? 1 : 2); }
constexpr int rloop_smem_vecs(int nts, int ty, int tz, int rgrp) { return 3 * nts * (2 * rloop_exch_arrays(ty, tz) + rgrp); }

// blockDim.x = nts = Lx * ty * tz sites of the tile (a multiple of 32, at most 128).  SGN = -1: D of eq. (2.2); +1: D^dagger.
template <int RECON, int SGN>
__global__ void __launch_bounds__(128, 2)
dslash_rloop_kernel(float *__restrict__ out, const float *__restrict__ in, const float *__restrict__ links, int Lx, int Ly, int Lz,
                    int Lt, int ty, int tz, long long V, float cdiag, int nrhs, int rgrp, int nchunk, int patch)
{
    constexpr int NVEC = LinkLayout<float, RECON>::NVEC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nts = blockDim.x, st = threadIdx.x;
    float4 *const smem = reinterpret_cast<float4 *>(smem_raw);
    const int rec = 3 * nts;                    // vectors of one [3][nts] record array
    const int nea = rloop_exch_arrays(ty, tz);  // record arrays per exchange buffer
    // exchange arrays: y0 = P psi for the site below (its forward hop), y1 = U_y^dag P psi for the site above (its backward
    // hop); a tile extent of 2 folds the two into one array (every site writes exactly one of them)
    const int off_y0 = 0, off_y1 = (ty == 2 ? 0 : rec), off_z0 = (ty == 2 ? rec : 2 * rec), off_z1 = off_z0 + (tz == 2 ? 0 : rec);
    float4 *const exch = smem;
    float4 *const carry = smem + 2 * nea * rec; // [rgrp][3][nts]

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    const int ngroups = (nrhs + rgrp - 1) / rgrp;
    int col, g, k;
    {
        const int item = blockIdx.x;
        if (patch > 0) { // (t-chunk, patch of patch x patch tile columns, column in patch, RHS group), group fastest
            const int per_chunk = ncol * ngroups;
            k = item / per_chunk;
            const int r = item - k * per_chunk;
            const int per_patch = patch * patch * ngroups;
            const int p = r / per_patch, w = r - p * per_patch;
            g = w % ngroups;
            const int c = w / ngroups;
            const int npy = ncy / patch;
            col = ((p % npy) * patch + c % patch) + ncy * ((p / npy) * patch + c / patch);
        } else { // (t-chunk, RHS group, tile column)
            col = item % ncol;
            const int kg = item / ncol;
            g = kg % ngroups;
            k = kg / ngroups;
        }
    }
    const int rhs0 = g * rgrp;
    const int nr = min(rgrp, nrhs - rhs0);
    const long long fs = 6 * padded_volume(V); // vectors per right-hand side
    in += (long long)rhs0 * 24 * padded_volume(V);
    out += (long long)rhs0 * 24 * padded_volume(V);

    const int row = st / Lx;
    const int x = st - row * Lx;
    const int yy = row % ty, zz = row / ty;
    const int lane = st & 31;
    const int lane_r = (lane & ~(Lx - 1)) | ((lane + 1) & (Lx - 1));
    const int lane_l = (lane & ~(Lx - 1)) | ((lane - 1) & (Lx - 1));
    const bool face_yb = (yy == 0), face_yf = (yy == ty - 1), face_zb = (zz == 0), face_zf = (zz == tz - 1);

    const long long S3 = (long long)Lx * Ly * Lz;
    const int t_begin = (int)((long long)Lt * k / nchunk), t_end = (int)((long long)Lt * (k + 1) / nchunk);
    const int cy = col % ncy, cz = col / ncy;
    const int y = cy * ty + yy, z = cz * tz + zz;
    const long long s3 = x + (long long)Lx * (y + (long long)Ly * z);
    // out-of-tile neighbour of a face thread (at most one per direction since ty, tz >= 2)
    const long long s3_y = face_yf ? s3 + (y + 1 == Ly ? -(long long)(Ly - 1) * Lx : (long long)Lx)
                                   : s3 + (y == 0 ? (long long)(Ly - 1) * Lx : -(long long)Lx);
    const long long s3_z = face_zf ? s3 + (z + 1 == Lz ? -(long long)(Lz - 1) * Lx * Ly : (long long)Lx * Ly)
                                   : s3 + (z == 0 ? (long long)(Lz - 1) * Lx * Ly : -(long long)Lx * Ly);
    // Lx*Ly*Lz is a multiple of the 32-site layout block: moving a site by whole slices moves its record by a multiple of
    // the record size, so one base pointer per stream plus a per-slice offset
    const float4 *const sp_own = spinor_ptr(in, s3), *const sp_y = spinor_ptr(in, s3_y), *const sp_z = spinor_ptr(in, s3_z);
    float4 *const out_own = const_cast<float4 *>(spinor_ptr(out, s3));
    // one lane per 32-site layout block asks L2 for the HBM streams ahead of time (a warp is one block when Lx = 32)
    const bool pf_lane = (Lx == 32) && lane == 0;

    if (t_begin >= t_end) return;
    { // ---- start of the march: the backward t products of slice t_begin, from slice t_begin - 1 ----
        const int tb = t_begin == 0 ? Lt - 1 : t_begin - 1;
        const long long site_tb = s3 + (long long)tb * S3;
        float u[18];
        load_link<3, float, RECON>(links, site_tb, u);
        for (int r = 0; r < nr; ++r) {
            float p[24], h[12], chi[12];
            ld_spinor(sp_own + r * fs + (long long)tb * S3 * 6, p);
            project<3, -SGN>(p, h);
            su3_dag_mul(u, h, chi);
            sts_half(carry + r * rec, nts, st, chi);
        }
        if (pf_lane) {
            for (int r = 0; r < nr; ++r) prefetch_l2(sp_own + r * fs + (long long)t_begin * S3 * 6, 6 * 512);
        }
    }

    int buf = 0;
    for (int t = t_begin; t < t_end; ++t) {
        const long long toff = (long long)t * S3;
        const long long toff_n = (long long)(t + 1 == Lt ? 0 : t + 1) * S3;
        float ux[18], uy[18], uz[18], ut[18];
        load_link<0, float, RECON>(links, s3 + toff, ux);
        load_link<1, float, RECON>(links, s3 + toff, uy);
        load_link<2, float, RECON>(links, s3 + toff, uz);
        load_link<3, float, RECON>(links, s3 + toff, ut);
        if (pf_lane && t + 1 < t_end) prefetch_l2(link_ptr<float, RECON>(links, s3 + toff_n), NVEC * 512);

        for (int r = 0; r < nr; ++r) {
            const float4 *const own_r = sp_own + r * fs;
            // the row of slice t+1 that a later iteration reads for the first time: two right-hand sides ahead
            if (pf_lane) {
                const int r2 = r + 2;
                if (r2 < nr) prefetch_l2(own_r + 2 * fs + toff_n * 6, 6 * 512);
                else if (t + 1 < t_end && r2 - nr < nr) prefetch_l2(sp_own + (r2 - nr) * fs + (long long)(t + 2 >= Lt ? t + 2 - Lt : t + 2) * S3 * 6, 6 * 512);
            }
            float psi[24], acc[24], h[12], g2[12], chi[12];
            ld_spinor(own_r + toff * 6, psi);
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = 0.f;
            // ---- x: both hops through warp shuffles ----
            project<0, SGN>(psi, h);
            shfl_half(g2, h, lane_r); // P psi(x+1)
            su3_mul(ux, g2, chi);
            reconstruct_add<0, SGN>(acc, chi);
            project<0, -SGN>(psi, h);
            su3_dag_mul(ux, h, chi); // U_x(x)^dag P psi(x): belongs to x+1
            shfl_half(g2, chi, lane_l);
            reconstruct_add<0, -SGN>(acc, g2);
            // ---- y, z: what the in-tile neighbours need from this site ----
            float4 *const eb = exch + buf * nea * rec;
            if (!face_yb) {
                project<1, SGN>(psi, h);
                sts_half(eb + off_y0, nts, st, h);
            }
            if (!face_yf) {
                project<1, -SGN>(psi, h);
                su3_dag_mul(uy, h, chi);
                sts_half(eb + off_y1, nts, st, chi);
            }
            if (!face_zb) {
                project<2, SGN>(psi, h);
                sts_half(eb + off_z0, nts, st, h);
            }
            if (!face_zf) {
                project<2, -SGN>(psi, h);
                su3_dag_mul(uz, h, chi);
                sts_half(eb + off_z1, nts, st, chi);
            }
            // ---- t: forward hop from slice t+1; backward product carried from slice t-1, the next one stored ----
            {
                float pn[24];
                ld_spinor(own_r + toff_n * 6, pn);
                project<3, SGN>(pn, h);
                su3_mul(ut, h, chi);
                reconstruct_add<3, SGN>(acc, chi);
                float4 *const cr = carry + r * rec;
                lds_half(cr, nts, st, chi);
                reconstruct_add<3, -SGN>(acc, chi);
                project<3, -SGN>(psi, h);
                su3_dag_mul(ut, h, chi);
                sts_half(cr, nts, st, chi);
            }
            // ---- y, z hops across the tile boundary: neighbour spinor (and link, backward) from global memory ----
            if (face_yf | face_yb) {
                float pn[24];
                ld_spinor(sp_y + r * fs + toff * 6, pn);
                if (face_yf) {
                    project<1, SGN>(pn, h);
                    su3_mul(uy, h, chi);
                    reconstruct_add<1, SGN>(acc, chi);
                } else {
                    float uf[18];
                    load_link<1, float, RECON>(links, s3_y + toff, uf);
                    project<1, -SGN>(pn, h);
                    su3_dag_mul(uf, h, chi);
                    reconstruct_add<1, -SGN>(acc, chi);
                }
            }
            if (face_zf | face_zb) {
                float pn[24];
                ld_spinor(sp_z + r * fs + toff * 6, pn);
                if (face_zf) {
                    project<2, SGN>(pn, h);
                    su3_mul(uz, h, chi);
                    reconstruct_add<2, SGN>(acc, chi);
                } else {
                    float uf[18];
                    load_link<2, float, RECON>(links, s3_z + toff, uf);
                    project<2, -SGN>(pn, h);
                    su3_dag_mul(uf, h, chi);
                    reconstruct_add<2, -SGN>(acc, chi);
                }
            }
            __syncthreads(); // the exchange buffer `buf` of this (slice, rhs) is complete
            if (!face_yf) {
                lds_half(eb + off_y0, nts, st + Lx, h);
                su3_mul(uy, h, chi);
                reconstruct_add<1, SGN>(acc, chi);
            }
            if (!face_yb) {
                lds_half(eb + off_y1, nts, st - Lx, chi);
                reconstruct_add<1, -SGN>(acc, chi);
            }
            if (!face_zf) {
                lds_half(eb + off_z0, nts, st + Lx * ty, h);
                su3_mul(uz, h, chi);
                reconstruct_add<2, SGN>(acc, chi);
            }
            if (!face_zb) {
                lds_half(eb + off_z1, nts, st - Lx * ty, chi);
                reconstruct_add<2, -SGN>(acc, chi);
            }
            // fused diagonal (step a6) and store (a7)
            float4 *const q = out_own + r * fs + toff * 6;
#pragma unroll
            for (int c = 0; c < 6; ++c)
                q[c * BLK] = make_float4(fmaf(cdiag, psi[4 * c], -0.5f * acc[4 * c]), fmaf(cdiag, psi[4 * c + 1], -0.5f * acc[4 * c + 1]),
                                         fmaf(cdiag, psi[4 * c + 2], -0.5f * acc[4 * c + 2]),
                                         fmaf(cdiag, psi[4 * c + 3], -0.5f * acc[4 * c + 3]));
            buf ^= 1;
        }
    }
}


// ---------------------------------------------------------------------------------------------
// Ring member: Lx = 32, tile 32 x 2 x 2 (one warp = one x-row = one 32-site layout block).  Same arithmetic and exchange as
// dslash_rloop_kernel, but no thread ever waits for global memory inside the right-hand-side loop: the four rows a warp
// needs per (slice, rhs) -- its own row, the same row of slice t+1, the out-of-tile y and z neighbour rows -- are contiguous
// 3 KB blocks of the native layout, and lane 0 copies each into a WARP-PRIVATE shared-memory slot with one cp.async.bulk
// (no LSU work, completion on an mbarrier) right after the warp has consumed the slot's previous content, i.e. one whole
// (slice, rhs) pass ahead of its use.  The face links of a slice (the same for every right-hand side) are rebuilt once per
// slice and parked in private shared-memory slots.
// Shared memory per CTA: ring 4 warps x 4 slots x 3 KB = 48 KB, exchange 24 KB, face links 10 KB, carried t products
// 6 KB x rgrp: rgrp <= 5 for two CTAs per SM.
constexpr int RING_ROWV = 6 * 32;                    // 16-byte vectors of one row slot
// UNI ("uniform roles"): every thread also holds U_y, U_z of the sites below it in registers and does its own backward hops, so
// that the four warps of a tile do the same number of SU(3) products per pass and no face links sit in shared memory
constexpr int ring_smem_vecs(int rgrp, bool uni) { return 4 * 4 * RING_ROWV + 2 * 2 * 3 * 128 + (uni ? 0 : 2 * 5 * 64) + rgrp * 3 * 128; }
constexpr size_t ring_smem_bytes(int rgrp, bool uni) { return (size_t)ring_smem_vecs(rgrp, uni) * 16 + 17 * 8; }

template <int RECON, int SGN, bool UNI>
__global__ void __launch_bounds__(128, 2)
dslash_rloop_ring_kernel(float *__restrict__ out, const float *__restrict__ in, const float *__restrict__ links, int Ly, int Lz, int Lt,
                         long long V, float cdiag, int nrhs, int rgrp, int nchunk, int patch)
{
    constexpr int Lx = 32, ty = 2, tz = 2, nts = 128;
    constexpr int NVEC = LinkLayout<float, RECON>::NVEC;
    constexpr int OWN = 0, TP = 1, FY = 2, FZ = 3;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int st = threadIdx.x, w = st >> 5, lane = st & 31;
    float4 *const smem = reinterpret_cast<float4 *>(smem_raw);
    float4 *const ring = smem + w * 4 * RING_ROWV;        // this warp's four row slots
    float4 *const exch = smem + 4 * 4 * RING_ROWV;        // [2 buffers][y, z][3][128]
    float4 *const fl = exch + 2 * 2 * 3 * nts;            // [y, z][5][64] face links (18 reals + 2 pad per site)
    float4 *const carry = fl + (UNI ? 0 : 2 * 5 * 64);    // [rgrp][3][128]
    unsigned long long *const mb0 = reinterpret_cast<unsigned long long *>(carry + rgrp * 3 * nts);
    unsigned long long *const mb = mb0 + w * 4; // this warp's four row slots
    unsigned long long *const xbar = mb0 + 16;  // the CTA's exchange barrier: arrive after the sends, wait before the receives

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    const int ngroups = (nrhs + rgrp - 1) / rgrp;
    int col, g, k;
    {
        const int item = blockIdx.x;
        if (patch > 0) {
            const int per_chunk = ncol * ngroups;
            k = item / per_chunk;
            const int r = item - k * per_chunk;
            const int per_patch = patch * patch * ngroups;
            const int p = r / per_patch, ww = r - p * per_patch;
            g = ww % ngroups;
            const int c = ww / ngroups;
            const int npy = ncy / patch;
            col = ((p % npy) * patch + c % patch) + ncy * ((p / npy) * patch + c / patch);
        } else {
            col = item % ncol;
            const int kg = item / ncol;
            g = kg % ngroups;
            k = kg / ngroups;
        }
    }
    const int rhs0 = g * rgrp;
    const int nr = min(rgrp, nrhs - rhs0);
    const long long fs = 6 * padded_volume(V);
    in += (long long)rhs0 * 24 * padded_volume(V);
    out += (long long)rhs0 * 24 * padded_volume(V);

    const int yy = w & 1, zz = w >> 1; // warp-uniform
    const int lane_r = (lane + 1) & 31, lane_l = (lane - 1) & 31;
    const long long S3 = (long long)Lx * Ly * Lz;
    const int t_begin = (int)((long long)Lt * k / nchunk), t_end = (int)((long long)Lt * (k + 1) / nchunk);
    const int cy = col % ncy, cz = col / ncy;
    const int y = cy * ty + yy, z = cz * tz + zz;
    const long long s3 = lane + (long long)Lx * (y + (long long)Ly * z);
    const long long s3_y = yy ? s3 + (y + 1 == Ly ? -(long long)(Ly - 1) * Lx : (long long)Lx)
                              : s3 + (y == 0 ? (long long)(Ly - 1) * Lx : -(long long)Lx);
    const long long s3_z = zz ? s3 + (z + 1 == Lz ? -(long long)(Lz - 1) * Lx * Ly : (long long)Lx * Ly)
                              : s3 + (z == 0 ? (long long)(Lz - 1) * Lx * Ly : -(long long)Lx * Ly);
    const float4 *const sp_own = spinor_ptr(in, s3), *const sp_y = spinor_ptr(in, s3_y), *const sp_z = spinor_ptr(in, s3_z);
    float4 *const out_own = const_cast<float4 *>(spinor_ptr(out, s3));
    // the row blocks as lane 0 sees them (its site is the first of the 32-site layout block)
    const float4 *const row_own = sp_own - lane, *const row_y = sp_y - lane, *const row_z = sp_z - lane;
    const int fl_y = zz * 32 + lane, fl_z = yy * 32 + lane; // face-link slots of the yy == 0 / zz == 0 sites

    if (t_begin >= t_end) return;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < 4; ++s) mbar_init(&mb[s], 1);
        if (w == 0) mbar_init(xbar, nts);
        fence_mbar_init();
    }
    __syncthreads();
    auto slot_off = [&](int t) { return (long long)t * S3 * 6; };
    auto wrap = [&](int t) { return t >= Lt ? t - Lt : t; };
    auto issue = [&](int slot, const float4 *src) { // lane 0 only
        mbar_expect(&mb[slot], RING_ROWV * 16);
        bulk_g2s(ring + slot * RING_ROWV, src, RING_ROWV * 16, &mb[slot]);
    };
    if (lane == 0) { // first pass of the march
        issue(OWN, row_own + slot_off(t_begin));
        issue(TP, row_own + slot_off(wrap(t_begin + 1)));
        issue(FY, row_y + slot_off(t_begin));
        issue(FZ, row_z + slot_off(t_begin));
        for (int r = 1; r < nr && r < 4; ++r) prefetch_l2(row_own + r * fs + slot_off(wrap(t_begin + 1)), RING_ROWV * 16);
    }
    { // backward t products of slice t_begin, from slice t_begin - 1
        const int tb = t_begin == 0 ? Lt - 1 : t_begin - 1;
        float u[18];
        load_link<3, float, RECON>(links, s3 + (long long)tb * S3, u);
        for (int r = 0; r < nr; ++r) {
            float p[24], h[12], chi[12];
            ld_spinor(sp_own + r * fs + slot_off(tb), p);
            project<3, -SGN>(p, h);
            su3_dag_mul(u, h, chi);
            sts_half(carry + r * 3 * nts, nts, st, chi);
        }
    }

    unsigned ph = 0;
    int buf = 0;
    for (int t = t_begin; t < t_end; ++t) {
        const long long toff = (long long)t * S3;
        float ux[18], uy[18], uz[18], ut[18];
        load_link<0, float, RECON>(links, s3 + toff, ux);
        load_link<1, float, RECON>(links, s3 + toff, uy);
        load_link<2, float, RECON>(links, s3 + toff, uz);
        load_link<3, float, RECON>(links, s3 + toff, ut);
        float uyb[18], uzb[18]; // UNI: U_y, U_z of the sites below (in the tile or not)
        if (UNI) {
            load_link<1, float, RECON>(links, (yy ? s3 - Lx : s3_y) + toff, uyb);
            load_link<2, float, RECON>(links, (zz ? s3 - (long long)Lx * Ly : s3_z) + toff, uzb);
        }
        if (!UNI && !yy) { // U_y of the out-of-tile site below: rebuilt once, read back per right-hand side
            float uf[18];
            load_link<1, float, RECON>(links, s3_y + toff, uf);
#pragma unroll
            for (int c = 0; c < 5; ++c)
                fl[c * 64 + fl_y] = make_float4(uf[4 * c], uf[4 * c + 1], c < 4 ? uf[4 * c + 2] : 0.f, c < 4 ? uf[4 * c + 3] : 0.f);
        }
        if (!UNI && !zz) {
            float uf[18];
            load_link<2, float, RECON>(links, s3_z + toff, uf);
#pragma unroll
            for (int c = 0; c < 5; ++c)
                fl[5 * 64 + c * 64 + fl_z] = make_float4(uf[4 * c], uf[4 * c + 1], c < 4 ? uf[4 * c + 2] : 0.f, c < 4 ? uf[4 * c + 3] : 0.f);
        }
        if (lane == 0 && t + 1 < t_end) prefetch_l2(link_ptr<float, RECON>(links, s3 + (long long)wrap(t + 1) * S3), NVEC * 512);

        for (int r = 0; r < nr; ++r) {
            // the pass after this one: (t, r + 1), or (t + 1, 0)
            const bool last_r = (r + 1 == nr);
            const int tn = last_r ? t + 1 : t, rn = last_r ? 0 : r + 1;
            const bool has_next = tn < t_end;
            const long long noff = rn * fs + slot_off(wrap(tn)), noff_tp = rn * fs + slot_off(wrap(tn + 1));
            if (lane == 0) { // the slice-(t+1) row that is copied three passes from now: ask L2 for it
                int r3 = r + 3, t3 = t;
                while (r3 >= nr) { r3 -= nr; ++t3; }
                if (t3 < t_end) prefetch_l2(row_own + r3 * fs + slot_off(wrap(t3 + 1)), RING_ROWV * 16);
            }
            float psi[24], acc[24], h[12], g2[12], chi[12];
            mbar_wait(&mb[OWN], ph);
#pragma unroll
            for (int c = 0; c < 6; ++c) unpack(ring[OWN * RING_ROWV + c * 32 + lane], &psi[4 * c]);
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = 0.f;
            // ---- x ----
            project<0, SGN>(psi, h);
            shfl_half(g2, h, lane_r);
            su3_mul(ux, g2, chi);
            reconstruct_add<0, SGN>(acc, chi);
            project<0, -SGN>(psi, h);
            su3_dag_mul(ux, h, chi);
            shfl_half(g2, chi, lane_l);
            reconstruct_add<0, -SGN>(acc, g2);
            // ---- y, z: what the in-tile neighbour needs from this site ----
            float4 *const ey = exch + buf * (2 * 3 * nts), *const ez = ey + 3 * nts;
            if (yy) { // the site below is in the tile: P psi for its forward hop
                project<1, SGN>(psi, h);
                sts_half(ey, nts, st, h);
            } else if (UNI) { // the site above is in the tile: P psi for its backward hop (it holds this site's link)
                project<1, -SGN>(psi, h);
                sts_half(ey, nts, st, h);
            } else {  // the site above is in the tile: U_y^dag P psi for its backward hop
                project<1, -SGN>(psi, h);
                su3_dag_mul(uy, h, chi);
                sts_half(ey, nts, st, chi);
            }
            if (zz) {
                project<2, SGN>(psi, h);
                sts_half(ez, nts, st, h);
            } else if (UNI) {
                project<2, -SGN>(psi, h);
                sts_half(ez, nts, st, h);
            } else {
                project<2, -SGN>(psi, h);
                su3_dag_mul(uz, h, chi);
                sts_half(ez, nts, st, chi);
            }
            mbar_arrive(xbar); // this thread's half spinors of the pass are in the exchange buffer
            // ---- t ----
            {
                float pn[24];
                mbar_wait(&mb[TP], ph);
#pragma unroll
                for (int c = 0; c < 6; ++c) unpack(ring[TP * RING_ROWV + c * 32 + lane], &pn[4 * c]);
                __syncwarp(); // every lane has read its words of the two slots: refill them for the next pass
                if (lane == 0 && has_next) {
                    fence_proxy_async(); // required (measured: without it a refill can overtake the reads above)
                    issue(OWN, row_own + noff);
                    issue(TP, row_own + noff_tp);
                }
                project<3, SGN>(pn, h);
                su3_mul(ut, h, chi);
                reconstruct_add<3, SGN>(acc, chi);
                float4 *const cr = carry + r * 3 * nts;
                lds_half(cr, nts, st, chi);
                reconstruct_add<3, -SGN>(acc, chi);
                project<3, -SGN>(psi, h);
                su3_dag_mul(ut, h, chi);
                sts_half(cr, nts, st, chi);
            }
            // ---- y, z hops across the tile boundary ----
            {
                float pn[24];
                mbar_wait(&mb[FY], ph);
#pragma unroll
                for (int c = 0; c < 6; ++c) unpack(ring[FY * RING_ROWV + c * 32 + lane], &pn[4 * c]);
                if (yy) {
                    project<1, SGN>(pn, h);
                    su3_mul(uy, h, chi);
                    reconstruct_add<1, SGN>(acc, chi);
                } else if (UNI) {
                    project<1, -SGN>(pn, h);
                    su3_dag_mul(uyb, h, chi);
                    reconstruct_add<1, -SGN>(acc, chi);
                } else {
                    float uf[20];
#pragma unroll
                    for (int c = 0; c < 5; ++c) unpack(fl[c * 64 + fl_y], &uf[4 * c]);
                    project<1, -SGN>(pn, h);
                    su3_dag_mul(reinterpret_cast<const float(&)[18]>(uf), h, chi);
                    reconstruct_add<1, -SGN>(acc, chi);
                }
            }
            {
                float pn[24];
                mbar_wait(&mb[FZ], ph);
#pragma unroll
                for (int c = 0; c < 6; ++c) unpack(ring[FZ * RING_ROWV + c * 32 + lane], &pn[4 * c]);
                __syncwarp();
                if (lane == 0 && has_next) {
                    fence_proxy_async(); // required (measured: without it a refill can overtake the reads above)
                    issue(FY, row_y + noff);
                    issue(FZ, row_z + noff);
                }
                if (zz) {
                    project<2, SGN>(pn, h);
                    su3_mul(uz, h, chi);
                    reconstruct_add<2, SGN>(acc, chi);
                } else if (UNI) {
                    project<2, -SGN>(pn, h);
                    su3_dag_mul(uzb, h, chi);
                    reconstruct_add<2, -SGN>(acc, chi);
                } else {
                    float uf[20];
#pragma unroll
                    for (int c = 0; c < 5; ++c) unpack(fl[5 * 64 + c * 64 + fl_z], &uf[4 * c]);
                    project<2, -SGN>(pn, h);
                    su3_dag_mul(reinterpret_cast<const float(&)[18]>(uf), h, chi);
                    reconstruct_add<2, -SGN>(acc, chi);
                }
            }
            mbar_wait(xbar, ph); // everybody's: the exchange buffer `buf` of this (slice, rhs) is complete
            if (yy && UNI) {
                lds_half(ey, nts, st - 32, h);
                su3_dag_mul(uyb, h, chi);
                reconstruct_add<1, -SGN>(acc, chi);
            } else if (yy) {
                lds_half(ey, nts, st - 32, chi);
                reconstruct_add<1, -SGN>(acc, chi);
            } else {
                lds_half(ey, nts, st + 32, h);
                su3_mul(uy, h, chi);
                reconstruct_add<1, SGN>(acc, chi);
            }
            if (zz && UNI) {
                lds_half(ez, nts, st - 64, h);
                su3_dag_mul(uzb, h, chi);
                reconstruct_add<2, -SGN>(acc, chi);
            } else if (zz) {
                lds_half(ez, nts, st - 64, chi);
                reconstruct_add<2, -SGN>(acc, chi);
            } else {
                lds_half(ez, nts, st + 64, h);
                su3_mul(uz, h, chi);
                reconstruct_add<2, SGN>(acc, chi);
            }
            float4 *const q = out_own + r * fs + toff * 6;
#pragma unroll
            for (int c = 0; c < 6; ++c)
                q[c * BLK] = make_float4(fmaf(cdiag, psi[4 * c], -0.5f * acc[4 * c]), fmaf(cdiag, psi[4 * c + 1], -0.5f * acc[4 * c + 1]),
                                         fmaf(cdiag, psi[4 * c + 2], -0.5f * acc[4 * c + 2]),
                                         fmaf(cdiag, psi[4 * c + 3], -0.5f * acc[4 * c + 3]));
            buf ^= 1;
            ph ^= 1;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
namespace {

template <int RECON, int SGN>
cudaError_t launch_rloop_s(const ApplyArgs &a, int ty, int tz)
{
    auto kern = dslash_rloop_kernel<RECON, SGN>;
    const int Lx = a.dims[0];
    const int nts = Lx * ty * tz;
    if (nts > 128 || nts % 32) return cudaErrorInvalidConfiguration;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    // right-hand sides per group: as many as leave room for two CTAs per SM (a group pays one link load per site and slice),
    // the groups equal in size; mrhs_rgrp overrides
    const int budget = 113 * 1024 / 16;
    int rmax = (budget - rloop_smem_vecs(nts, ty, tz, 0)) / (3 * nts);
    if (rmax < 1) return cudaErrorInvalidConfiguration;
    if (tn.mrhs_rgrp >= 1) { // forced group size, up to what one CTA per SM can hold
        const int rcap = (227 * 1024 / 16 - rloop_smem_vecs(nts, ty, tz, 0)) / (3 * nts);
        rmax = tn.mrhs_rgrp < rcap ? tn.mrhs_rgrp : rcap;
    }
    int ngroups = (a.nrhs + rmax - 1) / rmax;
    const int rgrp = (a.nrhs + ngroups - 1) / ngroups;
    ngroups = (a.nrhs + rgrp - 1) / rgrp;
    const size_t smem = (size_t)rloop_smem_vecs(nts, ty, tz, rgrp) * sizeof(float4);
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    // slices per t-chunk (tile_tc / tile_nchunk override): the start of a march costs about one right-hand-side pass
    const int tc = tn.tile_tc >= 1 ? tn.tile_tc : 16;
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (tn.tile_nchunk >= 1 && tn.tile_nchunk <= a.dims[3]) nchunk = tn.tile_nchunk;
    if (nchunk < 1) nchunk = 1;
    const int ncyh = a.dims[1] / ty, nczh = a.dims[2] / tz;
    const long long nitems = (long long)ncyh * nczh * nchunk * ngroups;
    if (nitems > 0x3fffffffLL) return cudaErrorInvalidConfiguration;
    int patch = tn.mrhs_patch >= 0 ? tn.mrhs_patch : 4;
    while (patch > 1 && (ncyh % patch || nczh % patch)) patch >>= 1;
    if (patch < 1 || ncyh % patch || nczh % patch) patch = 0;
    const float cdiag = (float)(4.0 + a.mass); // formed in double, rounded once (reading S8)
    kern<<<(unsigned)nitems, nts, smem, a.stream>>>((float *)a.out, (const float *)a.in, (const float *)a.links, a.dims[0], a.dims[1],
                                                     a.dims[2], a.dims[3], ty, tz, a.V, cdiag, a.nrhs, rgrp, nchunk, patch);
    count_launch();
    return cudaGetLastError();
}

template <int RECON, int SGN, bool UNI>
cudaError_t launch_ring_s(const ApplyArgs &a)
{
    auto kern = dslash_rloop_ring_kernel<RECON, SGN, UNI>;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    int rmax = UNI ? 6 : 5; // two CTAs per SM
    if (tn.mrhs_rgrp >= 1) { // forced group size, up to what one CTA per SM can hold
        const int rcap = (int)((227 * 1024 - ring_smem_bytes(0, UNI)) / (3 * 128 * 16));
        rmax = tn.mrhs_rgrp < rcap ? tn.mrhs_rgrp : rcap;
    }
    int ngroups = (a.nrhs + rmax - 1) / rmax;
    const int rgrp = (a.nrhs + ngroups - 1) / ngroups;
    ngroups = (a.nrhs + rgrp - 1) / rgrp;
    const size_t smem = ring_smem_bytes(rgrp, UNI);
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    const int tc = tn.tile_tc >= 1 ? tn.tile_tc : 16;
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (tn.tile_nchunk >= 1 && tn.tile_nchunk <= a.dims[3]) nchunk = tn.tile_nchunk;
    if (nchunk < 1) nchunk = 1;
    const int ncyh = a.dims[1] / 2, nczh = a.dims[2] / 2;
    const long long nitems = (long long)ncyh * nczh * nchunk * ngroups;
    if (nitems > 0x3fffffffLL) return cudaErrorInvalidConfiguration;
    int patch = tn.mrhs_patch >= 0 ? tn.mrhs_patch : 4;
    while (patch > 1 && (ncyh % patch || nczh % patch)) patch >>= 1;
    if (patch < 1 || ncyh % patch || nczh % patch) patch = 0;
    const float cdiag = (float)(4.0 + a.mass);
    kern<<<(unsigned)nitems, 128, smem, a.stream>>>((float *)a.out, (const float *)a.in, (const float *)a.links, a.dims[1], a.dims[2],
                                                     a.dims[3], a.V, cdiag, a.nrhs, rgrp, nchunk, patch);
    count_launch();
    return cudaGetLastError();
}

template <int RECON> cudaError_t launch_rloop_r(const ApplyArgs &a, int ty, int tz)
{
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    if (tn.mrhs_reg != 1 && a.dims[0] == 32 && ty == 2 && tz == 2) // the ring member wherever it applies
    {
        if (tn.mrhs_reg == 3 || tn.mrhs_reg < 0) return a.dagger ? launch_ring_s<RECON, +1, true>(a) : launch_ring_s<RECON, -1, true>(a);
        return a.dagger ? launch_ring_s<RECON, +1, false>(a) : launch_ring_s<RECON, -1, false>(a);
    }
    return a.dagger ? launch_rloop_s<RECON, +1>(a, ty, tz) : launch_rloop_s<RECON, -1>(a, ty, tz);
}

} // namespace

// fp32, Lx a power of two, tile of at most 128 sites (the caller checks); D and D^dagger, 18 / 12 / 8-real links
cudaError_t launch_rloop(const ApplyArgs &a, int ty, int tz)
{
    return a.recon == 18 ? launch_rloop_r<18>(a, ty, tz) : a.recon == 12 ? launch_rloop_r<12>(a, ty, tz) : launch_rloop_r<8>(a, ty, tz);
}

} // namespace wd
