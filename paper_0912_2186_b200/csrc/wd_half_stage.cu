// wd_half_stage.cu -- the staged (t-marching, cp.async) member for half-precision STORAGE (reading RH; wd_half.cu holds the
// format, the general one-thread-per-site kernel and the pack / unpack kernels).
//
// Same decomposition and copy-group bookkeeping as wd_dslash_stage.cu (a CTA owns a tile Lx x ty x tz of one time slice
// and marches along t; x hops by warp shuffles, y/z hops through the staged slice, backward hops computed at the source
// site and handed over through shared memory, t hops in registers; every global read is a cp.async issued half a step to
// a full step before its LDS), with these differences:
//   * what is staged is the RAW binary16 data: 3 vectors of 8 halves + one float scale per spinor, RECON/2 vectors per
//     site of links; conversion to float (and the multiplication by the scale) happens at the LDS;
//   * the exchange buffers hold the link-multiplied half spinors in float;
//   * links x,y and links z,t are staged in SEPARATE slot groups even where a 16-byte vector straddles the two (18 halves
//     per link): that vector is copied into both groups, so a group can be refilled for the next slice while the other
//     is still in use;
//   * the result is requantised per site (scale = max |component|) in the epilogue;
//   * 400 B of shared memory per site with 12-real links (fp32: 840 B): three CTAs of 128 sites per SM.
// Lx must be a power of two (4..32); other lattices take the general kernel of wd_half.cu.
#include <cuda_fp16.h>
#include "wd_half.cuh"
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_async.cuh"
#define WD_USE_F32X2
#include "wd_math.cuh"

namespace wd {

namespace {



// staged half spinor [3][stride] + scale -> 24 floats
__device__ __forceinline__ void lds_spinor(const uint4 *buf, const float *scale, int stride, int slot, float (&p)[24])
{
    const float s = scale[slot];
#pragma unroll
    for (int c = 0; c < 3; ++c) unpack8(buf[c * stride + slot], &p[8 * c]);
#pragma unroll
    for (int i = 0; i < 24; ++i) p[i] *= s;
}
__device__ __forceinline__ void lds_half12(const float4 *buf, int stride, int slot, float (&h)[12])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float4 v = buf[c * stride + slot];
        h[4 * c] = v.x; h[4 * c + 1] = v.y; h[4 * c + 2] = v.z; h[4 * c + 3] = v.w;
    }
}
__device__ __forceinline__ void sts_half12(float4 *buf, int stride, int slot, const float (&h)[12])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) buf[c * stride + slot] = make_float4(h[4 * c], h[4 * c + 1], h[4 * c + 2], h[4 * c + 3]);
}

// vectors (of 8 halves) of a site's link record that hold link MU
template <int MU, int RECON> struct HLinkVecs {
    static constexpr int first = (MU * RECON) / 8, last = (MU * RECON + RECON - 1) / 8, n = last - first + 1;
    static constexpr int skip = MU * RECON - first * 8;
};

// link MU out of a staged group: `base` points at vector `first0` of the record, slots `stride` apart
template <int MU, int RECON>
__device__ __forceinline__ void lds_link(const uint4 *base, int first0, int stride, int slot, float (&u)[18])
{
    using LV = HLinkVecs<MU, RECON>;
    float tmp[LV::n * 8];
#pragma unroll
    for (int j = 0; j < LV::n; ++j) unpack8(base[(LV::first - first0 + j) * stride + slot], &tmp[8 * j]);
#pragma unroll
    for (int i = 0; i < RECON; ++i) u[i] = tmp[LV::skip + i];
    if (RECON == 12) reconstruct_row2(u);
    if (RECON == 8) reconstruct_from8(u);
}

__device__ __forceinline__ void shfl12(float (&dst)[12], const float (&src)[12], int src_lane)
{
#pragma unroll
    for (int i = 0; i < 12; ++i) dst[i] = __shfl_sync(0xffffffffu, src[i], src_lane);
}

template <int RECON> struct HGeom {
    static constexpr int NVEC = RECON / 2;
    static constexpr int A_N = HLinkVecs<1, RECON>::last + 1;       // links x,y: vectors [0, A_N)
    static constexpr int B_FIRST = HLinkVecs<2, RECON>::first;      // links z,t: vectors [B_FIRST, NVEC)
    static constexpr int B_N = NVEC - B_FIRST;
    static constexpr int T_FIRST = HLinkVecs<3, RECON>::first;
};

} // namespace

// 16-byte units of shared memory of one CTA
template <int RECON> constexpr int half_stage_smem_units(int nt, int nyb, int nzb)
{
    return nt * (2 * 3 + 2 * 3 + HGeom<RECON>::A_N + HGeom<RECON>::B_N + 2 * 3) + nyb * HLinkVecs<1, RECON>::n +
           nzb * HLinkVecs<2, RECON>::n + (4 * nt + 3) / 4;
}

// gridDim.x = nchunk * nrhs * ncol, ordered (t-chunk, right-hand side, tile column); blockDim.x = Lx * ty * tz
template <int RECON, int NT, int SGN>
__global__ void __launch_bounds__(NT ? NT : 256, NT == 128 ? 3 : 1)
dslash_half_stage_kernel(uint4 *__restrict__ out, float *__restrict__ out_scale, const uint4 *__restrict__ in,
                         const float *__restrict__ in_scale, const uint4 *__restrict__ links, int Lx, int Ly, int Lz, int Lt, int ty,
                         int tz, long long V, float cdiag, int nrhs, int nchunk)
{
    constexpr int FS = SGN, BS = -SGN;
    using G = HGeom<RECON>;
    using FY = HLinkVecs<1, RECON>;
    using FZ = HLinkVecs<2, RECON>;
    constexpr int NVEC = G::NVEC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nt = NT ? NT : (int)blockDim.x, tid = threadIdx.x;
    const int nyb = Lx * tz, nzb = Lx * ty;
    uint4 *plane0 = reinterpret_cast<uint4 *>(smem_raw);            // two slice buffers [3][nt]
    const int plane_sz = 3 * nt;
    float4 *xchg_y = reinterpret_cast<float4 *>(plane0 + 2 * plane_sz); // [3][nt] U_y^dag P psi, float
    float4 *xchg_z = xchg_y + 3 * nt;
    uint4 *lnkA = reinterpret_cast<uint4 *>(xchg_z + 3 * nt);       // [A_N][nt] vectors 0 .. A_N-1 of the site's links
    uint4 *lnkB = lnkA + G::A_N * nt;                               // [B_N][nt] vectors B_FIRST .. NVEC-1
    uint4 *fy = lnkB + G::B_N * nt;                                 // [3][nt] out-of-tile y neighbour (face threads)
    uint4 *fz = fy + 3 * nt;
    uint4 *fly = fz + 3 * nt;                                       // [FY::n][nyb] U_y of the -y neighbour (yy == 0)
    uint4 *flz = fly + FY::n * nyb;                                 // [FZ::n][nzb]
    float *sc_plane = reinterpret_cast<float *>(flz + FZ::n * nzb); // [2][nt] scales of the slice buffers
    float *sc_fy = sc_plane + 2 * nt, *sc_fz = sc_fy + nt;

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    const int col = blockIdx.x % ncol;
    const int kg = blockIdx.x / ncol;
    const int rhs = kg % nrhs, k = kg / nrhs;
    const long long Vp = padded_volume(V);
    in += (long long)rhs * Vp * 3;
    out += (long long)rhs * Vp * 3;
    in_scale += (long long)rhs * Vp;
    out_scale += (long long)rhs * Vp;

    const int row = tid / Lx;
    const int x = tid - row * Lx;
    const int yy = row % ty, zz = row / ty;
    const int lane = tid & 31;
    const int lane_r = (lane & ~(Lx - 1)) | ((lane + 1) & (Lx - 1));
    const int lane_l = (lane & ~(Lx - 1)) | ((lane - 1) & (Lx - 1));
    const int slot_yb = tid - Lx, slot_yf = tid + Lx;
    const int slot_zb = tid - Lx * ty, slot_zf = tid + Lx * ty;
    const bool face_yb = (yy == 0), face_yf = (yy == ty - 1), face_zb = (zz == 0), face_zf = (zz == tz - 1);
    const int rank_y = zz * Lx + x, rank_z = yy * Lx + x;

    const long long S3 = (long long)Lx * Ly * Lz;
    const int t_begin = (int)((long long)Lt * k / nchunk), t_end = (int)((long long)Lt * (k + 1) / nchunk);
    const int cy = col % ncy, cz = col / ncy;
    const int y = cy * ty + yy, z = cz * tz + zz;
    const long long s3 = x + (long long)Lx * (y + (long long)Ly * z);
    const long long s3_y = face_yf ? s3 + (y + 1 == Ly ? -(long long)(Ly - 1) * Lx : (long long)Lx)
                                   : s3 + (y == 0 ? (long long)(Ly - 1) * Lx : -(long long)Lx);
    const long long s3_z = face_zf ? s3 + (z + 1 == Lz ? -(long long)(Lz - 1) * Lx * Ly : (long long)Lx * Ly)
                                   : s3 + (z == 0 ? (long long)(Lz - 1) * Lx * Ly : -(long long)Lx * Ly);
    // vector 0 of a site's record; S3 is a multiple of 32, so a slice offset toff moves a record by toff * (vectors per site)
    auto sp = [&](const uint4 *f, long long s) { return f + (s >> 5) * (3 * BLK) + (s & (BLK - 1)); };
    auto lk = [&](long long s) { return links + (s >> 5) * (NVEC * BLK) + (s & (BLK - 1)); };
    const uint4 *sp_own = sp(in, s3), *sp_y = sp(in, s3_y), *sp_z = sp(in, s3_z);
    const uint4 *lk_own = lk(s3), *lk_y = lk(s3_y), *lk_z = lk(s3_z);
    uint4 *out_own = out + (s3 >> 5) * (3 * BLK) + (s3 & (BLK - 1));

    auto stage_spinor = [&](uint4 *dst, float *sdst, const uint4 *base, long long s3n, long long toff) {
        const uint4 *q = base + toff * 3;
#pragma unroll
        for (int c = 0; c < 3; ++c) cpa16(dst + c * nt + tid, q + c * BLK);
        cpa4(sdst + tid, in_scale + s3n + toff);
    };
    auto stage_A = [&](long long toff) { // links x,y of the own site + y face, slice offset toff
        const uint4 *q = lk_own + toff * NVEC;
#pragma unroll
        for (int j = 0; j < G::A_N; ++j) cpa16(lnkA + j * nt + tid, q + j * BLK);
        if (face_yf | face_yb) stage_spinor(fy, sc_fy, sp_y, s3_y, toff);
        if (face_yb) {
            const uint4 *f = lk_y + toff * NVEC;
#pragma unroll
            for (int j = 0; j < FY::n; ++j) cpa16(fly + j * nyb + rank_y, f + (FY::first + j) * BLK);
        }
    };
    auto stage_B = [&](long long toff) { // links z,t of the own site + z face
        const uint4 *q = lk_own + toff * NVEC;
#pragma unroll
        for (int j = 0; j < G::B_N; ++j) cpa16(lnkB + j * nt + tid, q + (G::B_FIRST + j) * BLK);
        if (face_zf | face_zb) stage_spinor(fz, sc_fz, sp_z, s3_z, toff);
        if (face_zb) {
            const uint4 *f = lk_z + toff * NVEC;
#pragma unroll
            for (int j = 0; j < FZ::n; ++j) cpa16(flz + j * nzb + rank_z, f + (FZ::first + j) * BLK);
        }
    };

    float chi_t[12];
    int cur = 0;
    if (t_begin < t_end) {
        const long long toff = (long long)t_begin * S3;
        stage_spinor(plane0 + cur * plane_sz, sc_plane + cur * nt, sp_own, s3, toff);
        cpa_commit();
        stage_A(toff);
        cpa_commit();
        stage_B(toff);
        cpa_commit();
        const int tb = t_begin == 0 ? Lt - 1 : t_begin - 1;
        const long long site_tb = s3 + (long long)tb * S3;
        // own spinor and U_t of slice t_begin - 1 straight from global memory (once per march)
        float p[24], h[12], u[18];
        {
            const uint4 *q = sp(in, site_tb);
            const float s = __ldg(in_scale + site_tb);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const uint4 v = __ldg(q + c * BLK);
                unpack8(v, &p[8 * c]);
            }
#pragma unroll
            for (int i = 0; i < 24; ++i) p[i] *= s;
            using LT = HLinkVecs<3, RECON>;
            const uint4 *l = lk(site_tb);
            float tmp[LT::n * 8];
#pragma unroll
            for (int j = 0; j < LT::n; ++j) {
                const uint4 v = __ldg(l + (LT::first + j) * BLK);
                unpack8(v, &tmp[8 * j]);
            }
#pragma unroll
            for (int i = 0; i < RECON; ++i) u[i] = tmp[LT::skip + i];
            if (RECON == 12) reconstruct_row2(u);
            if (RECON == 8) reconstruct_from8(u);
        }
        project<3, BS>(p, h);
        su3_dag_mul(u, h, chi_t);
    }

    for (int t = t_begin; t < t_end; ++t) {
        const long long toff = (long long)t * S3;
        const long long toff_n = (long long)(t + 1 == Lt ? 0 : t + 1) * S3;
        const bool more = (t + 1 < t_end);
        stage_spinor(plane0 + (cur ^ 1) * plane_sz, sc_plane + (cur ^ 1) * nt, sp_own, s3, toff_n); // P
        cpa_commit();
        cpa_wait<2>();
        __syncthreads(); // (A) slice t complete for every thread

        const uint4 *pl = plane0 + cur * plane_sz;
        const float *ps = sc_plane + cur * nt;
        float acc[24], psi[24], u[18];
        lds_spinor(pl, ps, nt, tid, psi);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0.f;
        reconstruct_add<3, BS>(acc, chi_t);

        // ---- x ----
        lds_link<0, RECON>(lnkA, 0, nt, tid, u);
        {
            float h[12], g[12], chi[12];
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
        lds_link<1, RECON>(lnkA, 0, nt, tid, u);
        {
            float pn[24], h[12], chi[12];
            if (face_yf) lds_spinor(fy, sc_fy, nt, tid, pn);
            else lds_spinor(pl, ps, nt, slot_yf, pn);
            hop_forward_s<1, SGN>(acc, u, pn);
            project<1, BS>(psi, h);
            su3_dag_mul(u, h, chi);
            sts_half12(xchg_y, nt, tid, chi);
            if (face_yb) {
                lds_link<1, RECON>(fly, FY::first, nyb, rank_y, u);
                lds_spinor(fy, sc_fy, nt, tid, pn);
                hop_backward_s<1, SGN>(acc, u, pn);
            }
        }
        if (more) stage_A(toff_n);
        cpa_commit();
        cpa_wait<2>(); // group B of slice t has landed
        // ---- z ----
        lds_link<2, RECON>(lnkB, G::B_FIRST, nt, tid, u);
        {
            float pn[24], h[12], chi[12];
            if (face_zf) lds_spinor(fz, sc_fz, nt, tid, pn);
            else lds_spinor(pl, ps, nt, slot_zf, pn);
            hop_forward_s<2, SGN>(acc, u, pn);
            project<2, BS>(psi, h);
            su3_dag_mul(u, h, chi);
            sts_half12(xchg_z, nt, tid, chi);
            if (face_zb) {
                lds_link<2, RECON>(flz, FZ::first, nzb, rank_z, u);
                lds_spinor(fz, sc_fz, nt, tid, pn);
                hop_backward_s<2, SGN>(acc, u, pn);
            }
        }
        // ---- t ----
        lds_link<3, RECON>(lnkB, G::B_FIRST, nt, tid, u);
        cpa_wait<1>(); // own spinor of slice t+1 has landed
        {
            float pn[24], h[12];
            lds_spinor(plane0 + (cur ^ 1) * plane_sz, sc_plane + (cur ^ 1) * nt, nt, tid, pn);
            hop_forward_s<3, SGN>(acc, u, pn);
            project<3, BS>(psi, h);
            su3_dag_mul(u, h, chi_t);
        }
        if (more) stage_B(toff_n);
        cpa_commit();
        __syncthreads(); // (B) exchange buffers complete
        if (!face_yb) {
            float chi[12];
            lds_half12(xchg_y, nt, slot_yb, chi);
            reconstruct_add<1, BS>(acc, chi);
        }
        if (!face_zb) {
            float chi[12];
            lds_half12(xchg_z, nt, slot_zb, chi);
            reconstruct_add<2, BS>(acc, chi);
        }
#pragma unroll
        for (int i = 0; i < 24; ++i) psi[i] = fmaf(cdiag, psi[i], -0.5f * acc[i]);
        { // requantise (reading RH) and store
            float s = 0.f;
#pragma unroll
            for (int i = 0; i < 24; ++i) s = fmaxf(s, fabsf(psi[i]));
#pragma unroll
            // (one reciprocal and 24 products instead of 24 IEEE divisions: the ratio may differ from psi / s by one float
            // ulp, far below the binary16 rounding that follows; wd_pack_spinor keeps the exact division of reading RH)
            const float rs = s > 0.f ? __frcp_rn(s) : 0.f;
#pragma unroll
            for (int i = 0; i < 24; ++i) psi[i] *= rs;
            uint4 *q = out_own + toff * 3;
#pragma unroll
            for (int c = 0; c < 3; ++c) q[c * BLK] = pack8(&psi[8 * c]);
            out_scale[s3 + toff] = s;
        }
        cur ^= 1;
    }
    cpa_wait<0>();
}

namespace {

bool half_stage_shape(const ApplyArgs &a, int &ty, int &tz)
{
    const int Lx = a.dims[0], Ly = a.dims[1], Lz = a.dims[2];
    if (Lx < 4 || Lx > 32 || (Lx & (Lx - 1))) return false;
    if (((long long)Lx * Ly * Lz) % BLK) return false;
    int best = 0;
    for (int cy = 2; cy <= Ly && cy <= 16; ++cy) {
        if (Ly % cy) continue;
        for (int cz = 2; cz <= cy && cz <= Lz; ++cz) {
            if (Lz % cz) continue;
            const int nt = Lx * cy * cz;
            if (nt % 32 || nt > 128) continue;
            const int score = nt * 64 - (cy - cz);
            if (score > best) {
                best = score;
                ty = cy;
                tz = cz;
            }
        }
    }
    return best > 0;
}

template <int RECON, int NT, int SGN> cudaError_t launch_hs(const ApplyArgs &a, int ty, int tz)
{
    auto kern = dslash_half_stage_kernel<RECON, NT, SGN>;
    const int nt = a.dims[0] * ty * tz;
    const size_t smem = (size_t)half_stage_smem_units<RECON>(nt, a.dims[0] * tz, a.dims[0] * ty) * 16;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    const int tc = tn.tile_tc >= 1 ? tn.tile_tc : 8; // (measured on 32^3 x 64: 8 > 16 > 32 with three CTAs per SM)
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (tn.tile_nchunk >= 1 && tn.tile_nchunk <= a.dims[3]) nchunk = tn.tile_nchunk;
    if (nchunk < 1) nchunk = 1;
    const long long ncol = (long long)(a.dims[1] / ty) * (a.dims[2] / tz);
    if (ncol * nchunk * a.nrhs > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const long long Vp = padded_volume(a.V);
    float *out_scale = (float *)((char *)a.out + (size_t)a.nrhs * Vp * 48);
    const float *in_scale = (const float *)((const char *)a.in + (size_t)a.nrhs * Vp * 48);
    kern<<<(unsigned)(ncol * nchunk * a.nrhs), nt, smem, a.stream>>>((uint4 *)a.out, out_scale, (const uint4 *)a.in, in_scale,
                                                                    (const uint4 *)a.links, a.dims[0], a.dims[1], a.dims[2],
                                                                    a.dims[3], ty, tz, a.V, (float)(4.0 + a.mass), a.nrhs, nchunk);
    count_launch();
    return cudaGetLastError();
}

template <int RECON> cudaError_t launch_hs_r(const ApplyArgs &a, int ty, int tz)
{
    const int nt = a.dims[0] * ty * tz;
    if (nt == 128) return a.dagger ? launch_hs<RECON, 128, +1>(a, ty, tz) : launch_hs<RECON, 128, -1>(a, ty, tz);
    return a.dagger ? launch_hs<RECON, 0, +1>(a, ty, tz) : launch_hs<RECON, 0, -1>(a, ty, tz);
}

} // namespace

bool half_stage_supported(const ApplyArgs &a)
{
    int ty, tz;
    return half_stage_shape(a, ty, tz);
}

cudaError_t launch_half_stage(const ApplyArgs &a)
{
    int ty = 0, tz = 0;
    if (!half_stage_shape(a, ty, tz)) return cudaErrorInvalidConfiguration;
    return a.recon == 18 ? launch_hs_r<18>(a, ty, tz) : a.recon == 12 ? launch_hs_r<12>(a, ty, tz) : launch_hs_r<8>(a, ty, tz);
}

} // namespace wd
