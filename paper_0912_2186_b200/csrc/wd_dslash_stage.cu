// wd_dslash_stage.cu -- WD_KERNEL_STAGE: the t-marching tile kernel with EVERY global read staged
// through shared memory by cp.async one step ahead (fp32 and fp64).
//
// eq. (2.2); SURVEY.md 8(a) steps a1-a7 in one launch.  Decomposition: a CTA owns a tile
// Lx x ty x tz of one time slice and marches along t over a chunk of slices; x hops by warp
// shuffles, y/z hops through a shared-memory slice, backward hops computed at the source site (which
// holds the link) and handed over through shared memory, t hops in registers.  The round-1 tile kernel
// with this decomposition but plain global loads was latency bound (profiles/r01_tile_stage_ncu.md: ~60 % of
// the stall samples were the first use of a link / face load); here no arithmetic ever waits for HBM or L2:
//
//   * the four links of the thread's site, its out-of-tile face neighbours (spinor, plus the link for
//     a backward face) and its own spinor of the next slice are all copied global -> shared by
//     16-byte cp.async into slots PRIVATE to the thread, issued half a step to a full step before
//     they are read back with LDS; a slot is refilled for slice t+1 right after slice t consumed it;
//   * cp.async group bookkeeping per slice (commit order):  P = own spinor of t+1 (top of slice),
//     A = links x,y + y face of t+1 (after the y hops), B = links z,t + z face of t+1 (after the t
//     hops);  waits: wait_group 2 at the top (P(t), A(t-1 issued) done), 2 before z, 1 before t.
//
// Registers are no longer held across memory latency, shared memory is: 840 B/site in fp32 (two CTAs
// of 128 sites per SM), twice that in fp64 (one CTA of 128 sites per SM).  Requires ty, tz >= 2 (a thread
// has at most one face per direction), 4 <= Lx <= 32 (a tile spans the whole x extent; a power-of-two Lx
// exchanges x neighbours by warp shuffles, any other Lx through shared memory), Lx*ty*tz and Lx*Ly*Lz
// multiples of 32.
#include <cstdio>
#include <cstdlib>
#define WD_USE_F32X2 // packed FFMA2 SU(3) products (wd_math.cuh)
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_async.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

namespace {


// NV 16-byte vectors [vec][slot stride] -> registers
template <int NV, typename Vec, typename T>
__device__ __forceinline__ void lds_vecs(const Vec *buf, int stride, int slot, T *r)
{
    constexpr int CR = 16 / sizeof(T);
#pragma unroll
    for (int c = 0; c < NV; ++c) unpack(buf[c * stride + slot], &r[c * CR]);
}

// vectors of a site's link record that hold link MU
template <int MU, int RECON, typename T> struct FaceLinkVecs {
    static constexpr int CR = 16 / sizeof(T);
    static constexpr int first = (MU * RECON) / CR, last = (MU * RECON + RECON - 1) / CR, n = last - first + 1;
    static constexpr int skip = MU * RECON - first * CR;
};

// link MU out of a staged record: `base` points at vector `first0` of the record, slots `stride` apart
template <int MU, int RECON, typename Vec, typename T>
__device__ __forceinline__ void lds_link_at(const Vec *base, int first0, int stride, int slot, T (&u)[18])
{
    using LV = FaceLinkVecs<MU, RECON, T>;
    T tmp[LV::n * LV::CR];
    lds_vecs<LV::n>(base + (LV::first - first0) * stride, stride, slot, tmp);
#pragma unroll
    for (int i = 0; i < RECON; ++i) u[i] = tmp[LV::skip + i];
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

// shared-memory 16-byte vectors of one CTA (see the kernel for the carve-up)
template <typename T, int RECON> constexpr int stage_smem_vecs(int nt, int nyb, int nzb, bool xs)
{
    return nt * (2 * SpinorLayout<T>::NCH + (xs ? 2 : 3) * (SpinorLayout<T>::NCH / 2) + LinkLayout<T, RECON>::NVEC +
                 2 * SpinorLayout<T>::NCH) +
           nyb * FaceLinkVecs<1, RECON, T>::n + nzb * FaceLinkVecs<2, RECON, T>::n;
}

// gridDim.x = nchunk * nrhs * ncol, ordered (t-chunk, right-hand side, tile column): all right-hand
// sides of a t-chunk run back to back, so the chunk's links come from HBM once and then from L2.
// NT: threads per CTA known at compile time (128, the default tile) or 0 = read blockDim.x; with a
// constant NT every shared-memory slot is an immediate offset from one base register.
// XS: x hops by warp shuffles (Lx a power of two); otherwise (e.g. Lx = 24) x is handled like y and z
// inside the tile -- forward hop from the slice buffer, backward product through an exchange buffer --
// with the periodic wrap in the slot arithmetic (the tile always spans the whole x extent).
// SGN = -1: D of eq. (2.2); SGN = +1: gamma5 D gamma5 = D^dagger, every projector 1 -+ gamma_mu swapped.
// patch > 0 (several right-hand sides): blocks ordered (t-chunk, patch of patch x patch tile columns, column in patch,
// right-hand side) with the right-hand side FASTEST, so the CTAs resident at any time are all right-hand sides of a few
// neighbouring columns marching through the same slices: a slice's links come from HBM once and from L2 for the others.
template <typename T, int RECON, int NT, bool XS, int SGN>
__global__ void __launch_bounds__(NT ? NT : 256, 1)
dslash_stage_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ links, int Lx, int Ly,
                    int Lz, int Lt, int ty, int tz, long long V, T cdiag, int nrhs, int nchunk, int tgauge, int patch)
{
    constexpr int FS = SGN, BS = -SGN; // projector signs of the forward / backward hops
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH, CR = SL::CR, HCH = NCH / 2; // vectors per spinor / reals per vector / per half spinor
    using LL = LinkLayout<T, RECON>;
    constexpr int NVEC = LL::NVEC;
    using FY = FaceLinkVecs<1, RECON, T>;
    using FZ = FaceLinkVecs<2, RECON, T>;
    constexpr int A_END = FY::last + 1; // links x,y = vectors [0, A_END), z,t = [A_END, NVEC)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nt = NT ? NT : (int)blockDim.x, tid = threadIdx.x;
    const int nyb = Lx * tz, nzb = Lx * ty;
    Vec *plane0 = reinterpret_cast<Vec *>(smem_raw); // two slice buffers [NCH][nt]
    const int plane_sz = NCH * nt;
    Vec *xchg_y = plane0 + 2 * plane_sz; // [HCH][nt]  U_y^dag P+_y psi, for the site at y+1
    Vec *xchg_z = xchg_y + HCH * nt;     // [HCH][nt]
    Vec *lnk = xchg_z + HCH * nt;        // [NVEC][nt] the four links of the thread's site
    Vec *fy = lnk + NVEC * nt;           // [NCH][nt]  out-of-tile y neighbour spinor (face threads)
    Vec *fz = fy + NCH * nt;             // [NCH][nt]  out-of-tile z neighbour spinor
    Vec *fly = fz + NCH * nt;            // [FY::n][nyb]  U_y of the -y neighbour (yy == 0 threads)
    Vec *flz = fly + FY::n * nyb;        // [FZ::n][nzb]  U_z of the -z neighbour (zz == 0 threads)
    Vec *xchg_x = flz + FZ::n * nzb;     // [HCH][nt]  U_x^dag P+_x psi, for the site at x+1 (only if !XS)

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    int col, rhs, k;
    if (patch > 0) {
        const int per_chunk = ncol * nrhs;
        k = blockIdx.x / per_chunk;
        const int r = blockIdx.x - k * per_chunk;
        const int per_patch = patch * patch * nrhs;
        const int p = r / per_patch, w = r - p * per_patch;
        rhs = w % nrhs;
        const int c = w / nrhs;      // column within the patch
        const int npy = ncy / patch; // patches along y
        col = (p % npy) * patch + c % patch + ncy * ((p / npy) * patch + c / patch);
    } else { // (t-chunk, right-hand side, tile column)
        col = blockIdx.x % ncol;
        const int kg = blockIdx.x / ncol;
        rhs = kg % nrhs;
        k = kg / nrhs;
    }
    in += (long long)rhs * 24 * padded_volume(V);
    out += (long long)rhs * 24 * padded_volume(V);

    const int row = tid / Lx;
    const int x = tid - row * Lx;
    const int yy = row % ty, zz = row / ty;
    const int lane = tid & 31;
    const int lane_r = (lane & ~(Lx - 1)) | ((lane + 1) & (Lx - 1)); // XS only
    const int lane_l = (lane & ~(Lx - 1)) | ((lane - 1) & (Lx - 1));
    const int slot_xf = tid + (x + 1 == Lx ? 1 - Lx : 1), slot_xb = tid + (x == 0 ? Lx - 1 : -1); // !XS only
    const int slot_yb = tid - Lx, slot_yf = tid + Lx;
    const int slot_zb = tid - Lx * ty, slot_zf = tid + Lx * ty;
    const bool face_yb = (yy == 0), face_yf = (yy == ty - 1), face_zb = (zz == 0), face_zf = (zz == tz - 1);
    const int rank_y = zz * Lx + x, rank_z = yy * Lx + x;

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

    // Native addresses: Lx*Ly*Lz is a multiple of the 32-site layout block, so moving a site by `toff`
    // (a whole number of slices) moves its record by toff * (vectors per site): one base pointer per
    // stream, computed once, plus a per-slice offset -- no per-copy index arithmetic.
    const Vec *sp_own = spinor_ptr(in, s3), *sp_y = spinor_ptr(in, s3_y), *sp_z = spinor_ptr(in, s3_z);
    const Vec *lk_own = link_ptr<T, RECON>(links, s3), *lk_y = link_ptr<T, RECON>(links, s3_y),
              *lk_z = link_ptr<T, RECON>(links, s3_z);
    Vec *out_own = const_cast<Vec *>(spinor_ptr(static_cast<const T *>(out), s3));

    // ---- staging helpers (slots private to the thread) ----
    auto stage_spinor = [&](Vec *dst, const Vec *base, long long toff) {
        const Vec *q = base + toff * NCH;
#pragma unroll
        for (int c = 0; c < NCH; ++c) cpa16(dst + c * nt + tid, q + c * BLK);
    };
    auto stage_A = [&](long long toff) { // links x,y of the own site + y face, slice offset toff
        const Vec *q = lk_own + toff * NVEC;
#pragma unroll
        for (int j = 0; j < A_END; ++j) cpa16(lnk + j * nt + tid, q + j * BLK);
        if (face_yf | face_yb) stage_spinor(fy, sp_y, toff);
        if (face_yb) {
            const Vec *f = lk_y + toff * NVEC;
#pragma unroll
            for (int j = 0; j < FY::n; ++j) cpa16(fly + j * nyb + rank_y, f + (FY::first + j) * BLK);
        }
    };
    // tgauge: the caller's links are in temporal gauge (U_t(x,t) = 1 for t < Lt-1; "temporal gauge
    // fixing"): on those slices the vectors that hold only U_t are neither copied nor read and the t hops skip
    // the colour multiplication.
    auto unit_t = [&](int t) { return tgauge && t != Lt - 1; };
    auto stage_B = [&](long long toff, int t) { // links z,t of the own site + z face
        const Vec *q = lk_own + toff * NVEC;
        const int jend = unit_t(t) ? FZ::last + 1 : NVEC;
#pragma unroll
        for (int j = A_END; j < NVEC; ++j)
            if (j < jend) cpa16(lnk + j * nt + tid, q + j * BLK);
        if (face_zf | face_zb) stage_spinor(fz, sp_z, toff);
        if (face_zb) {
            const Vec *f = lk_z + toff * NVEC;
#pragma unroll
            for (int j = 0; j < FZ::n; ++j) cpa16(flz + j * nzb + rank_z, f + (FZ::first + j) * BLK);
        }
    };

    T chi_t[12]; // U_t(t-1)^dag P+_t psi(t-1) of this site
    int cur = 0;
    if (t_begin < t_end) { // ---- start the march at slice t_begin ----
        const long long toff = (long long)t_begin * S3;
        stage_spinor(plane0 + cur * plane_sz, sp_own, toff);
        cpa_commit(); // P'
        stage_A(toff);
        cpa_commit(); // A'
        stage_B(toff, t_begin);
        cpa_commit(); // B'
        const int tb = t_begin == 0 ? Lt - 1 : t_begin - 1;
        const long long site_tb = s3 + (long long)tb * S3;
        T u[18], p[24], h[12];
        load_spinor(in, site_tb, p);
        project<3, BS>(p, h);
        if (unit_t(tb)) {
#pragma unroll
            for (int i = 0; i < 12; ++i) chi_t[i] = h[i];
        } else {
            load_link<3, T, RECON>(links, site_tb, u);
            su3_dag_mul(u, h, chi_t);
        }
    }

    for (int t = t_begin; t < t_end; ++t) {
        const long long toff = (long long)t * S3;
        const long long toff_n = (long long)(t + 1 == Lt ? 0 : t + 1) * S3;
        const bool more = (t + 1 < t_end); // the next slice is still ours: keep its links and faces coming
        // P: own spinor of slice t+1 -> the other slice buffer (its old content, slice t-1, is dead)
        stage_spinor(plane0 + (cur ^ 1) * plane_sz, sp_own, toff_n);
        cpa_commit();
        cpa_wait<2>();   // own spinor of slice t (earlier P) and group A of slice t have landed
        __syncthreads(); // (A) slice t complete for every thread

        const Vec *pl = plane0 + cur * plane_sz;
        T acc[24], psi[24], u[18];
        lds_vecs<NCH>(pl, nt, tid, psi);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = (T)0;
        reconstruct_add<3, BS>(acc, chi_t); // backward t hop, product carried from the previous slice

        // ---- x: both hops through warp shuffles ----
        lds_link_at<0, RECON>(lnk, 0, nt, tid, u);
        if (XS) {
            T h[12], g[12], chi[12];
            project<0, FS>(psi, h);
            shfl12(g, h, lane_r); // P-_x psi(x+1)
            su3_mul(u, g, chi);
            reconstruct_add<0, FS>(acc, chi);
            project<0, BS>(psi, h);
            su3_dag_mul(u, h, chi); // U_x(x)^dag P+_x psi(x): belongs to x+1
            shfl12(g, chi, lane_l);
            reconstruct_add<0, BS>(acc, g);
        } else {
            T pn[24], h[12], chi[12];
            lds_vecs<NCH>(pl, nt, slot_xf, pn);
            hop_forward_s<0, SGN>(acc, u, pn);
            project<0, BS>(psi, h);
            su3_dag_mul(u, h, chi);
#pragma unroll
            for (int c = 0; c < HCH; ++c) pack(xchg_x[c * nt + tid], &chi[c * CR]);
        }
        // ---- y ----
        lds_link_at<1, RECON>(lnk, 0, nt, tid, u);
        {
            T pn[24], h[12], chi[12];
            if (face_yf) lds_vecs<NCH>(fy, nt, tid, pn);
            else lds_vecs<NCH>(pl, nt, slot_yf, pn);
            hop_forward_s<1, SGN>(acc, u, pn);
            project<1, BS>(psi, h);
            su3_dag_mul(u, h, chi);
#pragma unroll
            for (int c = 0; c < HCH; ++c) pack(xchg_y[c * nt + tid], &chi[c * CR]);
            if (face_yb) { // the site below is outside the tile: do its backward hop here
                lds_link_at<1, RECON>(fly, FY::first, nyb, rank_y, u);
                lds_vecs<NCH>(fy, nt, tid, pn);
                hop_backward_s<1, SGN>(acc, u, pn);
            }
        }
        if (more) stage_A(toff_n); // slots of links x,y and the y face are free again
        cpa_commit();
        cpa_wait<2>(); // group B of slice t (links z,t, z face) has landed
        // ---- z ----
        lds_link_at<2, RECON>(lnk, 0, nt, tid, u);
        {
            T pn[24], h[12], chi[12];
            if (face_zf) lds_vecs<NCH>(fz, nt, tid, pn);
            else lds_vecs<NCH>(pl, nt, slot_zf, pn);
            hop_forward_s<2, SGN>(acc, u, pn);
            project<2, BS>(psi, h);
            su3_dag_mul(u, h, chi);
#pragma unroll
            for (int c = 0; c < HCH; ++c) pack(xchg_z[c * nt + tid], &chi[c * CR]);
            if (face_zb) {
                lds_link_at<2, RECON>(flz, FZ::first, nzb, rank_z, u);
                lds_vecs<NCH>(fz, nt, tid, pn);
                hop_backward_s<2, SGN>(acc, u, pn);
            }
        }
        // ---- t: forward hop now, backward product for the next slice ----
        const bool ut = unit_t(t);
        if (!ut) lds_link_at<3, RECON>(lnk, 0, nt, tid, u);
        cpa_wait<1>(); // own spinor of slice t+1 (this slice's P) has landed
        {
            T pn[24], h[12];
            lds_vecs<NCH>(plane0 + (cur ^ 1) * plane_sz, nt, tid, pn);
            if (ut) { // U_t(x,t) = 1: the hops are projection and reconstruction only
                project<3, FS>(pn, h);
                reconstruct_add<3, FS>(acc, h);
                project<3, BS>(psi, chi_t);
            } else {
                hop_forward_s<3, SGN>(acc, u, pn);
                project<3, BS>(psi, h);
                su3_dag_mul(u, h, chi_t);
            }
        }
        if (more) stage_B(toff_n, t + 1 == Lt ? 0 : t + 1); // slots of links z,t and the z face are free again
        cpa_commit();
        __syncthreads(); // (B) exchange buffers complete
        if (!XS) {
            T chi[12];
            lds_vecs<HCH>(xchg_x, nt, slot_xb, chi);
            reconstruct_add<0, BS>(acc, chi);
        }
        if (!face_yb) {
            T chi[12];
            lds_vecs<HCH>(xchg_y, nt, slot_yb, chi);
            reconstruct_add<1, BS>(acc, chi);
        }
        if (!face_zb) {
            T chi[12];
            lds_vecs<HCH>(xchg_z, nt, slot_zb, chi);
            reconstruct_add<2, BS>(acc, chi);
        }
        // fused diagonal (step a6) and store (a7)
#pragma unroll
        for (int i = 0; i < 24; ++i) psi[i] = fma(cdiag, psi[i], (T)-0.5 * acc[i]);
        {
            Vec *q = out_own + toff * NCH;
#pragma unroll
            for (int c = 0; c < NCH; ++c) pack(q[c * BLK], &psi[c * CR]);
        }
        cur ^= 1;
    }
    cpa_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
cudaError_t ensure_dynamic_smem(const void *kernel, size_t bytes, size_t *per_device_cache)
{
    // the attribute is per device; the cache is an array of 64 entries (device ordinal), updated with relaxed atomics
    // (a race sets the same attribute twice, which is harmless)
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    size_t have = __atomic_load_n(&per_device_cache[dev], __ATOMIC_RELAXED);
    if (bytes <= have) return cudaSuccess;
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes)) != cudaSuccess) return e;
    __atomic_store_n(&per_device_cache[dev], bytes, __ATOMIC_RELAXED);
    return cudaSuccess;
}

int sm_count()
{
    static int cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    int n = __atomic_load_n(&cache[dev], __ATOMIC_RELAXED);
    if (n > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    __atomic_store_n(&cache[dev], n, __ATOMIC_RELAXED);
    return n;
}

namespace {

struct StageShape {
    int ty, tz, nt;
};

bool stage_shape(const ApplyArgs &a, StageShape &s)
{
    const int Lx = a.dims[0], Ly = a.dims[1], Lz = a.dims[2];
    if (Lx < 4 || Lx > 32) return false; // a tile spans the whole x extent; power-of-two Lx uses warp shuffles in x
    if (((long long)Lx * Ly * Lz) % BLK) return false;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    if (tn.tile_ty >= 2 && tn.tile_tz >= 2) {
        const int ty = tn.tile_ty, tz = tn.tile_tz;
        if (Ly % ty == 0 && Lz % tz == 0 && (Lx * ty * tz) % 32 == 0 && Lx * ty * tz <= 256) {
            s = {ty, tz, Lx * ty * tz};
            return true;
        }
    }
    int best = 0;
    for (int ty = 2; ty <= Ly && ty <= 16; ++ty) {
        if (Ly % ty) continue;
        for (int tz = 2; tz <= ty && tz <= Lz; ++tz) {
            if (Lz % tz) continue;
            const int nt = Lx * ty * tz;
            if (nt % 32 || nt > 128) continue; // 128 sites per tile: two CTAs per SM
            const int score = nt * 64 - (ty - tz);
            if (score > best) {
                best = score;
                s = {ty, tz, nt};
            }
        }
    }
    return best > 0;
}

template <typename T, int RECON> size_t stage_smem_bytes(const ApplyArgs &a, const StageShape &s)
{
    const bool xs = (a.dims[0] & (a.dims[0] - 1)) == 0;
    return (size_t)stage_smem_vecs<T, RECON>(s.nt, a.dims[0] * s.tz, a.dims[0] * s.ty, xs) * 16;
}

template <typename T, int RECON, int NT, bool XS, int SGN>
cudaError_t launch_stage_sgn(const ApplyArgs &a, const StageShape &s)
{
    auto kern = dslash_stage_kernel<T, RECON, NT, XS, SGN>;
    const size_t smem = stage_smem_bytes<T, RECON>(a, s);
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    // t-chunks of 16 slices (tile_tc / tile_nchunk override; measured 16 > 8 > 32 on 32^3 x 64 in both
    // precisions): the start of a march is the one place where this kernel waits for memory, so chunks
    // are not shorter than that
    const int tc = tn.tile_tc >= 1 ? tn.tile_tc : 16;
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (tn.tile_nchunk >= 1 && tn.tile_nchunk <= a.dims[3]) nchunk = tn.tile_nchunk;
    if (nchunk < 1) nchunk = 1;
    const int ncy = a.dims[1] / s.ty, ncz = a.dims[2] / s.tz;
    const long long ncol = (long long)ncy * ncz;
    if (ncol * nchunk * a.nrhs > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    // several right-hand sides through this kernel (fp64, or tile shapes the multi-RHS kernel does not take): order
    // the blocks so that all right-hand sides of a patch of columns are resident together and share the links in L2
    int patch = 0;
    if (a.nrhs > 1) {
        patch = tn.mrhs_patch >= 0 ? tn.mrhs_patch : 4;
        while (patch > 1 && (ncy % patch || ncz % patch)) patch >>= 1;
        if (patch < 1 || ncy % patch || ncz % patch) patch = 0;
    }
    dim3 grid((unsigned)(ncol * nchunk * a.nrhs));
    const T cdiag = (T)(4.0 + a.mass); // formed in double, rounded once (reading S8)
    kern<<<grid, s.nt, smem, a.stream>>>((T *)a.out, (const T *)a.in, (const T *)a.links, a.dims[0], a.dims[1], a.dims[2],
                                          a.dims[3], s.ty, s.tz, a.V, cdiag, a.nrhs, nchunk, a.tgauge, patch);
    count_launch();
    return cudaGetLastError();
}

template <typename T, int RECON, int NT, bool XS>
cudaError_t launch_stage_nt(const ApplyArgs &a, const StageShape &s)
{
    return a.dagger ? launch_stage_sgn<T, RECON, NT, XS, +1>(a, s) : launch_stage_sgn<T, RECON, NT, XS, -1>(a, s);
}

template <typename T, int RECON>
cudaError_t launch_stage_t(const ApplyArgs &a)
{
    StageShape s;
    if (!stage_shape(a, s)) return cudaErrorInvalidConfiguration;
    if (a.dims[0] & (a.dims[0] - 1)) return s.nt == 96 ? launch_stage_nt<T, RECON, 96, false>(a, s) : launch_stage_nt<T, RECON, 0, false>(a, s);
    return s.nt == 128 ? launch_stage_nt<T, RECON, 128, true>(a, s) : launch_stage_nt<T, RECON, 0, true>(a, s);
}

} // namespace

bool stage_supported(const ApplyArgs &a)
{
    StageShape s;
    if (a.nrhs < 1 || !stage_shape(a, s)) return false;
    // the tile's staging area must fit the 227 KB of shared memory a CTA can have (fp64 needs twice fp32's)
    const size_t smem =
        a.precision == 32
            ? (a.recon == 18 ? stage_smem_bytes<float, 18>(a, s) : a.recon == 12 ? stage_smem_bytes<float, 12>(a, s) : stage_smem_bytes<float, 8>(a, s))
            : (a.recon == 18 ? stage_smem_bytes<double, 18>(a, s) : a.recon == 12 ? stage_smem_bytes<double, 12>(a, s) : stage_smem_bytes<double, 8>(a, s));
    return smem <= 227 * 1024;
}

cudaError_t launch_mrhs(const ApplyArgs &a, int ty, int tz);  // wd_dslash_mrhs.cu
cudaError_t launch_rloop(const ApplyArgs &a, int ty, int tz); // wd_dslash_rloop.cu
cudaError_t launch_stage_bulk(const ApplyArgs &a);             // wd_dslash_stage_bulk.cu

cudaError_t launch_stage(const ApplyArgs &a)
{
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    // several fp32 right-hand sides: the kernel that shares the staged links between them in shared memory when Lx is
    // a power of two (measured, profiles/r02_mrhs.md: 24 RHS on 32^3 x 64 3.0 ms against 3.6 ms for the single-RHS member
    // in the patch order); for other Lx (x hops through shared memory) the single-RHS member in the (patch, column,
    // right-hand side) order, which shares the links through L2, is the faster one (20 RHS on 24^3 x 64: 1.30 against
    // 1.39 ms).  stage_no_mrhs = 0 / 1 forces the choice.
    const bool pow2 = !(a.dims[0] & (a.dims[0] - 1));
    // links in registers, loop over the right-hand sides (wd_dslash_rloop.cu): by measurement (profiles/r02_ncu.md section 10)
    // the default only for 8-real links on Lx = 32, where the rebuild is paid once per group of right-hand sides instead
    // of once per right-hand side (24 RHS on 32^3 x 64: 3.94 against 4.19 ms); mrhs_reg = 0 / 1 / 2 forces off / the
    // plain-load member / the ring member
    if (a.precision == 32 && a.nrhs > 1 && pow2 &&
        (tn.mrhs_reg > 0 || (tn.mrhs_reg < 0 && a.recon == 8 && a.dims[0] == 32 && !a.dagger))) {
        StageShape s;
        if (!stage_shape(a, s)) return cudaErrorInvalidConfiguration;
        if (s.nt <= 128) return launch_rloop(a, s.ty, s.tz);
    }
    if (a.precision == 32 && a.recon != 8 && a.nrhs > 1 && (tn.stage_no_mrhs < 0 ? pow2 : tn.stage_no_mrhs == 0)) {
        StageShape s;
        if (!stage_shape(a, s)) return cudaErrorInvalidConfiguration;
        // (D^dagger: the multi-RHS kernel has its sign-swapped member for the default 128-site tile of a power-of-two Lx)
        if (s.nt <= 128 && (!a.dagger || (pow2 && s.nt == 128))) return launch_mrhs(a, s.ty, s.tz); // (a forced bigger tile runs through the single-RHS kernel below)
    }
    if (a.dims[0] == 32 && tn.stage_bulk > 0) { // bulk-copy member: one warp = one x-row = one layout block
        StageShape s;
        if (!stage_shape(a, s)) return cudaErrorInvalidConfiguration;
        if (s.ty == 2 && s.tz == 2) return launch_stage_bulk(a);
    }
    if (a.precision == 32)
        return a.recon == 18 ? launch_stage_t<float, 18>(a) : a.recon == 12 ? launch_stage_t<float, 12>(a) : launch_stage_t<float, 8>(a);
    return a.recon == 18 ? launch_stage_t<double, 18>(a) : a.recon == 12 ? launch_stage_t<double, 12>(a) : launch_stage_t<double, 8>(a);
}

} // namespace wd
