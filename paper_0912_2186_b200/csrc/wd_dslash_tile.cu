// wd_dslash_tile.cu -- WD_KERNEL_TILE: shared-memory, t-marching Wilson-Dirac kernel for sm_100a.
//
// eq. (2.2); SURVEY.md 8(a) steps a1-a7 in one launch.  Why it exists: the site
// kernel requests ~1200 B/site from L2 for 480 B/site of compulsory HBM traffic
// (profiles/r01_site_ncu.md); the L2->SM path and load latency, not HBM, hold it back.  Here every
// spinor and every link enters an SM (almost) once:
//
//   * A CTA owns a tile  Lx x TY x TZ  of one time slice (one thread per site, a warp = x-rows)
//     and MARCHES along t over a chunk of slices.  Blocks are ordered (t-chunk, RHS group, tile
//     column), so the resident CTAs march through the same slices together (face neighbours in L2).
//   * t direction lives in registers: the thread that owns (x,y,z) at slice t loads U_t(x,t)
//     once, uses it for the forward hop  U_t(t) P- psi(t+1)  and, one step later, for the backward
//     hop into slice t+1,  U_t(t)^dag P+ psi(t)  (12 registers carried across the step).
//   * x direction is exchanged with warp shuffles (Lx is a power of two <= 32, so x-neighbours
//     are lanes of the same warp, periodic wrap = lane arithmetic): the projected half spinor
//     P-_x psi travels from lane x+1, the finished backward product U_x^dag P+_x psi from lane x-1.
//   * y, z directions go through shared memory: slice t of the tile sits in smem (filled one step
//     ahead with 16-byte cp.async straight from HBM/L2, double buffered), forward hops read the
//     neighbour's spinor there; backward hops are computed AT THE SOURCE SITE (which has the link
//     in registers already) and the 12-real result is handed to the site above through smem, so
//     every link is loaded by exactly one thread of the tile.
//   * sites on the tile's y/z faces fetch their out-of-tile neighbour (spinor, and for the
//     backward hop the link) straight from global memory, periodic wrap included; these branches
//     are warp-uniform for Lx = 32.
//
// Two __syncthreads per slice.  No atomics: results are deterministic.
#include <cstdio>
#include <cstdlib>
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

namespace {

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// spinor of one site from a smem slice buffer laid out [chunk][thread slot]
template <typename T>
__device__ __forceinline__ void lds_spinor(const typename SpinorLayout<T>::Vec *buf, int nt, int slot, T (&p)[24])
{
    using L = SpinorLayout<T>;
#pragma unroll
    for (int c = 0; c < L::NCH; ++c) unpack(buf[c * nt + slot], &p[c * L::CR]);
}

// half spinor (12 reals) to / from a smem exchange buffer laid out [chunk][thread slot]
template <typename T>
__device__ __forceinline__ void sts_half(typename SpinorLayout<T>::Vec *buf, int nt, int slot, const T (&h)[12])
{
    using L = SpinorLayout<T>;
#pragma unroll
    for (int c = 0; c < L::NCH / 2; ++c) {
        typename L::Vec v;
        pack(v, &h[c * L::CR]);
        buf[c * nt + slot] = v;
    }
}
template <typename T>
__device__ __forceinline__ void lds_half(const typename SpinorLayout<T>::Vec *buf, int nt, int slot, T (&h)[12])
{
    using L = SpinorLayout<T>;
#pragma unroll
    for (int c = 0; c < L::NCH / 2; ++c) unpack(buf[c * nt + slot], &h[c * L::CR]);
}

template <typename T>
__device__ __forceinline__ void shfl_half(T (&dst)[12], const T (&src)[12], int src_lane)
{
#pragma unroll
    for (int i = 0; i < 12; ++i) dst[i] = __shfl_sync(0xffffffffu, src[i], src_lane);
}

} // namespace

// smem bytes of one CTA: two slice buffers (24 reals/site) + two exchange buffers (12 reals/site)
template <typename T> constexpr size_t tile_smem_bytes(int nt) { return (size_t)nt * (2 * 24 + 2 * 12) * sizeof(T); }

// One launch = out[r] = D in[r] for all right-hand sides.
//   dims Lx (power of two, 4..32), Ly % ty == 0, Lz % tz == 0,
//   blockDim.x = Lx*ty*tz*nrb: the tile's sites times nrb right-hand sides (step a'): the nrb
//   threads of a site load the same links, one from L2, the others from L1.
//   gridDim.x = nchunk * ngroups * ncol, ordered (t-chunk, RHS group, tile column): all RHS groups
//   of a t-chunk run back to back, so the chunk's links come from HBM once and then from L2.
template <typename T, int RECON, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB)
dslash_tile_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ links, int Lx, int Ly, int Lz,
                   int Lt, int ty, int tz, long long V, T cdiag, int nrhs, int nrb, int nchunk)
{
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nt = blockDim.x, tid = threadIdx.x;
    Vec *plane0 = reinterpret_cast<Vec *>(smem_raw); // two slice buffers, plane0 + cur * NCH * nt
    const int plane_sz = NCH * nt;
    Vec *xchg_y = plane0 + 2 * plane_sz;     // U_y^dag P+_y psi of every tile site, for the site at y+1
    Vec *xchg_z = xchg_y + (NCH / 2) * nt;   // same for z

    const int ncy = Ly / ty;
    const int ncol = ncy * (Lz / tz);
    const int ngroups = (nrhs + nrb - 1) / nrb;
    // Work item = (t-chunk k, RHS group g, tile column col), k-major in blockIdx.x: the block
    // scheduler hands out CTAs in index order, so at any time the resident CTAs cover ALL columns of
    // a few consecutive (chunk, group) pairs and march through the same slices together -- a face
    // site's out-of-tile neighbour has just been (or is about to be) loaded by the neighbouring CTA
    // and is served from L2, not HBM.
    const int col = blockIdx.x % ncol;
    const int kg = blockIdx.x / ncol;
    const int g = kg % ngroups, k = kg / ngroups;

    // thread <-> (site of the tile, RHS of the group): x fastest, then y, z, RHS (x-rows are
    // (parts of) warps; shared-memory slots are indexed by tid, so neighbours stay within one RHS)
    const int x = tid & (Lx - 1);
    const int row = tid / Lx;
    const int yy = row % ty, zz = (row / ty) % tz;
    const int rhs = g * nrb + row / (ty * tz);
    const bool live = rhs < nrhs; // a partial last group computes a duplicate and does not store it
    in += (long long)(live ? rhs : nrhs - 1) * 24 * padded_volume(V);
    out += (long long)(live ? rhs : nrhs - 1) * 24 * padded_volume(V);
    const int lane = tid & 31;
    const int lane_r = (lane & ~(Lx - 1)) | ((lane + 1) & (Lx - 1)); // x+1, periodic
    const int lane_l = (lane & ~(Lx - 1)) | ((lane - 1) & (Lx - 1)); // x-1, periodic
    const int slot_yb = tid - Lx, slot_yf = tid + Lx;
    const int slot_zb = tid - Lx * ty, slot_zf = tid + Lx * ty;
    const bool face_yb = (yy == 0), face_yf = (yy == ty - 1), face_zb = (zz == 0), face_zf = (zz == tz - 1);

    const long long S3 = (long long)Lx * Ly * Lz;
    const int t_begin = (int)((long long)Lt * k / nchunk), t_end = (int)((long long)Lt * (k + 1) / nchunk);

    const int cy = col % ncy, cz = col / ncy;
    const int y = cy * ty + yy, z = cz * tz + zz;
    const long long s3 = x + (long long)Lx * (y + (long long)Ly * z); // slice-local site indices
    const long long s3_yf = s3 + (y + 1 == Ly ? -(long long)(Ly - 1) * Lx : (long long)Lx);
    const long long s3_yb = s3 + (y == 0 ? (long long)(Ly - 1) * Lx : -(long long)Lx);
    const long long s3_zf = s3 + (z + 1 == Lz ? -(long long)(Lz - 1) * Lx * Ly : (long long)Lx * Ly);
    const long long s3_zb = s3 + (z == 0 ? (long long)(Lz - 1) * Lx * Ly : -(long long)Lx * Ly);

    T chi_t[12]; // U_t(t-1)^dag P+_t psi(t-1) of this site
    int cur = 0;
    {   // ---- start the march at slice t_begin ----
        const long long site = s3 + (long long)t_begin * S3;
#pragma unroll
        for (int c = 0; c < NCH; ++c) cp_async16(&plane0[cur * plane_sz + c * nt + tid], spinor_ptr(in, site) + c * BLK);
        cp_async_commit();
        const long long site_tb = s3 + (long long)(t_begin == 0 ? Lt - 1 : t_begin - 1) * S3;
        T u[18], p[24], h[12];
        load_link<3, T, RECON>(links, site_tb, u);
        load_spinor(in, site_tb, p);
        project<3, +1>(p, h);
        su3_dag_mul(u, h, chi_t);
    }

    for (int t = t_begin; t < t_end; ++t) {
        const long long site = s3 + (long long)t * S3;
        const long long toff = (long long)t * S3;
        {   // slice t+1 of this tile -> the other buffer (its previous content, slice t-1, is no longer read)
            const long long site_tf = s3 + (long long)(t + 1 == Lt ? 0 : t + 1) * S3;
#pragma unroll
            for (int c = 0; c < NCH; ++c) cp_async16(&plane0[(cur ^ 1) * plane_sz + c * nt + tid], spinor_ptr(in, site_tf) + c * BLK);
            cp_async_commit();
        }
        asm volatile("cp.async.wait_group 1;\n" ::: "memory"); // slice t has landed (own part)
        __syncthreads();                                        // (A) ... and everybody else's

        const Vec *pl = plane0 + cur * plane_sz;
        T acc[24], psi[24], u[18];
        lds_spinor<T>(pl, nt, tid, psi);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = (T)0;
        reconstruct_add<3, +1>(acc, chi_t); // backward t hop, product carried from the previous slice

        // ---- x: both hops through warp shuffles ----
        load_link<0, T, RECON>(links, site, u);
        {
            T h[12], g[12], chi[12];
            project<0, -1>(psi, h);
            shfl_half(g, h, lane_r); // P-_x psi(x+1)
            su3_mul(u, g, chi);
            reconstruct_add<0, -1>(acc, chi);
            project<0, +1>(psi, h);
            su3_dag_mul(u, h, chi);  // U_x(x)^dag P+_x psi(x): belongs to x+1
            shfl_half(g, chi, lane_l);
            reconstruct_add<0, +1>(acc, g);
        }
        // ---- y ----
        load_link<1, T, RECON>(links, site, u);
        {
            T pn[24], h[12], chi[12];
            if (face_yf) load_spinor(in, s3_yf + toff, pn);
            else lds_spinor<T>(pl, nt, slot_yf, pn);
            hop_forward<1>(acc, u, pn);
            project<1, +1>(psi, h);
            su3_dag_mul(u, h, chi);
            sts_half<T>(xchg_y, nt, tid, chi);
            if (face_yb) { // the site below is outside the tile: do its backward hop here
                load_link<1, T, RECON>(links, s3_yb + toff, u);
                load_spinor(in, s3_yb + toff, pn);
                hop_backward<1>(acc, u, pn);
            }
        }
        // ---- z ----
        load_link<2, T, RECON>(links, site, u);
        {
            T pn[24], h[12], chi[12];
            if (face_zf) load_spinor(in, s3_zf + toff, pn);
            else lds_spinor<T>(pl, nt, slot_zf, pn);
            hop_forward<2>(acc, u, pn);
            project<2, +1>(psi, h);
            su3_dag_mul(u, h, chi);
            sts_half<T>(xchg_z, nt, tid, chi);
            if (face_zb) {
                load_link<2, T, RECON>(links, s3_zb + toff, u);
                load_spinor(in, s3_zb + toff, pn);
                hop_backward<2>(acc, u, pn);
            }
        }
        // ---- t: forward hop now, backward product for the next slice ----
        load_link<3, T, RECON>(links, site, u);
        cp_async_wait_all(); // own spinor of slice t+1 has landed in the other buffer
        {
            T pn[24], h[12];
            lds_spinor<T>(plane0 + (cur ^ 1) * plane_sz, nt, tid, pn);
            hop_forward<3>(acc, u, pn);
            project<3, +1>(psi, h);
            su3_dag_mul(u, h, chi_t);
        }
        __syncthreads(); // (B) exchange buffers complete
        if (!face_yb) {
            T chi[12];
            lds_half<T>(xchg_y, nt, slot_yb, chi);
            reconstruct_add<1, +1>(acc, chi);
        }
        if (!face_zb) {
            T chi[12];
            lds_half<T>(xchg_z, nt, slot_zb, chi);
            reconstruct_add<2, +1>(acc, chi);
        }
        // fused diagonal (step a6) and store (a7)
#pragma unroll
        for (int i = 0; i < 24; ++i) psi[i] = fma(cdiag, psi[i], (T)-0.5 * acc[i]);
        if (live) store_spinor(out, site, psi);
        cur ^= 1;
    }
    cp_async_wait_all();
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
namespace {

struct TileShape {
    int ty, tz, nt;
};

bool pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// Tile shape: Lx x ty x tz threads, ty | Ly, tz | Lz, a multiple of 32 and at most max_threads.
// WD_TILE_SHAPE="ty,tz" overrides the choice (tuning / tests); otherwise the largest tile of at
// most 128 sites wins, squarer tiles first (less face traffic).
bool choose_shape(const ApplyArgs &a, int max_threads, TileShape &s)
{
    const int Lx = a.dims[0], Ly = a.dims[1], Lz = a.dims[2];
    if (!pow2(Lx) || Lx < 4 || Lx > 32) return false;
    if (const char *e = getenv("WD_TILE_SHAPE")) {
        int ty = 0, tz = 0;
        if (sscanf(e, "%d,%d", &ty, &tz) == 2 && ty >= 1 && tz >= 1 && Ly % ty == 0 && Lz % tz == 0 &&
            (Lx * ty * tz) % 32 == 0 && Lx * ty * tz <= max_threads) {
            s = {ty, tz, Lx * ty * tz};
            return true;
        }
    }
    int best = 0;
    for (int ty = 1; ty <= Ly && ty <= 16; ++ty) {
        if (Ly % ty) continue;
        for (int tz = 1; tz <= ty && tz <= Lz; ++tz) {
            if (Lz % tz) continue;
            const int nt = Lx * ty * tz;
            if (nt % 32 || nt > 128) continue; // 128 sites per tile measured best (profiles/)
            const int score = nt * 64 - (ty - tz); // bigger first, then squarer
            if (score > best) {
                best = score;
                s = {ty, tz, nt};
            }
        }
    }
    return best > 0;
}

template <typename T> constexpr int tile_max_threads() { return sizeof(T) == 4 ? 256 : 128; }

template <typename T, int RECON>
cudaError_t launch_tile_t(const ApplyArgs &a)
{
    constexpr int MAXT = tile_max_threads<T>();
    constexpr int MINB = 2;
    auto kern = dslash_tile_kernel<T, RECON, MAXT, MINB>;
    TileShape s;
    if (!choose_shape(a, MAXT, s)) return cudaErrorInvalidConfiguration;
    // right-hand sides per CTA: fill the CTA up to MAXT threads (WD_TILE_NRB overrides)
    int nrb = MAXT / s.nt;
    if (const char *ev = getenv("WD_TILE_NRB")) {
        const int v = atoi(ev);
        if (v >= 1 && v * s.nt <= MAXT) nrb = v;
    }
    if (nrb > a.nrhs) nrb = a.nrhs;
    if (nrb < 1) nrb = 1;
    const int ngroups = (a.nrhs + nrb - 1) / nrb;
    const int nthreads = s.nt * nrb;
    const size_t smem = tile_smem_bytes<T>(nthreads);

    static size_t smem_set = 0;
    cudaError_t e;
    if (smem > smem_set) {
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        smem_set = smem;
    }
    // t is cut into chunks of 4 slices (WD_TILE_TC / WD_TILE_NCHUNK override; measured best on B200 for
    // 32^3 x 64): the start of a march costs one extra spinor + link per site (served from L2, the
    // previous chunk has just used them), short chunks give many CTAs per SM slot (load balance).
    int tc = 4;
    if (const char *ev = getenv("WD_TILE_TC")) {
        const int v = atoi(ev);
        if (v >= 1) tc = v;
    }
    int nchunk = (a.dims[3] + tc - 1) / tc;
    if (const char *ev = getenv("WD_TILE_NCHUNK")) {
        const int v = atoi(ev);
        if (v >= 1 && v <= a.dims[3]) nchunk = v;
    }
    if (nchunk < 1) nchunk = 1;
    const long long ncol = (long long)(a.dims[1] / s.ty) * (a.dims[2] / s.tz);
    if (ncol * nchunk * ngroups > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)(ncol * nchunk * ngroups));
    const T cdiag = (T)(4.0 + a.mass); // formed in double, rounded once (reading S8)
    kern<<<grid, nthreads, smem, a.stream>>>((T *)a.out, (const T *)a.in, (const T *)a.links, a.dims[0], a.dims[1],
                                              a.dims[2], a.dims[3], s.ty, s.tz, a.V, cdiag, a.nrhs, nrb, nchunk);
    count_launch();
    return cudaGetLastError();
}

} // namespace

bool tile_supported(const ApplyArgs &a)
{
    if (a.nrhs < 1) return false;
    TileShape s;
    return choose_shape(a, a.precision == 32 ? tile_max_threads<float>() : tile_max_threads<double>(), s);
}

cudaError_t launch_tile(const ApplyArgs &a)
{
    if (a.precision == 32) return a.recon == 18 ? launch_tile_t<float, 18>(a) : launch_tile_t<float, 12>(a);
    return a.recon == 18 ? launch_tile_t<double, 18>(a) : launch_tile_t<double, 12>(a);
}

} // namespace wd
