// wd_dslash_eo.cu -- red/black (even-odd) hopping blocks of the Wilson-Dirac operator (first cut).
//
// SURVEY.md 8(f) row f1; PAPER.md:126 ("red/black preconditioning"), PAPER.md:157 (the paper's own GPU
// kernel is the even-odd matvec).  Site parity p(x) = (x+y+z+t) mod 2; with every extent even
//     D = [ (4+m) 1    H_eo   ]     H_pq = hopping term of eq. (2.2) from parity q to parity p, factor -1/2 included
//         [  H_oe    (4+m) 1  ]
// One kernel:   out_p = alpha * x_p + beta * sum_mu [ (1-g_mu) U_mu(x) in_q(x+mu) + (1+g_mu) U_mu(x-mu)^dag in_q(x-mu) ]
// which gives H_pq (alpha = 0, beta = -1/2) and, in two launches, the even-odd preconditioned operator
//     Mhat psi_p = (4+m) psi_p - H_pq (4+m)^-1 H_qp psi_p          (second launch: alpha = 4+m, beta = 1/(2(4+m))).
//
// Fields of one parity ("half fields") use the blocked native spinor layout of wd_layout.cuh over the
// checkerboard index  cb = lex / 2  (lex = x + Lx*(y + Ly*(z + Lz*t)), Lx even), Vh = V/2 sites.  The links
// are a parity-ordered copy of the gauge handle's native link records (wd_gauge::links_eo: the records of the even
// sites, then those of the odd sites, each half in the blocked layout over cb), made once per gauge handle: with the
// full-lattice array a warp of one parity touched every other 16-byte lane, i.e. half of every 32-byte sector it
// pulled through L1.  One thread per output site, neighbours straight from global memory (the structure of
// WD_KERNEL_SITE): every link of the lattice is used exactly once per launch (forward at parity p, daggered at
// parity q), every input spinor eight times.
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

constexpr int EO_THREADS = 128;
#ifndef WD_EO_NR32
#define WD_EO_NR32 2 // right-hand sides per thread of the multi-RHS member, fp32
#endif
#ifndef WD_EO_NR64
#define WD_EO_NR64 2 // ... fp64
#endif

// SGN = -1: blocks of D; SGN = +1: blocks of gamma5 D gamma5 = D^dagger (all projectors swapped)
template <typename T, int RECON, int SGN>
__global__ void __launch_bounds__(EO_THREADS)
dslash_eo_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ xin, const T *__restrict__ links_p,
                 const T *__restrict__ links_q,
                 int Lx, int Ly, int Lz, int Lt, long long Vh, T alpha, T beta, int parity, double *__restrict__ norm_part, int nrhs,
                 const T *__restrict__ dot_y, double *__restrict__ dot_part, int tgauge)
{
    // gridDim.x = (site blocks) * nrhs with the right-hand side FASTEST: the CTAs resident at any time are all right-hand
    // sides of a few site blocks, so the links of a block come from HBM once and from L1/L2 for the others
    const int rhs = (int)(blockIdx.x % (unsigned)nrhs);
    const long long blk = blockIdx.x / (unsigned)nrhs, nblk = gridDim.x / (unsigned)nrhs;
    // norm_part (may be NULL): per-CTA partial sums of |out|^2 in fp64, fixed order -- lets a solver take the norm of
    // the result without another pass over it (wd_cg.cu)
    const long long cb_raw = blk * EO_THREADS + threadIdx.x;
    const bool valid = cb_raw < Vh;
    if (!valid && !norm_part && !dot_part) return;
    const long long cb = valid ? cb_raw : Vh - 1; // (only the last CTA has such threads; they redo a site and drop it)
    const long long Vhp = padded_volume(Vh); // sites per right-hand side of a half field
    in += (long long)rhs * 24 * Vhp;
    out += (long long)rhs * 24 * Vhp;

    const int Lxh = Lx / 2;
    long long rem = cb;
    const int xh = (int)(rem % Lxh); rem /= Lxh;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const int t = (int)(rem / Lz);
    const int x = 2 * xh + ((y + z + t + parity) & 1);
    const long long sy = Lx, sz = (long long)Lx * Ly, st = (long long)Lx * Ly * Lz;
    const long long site = x + sy * y + sz * z + st * t; // full-lattice index (links)
    const long long xf = site + (x + 1 == Lx ? -(long long)(Lx - 1) : 1), xb = site + (x == 0 ? (long long)(Lx - 1) : -1);
    const long long yf = site + (y + 1 == Ly ? -(Ly - 1) * sy : sy), yb = site + (y == 0 ? (Ly - 1) * sy : -sy);
    const long long zf = site + (z + 1 == Lz ? -(Lz - 1) * sz : sz), zb = site + (z == 0 ? (Lz - 1) * sz : -sz);
    const long long tf = site + (t + 1 == Lt ? -(Lt - 1) * st : st), tb = site + (t == 0 ? (Lt - 1) * st : -st);

    T acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = (T)0;
    T u[18], p[24];
    // neighbours have the opposite parity; their half-field index is lex / 2.  links_p / links_q: link records of the sites
    // of parity p / 1-p in half-field order, so that a warp's forward links (own sites) and daggered links (neighbour sites)
    // are 32 consecutive 16-byte lanes like its spinors (with the full-lattice link array they were every other lane)
    load_link<0, T, RECON>(links_p, cb, u);      load_spinor(in, xf >> 1, p); hop_forward_s<0, SGN>(acc, u, p);
    load_link<0, T, RECON>(links_q, xb >> 1, u); load_spinor(in, xb >> 1, p); hop_backward_s<0, SGN>(acc, u, p);
    load_link<1, T, RECON>(links_p, cb, u);      load_spinor(in, yf >> 1, p); hop_forward_s<1, SGN>(acc, u, p);
    load_link<1, T, RECON>(links_q, yb >> 1, u); load_spinor(in, yb >> 1, p); hop_backward_s<1, SGN>(acc, u, p);
    load_link<2, T, RECON>(links_p, cb, u);      load_spinor(in, zf >> 1, p); hop_forward_s<2, SGN>(acc, u, p);
    load_link<2, T, RECON>(links_q, zb >> 1, u); load_spinor(in, zb >> 1, p); hop_backward_s<2, SGN>(acc, u, p);
    // tgauge: the caller's links are in temporal gauge (U_t(x,t) = 1 for t < Lt-1; Fig. 4 "GF"): those
    // links are neither loaded nor multiplied -- a quarter of the link bytes
    load_spinor(in, tf >> 1, p);
    if (tgauge && t != Lt - 1) {
        T h[12];
        project<3, SGN>(p, h);
        reconstruct_add<3, SGN>(acc, h);
    } else {
        load_link<3, T, RECON>(links_p, cb, u);
        hop_forward_s<3, SGN>(acc, u, p);
    }
    load_spinor(in, tb >> 1, p);
    if (tgauge && t != 0) {
        T h[12];
        project<3, -SGN>(p, h);
        reconstruct_add<3, -SGN>(acc, h);
    } else {
        load_link<3, T, RECON>(links_q, tb >> 1, u);
        hop_backward_s<3, SGN>(acc, u, p);
    }

    if (xin) {
        load_spinor(xin + (long long)rhs * 24 * Vhp, cb, p);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = fma(alpha, p[i], beta * acc[i]);
    } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = beta * acc[i];
    }
    if (valid) store_spinor(out, cb, acc);
    if (norm_part) {
        __shared__ double sh[EO_THREADS / 32];
        double s2 = 0.0;
        if (valid)
#pragma unroll
            for (int i = 0; i < 24; ++i) s2 += (double)acc[i] * acc[i];
        for (int o = 16; o > 0; o >>= 1) s2 += __shfl_down_sync(0xffffffffu, s2, o);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s2;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
#pragma unroll
            for (int i = 0; i < EO_THREADS / 32; ++i) t += sh[i];
            norm_part[(long long)rhs * nblk + blk] = t;
        }
    }
    // dot_part (may be NULL; one right-hand side): per-CTA partials of <y, out> = sum conj(y) out over the sites, real parts in
    // [0, nblk), imaginary parts in [nblk, 2 nblk) -- the inner products BiCGstab takes with the result of a matvec
    if (dot_part) {
        __shared__ double shd[2][EO_THREADS / 32];
        double re = 0.0, im = 0.0;
        if (valid) {
            load_spinor(dot_y, cb, p);
#pragma unroll
            for (int i = 0; i < 24; i += 2) {
                re += (double)p[i] * acc[i] + (double)p[i + 1] * acc[i + 1];
                im += (double)p[i] * acc[i + 1] - (double)p[i + 1] * acc[i];
            }
        }
        for (int o = 16; o > 0; o >>= 1) {
            re += __shfl_down_sync(0xffffffffu, re, o);
            im += __shfl_down_sync(0xffffffffu, im, o);
        }
        if ((threadIdx.x & 31) == 0) {
            shd[0][threadIdx.x >> 5] = re;
            shd[1][threadIdx.x >> 5] = im;
        }
        __syncthreads();
        if (threadIdx.x < 2) {
            double t = 0.0;
#pragma unroll
            for (int i = 0; i < EO_THREADS / 32; ++i) t += shd[threadIdx.x][i];
            dot_part[threadIdx.x * nblk + blk] = t;
        }
    }
}

// Several right-hand sides: NR of them per thread, so that a link is loaded (and, for 12- / 8-real links, rebuilt) once for
// NR hops.  gridDim.x = (site blocks) * (groups of NR right-hand sides), the group FASTEST as above.  Per right-hand side
// the arithmetic and its order are those of dslash_eo_kernel.  No inner-product epilogue (one right-hand side only).
template <typename T, int RECON, int SGN, int NR>
__global__ void __launch_bounds__(EO_THREADS)
dslash_eo_nr_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ xin, const T *__restrict__ links_p,
                    const T *__restrict__ links_q, int Lx, int Ly, int Lz, int Lt, long long Vh, T alpha, T beta, int parity,
                    double *__restrict__ norm_part, int nrhs, int tgauge)
{
    const unsigned ngroups = (unsigned)((nrhs + NR - 1) / NR);
    const int rhs0 = (int)(blockIdx.x % ngroups) * NR;
    const long long blk = blockIdx.x / ngroups, nblk = gridDim.x / ngroups;
    const long long cb_raw = blk * EO_THREADS + threadIdx.x;
    const bool valid = cb_raw < Vh;
    if (!valid && !norm_part) return;
    const long long cb = valid ? cb_raw : Vh - 1;
    const long long Vhp = padded_volume(Vh), fs = 24 * Vhp; // reals per right-hand side of a half field
    in += (long long)rhs0 * fs;
    out += (long long)rhs0 * fs;
    const int nr = nrhs - rhs0 < NR ? nrhs - rhs0 : NR; // live right-hand sides of this group (uniform in the CTA)

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

    T acc[NR][24];
#pragma unroll
    for (int r = 0; r < NR; ++r)
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[r][i] = (T)0;
    T u[18], p[24];
#define WD_EO_NR_HOP(MU, LINKS, LSITE, NB, FWD)                                                              \
    load_link<MU, T, RECON>(LINKS, LSITE, u);                                                                \
    _Pragma("unroll") for (int r = 0; r < NR; ++r) if (r < nr) {                                             \
        load_spinor(in + r * fs, (NB) >> 1, p);                                                              \
        if (FWD) hop_forward_s<MU, SGN>(acc[r], u, p);                                                       \
        else hop_backward_s<MU, SGN>(acc[r], u, p);                                                          \
    }
    WD_EO_NR_HOP(0, links_p, cb, xf, true)
    WD_EO_NR_HOP(0, links_q, xb >> 1, xb, false)
    WD_EO_NR_HOP(1, links_p, cb, yf, true)
    WD_EO_NR_HOP(1, links_q, yb >> 1, yb, false)
    WD_EO_NR_HOP(2, links_p, cb, zf, true)
    WD_EO_NR_HOP(2, links_q, zb >> 1, zb, false)
    if (tgauge && t != Lt - 1) { // unit link (temporal gauge): projection and reconstruction only
#pragma unroll
        for (int r = 0; r < NR; ++r)
            if (r < nr) {
                T h[12];
                load_spinor(in + r * fs, tf >> 1, p);
                project<3, SGN>(p, h);
                reconstruct_add<3, SGN>(acc[r], h);
            }
    } else {
        WD_EO_NR_HOP(3, links_p, cb, tf, true)
    }
    if (tgauge && t != 0) {
#pragma unroll
        for (int r = 0; r < NR; ++r)
            if (r < nr) {
                T h[12];
                load_spinor(in + r * fs, tb >> 1, p);
                project<3, -SGN>(p, h);
                reconstruct_add<3, -SGN>(acc[r], h);
            }
    } else {
        WD_EO_NR_HOP(3, links_q, tb >> 1, tb, false)
    }
#undef WD_EO_NR_HOP

    __shared__ double sh[NR][EO_THREADS / 32];
#pragma unroll
    for (int r = 0; r < NR; ++r)
        if (r < nr) {
            if (xin) {
                load_spinor(xin + (long long)(rhs0 + r) * fs, cb, p);
#pragma unroll
                for (int i = 0; i < 24; ++i) acc[r][i] = fma(alpha, p[i], beta * acc[r][i]);
            } else {
#pragma unroll
                for (int i = 0; i < 24; ++i) acc[r][i] = beta * acc[r][i];
            }
            if (valid) store_spinor(out + r * fs, cb, acc[r]);
            if (norm_part) {
                double s2 = 0.0;
                if (valid)
#pragma unroll
                    for (int i = 0; i < 24; ++i) s2 += (double)acc[r][i] * acc[r][i];
                for (int o = 16; o > 0; o >>= 1) s2 += __shfl_down_sync(0xffffffffu, s2, o);
                if ((threadIdx.x & 31) == 0) sh[r][threadIdx.x >> 5] = s2;
            }
        }
    if (norm_part) {
        __syncthreads();
        if (threadIdx.x < nr) {
            double tt = 0.0;
#pragma unroll
            for (int i = 0; i < EO_THREADS / 32; ++i) tt += sh[threadIdx.x][i];
            norm_part[(long long)(rhs0 + threadIdx.x) * nblk + blk] = tt;
        }
    }
}

template <typename T, int RECON>
static cudaError_t launch_eo_t(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger,
                               double *norm_part, const void *dot_y, double *dot_part)
{
    if (dot_part && (a.nrhs != 1 || !dot_y)) return cudaErrorInvalidValue;
    const long long Vh = a.V / 2;
    const long long nb = (Vh + EO_THREADS - 1) / EO_THREADS;
    if (nb * a.nrhs > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (!a.links_eo) return cudaErrorInvalidValue; // the API builds the parity-ordered links before any red/black launch
    if (a.nrhs >= 2 && !dot_part) { // several right-hand sides: NR per thread share every link load
        constexpr int NR = sizeof(T) == 4 ? WD_EO_NR32 : WD_EO_NR64;
        const long long ng = (a.nrhs + NR - 1) / NR;
        const char *le = (const char *)a.links_eo;
        const size_t half = eo_links_half_bytes(a.V, a.precision, a.recon);
        auto kn = dagger ? dslash_eo_nr_kernel<T, RECON, +1, NR> : dslash_eo_nr_kernel<T, RECON, -1, NR>;
        kn<<<(unsigned)(nb * ng), EO_THREADS, 0, a.stream>>>((T *)a.out, (const T *)a.in, (const T *)xin, (const T *)(le + parity * half),
                                                            (const T *)(le + (1 - parity) * half), a.dims[0], a.dims[1], a.dims[2],
                                                            a.dims[3], Vh, (T)alpha, (T)beta, parity, norm_part, a.nrhs, a.tgauge);
        count_launch();
        return cudaGetLastError();
    }
    dim3 grid((unsigned)(nb * a.nrhs));
    auto kern = dagger ? dslash_eo_kernel<T, RECON, +1> : dslash_eo_kernel<T, RECON, -1>;
    if (!a.links_eo) return cudaErrorInvalidValue; // the API builds the parity-ordered links before any red/black launch
    const char *le = (const char *)a.links_eo;
    const size_t half = eo_links_half_bytes(a.V, a.precision, a.recon);
    kern<<<grid, EO_THREADS, 0, a.stream>>>((T *)a.out, (const T *)a.in, (const T *)xin, (const T *)(le + parity * half),
                                             (const T *)(le + (1 - parity) * half), a.dims[0],
                                             a.dims[1], a.dims[2], a.dims[3], Vh, (T)alpha, (T)beta, parity, norm_part, a.nrhs,
                                             (const T *)dot_y, dot_part, a.tgauge);
    count_launch();
    return cudaGetLastError();
}

// out_p = alpha * xin_p + beta * (sum of the eight projected, link-multiplied hops from parity 1-p); xin may be NULL
// norm_part: NULL, or ceil(Vh / 128) * nrhs doubles that receive per-CTA partial sums of |out|^2
// dot_part:  NULL, or 2 * ceil(Vh / 128) doubles that receive per-CTA partial sums of <dot_y, out> (nrhs = 1)
cudaError_t launch_eo(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger,
                      double *norm_part, const void *dot_y, double *dot_part)
{
    if (a.precision == 16) // half storage: no epilogues (the solvers do not run on it)
        return norm_part || dot_part ? cudaErrorInvalidValue : launch_eo_half(a, xin, alpha, beta, parity, dagger);
    if (a.precision == 32)
        return a.recon == 18 ? launch_eo_t<float, 18>(a, xin, alpha, beta, parity, dagger, norm_part, dot_y, dot_part)
               : a.recon == 12 ? launch_eo_t<float, 12>(a, xin, alpha, beta, parity, dagger, norm_part, dot_y, dot_part)
                               : launch_eo_t<float, 8>(a, xin, alpha, beta, parity, dagger, norm_part, dot_y, dot_part);
    return a.recon == 18 ? launch_eo_t<double, 18>(a, xin, alpha, beta, parity, dagger, norm_part, dot_y, dot_part)
           : a.recon == 12 ? launch_eo_t<double, 12>(a, xin, alpha, beta, parity, dagger, norm_part, dot_y, dot_part)
                           : launch_eo_t<double, 8>(a, xin, alpha, beta, parity, dagger, norm_part, dot_y, dot_part);
}

// ---- parity-ordered link records (pure data movement) ----
size_t eo_links_half_bytes(long long V, int precision, int recon)
{
    const size_t nvec = (size_t)recon * (size_t)(precision / 8) / 4; // 16-byte vectors per site: four links of `recon` reals
    return (size_t)((V / 2 + BLK - 1) / BLK) * nvec * BLK * 16;
}

__global__ void links_to_eo_kernel(uint4 *__restrict__ dst, const uint4 *__restrict__ src, int Lx, int Ly, int Lz, long long V,
                                   int nvec, long long half_vecs)
{
    const long long site = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= V) return;
    long long rem = site;
    const int x = (int)(rem % Lx); rem /= Lx;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const long long t = rem / Lz;
    const int par = (int)((x + y + z + t) & 1);
    const long long cb = site >> 1;
    const uint4 *q = src + (site >> 5) * ((long long)nvec * BLK) + (site & (BLK - 1));
    uint4 *d = dst + par * half_vecs + (cb >> 5) * ((long long)nvec * BLK) + (cb & (BLK - 1));
    for (int v = 0; v < nvec; ++v) d[(long long)v * BLK] = q[(long long)v * BLK];
}

cudaError_t launch_links_to_eo(void *links_eo, const void *links, const int dims[4], long long V, int precision, int recon,
                               cudaStream_t s)
{
    const int nvec = recon * (precision / 8) / 4;
    const long long half_vecs = (long long)(eo_links_half_bytes(V, precision, recon) / 16);
    links_to_eo_kernel<<<(unsigned)((V + 127) / 128), 128, 0, s>>>((uint4 *)links_eo, (const uint4 *)links, dims[0], dims[1], dims[2],
                                                                   V, nvec, half_vecs);
    count_launch();
    return cudaGetLastError();
}

// canonical full-lattice field <-> native half field of one parity (pure data movement)
template <typename T, bool TO_NATIVE>
__global__ void parity_copy_kernel(T *__restrict__ native, T *__restrict__ canon, int Lx, int Ly, int Lz, long long V,
                                   int parity)
{
    using L = SpinorLayout<T>;
    const long long Vh = V / 2, Vhp = padded_volume(Vh);
    const long long cb = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    const int Lxh = Lx / 2;
    long long rem = cb;
    const int xh = (int)(rem % Lxh); rem /= Lxh;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const long long t = rem / Lz;
    const int x = 2 * xh + (int)((y + z + t + parity) & 1);
    const long long site = x + (long long)Lx * (y + (long long)Ly * (z + (long long)Lz * t));
    T *c = canon + ((long long)blockIdx.y * V + site) * 24;
    typename L::Vec *q = reinterpret_cast<typename L::Vec *>(native + (long long)blockIdx.y * 24 * Vhp) +
                         (cb >> 5) * (L::NCH * BLK) + (cb & (BLK - 1));
#pragma unroll
    for (int v = 0; v < L::NCH; ++v) {
        if (TO_NATIVE) {
            typename L::Vec w;
            pack(w, c + v * L::CR);
            q[v * BLK] = w;
        } else {
            unpack(q[v * BLK], c + v * L::CR);
        }
    }
}

cudaError_t launch_parity_copy(void *native, void *canon, const int dims[4], long long V, int nrhs, int precision,
                               int parity, bool to_native, cudaStream_t s)
{
    const long long Vh = V / 2;
    if (Vh <= 0 || nrhs <= 0) return cudaSuccess;
    dim3 grid((unsigned)((Vh + 127) / 128), (unsigned)nrhs);
    if (precision == 32) {
        if (to_native) parity_copy_kernel<float, true><<<grid, 128, 0, s>>>((float *)native, (float *)canon, dims[0], dims[1], dims[2], V, parity);
        else parity_copy_kernel<float, false><<<grid, 128, 0, s>>>((float *)native, (float *)canon, dims[0], dims[1], dims[2], V, parity);
    } else {
        if (to_native) parity_copy_kernel<double, true><<<grid, 128, 0, s>>>((double *)native, (double *)canon, dims[0], dims[1], dims[2], V, parity);
        else parity_copy_kernel<double, false><<<grid, 128, 0, s>>>((double *)native, (double *)canon, dims[0], dims[1], dims[2], V, parity);
    }
    count_launch();
    return cudaGetLastError();
}

} // namespace wd
