// wd_transfer.cu -- transfer operators of the adaptive multigrid set-up (first cut): eq. (2.7) of arXiv:0912.2186
// on 4^4 space-time blocks with the chirality split of PAPER.md:116.
//
//   wd_block_orthonormalise : N_v global vectors -> P_{x; xhat, alpha} = orthonormal basis of { theta_xhat(x) psi^(alpha)_x },
//                             modified Gram-Schmidt over alpha in the given order inside every (block, chirality)
//                             (the reading of oracle/wd_coarsen.py), in place
//   wd_restrict  (P^dagger) : c[block][sigma][alpha] = sum_{x in block, spin in sigma, colour} conj(W_alpha(x)) psi(x)
//   wd_prolong   (P)        : psi(x) = sum_alpha c[block(x)][sigma(spin)][alpha] W_alpha(x)
//
// One CTA of 256 threads per block, one thread per site of the block (x fastest); fields in the native blocked layout
// (wd_layout.cuh), the N_v vectors as N_v right-hand sides of one buffer.  Inner products are accumulated in fp64 and
// reduced in a fixed order (deterministic).  Coarse vectors: [bt][bz][by][bx][sigma 0..1][alpha][re, im] in the working
// precision.  Set-up code: simple and correct first, it is not on the timed matvec path.
#include "wd_internal.h"
#include "wd_layout.cuh"

namespace wd {

namespace {

constexpr int TB = 256; // 4^4 sites per block

// sum of v over the CTA, returned to every thread; fixed order
__device__ __forceinline__ double cta_sum(double v, double *sh)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads(); // sh may still be read from the previous call
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < TB / 32; ++i) s += sh[i];
    return s;
}

// lexicographic site of thread `tid` of block `b`
__device__ __forceinline__ long long block_site(int tid, long long b, int Lx, int Ly, int Lz)
{
    const int nbx = Lx / 4, nby = Ly / 4, nbz = Lz / 4;
    const int bx = (int)(b % nbx), by = (int)((b / nbx) % nby), bz = (int)((b / ((long long)nbx * nby)) % nbz);
    const long long bt = b / ((long long)nbx * nby * nbz);
    const int x = bx * 4 + (tid & 3), y = by * 4 + ((tid >> 2) & 3), z = bz * 4 + ((tid >> 4) & 3);
    const long long t = bt * 4 + (tid >> 6);
    return x + (long long)Lx * (y + (long long)Ly * (z + (long long)Lz * t));
}

// <a, b> restricted to chirality 0 (reals 0..11) and 1 (reals 12..23): d[0..1] = sigma 0 (re, im), d[2..3] = sigma 1
template <typename T> __device__ __forceinline__ void chiral_dots(const T (&a)[24], const T (&b)[24], double (&d)[4])
{
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        double re = 0.0, im = 0.0;
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const double ar = a[s * 12 + 2 * i], ai = a[s * 12 + 2 * i + 1], br = b[s * 12 + 2 * i], bi = b[s * 12 + 2 * i + 1];
            re += ar * br + ai * bi;
            im += ar * bi - ai * br;
        }
        d[2 * s] = re;
        d[2 * s + 1] = im;
    }
}

template <typename T>
__global__ void __launch_bounds__(TB) block_orthonormalise_kernel(T *vecs, int Lx, int Ly, int Lz, long long V, int nv)
{
    __shared__ double sh[TB / 32];
    const long long site = block_site(threadIdx.x, blockIdx.x, Lx, Ly, Lz);
    const long long stride = 24 * padded_volume(V);
    for (int a = 0; a < nv; ++a) {
        T v[24];
        load_spinor_rw(vecs + a * stride, site, v); // coherent loads: this launch rewrites `vecs`
        for (int b = 0; b < a; ++b) { // modified Gram-Schmidt: v -= <w_b, v> w_b with the CURRENT v
            T w[24];
            load_spinor_rw(vecs + b * stride, site, w);
            double d[4];
            chiral_dots(w, v, d);
#pragma unroll
            for (int i = 0; i < 4; ++i) d[i] = cta_sum(d[i], sh);
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int i = 0; i < 6; ++i) {
                    const double wr = w[s * 12 + 2 * i], wi = w[s * 12 + 2 * i + 1];
                    v[s * 12 + 2 * i] = (T)(v[s * 12 + 2 * i] - (d[2 * s] * wr - d[2 * s + 1] * wi));
                    v[s * 12 + 2 * i + 1] = (T)(v[s * 12 + 2 * i + 1] - (d[2 * s] * wi + d[2 * s + 1] * wr));
                }
        }
        double n[2] = {0.0, 0.0};
#pragma unroll
        for (int i = 0; i < 24; ++i) n[i / 12] += (double)v[i] * v[i];
        n[0] = cta_sum(n[0], sh);
        n[1] = cta_sum(n[1], sh);
        const double r0 = rsqrt(n[0]), r1 = rsqrt(n[1]);
#pragma unroll
        for (int i = 0; i < 24; ++i) v[i] = (T)(v[i] * (i < 12 ? r0 : r1));
        store_spinor(vecs + a * stride, site, v);
        __syncthreads(); // the next vector reads this one (same thread, same site: ordering only)
    }
}

// restrict: the N_v inner products are taken CH at a time -- CH independent vector loads in flight, 4*CH partial
// sums reduced by warp shuffles, one shared-memory hand-off (two barriers) per chunk instead of per vector
template <typename T>
__global__ void __launch_bounds__(TB)
restrict_kernel(T *__restrict__ coarse, const T *__restrict__ W, const T *__restrict__ psi, int Lx, int Ly, int Lz, long long V, int nv)
{
    constexpr int CH = 4;
    __shared__ double sh[TB / 32][4 * CH];
    const long long site = block_site(threadIdx.x, blockIdx.x, Lx, Ly, Lz);
    const long long stride = 24 * padded_volume(V);
    T p[24];
    load_spinor(psi, site, p);
    T *c = coarse + ((long long)blockIdx.x * 2 * nv) * 2;
    for (int a0 = 0; a0 < nv; a0 += CH) {
        double d[CH][4];
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            if (a0 + k < nv) { // block-uniform
                T w[24];
                load_spinor(W + (a0 + k) * stride, site, w);
                chiral_dots(w, p, d[k]);
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) d[k][i] = 0.0;
            }
        }
#pragma unroll
        for (int k = 0; k < CH; ++k)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                double v = d[k][i];
                for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
                d[k][i] = v;
            }
        __syncthreads(); // sh free again
        if ((threadIdx.x & 31) == 0)
#pragma unroll
            for (int k = 0; k < CH; ++k)
#pragma unroll
                for (int i = 0; i < 4; ++i) sh[threadIdx.x >> 5][4 * k + i] = d[k][i];
        __syncthreads();
        if (threadIdx.x < 4 * CH) { // thread j finishes sum j = 4*k + i in a fixed order
            double sum = 0.0;
#pragma unroll
            for (int wp = 0; wp < TB / 32; ++wp) sum += sh[wp][threadIdx.x];
            const int k = threadIdx.x >> 2, i = threadIdx.x & 3, a = a0 + k;
            if (a < nv) c[((i >> 1) * nv + a) * 2 + (i & 1)] = (T)sum;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(TB)
prolong_kernel(T *__restrict__ psi, const T *__restrict__ W, const T *__restrict__ coarse, int Lx, int Ly, int Lz, long long V, int nv)
{
    const long long site = block_site(threadIdx.x, blockIdx.x, Lx, Ly, Lz);
    const long long stride = 24 * padded_volume(V);
    const T *c = coarse + ((long long)blockIdx.x * 2 * nv) * 2;
    T acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = (T)0;
    for (int a = 0; a < nv; ++a) {
        T w[24];
        load_spinor(W + a * stride, site, w);
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const T cr = c[(s * nv + a) * 2], ci = c[(s * nv + a) * 2 + 1];
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                const T wr = w[s * 12 + 2 * i], wi = w[s * 12 + 2 * i + 1];
                acc[s * 12 + 2 * i] += cr * wr - ci * wi;
                acc[s * 12 + 2 * i + 1] += cr * wi + ci * wr;
            }
        }
    }
    store_spinor(psi, site, acc);
}

} // namespace

// what: 0 = orthonormalise (a = vecs), 1 = restrict (a = coarse out, b = W, c = psi), 2 = prolong (a = psi out, b = W, c = coarse)
cudaError_t launch_transfer(int what, void *a, const void *b, const void *c, const int dims[4], long long V, int nv,
                            int precision, cudaStream_t s)
{
    const long long nblocks = V / TB;
    if (nblocks < 1 || nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const unsigned g = (unsigned)nblocks;
    if (precision == 32) {
        if (what == 0) block_orthonormalise_kernel<float><<<g, TB, 0, s>>>((float *)a, dims[0], dims[1], dims[2], V, nv);
        else if (what == 1) restrict_kernel<float><<<g, TB, 0, s>>>((float *)a, (const float *)b, (const float *)c, dims[0], dims[1], dims[2], V, nv);
        else prolong_kernel<float><<<g, TB, 0, s>>>((float *)a, (const float *)b, (const float *)c, dims[0], dims[1], dims[2], V, nv);
    } else {
        if (what == 0) block_orthonormalise_kernel<double><<<g, TB, 0, s>>>((double *)a, dims[0], dims[1], dims[2], V, nv);
        else if (what == 1) restrict_kernel<double><<<g, TB, 0, s>>>((double *)a, (const double *)b, (const double *)c, dims[0], dims[1], dims[2], V, nv);
        else prolong_kernel<double><<<g, TB, 0, s>>>((double *)a, (const double *)b, (const double *)c, dims[0], dims[1], dims[2], V, nv);
    }
    count_launch();
    return cudaGetLastError();
}

} // namespace wd
