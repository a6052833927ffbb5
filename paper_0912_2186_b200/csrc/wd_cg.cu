// wd_cg.cu -- Krylov shell around the even-odd matvec: CGNR for  Mhat x = b  on one parity (first cut).
//
// SURVEY.md 8(f) row f2; PAPER.md:116 ("CG on the normal equations"), PAPER.md:153-167 (CG built on the
// even-odd matvec, Table 2).  Algorithm = oracle/wd_solvers.py:cgnr_schur, step for step:
//     x = 0, r = b, z = Mhat^dag r, p = z, zz = <z,z>
//     loop:  w = Mhat p;  alpha = zz/<w,w>;  x += alpha p;  r -= alpha w;  z = Mhat^dag r;
//            zz' = <z,z>;  beta = zz'/zz;  p = z + beta p
// (<w,w> and <z,z> are produced by the epilogue of the matvec kernel itself: no extra pass over w and z)
// B200 shape of it: the whole iteration is enqueued on the gauge's stream with NO host synchronisation -- every
// scalar lives in device memory.  Reductions are deterministic two-level sums in fp64: each of RED_BLOCKS CTAs
// writes one partial in a fixed order, and every CTA of the kernel that needs the scalar re-adds the partials
// itself (a few hundred L2-resident doubles) instead of a separate finalise launch.  The host only reads the
// residual history back every CHECK iterations when a tolerance is set.
#include <cmath>
#include <cstdio>
#include <vector>
#include "wd_internal.h"
#include "wd_layout.cuh"

namespace wd {

namespace {

constexpr int RED_BLOCKS = 592; // 4 CTAs of 256 threads per SM on 148 SMs
constexpr int RED_THREADS = 256;

// Sum of the RED_BLOCKS partials, the same bits in every CTA and every run: warp 0 adds them in a fixed
// pattern (lane l takes partials l, l+32, ... in order, then a fixed shuffle tree) and broadcasts through shared
// memory.  Every thread of the CTA must call it (it contains a barrier).
__device__ __forceinline__ double sum_partials(const double *part, int n = RED_BLOCKS)
{
    __shared__ double total;
    if (n > 2048) { // the per-CTA partials of a matvec epilogue (thousands): every warp takes a share, same fixed pattern
        __shared__ double wsum[RED_THREADS / 32];
        double s = 0.0;
        for (int i = threadIdx.x; i < n; i += RED_THREADS) s += part[i];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int i = 0; i < RED_THREADS / 32; ++i) t += wsum[i];
            total = t;
        }
    } else if (threadIdx.x < 32) {
        double s = 0.0;
        for (int i = threadIdx.x; i < n; i += 32) s += part[i];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) total = s;
    }
    __syncthreads();
    const double t = total;
    __syncthreads(); // `total` may be reused by the next call
    return t;
}

// a / b with the breakdown guard of the solvers: an exact zero denominator (b = 0 right-hand side, a converged or
// broken-down recurrence) gives a zero step instead of 0/0 = NaN in x
__device__ __forceinline__ double safe_div(double a, double b) { return b != 0.0 ? a / b : 0.0; }

__device__ __forceinline__ double block_sum(double v, double *sh)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < RED_THREADS / 32; ++i) s += sh[i];
    return s; // valid in thread 0
}

template <typename Vec> __device__ __forceinline__ double norm2_vec(const Vec &v);
template <> __device__ __forceinline__ double norm2_vec<float4>(const float4 &v)
{
    return (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z + (double)v.w * v.w;
}
template <> __device__ __forceinline__ double norm2_vec<double2>(const double2 &v) { return v.x * v.x + v.y * v.y; }

__device__ __forceinline__ float4 axpy_vec(double a, const float4 &x, const float4 &y)
{
    const float f = (float)a;
    return make_float4(fmaf(f, x.x, y.x), fmaf(f, x.y, y.y), fmaf(f, x.z, y.z), fmaf(f, x.w, y.w));
}
__device__ __forceinline__ double2 axpy_vec(double a, const double2 &x, const double2 &y)
{
    return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y));
}

// is vector index i (layout [block][vector][lane], NCH vectors per site) a real site (not a pad lane)?
template <int NCH> __device__ __forceinline__ bool real_site(long long i, long long Vh)
{
    return (i / (NCH * BLK)) * BLK + (i % BLK) < Vh;
}

// part[b] = sum over this CTA's grid-stride share of |v|^2
template <typename Vec, int NCH>
__global__ void __launch_bounds__(RED_THREADS) norm2_kernel(const Vec *v, long long nvec, long long Vh, double *part)
{
    // blockIdx.y = right-hand side of a block solve (fields nvec apart, partials RED_BLOCKS apart); 0 for one right-hand side
    v += (long long)blockIdx.y * nvec;
    part += (long long)blockIdx.y * RED_BLOCKS;
    __shared__ double sh[RED_THREADS / 32];
    double s = 0.0;
    constexpr int UNR = 4;
    const long long stride = (long long)RED_BLOCKS * RED_THREADS;
    for (long long i0 = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i0 < nvec; i0 += UNR * stride) {
        Vec vv[UNR];
#pragma unroll
        for (int u = 0; u < UNR; ++u)
            if (i0 + u * stride < nvec) vv[u] = v[i0 + u * stride];
#pragma unroll
        for (int u = 0; u < UNR; ++u)
            if (i0 + u * stride < nvec && real_site<NCH>(i0 + u * stride, Vh)) s += norm2_vec(vv[u]);
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// alpha = zz / ww;  r -= alpha w;  rr_part = |r|^2 partials   (x += alpha p is done by update_px_kernel, which reads p anyway)
template <typename Vec, int NCH>
__global__ void __launch_bounds__(RED_THREADS)
update_r_kernel(Vec *r, const Vec *w, long long nvec, long long Vh, const double *zz_part, const double *ww_part, int npart,
                double *rr_part)
{
    {   // blockIdx.y = right-hand side of a block solve
        const long long rhs = blockIdx.y;
        r += rhs * nvec; w += rhs * nvec;
        zz_part += rhs * npart; ww_part += rhs * npart; rr_part += rhs * RED_BLOCKS;
    }
    __shared__ double sh[RED_THREADS / 32];
    const double alpha = safe_div(sum_partials(zz_part, npart), sum_partials(ww_part, npart));
    double s = 0.0;
    constexpr int UNR = 4; // independent vectors per thread and trip
    const long long stride = (long long)RED_BLOCKS * RED_THREADS;
    for (long long i0 = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i0 < nvec; i0 += UNR * stride) {
        Vec wv[UNR], rv[UNR];
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const long long i = i0 + u * stride;
            if (i < nvec) { wv[u] = w[i]; rv[u] = r[i]; }
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const long long i = i0 + u * stride;
            if (i < nvec) {
                const Vec rn = axpy_vec(-alpha, wv[u], rv[u]);
                r[i] = rn;
                if (real_site<NCH>(i, Vh)) s += norm2_vec(rn);
            }
        }
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) rr_part[blockIdx.x] = s;
}

// alpha = zz_old / ww (the step just taken);  x += alpha p;  beta = zz_new / zz_old;  p = z + beta p;
// hist[k] = sqrt(rr) (block 0)
template <typename Vec>
__global__ void __launch_bounds__(RED_THREADS)
update_px_kernel(Vec *x, Vec *p, const Vec *z, long long nvec, const double *zz_new_part, const double *zz_old_part,
                 const double *ww_part, int npart, const double *rr_part, double *hist_k, long long hist_stride = 0)
{
    {   // blockIdx.y = right-hand side of a block solve
        const long long rhs = blockIdx.y;
        x += rhs * nvec; p += rhs * nvec; z += rhs * nvec;
        zz_new_part += rhs * npart; zz_old_part += rhs * npart; ww_part += rhs * npart; rr_part += rhs * RED_BLOCKS;
        hist_k += rhs * hist_stride;
    }
    const double zz_old = sum_partials(zz_old_part, npart);
    const double alpha = safe_div(zz_old, sum_partials(ww_part, npart));
    const double beta = safe_div(sum_partials(zz_new_part, npart), zz_old);
    if (blockIdx.x == 0) { // (block-uniform branch: sum_partials has barriers)
        const double rr = sum_partials(rr_part);
        if (threadIdx.x == 0) *hist_k = sqrt(rr);
    }
    constexpr int UNR = 2; // three streams x 2 loads in flight
    const long long stride = (long long)RED_BLOCKS * RED_THREADS;
    for (long long i0 = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i0 < nvec; i0 += UNR * stride) {
        Vec pv[UNR], zv[UNR], xv[UNR];
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const long long i = i0 + u * stride;
            if (i < nvec) { pv[u] = p[i]; zv[u] = z[i]; xv[u] = x[i]; }
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            const long long i = i0 + u * stride;
            if (i < nvec) {
                x[i] = axpy_vec(alpha, pv[u], xv[u]);
                p[i] = axpy_vec(beta, pv[u], zv[u]);
            }
        }
    }
}

template <typename Vec>
__global__ void __launch_bounds__(RED_THREADS) zero_kernel(Vec *__restrict__ v, long long nvec)
{
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS) v[i] = Vec{};
}

__global__ void sqrt_of_sum_kernel(const double *part, double *out, long long out_stride = 0) // one CTA of 32 threads per RHS
{
    part += (long long)blockIdx.x * RED_BLOCKS;
    out += (long long)blockIdx.x * out_stride;
    const double t = sum_partials(part);
    if (threadIdx.x == 0) *out = sqrt(t);
}

// ---- BiCGstab pieces: complex inner products on the (re, im) pair layout, scalars as double2 in device memory ----
struct cplxd {
    double re, im;
};
__device__ __forceinline__ cplxd cmul(cplxd a, cplxd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cplxd cdiv(cplxd a, cplxd b)
{
    const double d = b.re * b.re + b.im * b.im;
    if (d == 0.0) return {0.0, 0.0}; // breakdown guard (see safe_div)
    return {(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}
__device__ __forceinline__ cplxd sum_partials_c(const double *part, int n = RED_BLOCKS) // part[0..n) = re, part[n..2n) = im
{
    cplxd r;
    r.re = sum_partials(part, n);
    r.im = sum_partials(part + n, n);
    return r;
}

// conj(a) * b summed over the complex numbers of one vector
__device__ __forceinline__ void cdot_vec(const float4 &a, const float4 &b, double &re, double &im)
{
    re += (double)a.x * b.x + (double)a.y * b.y + (double)a.z * b.z + (double)a.w * b.w;
    im += (double)a.x * b.y - (double)a.y * b.x + (double)a.z * b.w - (double)a.w * b.z;
}
__device__ __forceinline__ void cdot_vec(const double2 &a, const double2 &b, double &re, double &im)
{
    re += a.x * b.x + a.y * b.y;
    im += a.x * b.y - a.y * b.x;
}
// y + c * x for complex c
__device__ __forceinline__ float4 caxpy_vec(cplxd c, const float4 &x, const float4 &y)
{
    const float cr = (float)c.re, ci = (float)c.im;
    return make_float4(y.x + cr * x.x - ci * x.y, y.y + cr * x.y + ci * x.x, y.z + cr * x.z - ci * x.w, y.w + cr * x.w + ci * x.z);
}
__device__ __forceinline__ double2 caxpy_vec(cplxd c, const double2 &x, const double2 &y)
{
    return make_double2(y.x + c.re * x.x - c.im * x.y, y.y + c.re * x.y + c.im * x.x);
}

// part = <a, b> (and, if TT, part2 = <a, a>) partials
template <typename Vec, int NCH, bool TT>
__global__ void __launch_bounds__(RED_THREADS)
cdot_kernel(const Vec *__restrict__ a, const Vec *__restrict__ b, long long nvec, long long Vh, double *part, double *part2)
{
    __shared__ double sh[RED_THREADS / 32];
    double re = 0.0, im = 0.0, aa = 0.0;
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS)
        if (real_site<NCH>(i, Vh)) {
            const Vec av = a[i], bv = b[i];
            cdot_vec(av, bv, re, im);
            if (TT) aa += norm2_vec(av);
        }
    re = block_sum(re, sh);
    __syncthreads();
    im = block_sum(im, sh);
    __syncthreads();
    if (TT) aa = block_sum(aa, sh);
    if (threadIdx.x == 0) {
        part[blockIdx.x] = re;
        part[RED_BLOCKS + blockIdx.x] = im;
        if (TT) part2[blockIdx.x] = aa;
    }
}

// scal = {rho, alpha, omega} (device).  rho' = sum(rho_part); beta = (rho'/rho)(alpha/omega); p = r + beta (p - omega v);
// block 0 stores rho <- rho' and the residual norm of the previous iteration into *hist_k
template <typename Vec>
__global__ void __launch_bounds__(RED_THREADS)
bicg_p_kernel(Vec *__restrict__ p, const Vec *__restrict__ r, const Vec *__restrict__ v, long long nvec, const double *rho_part,
              cplxd *scal, const double *rr_part, double *hist_k)
{
    const cplxd rho_new = sum_partials_c(rho_part);
    const cplxd rho = scal[0], alpha = scal[1], omega = scal[2];
    const cplxd beta = cmul(cdiv(rho_new, rho), cdiv(alpha, omega));
    const cplxd mbo = {-(beta.re * omega.re - beta.im * omega.im), -(beta.re * omega.im + beta.im * omega.re)};
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS)
        p[i] = caxpy_vec(mbo, v[i], caxpy_vec(beta, p[i], r[i])); // r + beta p - beta omega v
    if (blockIdx.x == 0) {
        const double rr = sum_partials(rr_part);
        __syncthreads(); // every thread has read scal[0] before it is overwritten
        if (threadIdx.x == 0) {
            scal[3] = rho_new; // becomes rho after the alpha kernel (other CTAs may still be reading scal[0])
            *hist_k = sqrt(rr);
        }
    }
}

// alpha = rho' / <rhat, v>;  s = r - alpha v  (s overwrites r);  block 0 stores alpha and rho <- rho'
template <typename Vec>
__global__ void __launch_bounds__(RED_THREADS)
bicg_s_kernel(Vec *__restrict__ r, const Vec *__restrict__ v, long long nvec, const double *rv_part, int npart, cplxd *scal)
{
    const cplxd alpha = cdiv(scal[3], sum_partials_c(rv_part, npart)); // <rhat, v> from the epilogue of the matvec that made v
    const cplxd ma = {-alpha.re, -alpha.im};
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS)
        r[i] = caxpy_vec(ma, v[i], r[i]);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        scal[1] = alpha;
        scal[0] = scal[3];
    }
}

// omega = <t, s> / <t, t>;  x += alpha p + omega s;  r = s - omega t (s lives in r);  |r|^2 partials; block 0 stores omega.
// st_part = per-CTA partials of <s, t> from the epilogue of the matvec that made t (<t, s> is its conjugate), tt_part those
// of |t|^2; rho_part receives the partials of <rhat, r> for the next iteration (rhat is read here instead of in a kernel
// of its own)
template <typename Vec, int NCH>
__global__ void __launch_bounds__(RED_THREADS)
bicg_x_kernel(Vec *__restrict__ x, Vec *__restrict__ r, const Vec *__restrict__ p, const Vec *__restrict__ t,
              const Vec *__restrict__ rhat, long long nvec, long long Vh, const double *st_part, const double *tt_part, int npart,
              cplxd *scal, double *rr_part, double *rho_part)
{
    __shared__ double sh[RED_THREADS / 32];
    const cplxd st = sum_partials_c(st_part, npart);
    const double tt = sum_partials(tt_part, npart);
    const cplxd omega = {safe_div(st.re, tt), safe_div(-st.im, tt)};
    const cplxd alpha = scal[1];
    const cplxd mo = {-omega.re, -omega.im};
    double s2 = 0.0, re = 0.0, im = 0.0;
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS) {
        const Vec sv = r[i];
        x[i] = caxpy_vec(omega, sv, caxpy_vec(alpha, p[i], x[i]));
        const Vec rn = caxpy_vec(mo, t[i], sv);
        r[i] = rn;
        if (real_site<NCH>(i, Vh)) {
            s2 += norm2_vec(rn);
            cdot_vec(rhat[i], rn, re, im);
        }
    }
    s2 = block_sum(s2, sh);
    __syncthreads();
    re = block_sum(re, sh);
    __syncthreads();
    im = block_sum(im, sh);
    if (threadIdx.x == 0) {
        rr_part[blockIdx.x] = s2;
        rho_part[blockIdx.x] = re;
        rho_part[RED_BLOCKS + blockIdx.x] = im;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) scal[2] = omega;
}

__global__ void bicg_init_kernel(cplxd *scal)
{
    for (int i = 0; i < 4; ++i) scal[i] = {1.0, 0.0};
}

} // namespace

static cudaError_t ensure_workspace(wd_gauge *g, size_t ws_bytes, size_t nsc);

// nrhs right-hand sides advance in lock step (a block solve): every vector kernel gets a right-hand-side dimension
// (gridDim.y), the operator is applied to all of them in one batched launch (dslash_eo with the right-hand side fastest,
// so a block of links serves all of them), every right-hand side has its own scalars and history.  Per right-hand side the
// arithmetic and its order are those of the single solve: the results are bit-identical to nrhs separate calls.
template <typename T>
static int cgnr_schur_t(wd_gauge *g, const ApplyArgs &shape, void *x_out, const void *b_in, double mass, int parity, int max_iter,
                        double tol, int *iters_out, double *hist_host, cudaError_t *err, int nrhs = 1)
{
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH;
    constexpr int CHECK = 8; // iterations between convergence checks (the only host synchronisations)
    const long long Vh = shape.V / 2;
    const long long nvec = padded_volume(Vh) * NCH;            // vectors per right-hand side
    const size_t hb = (size_t)nvec * sizeof(Vec) * (size_t)nrhs; // bytes of one block of nrhs half fields
    cudaStream_t s = shape.stream;
    const double a0 = 4.0 + mass;
    const long long hs = (long long)max_iter + 1; // history entries per right-hand side

    // workspace lives in the gauge handle (a 0.5 GB cudaMalloc / cudaFree per solve costs up to a second)
    // |Mhat p|^2 and |Mhat^dag r|^2 come out of the matvec's epilogue as one partial per CTA of that kernel
    const int npart = (int)((Vh + 127) / 128);
    const size_t nsc = (size_t)nrhs * (3 * (size_t)npart + RED_BLOCKS + (size_t)hs); // zz_part[2] | ww_part | rr_part | hist
    if ((*err = ensure_workspace(g, 5 * hb, nsc)) != cudaSuccess) return -1;
    char *ws = (char *)g->cg_ws;
    double *sc = g->cg_sc;
    Vec *r = (Vec *)ws, *p = (Vec *)(ws + hb), *z = (Vec *)(ws + 2 * hb), *w = (Vec *)(ws + 3 * hb), *tmp = (Vec *)(ws + 4 * hb);
    Vec *x = (Vec *)x_out;
    const size_t np_all = (size_t)nrhs * npart;
    double *zz_part[2] = {sc, sc + np_all}, *ww_part = sc + 2 * np_all, *rr_part = sc + 3 * np_all;
    double *hist = rr_part + (size_t)nrhs * RED_BLOCKS;
    const dim3 vgrid(RED_BLOCKS, (unsigned)nrhs);

    ApplyArgs a = shape;
    a.nrhs = nrhs;
    // out = Mhat in  or  Mhat^dagger in;  norm_part receives the per-CTA partials of |out|^2
    auto schur = [&](Vec *out, const Vec *in, bool dagger, double *norm_part) -> cudaError_t {
        a.out = tmp;
        a.in = in;
        cudaError_t e = launch_eo(a, nullptr, 0.0, -0.5, 1 - parity, dagger);
        if (e != cudaSuccess) return e;
        a.out = out;
        a.in = tmp;
        return launch_eo(a, in, a0, 0.5 / a0, parity, dagger, norm_part);
    };
    int rc = 0, k = 0;
    std::vector<double> h0(nrhs, 0.0), hk(nrhs, 0.0);
    auto fail_cuda = [&](cudaError_t e) {
        *err = e;
        rc = -1;
    };
    // entry `col` of every right-hand side's history -> host
    auto fetch = [&](std::vector<double> &dst, int col) -> cudaError_t {
        cudaError_t e = cudaMemcpy2DAsync(dst.data(), sizeof(double), hist + col, (size_t)hs * sizeof(double), sizeof(double), nrhs,
                                          cudaMemcpyDeviceToHost, s);
        return e == cudaSuccess ? cudaStreamSynchronize(s) : e;
    };
    do {
        cudaError_t e;
        zero_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(x, nvec * nrhs);
        count_launch();
        if ((e = cudaMemcpyAsync(r, b_in, hb, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) { fail_cuda(e); break; }
        int cur = 0;
        if ((e = schur(z, r, true, zz_part[cur])) != cudaSuccess) { fail_cuda(e); break; }
        if ((e = cudaMemcpyAsync(p, z, hb, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) { fail_cuda(e); break; }
        norm2_kernel<Vec, NCH><<<vgrid, RED_THREADS, 0, s>>>(r, nvec, Vh, rr_part);
        count_launch();
        sqrt_of_sum_kernel<<<nrhs, 32, 0, s>>>(rr_part, hist, hs);
        count_launch();
        if (tol > 0.0) {
            if ((e = fetch(h0, 0)) != cudaSuccess) { fail_cuda(e); break; }
            bool all_zero = true;
            for (double v : h0) all_zero = all_zero && v == 0.0;
            if (all_zero) break; // b = 0: x = 0 is the solution
        }
        for (k = 0; k < max_iter; ++k) {
            if ((e = schur(w, p, false, ww_part)) != cudaSuccess) { fail_cuda(e); break; }
            update_r_kernel<Vec, NCH><<<vgrid, RED_THREADS, 0, s>>>(r, w, nvec, Vh, zz_part[cur], ww_part, npart, rr_part);
            count_launch();
            if ((e = schur(z, r, true, zz_part[cur ^ 1])) != cudaSuccess) { fail_cuda(e); break; }
            update_px_kernel<Vec><<<vgrid, RED_THREADS, 0, s>>>(x, p, z, nvec, zz_part[cur ^ 1], zz_part[cur], ww_part, npart, rr_part,
                                                                 hist + k + 1, hs);
            count_launch();
            cur ^= 1;
            if (tol > 0.0 && ((k + 1) % CHECK == 0 || k + 1 == max_iter)) {
                if ((e = fetch(hk, k + 1)) != cudaSuccess) { fail_cuda(e); break; }
                bool done = true;
                for (int i = 0; i < nrhs; ++i) done = done && hk[i] <= tol * h0[i];
                if (done) {
                    ++k;
                    break;
                }
            }
        }
        if (rc) break;
        if ((e = cudaGetLastError()) != cudaSuccess) { fail_cuda(e); break; }
        if (hist_host) { // [rhs][max_iter + 1], entries 0..k of every right-hand side
            e = cudaMemcpy2DAsync(hist_host, (size_t)hs * sizeof(double), hist, (size_t)hs * sizeof(double), ((size_t)k + 1) * sizeof(double),
                                  nrhs, cudaMemcpyDeviceToHost, s);
            if (e != cudaSuccess) { fail_cuda(e); break; }
        }
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
        if (hist_host)
            for (int i = 0; i < nrhs; ++i) {
                const double n0 = hist_host[(size_t)i * hs];
                if (n0 > 0.0)
                    for (int j = 0; j <= k; ++j) hist_host[(size_t)i * hs + j] /= n0; // relative residual |r_k| / |b|
            }
    } while (false);
    if (iters_out) *iters_out = k;
    return rc;
}

static cudaError_t ensure_workspace(wd_gauge *g, size_t ws_bytes, size_t nsc)
{
    cudaError_t e;
    if (g->cg_ws_bytes < ws_bytes) {
        cudaFree(g->cg_ws);
        g->cg_ws = nullptr;
        g->cg_ws_bytes = 0;
        if ((e = cudaMalloc(&g->cg_ws, ws_bytes)) != cudaSuccess) return e;
        g->cg_ws_bytes = ws_bytes;
    }
    if (g->cg_sc_count < nsc) {
        cudaFree(g->cg_sc);
        g->cg_sc = nullptr;
        g->cg_sc_count = 0;
        if ((e = cudaMalloc(&g->cg_sc, nsc * sizeof(double))) != cudaSuccess) return e;
        g->cg_sc_count = nsc;
    }
    return cudaSuccess;
}

// BiCGstab for Mhat x = b, x_0 = 0: oracle/wd_solvers.py:bicgstab_schur step for step; same execution model as CGNR
template <typename T>
static int bicgstab_schur_t(wd_gauge *g, const ApplyArgs &shape, void *x_out, const void *b_in, double mass, int parity,
                            int max_iter, double tol, int *iters_out, double *hist_host, cudaError_t *err)
{
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH;
    constexpr int CHECK = 8;
    const long long Vh = shape.V / 2;
    const long long nvec = padded_volume(Vh) * NCH;
    const size_t hb = (size_t)nvec * sizeof(Vec);
    cudaStream_t s = shape.stream;
    const double a0 = 4.0 + mass;
    const int npart = (int)((Vh + 127) / 128); // per-CTA partials of the matvec epilogues
    const size_t nsc = 3 * (size_t)RED_BLOCKS + 5 * (size_t)npart + 8 + (size_t)max_iter + 1;
    if ((*err = ensure_workspace(g, 6 * hb, nsc)) != cudaSuccess) return -1;
    char *ws = (char *)g->cg_ws;
    Vec *r = (Vec *)ws, *rhat = (Vec *)(ws + hb), *p = (Vec *)(ws + 2 * hb), *v = (Vec *)(ws + 3 * hb), *t = (Vec *)(ws + 4 * hb),
        *tmp = (Vec *)(ws + 5 * hb);
    Vec *x = (Vec *)x_out;
    double *sc = g->cg_sc;
    double *rho_part = sc, *rr_part = sc + 2 * RED_BLOCKS, *rv_part = sc + 3 * RED_BLOCKS, *st_part = rv_part + 2 * (size_t)npart,
           *tt_part = st_part + 2 * (size_t)npart;
    cplxd *scal = (cplxd *)(tt_part + npart);
    double *hist = (double *)(scal + 4);

    ApplyArgs a = shape;
    // out = Mhat in; the second launch also leaves the per-CTA partials of <y, out> in dot_part and of |out|^2 in norm_part
    auto schur = [&](Vec *out, const Vec *in, const Vec *y, double *dot_part, double *norm_part) -> cudaError_t {
        a.out = tmp;
        a.in = in;
        cudaError_t e = launch_eo(a, nullptr, 0.0, -0.5, 1 - parity, false);
        if (e != cudaSuccess) return e;
        a.out = out;
        a.in = tmp;
        return launch_eo(a, in, a0, 0.5 / a0, parity, false, norm_part, y, dot_part);
    };
    int rc = 0, k = 0;
    double h0 = 0.0;
    auto fail_cuda = [&](cudaError_t e) {
        *err = e;
        rc = -1;
    };
    do {
        cudaError_t e;
        zero_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(x, nvec);
        zero_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(p, nvec);
        zero_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(v, nvec);
        bicg_init_kernel<<<1, 1, 0, s>>>(scal);
        count_launch(4);
        if ((e = cudaMemcpyAsync(r, b_in, hb, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) { fail_cuda(e); break; }
        if ((e = cudaMemcpyAsync(rhat, b_in, hb, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) { fail_cuda(e); break; }
        norm2_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>(r, nvec, Vh, rr_part);
        sqrt_of_sum_kernel<<<1, 32, 0, s>>>(rr_part, hist);
        count_launch(2);
        if (tol > 0.0) {
            if ((e = cudaMemcpyAsync(&h0, hist, sizeof(double), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { fail_cuda(e); break; }
            if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
            if (h0 == 0.0) break;
        }
        // rho_0 = <rhat, r_0>; every later rho comes out of bicg_x_kernel, <rhat, v>, <s, t> and |t|^2 out of the matvec
        // epilogues: 7 launches and 15 spinor passes per iteration (10 and 19 with separate inner-product kernels)
        cdot_kernel<Vec, NCH, false><<<RED_BLOCKS, RED_THREADS, 0, s>>>(rhat, r, nvec, Vh, rho_part, nullptr);
        count_launch();
        for (k = 0; k < max_iter; ++k) {
            bicg_p_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(p, r, v, nvec, rho_part, scal, rr_part, hist + k);
            count_launch();
            if ((e = schur(v, p, rhat, rv_part, nullptr)) != cudaSuccess) { fail_cuda(e); break; }
            bicg_s_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(r, v, nvec, rv_part, npart, scal);
            count_launch();
            if ((e = schur(t, r, r, st_part, tt_part)) != cudaSuccess) { fail_cuda(e); break; }
            bicg_x_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>(x, r, p, t, rhat, nvec, Vh, st_part, tt_part, npart, scal, rr_part,
                                                                      rho_part);
            count_launch();
            if (tol > 0.0 && ((k + 1) % CHECK == 0 || k + 1 == max_iter)) {
                double hk = 0.0;
                sqrt_of_sum_kernel<<<1, 32, 0, s>>>(rr_part, hist + k + 1);
                count_launch();
                if ((e = cudaMemcpyAsync(&hk, hist + k + 1, sizeof(double), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { fail_cuda(e); break; }
                if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
                if (hk <= tol * h0) {
                    ++k;
                    break;
                }
            }
        }
        if (rc) break;
        sqrt_of_sum_kernel<<<1, 32, 0, s>>>(rr_part, hist + k); // |r_k| of the last iterate
        count_launch();
        if ((e = cudaGetLastError()) != cudaSuccess) { fail_cuda(e); break; }
        if (hist_host) {
            if ((e = cudaMemcpyAsync(hist_host, hist, ((size_t)k + 1) * sizeof(double), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { fail_cuda(e); break; }
        }
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
        if (hist_host && hist_host[0] > 0.0) {
            const double n0 = hist_host[0];
            for (int i = 0; i <= k; ++i) hist_host[i] /= n0;
        }
    } while (false);
    if (iters_out) *iters_out = k;
    return rc;
}

int bicgstab_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter,
                   double tol, int *iters_out, double *hist_host, cudaError_t *err)
{
    return shape.precision == 32
               ? bicgstab_schur_t<float>(g, shape, x, b, mass, parity, max_iter, tol, iters_out, hist_host, err)
               : bicgstab_schur_t<double>(g, shape, x, b, mass, parity, max_iter, tol, iters_out, hist_host, err);
}

// ---- GCR(m) pieces ----
constexpr int GCR_GROUP = 8; // earlier directions handled per pass over the new one (GCR(8): all of them)

// part[(2 i + c) * RED_BLOCKS + b] = partials of <q_{i0+i}, q_j> (c = 0 real, 1 imaginary part), i < ni <= GCR_GROUP:
// q_j is read once for all of them.  q_i = qbase + i * stride
// (RED_BLOCKS is 4 CTAs per SM: the register cap keeps all of them resident -- at 80 registers only three fit and the fourth
// ran as a second, nearly empty wave: 116 us for two passes over the vectors where the plain inner-product kernel takes 37)
template <typename Vec, int NCH>
__global__ void __launch_bounds__(RED_THREADS, 4)
gcr_dots_kernel(const Vec *__restrict__ qbase, long long stride, int i0, int ni, const Vec *__restrict__ qj, long long nvec,
                long long Vh, double *part)
{
    __shared__ double sh[RED_THREADS / 32];
    double re[GCR_GROUP], im[GCR_GROUP];
#pragma unroll
    for (int i = 0; i < GCR_GROUP; ++i) re[i] = im[i] = 0.0;
    for (long long k = (long long)blockIdx.x * RED_THREADS + threadIdx.x; k < nvec; k += (long long)RED_BLOCKS * RED_THREADS)
        if (real_site<NCH>(k, Vh)) {
            const Vec b = qj[k];
#pragma unroll
            for (int i = 0; i < GCR_GROUP; ++i)
                if (i < ni) cdot_vec(qbase[(i0 + i) * stride + k], b, re[i], im[i]);
        }
#pragma unroll
    for (int i = 0; i < GCR_GROUP; ++i)
        if (i < ni) { // (ni is uniform: the barriers inside block_sum are reached by every thread)
            double v = block_sum(re[i], sh);
            if (threadIdx.x == 0) part[(2 * i) * RED_BLOCKS + blockIdx.x] = v;
            __syncthreads();
            v = block_sum(im[i], sh);
            if (threadIdx.x == 0) part[(2 * i + 1) * RED_BLOCKS + blockIdx.x] = v;
            __syncthreads();
        }
}

// beta_i = <q_i, q_j> / qq_i for the ni directions from i0;  p_j = psrc - sum beta_i p_i;  q_j -= sum beta_i q_i: one pass
// over p_j and q_j for the whole group.  The inner products were all taken with the q_j that entered the group
// (classical Gram-Schmidt inside a group; the q_i are mutually orthogonal, so in exact arithmetic this is the modified
// form the oracle writes out).  psrc may be p_j itself, or r for an unpreconditioned direction (p_j = r needs no copy).
// FINAL (the last group): also the partials of <q_j, r> and |q_j|^2 of the finished direction.
template <typename Vec, int NCH, bool FINAL>
__global__ void __launch_bounds__(RED_THREADS, 4)
gcr_orth_kernel(Vec *pj, const Vec *psrc, Vec *__restrict__ qj, const Vec *__restrict__ pbase, const Vec *__restrict__ qbase,
                long long stride, int i0, int ni, long long nvec, long long Vh, const double *part, const double *qq,
                const Vec *__restrict__ r, double *qr_part, double *qq_part)
{
    __shared__ double sh[RED_THREADS / 32];
    cplxd mb[GCR_GROUP];
#pragma unroll
    for (int i = 0; i < GCR_GROUP; ++i) {
        mb[i] = {0.0, 0.0};
        if (i < ni) {
            const cplxd d = sum_partials_c(part + (size_t)(2 * i) * RED_BLOCKS);
            const double q2 = qq[i0 + i];
            mb[i] = {-safe_div(d.re, q2), -safe_div(d.im, q2)};
        }
    }
    double re = 0.0, im = 0.0, q2 = 0.0;
    for (long long k = (long long)blockIdx.x * RED_THREADS + threadIdx.x; k < nvec; k += (long long)RED_BLOCKS * RED_THREADS) {
        Vec pv = psrc[k], qv = qj[k];
#pragma unroll
        for (int i = 0; i < GCR_GROUP; ++i)
            if (i < ni) {
                pv = caxpy_vec(mb[i], pbase[(i0 + i) * stride + k], pv);
                qv = caxpy_vec(mb[i], qbase[(i0 + i) * stride + k], qv);
            }
        pj[k] = pv;
        qj[k] = qv;
        if (FINAL && real_site<NCH>(k, Vh)) {
            cdot_vec(qv, r[k], re, im);
            q2 += norm2_vec(qv);
        }
    }
    if (FINAL) {
        re = block_sum(re, sh);
        __syncthreads();
        im = block_sum(im, sh);
        __syncthreads();
        q2 = block_sum(q2, sh);
        if (threadIdx.x == 0) {
            qr_part[blockIdx.x] = re;
            qr_part[RED_BLOCKS + blockIdx.x] = im;
            qq_part[blockIdx.x] = q2;
        }
    }
}

// alpha = <q, r> / <q, q>;  x += alpha p;  r -= alpha q;  |r|^2 partials;  block 0 stores <q, q>
template <typename Vec, int NCH>
__global__ void __launch_bounds__(RED_THREADS)
gcr_update_kernel(Vec *__restrict__ x, Vec *__restrict__ r, const Vec *__restrict__ p, const Vec *__restrict__ q, long long nvec,
                  long long Vh, const double *qr_part, const double *qq_part, double *qq_out, double *rr_part)
{
    __shared__ double sh[RED_THREADS / 32];
    const cplxd qr = sum_partials_c(qr_part);
    const double qq = sum_partials(qq_part);
    const cplxd alpha = {safe_div(qr.re, qq), safe_div(qr.im, qq)};
    const cplxd ma = {-alpha.re, -alpha.im};
    double s2 = 0.0;
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS) {
        x[i] = caxpy_vec(alpha, p[i], x[i]);
        const Vec rn = caxpy_vec(ma, q[i], r[i]);
        r[i] = rn;
        if (real_site<NCH>(i, Vh)) s2 += norm2_vec(rn);
    }
    s2 = block_sum(s2, sh);
    if (threadIdx.x == 0) rr_part[blockIdx.x] = s2;
    if (blockIdx.x == 0 && threadIdx.x == 0) *qq_out = qq;
}

// restarted GCR(m) for Mhat x = b, x_0 = 0: oracle/wd_solvers.py:gcr_schur step for step.  precond != NULL: the search
// direction is p_j = K r with K applied by the caller's function (the multigrid cycle is "a preconditioner
// for a GCR(8) outer Krylov solver"; K may change from call to call -- GCR is flexible); it must enqueue its work on the
// stream it is given and must not call the wd_*_schur solvers of this gauge (they share its workspace).
template <typename T>
static int gcr_schur_t(wd_gauge *g, const ApplyArgs &shape, void *x_out, const void *b_in, double mass, int parity, int max_iter,
                       int restart, double tol, int *iters_out, double *hist_host, cudaError_t *err, precond_fn precond, void *ctx)
{
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH;
    constexpr int CHECK = 8;
    const long long Vh = shape.V / 2;
    const long long nvec = padded_volume(Vh) * NCH;
    const size_t hb = (size_t)nvec * sizeof(Vec);
    cudaStream_t s = shape.stream;
    const double a0 = 4.0 + mass;
    const size_t nsc = (2 * GCR_GROUP + 4) * (size_t)RED_BLOCKS + (size_t)restart + (size_t)max_iter + 1;
    if ((*err = ensure_workspace(g, (size_t)(2 * restart + 2) * hb, nsc)) != cudaSuccess) return -1;
    char *ws = (char *)g->cg_ws;
    Vec *r = (Vec *)ws, *tmp = (Vec *)(ws + hb);
    auto P = [&](int j) { return (Vec *)(ws + (size_t)(2 + j) * hb); };
    auto Q = [&](int j) { return (Vec *)(ws + (size_t)(2 + restart + j) * hb); };
    Vec *x = (Vec *)x_out;
    double *sc = g->cg_sc;
    double *dot_part = sc, *qr_part = sc + 2 * GCR_GROUP * RED_BLOCKS, *qq_part = qr_part + 2 * RED_BLOCKS, *rr_part = qq_part + RED_BLOCKS;
    double *qq = rr_part + RED_BLOCKS, *hist = qq + restart;

    ApplyArgs a = shape;
    auto schur = [&](Vec *out, const Vec *in) -> cudaError_t {
        a.out = tmp;
        a.in = in;
        cudaError_t e = launch_eo(a, nullptr, 0.0, -0.5, 1 - parity, false);
        if (e != cudaSuccess) return e;
        a.out = out;
        a.in = tmp;
        return launch_eo(a, in, a0, 0.5 / a0, parity, false);
    };
    int rc = 0, k = 0;
    double h0 = 0.0;
    auto fail_cuda = [&](cudaError_t e) {
        *err = e;
        rc = -1;
    };
    do {
        cudaError_t e;
        zero_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>(x, nvec);
        if ((e = cudaMemcpyAsync(r, b_in, hb, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) { fail_cuda(e); break; }
        norm2_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>(r, nvec, Vh, rr_part);
        sqrt_of_sum_kernel<<<1, 32, 0, s>>>(rr_part, hist);
        count_launch(3);
        if (tol > 0.0) {
            if ((e = cudaMemcpyAsync(&h0, hist, sizeof(double), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { fail_cuda(e); break; }
            if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
            if (h0 == 0.0) break;
        }
        for (k = 0; k < max_iter; ++k) {
            const int j = k % restart;
            // the new direction: K r (written to P(j) by the caller's function) or r itself (copied into P(j) by the
            // orthogonalisation pass, or by a plain copy when there is nothing to orthogonalise against)
            const Vec *psrc = r;
            if (precond) {
                if (precond(ctx, P(j), r, (void *)s) != 0) { fail_cuda(cudaErrorUnknown); break; }
                psrc = P(j);
            }
            if ((e = schur(Q(j), psrc)) != cudaSuccess) { fail_cuda(e); break; }
            if (j == 0) {
                if (!precond && (e = cudaMemcpyAsync(P(0), r, hb, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) { fail_cuda(e); break; }
                cdot_kernel<Vec, NCH, true><<<RED_BLOCKS, RED_THREADS, 0, s>>>(Q(0), r, nvec, Vh, qr_part, qq_part);
                count_launch();
            }
            // Gram-Schmidt against the cycle's earlier directions, GCR_GROUP of them per pass over p_j and q_j; the last
            // pass also takes <q_j, r> and |q_j|^2
            for (int i0 = 0; i0 < j; i0 += GCR_GROUP) {
                const int ni = j - i0 < GCR_GROUP ? j - i0 : GCR_GROUP;
                gcr_dots_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>(Q(0), nvec, i0, ni, Q(j), nvec, Vh, dot_part);
                if (i0 + ni == j)
                    gcr_orth_kernel<Vec, NCH, true><<<RED_BLOCKS, RED_THREADS, 0, s>>>(P(j), i0 == 0 ? psrc : P(j), Q(j), P(0), Q(0), nvec, i0, ni,
                                                                                     nvec, Vh, dot_part, qq, r, qr_part, qq_part);
                else
                    gcr_orth_kernel<Vec, NCH, false><<<RED_BLOCKS, RED_THREADS, 0, s>>>(P(j), i0 == 0 ? psrc : P(j), Q(j), P(0), Q(0), nvec, i0, ni,
                                                                                      nvec, Vh, dot_part, qq, r, qr_part, qq_part);
                count_launch(2);
            }
            gcr_update_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>(x, r, P(j), Q(j), nvec, Vh, qr_part, qq_part, qq + j, rr_part);
            sqrt_of_sum_kernel<<<1, 32, 0, s>>>(rr_part, hist + k + 1);
            count_launch(3);
            if (tol > 0.0 && ((k + 1) % CHECK == 0 || k + 1 == max_iter)) {
                double hk = 0.0;
                if ((e = cudaMemcpyAsync(&hk, hist + k + 1, sizeof(double), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { fail_cuda(e); break; }
                if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
                if (hk <= tol * h0) {
                    ++k;
                    break;
                }
            }
        }
        if (rc) break;
        if ((e = cudaGetLastError()) != cudaSuccess) { fail_cuda(e); break; }
        if (hist_host) {
            if ((e = cudaMemcpyAsync(hist_host, hist, ((size_t)k + 1) * sizeof(double), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { fail_cuda(e); break; }
        }
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { fail_cuda(e); break; }
        if (hist_host && hist_host[0] > 0.0) {
            const double n0 = hist_host[0];
            for (int i = 0; i <= k; ++i) hist_host[i] /= n0;
        }
    } while (false);
    if (iters_out) *iters_out = k;
    return rc;
}

int gcr_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter, int restart,
              double tol, int *iters_out, double *hist_host, cudaError_t *err, precond_fn precond, void *ctx)
{
    return shape.precision == 32
               ? gcr_schur_t<float>(g, shape, x, b, mass, parity, max_iter, restart, tol, iters_out, hist_host, err, precond, ctx)
               : gcr_schur_t<double>(g, shape, x, b, mass, parity, max_iter, restart, tol, iters_out, hist_host, err, precond, ctx);
}

// ---- true-residual control (tol > 0) ----------------------------------------------------------------------------
// The solvers above iterate on the RECURSIVELY updated residual; in fp32 it keeps falling below what |b - Mhat x| can
// reach.  With a tolerance the public entry points therefore (1) run the solver, (2) recompute r = b - Mhat x with one
// extra operator application, (3) put that true value into the history, and (4) while it is still above tol * |b| and
// iterations are left, solve Mhat e = r for a correction and add it (defect correction), stopping when a round no
// longer halves the true residual.  What is reported as converged is converged.
namespace {
__device__ __forceinline__ void sub_vec(float4 &a, const float4 &b) { a.x -= b.x; a.y -= b.y; a.z -= b.z; a.w -= b.w; }
__device__ __forceinline__ void sub_vec(double2 &a, const double2 &b) { a.x -= b.x; a.y -= b.y; }
__device__ __forceinline__ void add_vec(float4 &a, const float4 &b) { a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w; }
__device__ __forceinline__ void add_vec(double2 &a, const double2 &b) { a.x += b.x; a.y += b.y; }
template <typename Vec, int NCH>
__global__ void __launch_bounds__(RED_THREADS)
true_residual_kernel(Vec *__restrict__ r, const Vec *__restrict__ b, const Vec *__restrict__ w, long long nvec, long long Vh, double *part)
{
    __shared__ double sh[RED_THREADS / 32];
    double s2 = 0.0;
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS) {
        Vec v = b[i];
        const Vec wv = w[i];
        sub_vec(v, wv);
        r[i] = v;
        if (real_site<NCH>(i, Vh)) s2 += norm2_vec(v);
    }
    s2 = block_sum(s2, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = s2;
}
template <typename Vec>
__global__ void __launch_bounds__(RED_THREADS) add_kernel(Vec *__restrict__ x, const Vec *__restrict__ e, long long nvec)
{
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < nvec; i += (long long)RED_BLOCKS * RED_THREADS) {
        Vec v = x[i];
        add_vec(v, e[i]);
        x[i] = v;
    }
}
} // namespace

template <typename T>
static int refined_t(wd_gauge *g, const ApplyArgs &shape, int kind, void *x_out, const void *b_in, double mass, int parity,
                     int max_iter, int restart, double tol, int *iters_out, double *hist_host, cudaError_t *err, precond_fn precond,
                     void *ctx)
{
    using SL = SpinorLayout<T>;
    using Vec = typename SL::Vec;
    constexpr int NCH = SL::NCH;
    auto inner = [&](void *x, const void *b, int iters, double t, int *done, double *hist) {
        return kind == 0   ? cgnr_schur(g, shape, x, b, mass, parity, iters, t, done, hist, err)
               : kind == 1 ? bicgstab_schur(g, shape, x, b, mass, parity, iters, t, done, hist, err)
                           : gcr_schur(g, shape, x, b, mass, parity, iters, restart, t, done, hist, err, precond, ctx);
    };
    if (!(tol > 0.0)) return inner(x_out, b_in, max_iter, tol, iters_out, hist_host);
    const long long Vh = shape.V / 2;
    const long long nvec = padded_volume(Vh) * NCH;
    const size_t hb = (size_t)nvec * sizeof(Vec);
    cudaStream_t s = shape.stream;
    if (g->rf_ws_bytes < 3 * hb + RED_BLOCKS * sizeof(double)) {
        cudaFree(g->rf_ws);
        g->rf_ws = nullptr;
        g->rf_ws_bytes = 0;
        if ((*err = cudaMalloc(&g->rf_ws, 3 * hb + RED_BLOCKS * sizeof(double))) != cudaSuccess) return -1;
        g->rf_ws_bytes = 3 * hb + RED_BLOCKS * sizeof(double);
    }
    Vec *r = (Vec *)g->rf_ws, *e = (Vec *)((char *)g->rf_ws + hb), *tmp = (Vec *)((char *)g->rf_ws + 2 * hb);
    double *part = (double *)((char *)g->rf_ws + 3 * hb);
    const double a0 = 4.0 + mass;
    ApplyArgs a = shape;
    // |v|: partials on the device, summed on the host in a fixed order (this path synchronises anyway)
    auto host_norm = [&](double &out) -> cudaError_t {
        static thread_local double h[RED_BLOCKS];
        cudaError_t ce = cudaMemcpyAsync(h, part, sizeof(h), cudaMemcpyDeviceToHost, s);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(s);
        double sum = 0.0;
        for (int i = 0; i < RED_BLOCKS; ++i) sum += h[i];
        out = sqrt(sum);
        return ce;
    };
    auto true_residual = [&](const Vec *x, double &nrm) -> cudaError_t { // r = b - Mhat x
        a.out = tmp;
        a.in = x;
        cudaError_t ce = launch_eo(a, nullptr, 0.0, -0.5, 1 - parity, false);
        if (ce != cudaSuccess) return ce;
        a.out = e; // (e is free here)
        a.in = tmp;
        if ((ce = launch_eo(a, x, a0, 0.5 / a0, parity, false)) != cudaSuccess) return ce;
        true_residual_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>(r, (const Vec *)b_in, e, nvec, Vh, part);
        count_launch();
        return host_norm(nrm);
    };
    double bnorm = 0.0;
    norm2_kernel<Vec, NCH><<<RED_BLOCKS, RED_THREADS, 0, s>>>((const Vec *)b_in, nvec, Vh, part);
    count_launch();
    if ((*err = host_norm(bnorm)) != cudaSuccess) return -1;
    int total = 0, done = 0;
    if (inner(x_out, b_in, max_iter, tol, &done, hist_host)) return -1;
    total = done;
    if (bnorm == 0.0) { // b = 0: x = 0
        if (iters_out) *iters_out = total;
        return 0;
    }
    double rn = 0.0;
    if ((*err = true_residual((const Vec *)x_out, rn)) != cudaSuccess) return -1;
    if (hist_host) hist_host[total] = rn / bnorm;
    while (rn > tol * bnorm && total < max_iter) {
        const double before = rn;
        const int off = total;
        if (inner(e, r, max_iter - total, tol * bnorm / rn, &done, hist_host ? hist_host + off : nullptr)) return -1;
        if (hist_host)
            for (int i = 0; i <= done; ++i) hist_host[off + i] *= before / bnorm; // the inner history is relative to |r|
        total += done;
        add_kernel<Vec><<<RED_BLOCKS, RED_THREADS, 0, s>>>((Vec *)x_out, e, nvec);
        count_launch();
        if ((*err = true_residual((const Vec *)x_out, rn)) != cudaSuccess) return -1;
        if (hist_host) hist_host[total] = rn / bnorm;
        if (done == 0 || rn > 0.5 * before) break; // stagnation at the working precision: report the true value
    }
    if (iters_out) *iters_out = total;
    return 0;
}

// block CGNR: nrhs right-hand sides in lock step, one batched operator application per step (no true-residual restarts:
// the caller gets the recursive history; wd_cgnr_schur on a single right-hand side has the residual control)
int cgnr_schur_block(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int nrhs, int max_iter,
                     double tol, int *iters_out, double *hist_host, cudaError_t *err)
{
    return shape.precision == 32
               ? cgnr_schur_t<float>(g, shape, x, b, mass, parity, max_iter, tol, iters_out, hist_host, err, nrhs)
               : cgnr_schur_t<double>(g, shape, x, b, mass, parity, max_iter, tol, iters_out, hist_host, err, nrhs);
}

int solve_schur(wd_gauge *g, const ApplyArgs &shape, int kind, void *x, const void *b, double mass, int parity, int max_iter,
                int restart, double tol, int *iters_out, double *hist_host, cudaError_t *err, precond_fn precond, void *ctx)
{
    return shape.precision == 32
               ? refined_t<float>(g, shape, kind, x, b, mass, parity, max_iter, restart, tol, iters_out, hist_host, err, precond, ctx)
               : refined_t<double>(g, shape, kind, x, b, mass, parity, max_iter, restart, tol, iters_out, hist_host, err, precond, ctx);
}

// x = approximate solution of Mhat x = b on `parity` after at most max_iter CGNR iterations (tol = 0: exactly
// max_iter, no host synchronisation inside the loop).  Returns 0, or -1 with *err set.
int cgnr_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter,
               double tol, int *iters_out, double *hist_host, cudaError_t *err)
{
    return shape.precision == 32 ? cgnr_schur_t<float>(g, shape, x, b, mass, parity, max_iter, tol, iters_out, hist_host, err)
                                 : cgnr_schur_t<double>(g, shape, x, b, mass, parity, max_iter, tol, iters_out, hist_host, err);
}

} // namespace wd
