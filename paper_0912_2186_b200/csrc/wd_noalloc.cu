// wd_noalloc.cu -- the even-odd preconditioned operator for callers that cannot allocate device memory (code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc):
//     Mhat psi_p = (4+m) psi_p - H_pq (4+m)^-1 H_qp psi_p          (wd_dslash_eo.cu)
// Two launches; the intermediate half field H_qp psi_p, which wd_apply_schur takes from the caller (`tmp_half_dev`), lives in
// a file-scope device array of WD_STATIC_SCRATCH_BYTES.  Every GPU that loads the library holds that array until the
// process exits.  Nothing here calls cudaMalloc / cudaFree or a routine that allocates:
//   * the links are the gauge handle's ordinary full-lattice native links, indexed by lex (wd_dslash_eo.cu reads a
//     parity-ordered COPY that the first red/black call allocates -- not available here), so this is a kernel of its own;
//   * in host code the array's name is a host-side stand-in, not a device address: the address comes from
//     cudaGetSymbolAddress, once per device with that device current, and is cached per device ordinal.
// All calls share the array and it keeps the last call's contents.  Nothing in it has to start at zero: the first launch
// writes every site of the intermediate field before the second launch reads it, and pad lanes are never read.  Calls
// that overlap on the GPU (different streams, or two host threads) race on it.
#include "../../include/wd.h"
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_link.cuh"
#include "wd_math.cuh"

namespace wd {

namespace {

constexpr int NA_THREADS = 128;

static __device__ __align__(256) unsigned char g_static_scratch[WD_STATIC_SCRATCH_BYTES];

// out_p = alpha * x_p + beta * sum_mu [ (1-g_mu) U_mu(x) in_q(x+mu) + (1+g_mu) U_mu(x-mu)^dag in_q(x-mu) ]
// half fields over cb = lex / 2 (wd_dslash_eo.cu); one thread per output site; gridDim.y = right-hand sides
template <typename T, int RECON>
__global__ void __launch_bounds__(NA_THREADS)
dslash_eo_lex_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ xin, const T *__restrict__ links, int Lx,
                     int Ly, int Lz, int Lt, long long Vh, T alpha, T beta, int parity)
{
    const long long cb = (long long)blockIdx.x * NA_THREADS + threadIdx.x;
    if (cb >= Vh) return;
    const long long Vhp = padded_volume(Vh), rhs = blockIdx.y;
    in += rhs * 24 * Vhp;
    out += rhs * 24 * Vhp;
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

    T acc[24], u[18], p[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = (T)0;
    // neighbours have the opposite parity; their half-field index is lex / 2
    load_link<0, T, RECON>(links, site, u); load_spinor(in, xf >> 1, p); hop_forward_s<0, -1>(acc, u, p);
    load_link<0, T, RECON>(links, xb, u);   load_spinor(in, xb >> 1, p); hop_backward_s<0, -1>(acc, u, p);
    load_link<1, T, RECON>(links, site, u); load_spinor(in, yf >> 1, p); hop_forward_s<1, -1>(acc, u, p);
    load_link<1, T, RECON>(links, yb, u);   load_spinor(in, yb >> 1, p); hop_backward_s<1, -1>(acc, u, p);
    load_link<2, T, RECON>(links, site, u); load_spinor(in, zf >> 1, p); hop_forward_s<2, -1>(acc, u, p);
    load_link<2, T, RECON>(links, zb, u);   load_spinor(in, zb >> 1, p); hop_backward_s<2, -1>(acc, u, p);
    load_link<3, T, RECON>(links, site, u); load_spinor(in, tf >> 1, p); hop_forward_s<3, -1>(acc, u, p);
    load_link<3, T, RECON>(links, tb, u);   load_spinor(in, tb >> 1, p); hop_backward_s<3, -1>(acc, u, p);
    if (xin) {
        load_spinor(xin + rhs * 24 * Vhp, cb, p);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = fma(alpha, p[i], beta * acc[i]);
    } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = beta * acc[i];
    }
    store_spinor(out, cb, acc);
}

// device address of the scratch array on the current device: cudaGetSymbolAddress once per device (with that device
// current), cached by device ordinal; a race between two threads stores the same address twice
cudaError_t static_scratch_ptr(void **ptr)
{
    static void *cache[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    void *p = (dev >= 0 && dev < 64) ? __atomic_load_n(&cache[dev], __ATOMIC_ACQUIRE) : nullptr;
    if (!p) {
        if ((e = cudaGetSymbolAddress(&p, g_static_scratch)) != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        if (dev >= 0 && dev < 64) __atomic_store_n(&cache[dev], p, __ATOMIC_RELEASE);
    }
    *ptr = p;
    return cudaSuccess;
}

template <typename T, int RECON>
cudaError_t schur_static_t(const ApplyArgs &a, void *scratch, int parity)
{
    const long long Vh = a.V / 2;
    const long long nb = (Vh + NA_THREADS - 1) / NA_THREADS;
    if (nb > 0x7fffffffLL || a.nrhs > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)nb, (unsigned)a.nrhs);
    const double a0 = 4.0 + a.mass;
    auto kern = dslash_eo_lex_kernel<T, RECON>;
    // scratch_q = H_qp in_p
    kern<<<grid, NA_THREADS, 0, a.stream>>>((T *)scratch, (const T *)a.in, nullptr, (const T *)a.links, a.dims[0], a.dims[1], a.dims[2],
                                            a.dims[3], Vh, (T)0.0, (T)-0.5, 1 - parity);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    // out_p = (4+m) in_p - H_pq scratch_q / (4+m) = (4+m) in_p + hops(scratch_q) / (2 (4+m))
    kern<<<grid, NA_THREADS, 0, a.stream>>>((T *)a.out, (const T *)scratch, (const T *)a.in, (const T *)a.links, a.dims[0], a.dims[1],
                                            a.dims[2], a.dims[3], Vh, (T)a0, (T)(0.5 / a0), parity);
    count_launch(2);
    return cudaGetLastError();
}

} // namespace

// bytes of the intermediate half field of a.nrhs right-hand sides (what the call needs of the static array)
size_t schur_static_need(const ApplyArgs &a)
{
    return (size_t)a.nrhs * (size_t)padded_volume(a.V / 2) * 24 * (a.precision == 32 ? 4 : 8);
}

// a.out = Mhat a.in on `parity` (fp32 / fp64, any link format); the caller has checked schur_static_need(a) against
// WD_STATIC_SCRATCH_BYTES
cudaError_t launch_schur_static(const ApplyArgs &a, int parity)
{
    if (schur_static_need(a) > (size_t)WD_STATIC_SCRATCH_BYTES) return cudaErrorInvalidValue;
    void *scratch = nullptr;
    cudaError_t e = static_scratch_ptr(&scratch);
    if (e != cudaSuccess) return e;
    if (a.precision == 32)
        return a.recon == 18 ? schur_static_t<float, 18>(a, scratch, parity)
               : a.recon == 12 ? schur_static_t<float, 12>(a, scratch, parity)
                               : schur_static_t<float, 8>(a, scratch, parity);
    return a.recon == 18 ? schur_static_t<double, 18>(a, scratch, parity)
           : a.recon == 12 ? schur_static_t<double, 12>(a, scratch, parity)
                           : schur_static_t<double, 8>(a, scratch, parity);
}

} // namespace wd
