// wd_dslash_site.cu -- WD_KERNEL_SITE: one thread per lattice site, neighbours fetched straight
// from global memory (L1/L2 provide the reuse).  Works for ANY extents >= 1, including the
// degenerate L = 1, 2 cases of reading S4 (coincident neighbours are simply fetched twice and
// both hops accumulate).  It is the general-purpose kernel and the fallback for lattices the
// tiled kernel does not take; eq. (2.2); SURVEY.md 8(a) steps a1-a7.
//
// A thread handles NR right-hand sides of its site: each link is loaded (and, for recon 12,
// rebuilt) once per direction and reused for the NR spinors (step a').
#include <cstdlib>
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

constexpr int SITE_THREADS = 128;

template <int MU, int SGN, typename T, int RECON, int NR>
__device__ __forceinline__ void hop_pair(T (&acc)[NR][24], const T *__restrict__ in, const T *__restrict__ links,
                                         long long Vp, long long site, long long sf, long long sb, int rhs0, int nrhs)
{
    T u[18];
    load_link<MU, T, RECON>(links, site, u); // U_mu(x)
#pragma unroll
    for (int r = 0; r < NR; ++r)
        if (rhs0 + r < nrhs) {
            T p[24];
            load_spinor(in + (long long)(rhs0 + r) * 24 * Vp, sf, p); // psi(x+mu)
            hop_forward_s<MU, SGN>(acc[r], u, p);
        }
    load_link<MU, T, RECON>(links, sb, u); // U_mu(x-mu)
#pragma unroll
    for (int r = 0; r < NR; ++r)
        if (rhs0 + r < nrhs) {
            T p[24];
            load_spinor(in + (long long)(rhs0 + r) * 24 * Vp, sb, p); // psi(x-mu)
            hop_backward_s<MU, SGN>(acc[r], u, p);
        }
}

// SGN = -1: D of eq. (2.2); SGN = +1: gamma5 D gamma5 = D^dagger, every projector swapped
template <typename T, int RECON, int NR, int SGN>
__global__ void __launch_bounds__(SITE_THREADS)
dslash_site_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ links, int Lx, int Ly, int Lz,
                   int Lt, long long V, T cdiag, int nrhs, int bps, long long site0, long long nsites)
{
    // Block order (step a'): the lattice is cut into SLABS of bps consecutive site blocks (a few time
    // slices); within a slab all RHS groups are swept one after the other, then the next slab.  The
    // links of a slab (sized to stay in L2) come from HBM once and serve every group; the spinors of
    // a group keep their short t-neighbour reuse distance.  (Measured on B200: one sweep of the whole
    // lattice per group re-reads the 604 MB gauge field 12 x from HBM; RHS group fastest loses the
    // spinors' t reuse instead and is slower still.)
    const int ngroups = (nrhs + NR - 1) / NR;
    const long long nb = (nsites + SITE_THREADS - 1) / SITE_THREADS; // the launch covers sites [site0, site0 + nsites)
    const long long bid = blockIdx.x;
    const long long slab = bid / ((long long)bps * ngroups);
    const long long nbl = min((long long)bps, nb - slab * bps); // site blocks in this slab
    const long long r = bid - slab * bps * ngroups;
    const long long site = site0 + (slab * bps + r % nbl) * SITE_THREADS + threadIdx.x;
    if (site >= site0 + nsites) return;
    const int rhs0 = (int)(r / nbl) * NR;
    const long long Vp = padded_volume(V); // sites per right-hand side in the native layout

    // periodic neighbours (step a1): coordinates from the lexicographic index, wrap by compare
    long long rem = site;
    const int x = (int)(rem % Lx); rem /= Lx;
    const int y = (int)(rem % Ly); rem /= Ly;
    const int z = (int)(rem % Lz);
    const int t = (int)(rem / Lz);
    const long long sx = 1, sy = Lx, sz = (long long)Lx * Ly, st = (long long)Lx * Ly * Lz;
    const long long xf = site + (x + 1 == Lx ? -(Lx - 1) * sx : sx), xb = site + (x == 0 ? (Lx - 1) * sx : -sx);
    const long long yf = site + (y + 1 == Ly ? -(Ly - 1) * sy : sy), yb = site + (y == 0 ? (Ly - 1) * sy : -sy);
    const long long zf = site + (z + 1 == Lz ? -(Lz - 1) * sz : sz), zb = site + (z == 0 ? (Lz - 1) * sz : -sz);
    const long long tf = site + (t + 1 == Lt ? -(Lt - 1) * st : st), tb = site + (t == 0 ? (Lt - 1) * st : -st);

    T acc[NR][24];
#pragma unroll
    for (int r = 0; r < NR; ++r)
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[r][i] = (T)0;

    hop_pair<0, SGN, T, RECON, NR>(acc, in, links, Vp, site, xf, xb, rhs0, nrhs);
    hop_pair<1, SGN, T, RECON, NR>(acc, in, links, Vp, site, yf, yb, rhs0, nrhs);
    hop_pair<2, SGN, T, RECON, NR>(acc, in, links, Vp, site, zf, zb, rhs0, nrhs);
    hop_pair<3, SGN, T, RECON, NR>(acc, in, links, Vp, site, tf, tb, rhs0, nrhs);

    // fused diagonal (step a6): out = (4+m) psi(x) - 1/2 acc
#pragma unroll
    for (int r = 0; r < NR; ++r)
        if (rhs0 + r < nrhs) {
            T p[24];
            load_spinor(in + (long long)(rhs0 + r) * 24 * Vp, site, p);
#pragma unroll
            for (int i = 0; i < 24; ++i) p[i] = fma(cdiag, p[i], (T)-0.5 * acc[r][i]);
            store_spinor(out + (long long)(rhs0 + r) * 24 * Vp, site, p);
        }
}

template <typename T, int RECON, int NR>
static cudaError_t launch_site_t(const ApplyArgs &a)
{
    const long long site0 = a.site_end > a.site_begin ? a.site_begin : 0;
    const long long nsites = a.site_end > a.site_begin ? a.site_end - a.site_begin : a.V;
    const long long nb = (nsites + SITE_THREADS - 1) / SITE_THREADS;
    const long long ngroups = (a.nrhs + NR - 1) / NR;
    if (nb * ngroups > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    // slab: ~32 MB of links (WD_SITE_SLAB_MB overrides) -- a fraction of the 126 MB L2, leaving room
    // for the spinor streams of the groups passing through
    const Tuning &tn = a.tune ? *a.tune : default_tuning();
    const double slab_mb = tn.site_slab_mb > 0 ? (double)tn.site_slab_mb : 32.0;
    long long bps = (long long)(slab_mb * 1e6 / ((double)SITE_THREADS * 4 * RECON * sizeof(T)));
    if (ngroups == 1 || bps > nb) bps = nb;
    if (bps < 1) bps = 1;
    dim3 grid((unsigned)(nb * ngroups));
    const T cdiag = (T)(4.0 + a.mass); // formed in double, rounded once (reading S8)
    auto kern = a.dagger ? dslash_site_kernel<T, RECON, NR, +1> : dslash_site_kernel<T, RECON, NR, -1>;
    kern<<<grid, SITE_THREADS, 0, a.stream>>>(
        (T *)a.out, (const T *)a.in, (const T *)a.links, a.dims[0], a.dims[1], a.dims[2], a.dims[3], a.V, cdiag, a.nrhs,
        (int)bps, site0, nsites);
    count_launch();
    return cudaGetLastError();
}

template <typename T, int RECON>
static cudaError_t launch_site_r(const ApplyArgs &a)
{
    if (a.nrhs >= 2 && sizeof(T) == 4) return launch_site_t<T, RECON, 2>(a);
    return launch_site_t<T, RECON, 1>(a);
}

cudaError_t launch_site(const ApplyArgs &a)
{
    if (a.precision == 32)
        return a.recon == 18 ? launch_site_r<float, 18>(a) : a.recon == 12 ? launch_site_r<float, 12>(a) : launch_site_r<float, 8>(a);
    return a.recon == 18 ? launch_site_r<double, 18>(a) : a.recon == 12 ? launch_site_r<double, 12>(a) : launch_site_r<double, 8>(a);
}

} // namespace wd
