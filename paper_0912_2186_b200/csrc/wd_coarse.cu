// wd_coarse.cu -- the coarse operator of the adaptive multigrid as an explicit nearest-neighbour stencil
// (PAPER.md:82-88 Galerkin form Dhat = P^dagger D P; PAPER.md:116 4^4 blocks x chirality; "the N_V x N_V
// complex matrix operations needed for the coarse operators").
//
// D of eq. (2.2) couples nearest neighbours only, so Dhat couples a block b to itself and to its 8 neighbouring blocks.
// Coarse index i = sigma * N_v + alpha (n = 2 N_v per block), W^sigma_alpha = basis vector restricted to chirality sigma:
//
//   S[b][0]      = A(b)    = sum_{x in b} W(x)^dag [ (4+m) W(x) + the 8 hops whose source site is also in b ]
//   S[b][1+mu]   = F_mu(b) = sum_{x in b, hop leaves through the +mu face} W(x)^dag [ -1/2 (1 - gamma_mu) U_mu(x)        W(x+mu) ]
//   S[b][5+mu]   = B_mu(b) = sum_{x in b, hop leaves through the -mu face} W(x)^dag [ -1/2 (1 + gamma_mu) U_mu(x-mu)^dag W(x-mu) ]
//   (Dhat c)(b)  = A(b) c(b) + sum_mu [ F_mu(b) c(b+mu) + B_mu(b) c(b-mu) ]     (periodic coarse lattice; coincident
//                                                                                neighbour blocks simply add, reading S4)
//
// Device layout of the stencil (wd.h): S[block][k 0..8][column j][row i][re, im] in the working precision -- column
// major, so that the n threads that own the rows of one matrix read consecutive addresses while they sweep the columns.
//
// wd_build_coarse: one CTA per (block, term d), d = 0 the diagonal term, 1..4 forward hops, 5..8 backward hops.  Sites
// are taken CS at a time: phase 1 computes t = U W_alpha'(x +- mu) (colour product on all four spin rows) and
// g = gamma_mu t for every (site, alpha') into shared memory, phase 2 gives each thread pairs (alpha, alpha') and
// accumulates the four chirality blocks  (sigma,sigma) = -1/2 W^sigma.t^sigma  and  (sigma, 1-sigma) = +-1/2 W^sigma.g^sigma
// over the sites in a fixed order (fp64 accumulators, no atomics: deterministic).  Hops that stay inside the block go
// to a scratch partial of A; a second kernel adds the nine partials in a fixed order.  Set-up code: correct and
// deterministic first; it runs once per set of near-null vectors, not in the solver loop.
//
// wd_apply_coarse: one CTA per coarse site, thread (k, i) owns row i of matrix k, sweeps its columns against the
// neighbour's coarse vector (staged in shared memory), the nine partial rows are added in a fixed order.  Per coarse
// site 9 n^2 complex matrix elements are streamed once: 8 flops per 2w bytes, i.e. HBM bound for one right-hand side
// (the case of the K-cycle); with R right-hand sides the matrix element is reused R times from registers.
#include "wd_internal.h"
#include "wd_layout.cuh"
#include "wd_math.cuh"
#include "wd_link.cuh"

namespace wd {

namespace {

constexpr int TB = 256; // 4^4 sites per block

// g = gamma_MU t (DeGrand-Rossi, wd_math.cuh header): t, g are [spin][colour][re,im]
template <typename T> __device__ __forceinline__ void gamma_mul(int mu, const T (&t)[24], T (&g)[24])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T t0r = t[(0 * 3 + c) * 2], t0i = t[(0 * 3 + c) * 2 + 1], t1r = t[(1 * 3 + c) * 2], t1i = t[(1 * 3 + c) * 2 + 1];
        const T t2r = t[(2 * 3 + c) * 2], t2i = t[(2 * 3 + c) * 2 + 1], t3r = t[(3 * 3 + c) * 2], t3i = t[(3 * 3 + c) * 2 + 1];
        T g0r, g0i, g1r, g1i, g2r, g2i, g3r, g3i;
        if (mu == 0) { // (i t3, i t2, -i t1, -i t0)
            g0r = -t3i; g0i = t3r; g1r = -t2i; g1i = t2r; g2r = t1i; g2i = -t1r; g3r = t0i; g3i = -t0r;
        } else if (mu == 1) { // (-t3, t2, t1, -t0)
            g0r = -t3r; g0i = -t3i; g1r = t2r; g1i = t2i; g2r = t1r; g2i = t1i; g3r = -t0r; g3i = -t0i;
        } else if (mu == 2) { // (i t2, -i t3, -i t0, i t1)
            g0r = -t2i; g0i = t2r; g1r = t3i; g1i = -t3r; g2r = t0i; g2i = -t0r; g3r = -t1i; g3i = t1r;
        } else { // (t2, t3, t0, t1)
            g0r = t2r; g0i = t2i; g1r = t3r; g1i = t3i; g2r = t0r; g2i = t0i; g3r = t1r; g3i = t1i;
        }
        g[(0 * 3 + c) * 2] = g0r; g[(0 * 3 + c) * 2 + 1] = g0i;
        g[(1 * 3 + c) * 2] = g1r; g[(1 * 3 + c) * 2 + 1] = g1i;
        g[(2 * 3 + c) * 2] = g2r; g[(2 * 3 + c) * 2 + 1] = g2i;
        g[(3 * 3 + c) * 2] = g3r; g[(3 * 3 + c) * 2 + 1] = g3i;
    }
}

template <typename T, int RECON> __device__ __forceinline__ void load_link_mu(int mu, const T *links, long long site, T (&u)[18])
{
    if (mu == 0) load_link<0, T, RECON>(links, site, u);
    else if (mu == 1) load_link<1, T, RECON>(links, site, u);
    else if (mu == 2) load_link<2, T, RECON>(links, site, u);
    else load_link<3, T, RECON>(links, site, u);
}

// t = U p (DAG = false) or U^dagger p (DAG = true) on all four spin rows
template <bool DAG, typename T> __device__ __forceinline__ void colour_mul(const T (&u)[18], const T (&p)[24], T (&t)[24])
{
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        T h[12], chi[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) h[i] = p[half * 12 + i];
        if (DAG) su3_dag_mul(u, h, chi);
        else su3_mul(u, h, chi);
#pragma unroll
        for (int i = 0; i < 12; ++i) t[half * 12 + i] = chi[i];
    }
}

// gridDim = (9, nblocks): term d = blockIdx.x, block b = blockIdx.y.  Shared memory: three arrays [CS][24][nv] of T.
// out_cross: S (matrix 1+mu / 5+mu of block b) for d >= 1; out_part: scratch [block][d][n*n complex] partials of A.
template <typename T, int RECON>
__global__ void __launch_bounds__(TB)
coarse_build_kernel(T *__restrict__ S, T *__restrict__ part, const T *__restrict__ W, const T *__restrict__ links, int Lx,
                    int Ly, int Lz, int Lt, long long V, int nv, T cdiag, int CS)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // [CS][24][nv] with the site pitch padded by one word: phase 1 writes with lanes = sites (32 different site slots,
    // same vector), and a pitch of 24 nv words would put all 32 lanes in one bank
    const int pitch = 24 * nv + 1;
    T *Wb = reinterpret_cast<T *>(smem_raw);
    T *Tb = Wb + (size_t)CS * pitch;
    T *Gb = Tb + (size_t)CS * pitch;
    const int d = blockIdx.x;
    const long long b = blockIdx.y;
    const int n = 2 * nv;
    const int mu = d == 0 ? 0 : (d - 1) & 3;
    const bool fwd = d >= 1 && d <= 4;
    const int nbx = Lx / 4, nby = Ly / 4, nbz = Lz / 4;
    const int bx = (int)(b % nbx), by = (int)((b / nbx) % nby), bz = (int)((b / ((long long)nbx * nby)) % nbz);
    const int bt = (int)(b / ((long long)nbx * nby * nbz));
    const long long stride = 24 * padded_volume(V);
    const int tid = threadIdx.x;

    // work items of phase 2: (pair of rows alpha = 2 ia, 2 ia + 1; column alpha'), item p = tid + 256 * q, q < NP.  The
    // hopped vector t, g of column alpha' is read from shared memory once for both rows (the phase is bound by
    // shared-memory bandwidth: 48 words of t, g per 96 FMAs with one row per thread, 48 per 192 with two).
    constexpr int NP = 2; // up to 512 items: nv <= 32
    const int npair = ((nv + 1) / 2) * nv;
    double acc[NP][2][2][8]; // [item][row 0/1][0 = leaves the block, 1 = stays inside][(s,s') 00, 11 (from t), 01, 10 (from g): re, im]
#pragma unroll
    for (int q = 0; q < NP; ++q)
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int i = 0; i < 8; ++i) acc[q][r][e][i] = 0.0;

    for (int c0 = 0; c0 < TB; c0 += CS) {
        __syncthreads(); // the previous chunk's buffers have been consumed
        // ---- phase 1: (site, alpha') work items ----
        for (int w = tid; w < CS * nv; w += TB) {
            const int ls = c0 + w % CS, a = w / CS;
            const int x = bx * 4 + (ls & 3), y = by * 4 + ((ls >> 2) & 3), z = bz * 4 + ((ls >> 4) & 3), t = bt * 4 + (ls >> 6);
            const long long site = x + (long long)Lx * (y + (long long)Ly * (z + (long long)Lz * t));
            T own[24], tt[24], gg[24];
            load_spinor(W + a * stride, site, own);
            if (d == 0) {
#pragma unroll
                for (int i = 0; i < 24; ++i) {
                    tt[i] = cdiag * own[i];
                    gg[i] = (T)0;
                }
            } else {
                int cc[4] = {x, y, z, (int)t};
                const int L[4] = {Lx, Ly, Lz, Lt};
                cc[mu] = fwd ? (cc[mu] + 1 == L[mu] ? 0 : cc[mu] + 1) : (cc[mu] == 0 ? L[mu] - 1 : cc[mu] - 1);
                const long long nsite = cc[0] + (long long)Lx * (cc[1] + (long long)Ly * (cc[2] + (long long)Lz * cc[3]));
                T u[18], p[24];
                load_link_mu<T, RECON>(mu, links, fwd ? site : nsite, u);
                load_spinor(W + a * stride, nsite, p);
                if (fwd) colour_mul<false>(u, p, tt);
                else colour_mul<true>(u, p, tt);
                gamma_mul(mu, tt, gg);
            }
            const int sl = w % CS;
#pragma unroll
            for (int i = 0; i < 24; ++i) {
                Wb[(size_t)sl * pitch + i * nv + a] = own[i];
                Tb[(size_t)sl * pitch + i * nv + a] = tt[i];
                Gb[(size_t)sl * pitch + i * nv + a] = gg[i];
            }
        }
        __syncthreads();
        // ---- phase 2: (two rows alpha, column alpha') items ----
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const int p = tid + TB * q;
            if (p < npair) {
                const int ia = p / nv, ap = p - ia * nv;
                const int a0 = 2 * ia, a1 = (2 * ia + 1 < nv) ? 2 * ia + 1 : a0; // (odd nv: the last item redoes row a0, not stored)
                for (int sl = 0; sl < CS; ++sl) {
                    const int ls = c0 + sl;
                    const int lc = mu == 0 ? (ls & 3) : mu == 1 ? ((ls >> 2) & 3) : mu == 2 ? ((ls >> 4) & 3) : (ls >> 6);
                    const int stays = (d == 0) ? 1 : (fwd ? (lc != 3) : (lc != 0));
                    const T *w0 = Wb + (size_t)sl * pitch + a0, *w1 = Wb + (size_t)sl * pitch + a1;
                    const T *tv = Tb + (size_t)sl * pitch + ap, *gv = Gb + (size_t)sl * pitch + ap;
                    T ds0[8], ds1[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) ds0[i] = ds1[i] = (T)0;
#pragma unroll
                    for (int s = 0; s < 2; ++s)
#pragma unroll
                        for (int i = 0; i < 6; ++i) {
                            const int k = s * 12 + 2 * i;
                            const T tr = tv[(size_t)k * nv], ti = tv[(size_t)(k + 1) * nv];
                            const T gr = gv[(size_t)k * nv], gi = gv[(size_t)(k + 1) * nv];
                            const T xr = w0[(size_t)k * nv], xi = w0[(size_t)(k + 1) * nv];
                            const T yr = w1[(size_t)k * nv], yi = w1[(size_t)(k + 1) * nv];
                            ds0[2 * s] += xr * tr + xi * ti;     // conj(w) t
                            ds0[2 * s + 1] += xr * ti - xi * tr;
                            ds0[4 + 2 * s] += xr * gr + xi * gi; // conj(w) g
                            ds0[4 + 2 * s + 1] += xr * gi - xi * gr;
                            ds1[2 * s] += yr * tr + yi * ti;
                            ds1[2 * s + 1] += yr * ti - yi * tr;
                            ds1[4 + 2 * s] += yr * gr + yi * gi;
                            ds1[4 + 2 * s + 1] += yr * gi - yi * gr;
                        }
                    const double m1 = stays ? 1.0 : 0.0, m0 = 1.0 - m1; // (no dynamic index into the register array)
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        acc[q][0][0][i] = fma(m0, (double)ds0[i], acc[q][0][0][i]);
                        acc[q][0][1][i] = fma(m1, (double)ds0[i], acc[q][0][1][i]);
                        acc[q][1][0][i] = fma(m0, (double)ds1[i], acc[q][1][0][i]);
                        acc[q][1][1][i] = fma(m1, (double)ds1[i], acc[q][1][1][i]);
                    }
                }
            }
        }
    }
    // ---- write: entry (row sigma*nv+a, column sigma'*nv+a'), column-major [col][row][re,im] ----
    const double ct = d == 0 ? 1.0 : -0.5;                 // coefficient of the chirality-preserving part
    const double cg = d == 0 ? 0.0 : (fwd ? 0.5 : -0.5);   // of the chirality-flipping part: -1/2 (1 -+ gamma) = -1/2 +- 1/2 gamma
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        const int p = tid + TB * q;
        if (p < npair) {
            const int ia = p / nv, ap = p - ia * nv;
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int a = 2 * ia + r;
                if (a >= nv) continue;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    T *dst = e == 0 ? (d == 0 ? nullptr : S + ((b * 9 + d) * (long long)n * n) * 2)
                                    : part + ((b * 9 + d) * (long long)n * n) * 2;
                    if (!dst) continue;
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const int row = s * nv + a;
                        // (s, s): from t ; (s, 1-s): from g (rows in s, source chirality 1-s)
                        const long long i0 = (((long long)(s * nv + ap)) * n + row) * 2,
                                        i1 = (((long long)((1 - s) * nv + ap)) * n + row) * 2;
                        dst[i0] = (T)(ct * acc[q][r][e][2 * s]);
                        dst[i0 + 1] = (T)(ct * acc[q][r][e][2 * s + 1]);
                        dst[i1] = (T)(cg * acc[q][r][e][4 + 2 * s]);
                        dst[i1 + 1] = (T)(cg * acc[q][r][e][4 + 2 * s + 1]);
                    }
                }
            }
        }
    }
}

// A(b) = sum of the nine partials in a fixed order
template <typename T>
__global__ void coarse_sum_kernel(T *__restrict__ S, const T *__restrict__ part, long long nblocks, int n)
{
    const long long per = (long long)n * n * 2;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nblocks * per) return;
    const long long b = i / per, e = i - b * per;
    double s = 0.0;
#pragma unroll
    for (int d = 0; d < 9; ++d) s += (double)part[(b * 9 + d) * per + e];
    S[(b * 9) * per + e] = (T)s;
}

// one CTA per coarse site; blockDim.x >= 9 * n; NR right-hand sides per pass
template <typename T, int NR>
__global__ void coarse_apply_kernel(T *__restrict__ out, const T *__restrict__ in, const T *__restrict__ S, int nbx, int nby,
                                    int nbz, int nbt, int nv, int nrhs)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = 2 * nv;
    T *cin = reinterpret_cast<T *>(smem_raw); // [NR][9][n][2]
    T *par = cin + (size_t)NR * 9 * n * 2;    // [NR][9][n][2]
    const long long b = blockIdx.x;
    const long long nblocks = (long long)nbx * nby * nbz * nbt;
    const int bx = (int)(b % nbx), by = (int)((b / nbx) % nby), bz = (int)((b / ((long long)nbx * nby)) % nbz);
    const int bt = (int)(b / ((long long)nbx * nby * nbz));
    const int tid = threadIdx.x;
    const int k = tid / n, i = tid - k * n;
    for (int r0 = 0; r0 < nrhs; r0 += NR) {
        __syncthreads();
        // stage the nine neighbours' coarse vectors
        for (int w = tid; w < NR * 9 * n; w += blockDim.x) {
            const int r = w / (9 * n), kk = (w / n) % 9, j = w % n;
            int c[4] = {bx, by, bz, bt};
            const int nb[4] = {nbx, nby, nbz, nbt};
            if (kk >= 1) {
                const int mu = (kk - 1) & 3;
                c[mu] = kk <= 4 ? (c[mu] + 1 == nb[mu] ? 0 : c[mu] + 1) : (c[mu] == 0 ? nb[mu] - 1 : c[mu] - 1);
            }
            const long long nbk = c[0] + (long long)nbx * (c[1] + (long long)nby * (c[2] + (long long)nbz * c[3]));
            const bool live = r0 + r < nrhs;
            const T *src = in + (((long long)(live ? r0 + r : 0) * nblocks + nbk) * n + j) * 2;
            cin[(size_t)w * 2] = live ? src[0] : (T)0;
            cin[(size_t)w * 2 + 1] = live ? src[1] : (T)0;
        }
        __syncthreads();
        if (k < 9) {
            T ar[NR], ai[NR];
#pragma unroll
            for (int r = 0; r < NR; ++r) ar[r] = ai[r] = (T)0;
            const T *m = S + (((b * 9 + k) * (long long)n) * n + i) * 2; // column 0, row i; next column + 2n
#pragma unroll 4
            for (int j = 0; j < n; ++j) {
                const T mr = m[(long long)j * n * 2], mi = m[(long long)j * n * 2 + 1];
#pragma unroll
                for (int r = 0; r < NR; ++r) {
                    const T cr = cin[(((size_t)r * 9 + k) * n + j) * 2], ci = cin[(((size_t)r * 9 + k) * n + j) * 2 + 1];
                    ar[r] = fma(mr, cr, ar[r]); ar[r] = fma(-mi, ci, ar[r]);
                    ai[r] = fma(mr, ci, ai[r]); ai[r] = fma(mi, cr, ai[r]);
                }
            }
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                par[(((size_t)r * 9 + k) * n + i) * 2] = ar[r];
                par[(((size_t)r * 9 + k) * n + i) * 2 + 1] = ai[r];
            }
        }
        __syncthreads();
        for (int w = tid; w < NR * n * 2; w += blockDim.x) {
            const int r = w / (2 * n), e = w % (2 * n);
            if (r0 + r < nrhs) {
                T s = (T)0;
#pragma unroll
                for (int kk = 0; kk < 9; ++kk) s += par[((size_t)r * 9 + kk) * n * 2 + e];
                out[(((long long)(r0 + r) * nblocks + b) * n) * 2 + e] = s;
            }
        }
    }
}

template <typename T, int RECON>
cudaError_t build_t(void *S, void *part, const void *W, const void *links, const int dims[4], long long V, int nv, double mass,
                    cudaStream_t s)
{
    const long long nblocks = V / TB;
    if (nblocks < 1 || nv < 1 || nv > 32) return cudaErrorInvalidConfiguration;
    int CS = 32;
    while (CS > 1 && (size_t)3 * CS * (24 * nv + 1) * sizeof(T) > 200 * 1024) CS >>= 1;
    const size_t smem = (size_t)3 * CS * (24 * nv + 1) * sizeof(T);
    auto kern = coarse_build_kernel<T, RECON>;
    static size_t smem_set[64];
    cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
    if (e != cudaSuccess) return e;
    // gridDim.y is limited to 65535 blocks = 16.7 M sites (checked by wd_build_coarse)
    const int n = 2 * nv;
    if (nblocks > 65535) return cudaErrorInvalidConfiguration;
    kern<<<dim3(9, (unsigned)nblocks), TB, smem, s>>>((T *)S, (T *)part, (const T *)W, (const T *)links, dims[0], dims[1], dims[2],
                                                     dims[3], V, nv, (T)(4.0 + mass), CS);
    count_launch();
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    const long long tot = nblocks * n * n * 2;
    coarse_sum_kernel<T><<<(unsigned)((tot + 255) / 256), 256, 0, s>>>((T *)S, (const T *)part, nblocks, n);
    count_launch();
    return cudaGetLastError();
}

template <typename T, int NR>
cudaError_t apply_nr(void *out, const void *in, const void *S, const int dims[4], int nv, int nrhs, cudaStream_t s)
{
    const int n = 2 * nv;
    const long long nblocks = (long long)(dims[0] / 4) * (dims[1] / 4) * (dims[2] / 4) * (dims[3] / 4);
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    int threads = ((9 * n + 31) / 32) * 32;
    if (threads > 1024) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)2 * NR * 9 * n * 2 * sizeof(T);
    auto kern = coarse_apply_kernel<T, NR>;
    static size_t smem_set[64];
    if (smem > 48 * 1024) {
        cudaError_t e = ensure_dynamic_smem((const void *)kern, smem, smem_set);
        if (e != cudaSuccess) return e;
    }
    kern<<<(unsigned)nblocks, threads, smem, s>>>((T *)out, (const T *)in, (const T *)S, dims[0] / 4, dims[1] / 4, dims[2] / 4,
                                                  dims[3] / 4, nv, nrhs);
    count_launch();
    return cudaGetLastError();
}

template <typename T> cudaError_t apply_t(void *out, const void *in, const void *S, const int dims[4], int nv, int nrhs, cudaStream_t s)
{
    if (nrhs >= 4) return apply_nr<T, 4>(out, in, S, dims, nv, nrhs, s);
    if (nrhs >= 2) return apply_nr<T, 2>(out, in, S, dims, nv, nrhs, s);
    return apply_nr<T, 1>(out, in, S, dims, nv, nrhs, s);
}

} // namespace

cudaError_t launch_coarse_build(void *S, void *part, const void *W, const void *links, const int dims[4], long long V, int nv,
                                double mass, int precision, int recon, cudaStream_t s)
{
    if (precision == 32)
        return recon == 18 ? build_t<float, 18>(S, part, W, links, dims, V, nv, mass, s)
               : recon == 12 ? build_t<float, 12>(S, part, W, links, dims, V, nv, mass, s)
                             : build_t<float, 8>(S, part, W, links, dims, V, nv, mass, s);
    return recon == 18 ? build_t<double, 18>(S, part, W, links, dims, V, nv, mass, s)
           : recon == 12 ? build_t<double, 12>(S, part, W, links, dims, V, nv, mass, s)
                         : build_t<double, 8>(S, part, W, links, dims, V, nv, mass, s);
}

cudaError_t launch_coarse_apply(void *out, const void *in, const void *S, const int dims[4], int nv, int nrhs, int precision,
                                cudaStream_t s)
{
    return precision == 32 ? apply_t<float>(out, in, S, dims, nv, nrhs, s) : apply_t<double>(out, in, S, dims, nv, nrhs, s);
}

} // namespace wd
