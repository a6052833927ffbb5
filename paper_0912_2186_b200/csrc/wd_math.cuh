// wd_math.cuh -- per-site arithmetic of the Wilson-Dirac hopping term (device only).
//
// Implements SURVEY.md section 8(a) steps a2-a6 for eq. (2.2) of arXiv:0912.2186
// (PAPER.md:69-73): 12-real link reconstruction, spin projection with (1 +- gamma_mu),
// SU(3) mat-vec on the two independent spin rows, reconstruction of rows 2,3 and
// accumulation.  Everything is written out for the DeGrand-Rossi basis (S2):
//
//   gamma_x = [[0,0,0,i],[0,0,i,0],[0,-i,0,0],[-i,0,0,0]]   gamma_y = [[0,0,0,-1],[0,0,1,0],[0,1,0,0],[-1,0,0,0]]
//   gamma_z = [[0,0,i,0],[0,0,0,-i],[-i,0,0,0],[0,i,0,0]]   gamma_t = [[0,0,1,0],[0,0,0,1],[1,0,0,0],[0,1,0,0]]
//
// Each projector (1 + S gamma_mu), S = +-1, has rank 2: rows 2,3 of (1 + S gamma_mu) psi are
// unit multiples of rows 0,1 ("h0", "h1"), so the colour matrix only multiplies h0 and h1:
//
//   mu   h0                 h1                 row 2        row 3
//   x    psi0 + S i psi3    psi1 + S i psi2    -S i h1      -S i h0
//   y    psi0 - S   psi3    psi1 + S   psi2     S   h1      -S   h0
//   z    psi0 + S i psi2    psi1 - S i psi3    -S i h0       S i h1
//   t    psi0 + S   psi2    psi1 + S   psi3     S   h0       S   h1
//
// Register layouts: spinor  p[24], index (spin*3 + colour)*2 + {0:re, 1:im}
//                   half    h[12], index (row*3  + colour)*2 + {0:re, 1:im}
//                   link    u[18], index (a*3 + b)*2 + {0:re, 1:im},  (U v)_a = sum_b U[a][b] v_b
#pragma once

namespace wd {

// h = rows 0,1 of (1 + S gamma_MU) p
template <int MU, int S, typename T>
__device__ __forceinline__ void project(const T (&p)[24], T (&h)[12])
{
    constexpr T s = (T)S;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T p0r = p[(0 * 3 + c) * 2], p0i = p[(0 * 3 + c) * 2 + 1];
        const T p1r = p[(1 * 3 + c) * 2], p1i = p[(1 * 3 + c) * 2 + 1];
        const T p2r = p[(2 * 3 + c) * 2], p2i = p[(2 * 3 + c) * 2 + 1];
        const T p3r = p[(3 * 3 + c) * 2], p3i = p[(3 * 3 + c) * 2 + 1];
        T h0r, h0i, h1r, h1i;
        if (MU == 0) {        // h0 = p0 + S i p3 ; h1 = p1 + S i p2
            h0r = p0r - s * p3i; h0i = p0i + s * p3r;
            h1r = p1r - s * p2i; h1i = p1i + s * p2r;
        } else if (MU == 1) { // h0 = p0 - S p3 ; h1 = p1 + S p2
            h0r = p0r - s * p3r; h0i = p0i - s * p3i;
            h1r = p1r + s * p2r; h1i = p1i + s * p2i;
        } else if (MU == 2) { // h0 = p0 + S i p2 ; h1 = p1 - S i p3
            h0r = p0r - s * p2i; h0i = p0i + s * p2r;
            h1r = p1r + s * p3i; h1i = p1i - s * p3r;
        } else {              // h0 = p0 + S p2 ; h1 = p1 + S p3
            h0r = p0r + s * p2r; h0i = p0i + s * p2i;
            h1r = p1r + s * p3r; h1i = p1i + s * p3i;
        }
        h[(0 * 3 + c) * 2] = h0r; h[(0 * 3 + c) * 2 + 1] = h0i;
        h[(1 * 3 + c) * 2] = h1r; h[(1 * 3 + c) * 2 + 1] = h1i;
    }
}

// chi_row = U h_row  (forward hop: the un-daggered link)
template <typename T>
__device__ __forceinline__ void su3_mul(const T (&u)[18], const T (&h)[12], T (&chi)[12])
{
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            T re = (T)0, im = (T)0;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const T ur = u[(a * 3 + b) * 2], ui = u[(a * 3 + b) * 2 + 1];
                const T hr = h[(r * 3 + b) * 2], hi = h[(r * 3 + b) * 2 + 1];
                re = fma(ur, hr, re); re = fma(-ui, hi, re);
                im = fma(ur, hi, im); im = fma(ui, hr, im);
            }
            chi[(r * 3 + a) * 2] = re; chi[(r * 3 + a) * 2 + 1] = im;
        }
}

// chi_row = U^dagger h_row  (backward hop):  (U^dag)[a][b] = conj(U[b][a])
template <typename T>
__device__ __forceinline__ void su3_dag_mul(const T (&u)[18], const T (&h)[12], T (&chi)[12])
{
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            T re = (T)0, im = (T)0;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const T ur = u[(b * 3 + a) * 2], ui = u[(b * 3 + a) * 2 + 1];
                const T hr = h[(r * 3 + b) * 2], hi = h[(r * 3 + b) * 2 + 1];
                re = fma(ur, hr, re); re = fma(ui, hi, re);
                im = fma(ur, hi, im); im = fma(-ui, hr, im);
            }
            chi[(r * 3 + a) * 2] = re; chi[(r * 3 + a) * 2 + 1] = im;
        }
}

// ---- fp32: packed two-lane FMA (Blackwell fma.rn.f32x2 -> SASS FFMA2) ------------------------
// The two independent spin rows h0, h1 of a half spinor are multiplied by the SAME link, so they
// ride in the two lanes of one f32x2 operand while the link element is the scalar (broadcast)
// operand: 36 FFMA2 instead of 72 FFMA per SU(3) x half-spinor product, i.e. half the issue slots
// for 60 % of the kernel's floating-point instructions.  Same products, same summation order per
// lane as the scalar code above.  Opt-in per translation unit (#define WD_USE_F32X2 before this
// header): measured on B200 it helps the cp.async-staged kernel, whose limit is issue slots, and
// slows the latency-bound site kernel (profiles/r01_tile_stage_ncu.md).
#ifdef WD_USE_F32X2
__device__ __forceinline__ unsigned long long f2_pack(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

template <bool DAG>
__device__ __forceinline__ void su3_mul_f2(const float (&u)[18], const float (&h)[12], float (&chi)[12])
{
    unsigned long long hre[3], him[3];
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        hre[b] = f2_pack(h[(0 * 3 + b) * 2], h[(1 * 3 + b) * 2]);
        him[b] = f2_pack(h[(0 * 3 + b) * 2 + 1], h[(1 * 3 + b) * 2 + 1]);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        unsigned long long re, im;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            // element (a,b) of U, or of U^dagger = conj(U[b][a])
            const float ur = DAG ? u[(b * 3 + a) * 2] : u[(a * 3 + b) * 2];
            const float ui = DAG ? -u[(b * 3 + a) * 2 + 1] : u[(a * 3 + b) * 2 + 1];
            const unsigned long long urr = f2_pack(ur, ur), uii = f2_pack(ui, ui), umi = f2_pack(-ui, -ui);
            if (b == 0) {
                re = f2_mul(urr, hre[b]);
                im = f2_mul(urr, him[b]);
            } else {
                re = f2_fma(urr, hre[b], re);
                im = f2_fma(urr, him[b], im);
            }
            re = f2_fma(umi, him[b], re);
            im = f2_fma(uii, hre[b], im);
        }
        f2_unpack(re, chi[(0 * 3 + a) * 2], chi[(1 * 3 + a) * 2]);
        f2_unpack(im, chi[(0 * 3 + a) * 2 + 1], chi[(1 * 3 + a) * 2 + 1]);
    }
}
__device__ __forceinline__ void su3_mul(const float (&u)[18], const float (&h)[12], float (&chi)[12])
{
    su3_mul_f2<false>(u, h, chi);
}
__device__ __forceinline__ void su3_dag_mul(const float (&u)[18], const float (&h)[12], float (&chi)[12])
{
    su3_mul_f2<true>(u, h, chi);
}
#endif

// acc += (1 + S gamma_MU)-reconstruction of chi (rows 0,1 = chi; rows 2,3 per the table above)
template <int MU, int S, typename T>
__device__ __forceinline__ void reconstruct_add(T (&acc)[24], const T (&chi)[12])
{
    constexpr T s = (T)S;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T c0r = chi[(0 * 3 + c) * 2], c0i = chi[(0 * 3 + c) * 2 + 1];
        const T c1r = chi[(1 * 3 + c) * 2], c1i = chi[(1 * 3 + c) * 2 + 1];
        acc[(0 * 3 + c) * 2] += c0r; acc[(0 * 3 + c) * 2 + 1] += c0i;
        acc[(1 * 3 + c) * 2] += c1r; acc[(1 * 3 + c) * 2 + 1] += c1i;
        if (MU == 0) {        // row2 = -S i chi1 ; row3 = -S i chi0      (-S i)(a+ib) = S b - S i a
            acc[(2 * 3 + c) * 2] += s * c1i; acc[(2 * 3 + c) * 2 + 1] -= s * c1r;
            acc[(3 * 3 + c) * 2] += s * c0i; acc[(3 * 3 + c) * 2 + 1] -= s * c0r;
        } else if (MU == 1) { // row2 = S chi1 ; row3 = -S chi0
            acc[(2 * 3 + c) * 2] += s * c1r; acc[(2 * 3 + c) * 2 + 1] += s * c1i;
            acc[(3 * 3 + c) * 2] -= s * c0r; acc[(3 * 3 + c) * 2 + 1] -= s * c0i;
        } else if (MU == 2) { // row2 = -S i chi0 ; row3 = S i chi1        (S i)(a+ib) = -S b + S i a
            acc[(2 * 3 + c) * 2] += s * c0i; acc[(2 * 3 + c) * 2 + 1] -= s * c0r;
            acc[(3 * 3 + c) * 2] -= s * c1i; acc[(3 * 3 + c) * 2 + 1] += s * c1r;
        } else {              // row2 = S chi0 ; row3 = S chi1
            acc[(2 * 3 + c) * 2] += s * c0r; acc[(2 * 3 + c) * 2 + 1] += s * c0i;
            acc[(3 * 3 + c) * 2] += s * c1r; acc[(3 * 3 + c) * 2 + 1] += s * c1i;
        }
    }
}

// Third row of a special-unitary matrix from the first two: row2 = conj(row0 x row1)
// ("stored as 12 ... floats").
template <typename T>
__device__ __forceinline__ void reconstruct_row2(T (&u)[18])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int j = (c + 1) % 3, k = (c + 2) % 3;
        const T ajr = u[(0 * 3 + j) * 2], aji = u[(0 * 3 + j) * 2 + 1];
        const T akr = u[(0 * 3 + k) * 2], aki = u[(0 * 3 + k) * 2 + 1];
        const T bjr = u[(1 * 3 + j) * 2], bji = u[(1 * 3 + j) * 2 + 1];
        const T bkr = u[(1 * 3 + k) * 2], bki = u[(1 * 3 + k) * 2 + 1];
        // z = a_j b_k - a_k b_j ;  row2[c] = conj(z)
        const T zr = ajr * bkr - aji * bki - (akr * bjr - aki * bji);
        const T zi = ajr * bki + aji * bkr - (akr * bji + aki * bjr);
        u[(2 * 3 + c) * 2] = zr;
        u[(2 * 3 + c) * 2 + 1] = -zi;
    }
}

// Full SU(3) link from 8 stored reals ("stored as 12 or 8 ... floats"; reading R8 in DESIGN.md section 2):
//   stored  (Re a2, Im a2, Re a3, Im a3, Re b1, Im b1, arg(a1)/pi, arg(c1)/pi)   for rows a, b, c of the link
//           (the two phases in units of pi, in [-1, 1]: sincospi needs no range reduction by an inexact pi)
//   |a1| = sqrt(1 - N), N = |a2|^2 + |a3|^2 (row 0 has unit length);  |c1| = sqrt(1 - |a1|^2 - |b1|^2) (so has column 0)
//   b perpendicular to a and c = conj(a x b) give two linear equations for (b2, b3):
//       b2 = -(conj(a1) b1 a2 + conj(a3 c1)) / N        b3 = (conj(a2 c1) - a3 conj(a1) b1) / N
//   c2 = conj(a3 b1 - a1 b3),  c3 = conj(a1 b2 - a2 b1)
// In place: u[0..7] hold the stored reals on entry.  N = 0 (a2 = a3 = 0, e.g. the unit matrix) cannot be represented;
// wd_load_gauge refuses such links.  Rounding is amplified by 1/N in b2, b3, c2, c3.
__device__ __forceinline__ void wd_sincospi(float x, float &s, float &c) { sincospif(x, &s, &c); }
__device__ __forceinline__ void wd_sincospi(double x, double &s, double &c) { sincospi(x, &s, &c); }
// square root and reciprocal of the rebuild: fp32 takes the 2-ulp hardware approximations (x * rsqrt(x), rcp) -- their error
// is of the size of the rounding the 1/N amplification already multiplies (tolerance R8) and they save ~25 instructions
// per link in a kernel that the rebuild makes instruction bound; fp64 is exact
__device__ __forceinline__ float wd_sqrt0(float x) { return x > 0.f ? x * rsqrtf(x) : 0.f; }
__device__ __forceinline__ double wd_sqrt0(double x) { return x > 0.0 ? sqrt(x) : 0.0; }
__device__ __forceinline__ float wd_rcp(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double wd_rcp(double x) { return 1.0 / x; }
template <typename T>
__device__ __forceinline__ void reconstruct_from8(T (&u)[18])
{
    const T a2r = u[0], a2i = u[1], a3r = u[2], a3i = u[3], b1r = u[4], b1i = u[5], tha = u[6], thc = u[7];
    const T N = a2r * a2r + a2i * a2i + a3r * a3r + a3i * a3i;
    const T inv = wd_rcp(N);
    const T ma1 = wd_sqrt0((T)1 - N);
    T sa, ca, sc, cc;
    wd_sincospi(tha, sa, ca);
    wd_sincospi(thc, sc, cc);
    const T a1r = ma1 * ca, a1i = ma1 * sa;
    const T mc1 = wd_sqrt0((T)1 - ma1 * ma1 - (b1r * b1r + b1i * b1i));
    const T c1r = mc1 * cc, c1i = mc1 * sc;
    const T pr = a1r * b1r + a1i * b1i, pi = a1r * b1i - a1i * b1r; // p = conj(a1) b1
    const T qr = a3r * c1r - a3i * c1i, qi = a3r * c1i + a3i * c1r; // q = a3 c1
    const T sr = a2r * c1r - a2i * c1i, si = a2r * c1i + a2i * c1r; // s = a2 c1
    const T b2r = -((pr * a2r - pi * a2i) + qr) * inv, b2i = -((pr * a2i + pi * a2r) - qi) * inv;
    const T b3r = (sr - (a3r * pr - a3i * pi)) * inv, b3i = (-si - (a3r * pi + a3i * pr)) * inv;
    // c2 = conj(a3 b1 - a1 b3), c3 = conj(a1 b2 - a2 b1)
    const T c2r = (a3r * b1r - a3i * b1i) - (a1r * b3r - a1i * b3i), c2i = -((a3r * b1i + a3i * b1r) - (a1r * b3i + a1i * b3r));
    const T c3r = (a1r * b2r - a1i * b2i) - (a2r * b1r - a2i * b1i), c3i = -((a1r * b2i + a1i * b2r) - (a2r * b1i + a2i * b1r));
    u[0] = a1r; u[1] = a1i; u[2] = a2r; u[3] = a2i; u[4] = a3r; u[5] = a3i;
    u[6] = b1r; u[7] = b1i; u[8] = b2r; u[9] = b2i; u[10] = b3r; u[11] = b3i;
    u[12] = c1r; u[13] = c1i; u[14] = c2r; u[15] = c2i; u[16] = c3r; u[17] = c3i;
}

// One forward + one backward hop in direction MU accumulated into acc:
//   acc += (1 - gamma_MU) U_f p_f  +  (1 + gamma_MU) U_b^dag p_b
template <int MU, typename T>
__device__ __forceinline__ void hop_forward(T (&acc)[24], const T (&u)[18], const T (&p)[24])
{
    T h[12], chi[12];
    project<MU, -1>(p, h);
    su3_mul(u, h, chi);
    reconstruct_add<MU, -1>(acc, chi);
}

template <int MU, typename T>
__device__ __forceinline__ void hop_backward(T (&acc)[24], const T (&u)[18], const T (&p)[24])
{
    T h[12], chi[12];
    project<MU, +1>(p, h);
    su3_dag_mul(u, h, chi);
    reconstruct_add<MU, +1>(acc, chi);
}

// Hops with the projector sign as a parameter: SGN = -1 is D of eq. (2.2) (hop_forward / hop_backward above),
// SGN = +1 is gamma5 D gamma5 = D^dagger, i.e. every projector 1 -+ gamma_mu swapped.
template <int MU, int SGN, typename T>
__device__ __forceinline__ void hop_forward_s(T (&acc)[24], const T (&u)[18], const T (&p)[24])
{
    T h[12], chi[12];
    project<MU, SGN>(p, h);
    su3_mul(u, h, chi);
    reconstruct_add<MU, SGN>(acc, chi);
}

template <int MU, int SGN, typename T>
__device__ __forceinline__ void hop_backward_s(T (&acc)[24], const T (&u)[18], const T (&p)[24])
{
    T h[12], chi[12];
    project<MU, -SGN>(p, h);
    su3_dag_mul(u, h, chi);
    reconstruct_add<MU, -SGN>(acc, chi);
}

} // namespace wd
