/*
 * wd_oracle.c -- CPU ORACLE for the fine Wilson-Dirac matvec D*psi.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no source,
 * header, table or index helper with the CUDA library under paper_0912_2186_b200/csrc/.
 *
 * What it computes (section 2, eq. (2.2), with the gauge-covariant link
 * convention fixed by BASELINE.json:north_star and the reading S1 listed in DESIGN.md):
 *
 *   (D psi)(x) = (4+m) psi(x)
 *              - 1/2 sum_{mu=1..4} [ (1 + sign*gamma_mu) (x) U_mu(x)         psi(x+mu)
 *                                  + (1 - sign*gamma_mu) (x) U_mu(x-mu)^dag  psi(x-mu) ]
 *
 * with sign = -1 for the operator D of the build (projector (1-gamma_mu) on the un-daggered
 * link, as eq. (2.2) pairs "(gamma_mu - 1)/2" with U and "(gamma_mu + 1)/2" with U^dagger)
 * and sign = +1 for gamma5 D gamma5 = D^dagger ("gamma5-Hermiticity").
 * gamma acts on spin, U on colour; x +- mu is taken modulo L_mu (periodic, no phase).
 * It is the literal definition, evaluated in fp64 with explicit dense 4x4 gamma matrices
 * and full 3x3 complex link products: no spin-projection trick, no blocking, no reordering.
 *
 * Gamma basis: DeGrand-Rossi (BASELINE.json:north_star; the paper only says "4x4 (sparse)
 * spinor matrices").  gamma5 = gamma_x gamma_y gamma_z gamma_t = diag(1,1,-1,-1).
 *
 * Canonical layouts (readings S5, S6), all C-contiguous doubles:
 *   psi [rhs][t][z][y][x][spin 0..3][colour 0..2][re,im]     dims = {Lx, Ly, Lz, Lt}
 *   U   [mu 0..3][t][z][y][x][row a][col b][re,im]           (U psi)_a = sum_b U[a][b] psi_b
 *   with recon == 12 the caller passes only rows a = 0,1:
 *   U12 [mu][t][z][y][x][row 0..1][col b][re,im]  and row 2 = conj(row0 x row1)
 *   ("Gauge field stored as 12 ... floats"; BASELINE.json:configs[2]).
 *   U_mu(x) sits on the link from x to x+mu.
 *
 * Tiny extents (reading S4): for L_mu = 2 the forward and backward neighbour coincide and
 * BOTH hops are accumulated; for L_mu = 1 both are self-hops.  Any L_mu >= 1 is accepted.
 *
 * Parity pins live in tests/test_oracle_pins.py (free-field closed form, gamma5-hermiticity,
 * gauge covariance, brute-force dense matrix, point source, translation covariance) and, for the
 * red/black pieces at the end of this file, in tests/test_oracle_pins_evenodd.py (block
 * decomposition of the pinned full operator, dense Schur complement, solve identity).
 * The paper prints no worked numeric example of D*psi, so the S1 choice (which projector
 * sits on the forward hop) is pinned only by BASELINE.json's convention + the point-source
 * test written from the displayed formula: "parity unpinned" for S1 alone.
 */
#include <complex.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* DeGrand-Rossi gamma matrices, rows then columns; index 0..3 = x,y,z,t. */
static const cplx GAMMA[4][4][4] = {
    /* gamma_x */
    {{0, 0, 0, I}, {0, 0, I, 0}, {0, -I, 0, 0}, {-I, 0, 0, 0}},
    /* gamma_y */
    {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* gamma_z */
    {{0, 0, I, 0}, {0, 0, 0, -I}, {-I, 0, 0, 0}, {0, I, 0, 0}},
    /* gamma_t */
    {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};

/* Export gamma_mu as 32 doubles [row][col][re,im] so tests can check the Clifford algebra. */
void wdo_gamma(int mu, double *out32)
{
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) {
            out32[(i * 4 + j) * 2 + 0] = creal(GAMMA[mu][i][j]);
            out32[(i * 4 + j) * 2 + 1] = cimag(GAMMA[mu][i][j]);
        }
}

int wdo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void wdo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Fetch link U_mu(site) as a full 3x3 matrix; rebuilds row 2 when only 12 reals are stored. */
static void load_link(cplx u[3][3], const double *U, int recon, size_t V, int mu, size_t site)
{
    const int rows = (recon == 12) ? 2 : 3;
    const double *p = U + ((size_t)mu * V + site) * (size_t)(rows * 3 * 2);
    for (int a = 0; a < rows; ++a)
        for (int b = 0; b < 3; ++b)
            u[a][b] = p[(a * 3 + b) * 2] + I * p[(a * 3 + b) * 2 + 1];
    if (recon == 12) {
        /* row2 = conj(row0 x row1): third row of a special unitary matrix */
        u[2][0] = conj(u[0][1] * u[1][2] - u[0][2] * u[1][1]);
        u[2][1] = conj(u[0][2] * u[1][0] - u[0][0] * u[1][2]);
        u[2][2] = conj(u[0][0] * u[1][1] - u[0][1] * u[1][0]);
    }
}

static void load_spinor(cplx s[4][3], const double *psi, size_t site)
{
    const double *p = psi + site * 24;
    for (int sp = 0; sp < 4; ++sp)
        for (int c = 0; c < 3; ++c)
            s[sp][c] = p[(sp * 3 + c) * 2] + I * p[(sp * 3 + c) * 2 + 1];
}

/*
 * out = D(U; mass, sign) psi   for nrhs independent right-hand sides.
 * Returns 0 on success, -1 on bad arguments.  Whole-lattice range.
 */
int wdo_apply_range(double *out, const double *psi, const double *U, const int dims[4],
                    double mass, int nrhs, int recon, int sign, long site_begin, long site_end);

int wdo_apply(double *out, const double *psi, const double *U, const int dims[4], double mass,
              int nrhs, int recon, int sign)
{
    if (!dims) return -1;
    long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    return wdo_apply_range(out, psi, U, dims, mass, nrhs, recon, sign, 0, V);
}

/*
 * Same, but only the output sites with lexicographic index in [site_begin, site_end) are
 * written (others untouched).  Lets bench.py time a bounded sample and lets the full-size
 * parity tests check sampled outputs "one by one" without a whole-lattice CPU apply.
 */
int wdo_apply_range(double *out, const double *psi, const double *U, const int dims[4],
                    double mass, int nrhs, int recon, int sign, long site_begin, long site_end)
{
    if (!out || !psi || !U || !dims) return -1;
    if (recon != 18 && recon != 12) return -1;
    if (sign != 1 && sign != -1) return -1;
    if (nrhs < 1) return -1;
    for (int d = 0; d < 4; ++d)
        if (dims[d] < 1) return -1;
    const int L[4] = {dims[0], dims[1], dims[2], dims[3]};
    const size_t V = (size_t)L[0] * L[1] * L[2] * L[3];
    if (site_begin < 0 || site_end > (long)V || site_begin > site_end) return -1;

    /* spin matrices (1 + sign*gamma_mu) for the forward hop, (1 - sign*gamma_mu) backward */
    cplx PF[4][4][4], PB[4][4][4];
    for (int mu = 0; mu < 4; ++mu)
        for (int i = 0; i < 4; ++i)
            for (int j = 0; j < 4; ++j) {
                cplx one = (i == j) ? 1.0 : 0.0;
                PF[mu][i][j] = one + (double)sign * GAMMA[mu][i][j];
                PB[mu][i][j] = one - (double)sign * GAMMA[mu][i][j];
            }

    for (int r = 0; r < nrhs; ++r) {
        const double *psi_r = psi + (size_t)r * V * 24;
        double *out_r = out + (size_t)r * V * 24;
#pragma omp parallel for schedule(static)
        for (long site = site_begin; site < site_end; ++site) {
            int x[4];
            size_t rem = (size_t)site;
            for (int d = 0; d < 4; ++d) {
                x[d] = (int)(rem % (size_t)L[d]);
                rem /= (size_t)L[d];
            }
            cplx acc[4][3];
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) acc[s][a] = 0.0;

            for (int mu = 0; mu < 4; ++mu) {
                int xf[4] = {x[0], x[1], x[2], x[3]};
                int xb[4] = {x[0], x[1], x[2], x[3]};
                xf[mu] = (x[mu] + 1) % L[mu];
                xb[mu] = (x[mu] - 1 + L[mu]) % L[mu];
                size_t sf = (size_t)xf[0] + (size_t)L[0] * (xf[1] + (size_t)L[1] * (xf[2] + (size_t)L[2] * xf[3]));
                size_t sb = (size_t)xb[0] + (size_t)L[0] * (xb[1] + (size_t)L[1] * (xb[2] + (size_t)L[2] * xb[3]));

                cplx Uf[3][3], Ub[3][3], pf[4][3], pb[4][3], tf[4][3], tb[4][3];
                load_link(Uf, U, recon, V, mu, (size_t)site); /* U_mu(x)      */
                load_link(Ub, U, recon, V, mu, sb);           /* U_mu(x - mu) */
                load_spinor(pf, psi_r, sf);                   /* psi(x + mu)  */
                load_spinor(pb, psi_r, sb);                   /* psi(x - mu)  */

                for (int s = 0; s < 4; ++s)
                    for (int a = 0; a < 3; ++a) {
                        cplx f = 0.0, b = 0.0;
                        for (int c = 0; c < 3; ++c) {
                            f += Uf[a][c] * pf[s][c];       /* U psi        */
                            b += conj(Ub[c][a]) * pb[s][c]; /* U^dagger psi */
                        }
                        tf[s][a] = f;
                        tb[s][a] = b;
                    }
                for (int s = 0; s < 4; ++s)
                    for (int a = 0; a < 3; ++a) {
                        cplx v = 0.0;
                        for (int s2 = 0; s2 < 4; ++s2)
                            v += PF[mu][s][s2] * tf[s2][a] + PB[mu][s][s2] * tb[s2][a];
                        acc[s][a] += v;
                    }
            }

            cplx ctr[4][3];
            load_spinor(ctr, psi_r, (size_t)site);
            double *o = out_r + (size_t)site * 24;
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) {
                    cplx v = (4.0 + mass) * ctr[s][a] - 0.5 * acc[s][a];
                    o[(s * 3 + a) * 2] = creal(v);
                    o[(s * 3 + a) * 2 + 1] = cimag(v);
                }
        }
    }
    return 0;
}

/*
 * ---- red/black (even-odd) pieces: SURVEY.md 8(f) row f1; PAPER.md:126 ("red/black
 * preconditioning"), PAPER.md:157 (the paper's GPU kernel is the even-odd matvec) ----
 *
 * Site parity p(x) = (x1+x2+x3+x4) mod 2.  With every extent even, all eight neighbours of a
 * site have the opposite parity, so in the ordering (even sites, odd sites)
 *
 *        D = [ (4+m) 1     H_eo   ]        H_pq = hopping term of eq. (2.2) from parity q to parity p
 *            [  H_oe     (4+m) 1  ]        (including its factor -1/2)
 *
 * wdo_hop_parity:  out(x) = (H psi)(x) = -1/2 sum_mu [ (1+sign*gamma_mu) U_mu(x) psi(x+mu)
 *                                                    + (1-sign*gamma_mu) U_mu(x-mu)^dag psi(x-mu) ]
 *                  for the sites x of parity `parity`; out(x) = 0 on the other sites.  psi is a
 *                  full-lattice field; only its values on the opposite parity are read.
 * wdo_schur:       the even-odd preconditioned operator on parity p (Schur complement of the
 *                  opposite-parity block, whose diagonal block (4+m) 1 is a scalar for Wilson):
 *                      Mhat psi_p = (4+m) psi_p - H_pq (4+m)^-1 H_qp psi_p ,   q = 1 - p
 *                  psi's values on parity q are ignored; out is 0 there.
 * Both are the definitions written out: same gamma tables, link loader and periodic indexing as
 * wdo_apply above.  Extents must be even (return -2 otherwise: the block form above needs it).
 */
static int site_parity(const int x[4]) { return (x[0] + x[1] + x[2] + x[3]) & 1; }

int wdo_hop_parity(double *out, const double *psi, const double *U, const int dims[4], int nrhs,
                   int recon, int sign, int parity)
{
    if (!out || !psi || !U || !dims) return -1;
    if (recon != 18 && recon != 12) return -1;
    if (sign != 1 && sign != -1) return -1;
    if (parity != 0 && parity != 1) return -1;
    if (nrhs < 1) return -1;
    for (int d = 0; d < 4; ++d) {
        if (dims[d] < 1) return -1;
        if (dims[d] % 2) return -2;
    }
    const int L[4] = {dims[0], dims[1], dims[2], dims[3]};
    const size_t V = (size_t)L[0] * L[1] * L[2] * L[3];
    cplx PF[4][4][4], PB[4][4][4];
    for (int mu = 0; mu < 4; ++mu)
        for (int i = 0; i < 4; ++i)
            for (int j = 0; j < 4; ++j) {
                cplx one = (i == j) ? 1.0 : 0.0;
                PF[mu][i][j] = one + (double)sign * GAMMA[mu][i][j];
                PB[mu][i][j] = one - (double)sign * GAMMA[mu][i][j];
            }
    for (int r = 0; r < nrhs; ++r) {
        const double *psi_r = psi + (size_t)r * V * 24;
        double *out_r = out + (size_t)r * V * 24;
#pragma omp parallel for schedule(static)
        for (long site = 0; site < (long)V; ++site) {
            int x[4];
            size_t rem = (size_t)site;
            for (int d = 0; d < 4; ++d) {
                x[d] = (int)(rem % (size_t)L[d]);
                rem /= (size_t)L[d];
            }
            double *o = out_r + (size_t)site * 24;
            if (site_parity(x) != parity) {
                for (int i = 0; i < 24; ++i) o[i] = 0.0;
                continue;
            }
            cplx acc[4][3];
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) acc[s][a] = 0.0;
            for (int mu = 0; mu < 4; ++mu) {
                int xf[4] = {x[0], x[1], x[2], x[3]};
                int xb[4] = {x[0], x[1], x[2], x[3]};
                xf[mu] = (x[mu] + 1) % L[mu];
                xb[mu] = (x[mu] - 1 + L[mu]) % L[mu];
                size_t sf = (size_t)xf[0] + (size_t)L[0] * (xf[1] + (size_t)L[1] * (xf[2] + (size_t)L[2] * xf[3]));
                size_t sb = (size_t)xb[0] + (size_t)L[0] * (xb[1] + (size_t)L[1] * (xb[2] + (size_t)L[2] * xb[3]));
                cplx Uf[3][3], Ub[3][3], pf[4][3], pb[4][3], tf[4][3], tb[4][3];
                load_link(Uf, U, recon, V, mu, (size_t)site); /* U_mu(x)      */
                load_link(Ub, U, recon, V, mu, sb);           /* U_mu(x - mu) */
                load_spinor(pf, psi_r, sf);                   /* psi(x + mu): opposite parity */
                load_spinor(pb, psi_r, sb);                   /* psi(x - mu): opposite parity */
                for (int s = 0; s < 4; ++s)
                    for (int a = 0; a < 3; ++a) {
                        cplx f = 0.0, b = 0.0;
                        for (int c = 0; c < 3; ++c) {
                            f += Uf[a][c] * pf[s][c];
                            b += conj(Ub[c][a]) * pb[s][c];
                        }
                        tf[s][a] = f;
                        tb[s][a] = b;
                    }
                for (int s = 0; s < 4; ++s)
                    for (int a = 0; a < 3; ++a) {
                        cplx v = 0.0;
                        for (int s2 = 0; s2 < 4; ++s2)
                            v += PF[mu][s][s2] * tf[s2][a] + PB[mu][s][s2] * tb[s2][a];
                        acc[s][a] += v;
                    }
            }
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) {
                    cplx v = -0.5 * acc[s][a];
                    o[(s * 3 + a) * 2] = creal(v);
                    o[(s * 3 + a) * 2 + 1] = cimag(v);
                }
        }
    }
    return 0;
}

int wdo_schur(double *out, const double *psi, const double *U, const int dims[4], double mass,
              int nrhs, int recon, int sign, int parity)
{
    if (!out || !psi || !U || !dims) return -1;
    if (parity != 0 && parity != 1) return -1;
    if (nrhs < 1) return -1;
    for (int d = 0; d < 4; ++d)
        if (dims[d] < 1) return -1;
    if (4.0 + mass == 0.0) return -3; /* the diagonal block is not invertible */
    const size_t n = (size_t)nrhs * dims[0] * dims[1] * dims[2] * dims[3] * 24;
    double *t1 = (double *)malloc(n * sizeof(double)); /* H_qp psi_p          (parity q) */
    double *t2 = (double *)malloc(n * sizeof(double)); /* H_pq (H_qp psi_p)   (parity p) */
    if (!t1 || !t2) {
        free(t1);
        free(t2);
        return -4;
    }
    int rc = wdo_hop_parity(t1, psi, U, dims, nrhs, recon, sign, 1 - parity);
    if (rc == 0) rc = wdo_hop_parity(t2, t1, U, dims, nrhs, recon, sign, parity);
    if (rc == 0) {
        const int L[4] = {dims[0], dims[1], dims[2], dims[3]};
        const size_t V = (size_t)L[0] * L[1] * L[2] * L[3];
        const double a = 4.0 + mass;
        for (int r = 0; r < nrhs; ++r)
            for (size_t site = 0; site < V; ++site) {
                int x[4];
                size_t rem = site;
                for (int d = 0; d < 4; ++d) {
                    x[d] = (int)(rem % (size_t)L[d]);
                    rem /= (size_t)L[d];
                }
                const size_t o = ((size_t)r * V + site) * 24;
                for (int i = 0; i < 24; ++i)
                    out[o + i] = site_parity(x) == parity ? a * psi[o + i] - t2[o + i] / a : 0.0;
            }
    }
    free(t1);
    free(t2);
    return rc;
}
