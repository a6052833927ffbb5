"""Pins for the red/black (even-odd) pieces of the oracle (oracle/wd_oracle.c: wdo_hop_parity, wdo_schur) --
SURVEY.md 8(f) row f1; PAPER.md:126 ("red/black preconditioning"), PAPER.md:157 (the paper's GPU kernel is
the even-odd matvec).  CPU only.  Each pin ties the new functions to something other than themselves:

  E1  block decomposition against the (already pinned) full operator:  D psi = (4+m) psi + H_eo psi_o + H_oe psi_e
  E2  the Schur complement of a brute-force DENSE matrix assembled in test_oracle_pins.dense_matrix
      (global shift permutations and Kronecker products, no code of the oracle):  A - D_pq A^-1 D_qp
  E3  the solve identity that makes red/black preconditioning work: if D psi = b then
      Mhat psi_p = b_p - H_pq (4+m)^-1 b_q   (dense solve on a tiny lattice)
  E4  gamma5-hermiticity is inherited: <phi, g5 Mhat g5 psi> = <Mhat phi, psi>, and sign=+1 gives Mhat^dagger
  E5  free field, constant spinor on one parity: H_qp maps it to -4 x the same constant on the other parity
      (eight hops, projectors (1-g)+(1+g) = 2, factor -1/2), hence Mhat c = [(4+m) - 16/(4+m)] c
  E6  odd extents are refused (the block form needs every neighbour on the opposite parity)
"""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from test_oracle_pins import G5, c2r, dense_matrix, r2c, random_fields, site_shape


def parity_mask(dims):
    """[Lt, Lz, Ly, Lx] array of (x+y+z+t) mod 2."""
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (x + y + z + t) % 2


def hop_c(oracle, psi_c, U_c, dims, parity, sign=-1):
    return r2c(oracle.hop_parity(c2r(psi_c), c2r(U_c), dims, parity, sign=sign))


def schur_c(oracle, psi_c, U_c, dims, mass, parity, sign=-1):
    return r2c(oracle.schur(c2r(psi_c), c2r(U_c), dims, mass, parity, sign=sign))


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 2), (4, 4, 4, 4), (2, 6, 4, 8)])
def test_e1_block_decomposition_of_the_full_operator(oracle, dims):
    U, psi = random_fields(dims, 101, nrhs=2)
    mass = -0.37
    full = r2c(oracle.apply(c2r(psi), c2r(U), dims, mass))
    pm = parity_mask(dims)
    for p in (0, 1):
        h = hop_c(oracle, psi, U, dims, p)
        on = (pm == p)[None, ..., None, None]
        assert np.all(h[np.broadcast_to(~on, h.shape)] == 0)  # nothing written on the other parity
        want = np.where(on, full - (4.0 + mass) * psi, 0)
        assert np.max(np.abs(h - want)) < 1e-13
        # only the opposite parity of the input is read
        other = np.where(on, 0, psi)
        assert np.array_equal(hop_c(oracle, other, U, dims, p), h)


@pytest.mark.parametrize("dims,parity", [((2, 2, 2, 2), 0), ((2, 2, 2, 2), 1), ((4, 2, 2, 2), 0), ((2, 2, 4, 2), 1)])
def test_e2_dense_schur_complement(oracle, dims, parity):
    U, psi = random_fields(dims, 103)
    mass = 0.21
    V = fields.volume(dims)
    M = dense_matrix(U, dims, mass)                           # (site, spin, colour) ordering, x fastest
    par = np.repeat(parity_mask(dims).reshape(V), 12)
    ip, iq = np.where(par == parity)[0], np.where(par != parity)[0]
    App, Apq, Aqp, Aqq = M[np.ix_(ip, ip)], M[np.ix_(ip, iq)], M[np.ix_(iq, ip)], M[np.ix_(iq, iq)]
    assert np.allclose(Aqq, (4.0 + mass) * np.eye(len(iq)))   # Wilson: the diagonal blocks are scalar
    S = App - Apq @ np.linalg.solve(Aqq, Aqp)
    vec = psi[0].reshape(12 * V)
    got = schur_c(oracle, psi, U, dims, mass, parity)[0].reshape(12 * V)
    assert np.max(np.abs(got[ip] - S @ vec[ip])) < 1e-13
    assert np.all(got[iq] == 0)
    # sign = +1 is the dagger of the Schur operator (gamma5-hermiticity of D carries over)
    gotd = schur_c(oracle, psi, U, dims, mass, parity, sign=+1)[0].reshape(12 * V)
    assert np.max(np.abs(gotd[ip] - S.conj().T @ vec[ip])) < 1e-13


def test_e3_solve_identity_of_red_black_preconditioning(oracle):
    dims = (2, 2, 2, 4)
    U, b = random_fields(dims, 107)
    mass = 0.3
    V = fields.volume(dims)
    M = dense_matrix(U, dims, mass)
    psi = np.linalg.solve(M, b[0].reshape(12 * V)).reshape(b.shape)      # D psi = b, dense
    pm = (parity_mask(dims) == 0)[None, ..., None, None]
    lhs = schur_c(oracle, psi, U, dims, mass, 0)                          # Mhat psi_e
    b_odd = np.where(pm, 0, b)
    rhs = np.where(pm, b, 0) - hop_c(oracle, b_odd, U, dims, 0) / (4.0 + mass)
    assert np.max(np.abs(lhs - rhs)) < 1e-12


@pytest.mark.parametrize("dims", [(4, 4, 2, 2), (2, 4, 6, 4)])
def test_e4_gamma5_hermiticity_of_the_schur_operator(oracle, dims):
    U, psi = random_fields(dims, 109)
    _, phi = random_fields(dims, 111)
    mass = -0.2
    g5 = np.diag(G5).real
    pm = (parity_mask(dims) == 1)[None, ..., None, None]
    psi, phi = np.where(pm, psi, 0), np.where(pm, phi, 0)
    g5psi = psi * g5[:, None]
    lhs = np.vdot(phi, schur_c(oracle, g5psi, U, dims, mass, 1) * g5[:, None])
    rhs = np.vdot(schur_c(oracle, phi, U, dims, mass, 1), psi)
    assert abs(lhs - rhs) < 1e-11
    # and the sign=+1 operator is that adjoint
    assert abs(np.vdot(phi, schur_c(oracle, psi, U, dims, mass, 1, sign=+1)) - rhs) < 1e-11


def test_e5_free_field_constant_on_one_parity(oracle):
    dims = (4, 2, 6, 4)
    mass = 0.15
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), (4,) + site_shape(dims) + (3, 3)).copy()
    rng = np.random.default_rng(5)
    c = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    even = (parity_mask(dims) == 0)[None, ..., None, None]
    psi = np.where(even, c, 0)                                   # constant spinor on the even sites
    h = hop_c(oracle, psi, U, dims, 1)                           # lands on the odd sites
    assert np.max(np.abs(h - np.where(even, 0, -4.0 * c))) < 1e-13
    m = schur_c(oracle, psi, U, dims, mass, 0)
    a = 4.0 + mass
    assert np.max(np.abs(m - np.where(even, (a - 16.0 / a) * c, 0))) < 1e-12


@pytest.mark.parametrize("dims", [(3, 2, 2, 2), (2, 2, 2, 5), (1, 1, 1, 1)])
def test_e6_odd_extents_are_refused(oracle, dims):
    U, psi = random_fields(dims, 113)
    with pytest.raises(RuntimeError):
        oracle.hop_parity(c2r(psi), c2r(U), dims, 0)
    with pytest.raises(RuntimeError):
        oracle.schur(c2r(psi), c2r(U), dims, 0.1, 0)
