"""Pins for oracle/wd_coarsen.py (eq. (2.7) prolongator, Galerkin coarse operator).  CPU only.
  C1  P^dagger P = 1 on the coarse space ("[P^dagger P] = delta"), and P P^dagger is a projector
  C2  the near-null vectors are reproduced exactly: P P^dagger psi^(alpha) = psi^(alpha)   (S = span(P))
  C3  sigma3 P = P gamma5: restricting gamma5 psi flips the sign of the sigma = 1 coarse components
  C4  gamma5-hermiticity survives coarsening: sigma3 Dhat sigma3 = Dhat^dagger
  C5  the paper's own example eq. (2.4): one vector, constant in a single spin-colour component on 4^4 blocks, gives
      P = theta / 2^d with d = 4, i.e. entries 1/16 inside the block
  C6  span: the first k columns span the same space as the first k input vectors on every block (Gram-Schmidt order)
  C7  the explicit 9-point stencil (coarse_stencil / coarse_apply_stencil) equals the composition P^dagger D P c of the
      pinned pieces (C1-C4 and the pinned D), on coarse lattices with extents 1, 2 and 3 (coincident neighbour blocks)
  C8  gamma5-hermiticity block by block: A = s3 A^dag s3 and B_mu(b) = s3 F_mu(b - mu)^dag s3
  C9  free field, the paper's piecewise-constant example: closed-form entries in tests/golden/coarse_free_field.txt
"""
import os

import numpy as np
import pytest

from oracle import wd_coarsen as wc
from test_oracle_pins import c2r, random_fields

DIMS = (8, 4, 4, 8)
G5 = np.array([1.0, 1.0, -1.0, -1.0])


def vectors(nv, seed=301, dims=DIMS):
    rng = np.random.default_rng(seed)
    shp = (nv, dims[3], dims[2], dims[1], dims[0], 4, 3)
    return rng.standard_normal(shp) + 1j * rng.standard_normal(shp)


def rand_coarse(nv, seed, dims=DIMS):
    rng = np.random.default_rng(seed)
    shp = (dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 2, nv)
    return rng.standard_normal(shp) + 1j * rng.standard_normal(shp)


def test_c1_c2_orthonormal_projector_and_reproduction():
    nv = 5
    psis = vectors(nv)
    W = wc.block_orthonormalise(psis, DIMS)
    c = rand_coarse(nv, 303)
    assert np.max(np.abs(wc.restrict(W, wc.prolong(W, c, DIMS), DIMS) - c)) < 1e-13          # P^dag P = 1
    phi = vectors(1, 305)[0]
    once = wc.prolong(W, wc.restrict(W, phi, DIMS), DIMS)
    twice = wc.prolong(W, wc.restrict(W, once, DIMS), DIMS)
    assert np.max(np.abs(once - twice)) < 1e-13                                              # projector
    for a in range(nv):
        back = wc.prolong(W, wc.restrict(W, psis[a], DIMS), DIMS)
        assert np.max(np.abs(back - psis[a])) < 1e-12                                        # C2


def test_c3_sigma3_p_equals_p_gamma5():
    W = wc.block_orthonormalise(vectors(4), DIMS)
    phi = vectors(1, 307)[0]
    c = wc.restrict(W, phi, DIMS)
    c5 = wc.restrict(W, phi * G5[:, None], DIMS)
    sig3 = np.array([1.0, -1.0])[:, None]
    assert np.max(np.abs(c5 - sig3 * c)) < 1e-13


def test_c4_coarse_gamma5_hermiticity():
    nv = 3
    W = wc.block_orthonormalise(vectors(nv), DIMS)
    U, _ = random_fields(DIMS, 309)
    a, b = rand_coarse(nv, 311), rand_coarse(nv, 313)
    sig3 = np.array([1.0, -1.0])[:, None]
    mass = -0.2
    lhs = np.vdot(a, sig3 * wc.coarse_apply(W, sig3 * b, c2r(U), DIMS, mass))
    rhs = np.vdot(wc.coarse_apply(W, a, c2r(U), DIMS, mass), b)
    assert abs(lhs - rhs) < 1e-11


def test_c5_paper_eq_2_4_piecewise_constant():
    psi = np.zeros((1, DIMS[3], DIMS[2], DIMS[1], DIMS[0], 4, 3), dtype=np.complex128)
    psi[0, ..., 0, 1] = 3.7          # constant, one spin-colour component (chirality sigma = 0)
    psi[0, ..., 3, 2] = -0.4j        # and one in the other chirality, so that both sub-blocks are non-empty
    W = wc.block_orthonormalise(psi, DIMS)
    assert np.allclose(np.abs(W[0, ..., 0, 1]), 1.0 / 2 ** 4)        # theta / 2^d, d = 4
    assert np.allclose(np.abs(W[0, ..., 3, 2]), 1.0 / 2 ** 4)
    assert np.all(W[0, ..., 1, :] == 0) and np.all(W[0, ..., 2, :] == 0)


def test_c6_nested_spans():
    nv = 4
    psis = vectors(nv, 315)
    W = wc.block_orthonormalise(psis, DIMS)
    for k in range(1, nv + 1):
        Wk = wc.block_orthonormalise(psis[:k], DIMS)
        assert np.max(np.abs(Wk - W[:k])) < 1e-13                      # Gram-Schmidt in the given order
        back = wc.prolong(W[:k], wc.restrict(W[:k], psis[k - 1], DIMS), DIMS)
        assert np.max(np.abs(back - psis[k - 1])) < 1e-12


def test_bad_dims_are_refused():
    with pytest.raises(ValueError):
        wc.block_orthonormalise(vectors(1, dims=(6, 4, 4, 8)), (6, 4, 4, 8))


@pytest.mark.parametrize("dims", [(8, 4, 4, 8), (12, 4, 8, 4), (4, 4, 4, 4)])
def test_c7_stencil_equals_the_galerkin_composition(dims):
    nv = 3
    W = wc.block_orthonormalise(vectors(nv, 321, dims), dims)
    U, _ = random_fields(dims, 323)
    mass = -0.2
    S = wc.coarse_stencil(W, c2r(U), dims, mass)
    assert S.shape == (dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 9, 2 * nv, 2 * nv)
    for seed in (325, 327):
        c = rand_coarse(nv, seed, dims)
        assert np.max(np.abs(wc.coarse_apply_stencil(S, c) - wc.coarse_apply(W, c, c2r(U), dims, mass))) < 1e-12


def test_c8_stencil_gamma5_hermiticity_block_by_block():
    dims, nv = (12, 4, 8, 8), 2
    W = wc.block_orthonormalise(vectors(nv, 331, dims), dims)
    U, _ = random_fields(dims, 333)
    S = wc.coarse_stencil(W, c2r(U), dims, 0.1)
    s3 = np.diag(np.repeat([1.0, -1.0], nv))
    dag = lambda M: np.conj(np.swapaxes(M, -1, -2))
    assert np.max(np.abs(S[..., 0, :, :] - s3 @ dag(S[..., 0, :, :]) @ s3)) < 1e-13
    for mu in range(4):
        F_shifted = np.roll(S[..., 1 + mu, :, :], +1, axis=3 - mu)       # F_mu(b - mu) at position b
        assert np.max(np.abs(S[..., 5 + mu, :, :] - s3 @ dag(F_shifted) @ s3)) < 1e-13
    assert np.max(np.abs(S[..., 1:, :, :])) > 1e-3                       # (not trivially zero)


def test_c9_free_field_golden_stencil():
    dims = (8, 4, 8, 4)
    psi = np.zeros((1, dims[3], dims[2], dims[1], dims[0], 4, 3), dtype=np.complex128)
    psi[0, ..., 0, 0] = 2.5
    psi[0, ..., 2, 0] = -1.5
    W = wc.block_orthonormalise(psi, dims)
    U = np.zeros((4, dims[3], dims[2], dims[1], dims[0], 3, 3, 2))
    for i in range(3):
        U[..., i, i, 0] = 1.0
    S = wc.coarse_stencil(W, U, dims, -0.25)
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "coarse_free_field.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 9
    sgn = np.sign(2.5) * np.sign(-1.5)                                  # relative sign of the two normalised columns
    for r in rows:
        k = int(r[0])
        v = [float(x) for x in r[1:]]
        want = np.array([[v[0] + 1j * v[1], sgn * (v[2] + 1j * v[3])], [sgn * (v[4] + 1j * v[5]), v[6] + 1j * v[7]]])
        assert np.max(np.abs(S[..., k, :, :] - want)) < 1e-14, k
