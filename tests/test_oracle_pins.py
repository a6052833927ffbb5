"""Pins for the CPU oracle (oracle/wd_oracle.c) against what the paper and mathematics fix.

The paper prints no worked example of D*psi, so the oracle is pinned by closed forms, invariants
and brute force (BASELINE.json:north_star lists P1-P4):
  P0  gamma algebra of the oracle's own tables
  P1  free-field plane waves: closed-form eigenvalues (tests/golden/free_field_eigs.txt) + S1 sign
  P2  gamma5-hermiticity <phi, g5 D g5 psi> = <D phi, psi>
  P3  gauge covariance D(U^g)(g psi) = g D(U) psi
  P4  brute-force dense matrix from Kronecker products + shift permutations on tiny lattices
  P5  point source: exactly which neighbours light up, and with which matrix   (eq. (2.2))
  P6  translation covariance,  P7 linearity / mass derivative,  P8 anisotropic shapes
  P9  12-real reconstruction
None of these use the oracle's own formula: the dense matrix is assembled a different way
(global shift matrices and Kronecker structure instead of a per-site stencil loop).
"""
import os

import numpy as np
import pytest

from paper_0912_2186_b200 import fields

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "free_field_eigs.txt")

# DeGrand-Rossi basis as stated in BASELINE.json:north_star / DESIGN.md S2 (typed here independently).
I_ = 1j
G = np.array([
    [[0, 0, 0, I_], [0, 0, I_, 0], [0, -I_, 0, 0], [-I_, 0, 0, 0]],
    [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],
    [[0, 0, I_, 0], [0, 0, 0, -I_], [-I_, 0, 0, 0], [0, I_, 0, 0]],
    [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],
], dtype=np.complex128)
G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)


def c2r(c):
    return np.stack([c.real, c.imag], axis=-1)


def r2c(r):
    return r[..., 0] + 1j * r[..., 1]


def rand_su3(rng, shape):
    z = rng.standard_normal(shape + (3, 3)) + 1j * rng.standard_normal(shape + (3, 3))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    q = q * (d / np.abs(d))[..., None, :]
    det = np.linalg.det(q)
    return q * np.exp(-1j * np.angle(det) / 3)[..., None, None]


def site_shape(dims):
    return (dims[3], dims[2], dims[1], dims[0])


def random_fields(dims, seed, nrhs=1):
    rng = np.random.default_rng(seed)
    U = rand_su3(rng, (4,) + site_shape(dims))
    psi = rng.standard_normal((nrhs,) + site_shape(dims) + (4, 3)) + 1j * rng.standard_normal(
        (nrhs,) + site_shape(dims) + (4, 3))
    return U, psi


def apply_c(oracle, psi_c, U_c, dims, mass, sign=-1):
    return r2c(oracle.apply(c2r(psi_c), c2r(U_c), dims, mass, sign=sign))


# ------------------------------------------------------------------ P0
def test_gamma_algebra(oracle):
    g = [oracle.gamma(mu) for mu in range(4)]
    for mu in range(4):
        assert np.array_equal(g[mu], G[mu])
        assert np.array_equal(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu), atol=0)
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    assert np.array_equal(g5, G5)
    for mu in range(4):
        assert np.array_equal(g5 @ g[mu] @ g5, -g[mu])


# ------------------------------------------------------------------ P1
def _golden_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            v = line.split()
            rows.append((tuple(int(a) for a in v[0:4]), tuple(int(a) for a in v[4:8]), float(v[8]),
                         float(v[9]), float(v[10])))
    return rows


def plane_wave(dims, k, u):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    p = [2 * np.pi * k[i] / dims[i] for i in range(4)]
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return phase[..., None, None] * u, p


@pytest.mark.parametrize("row", _golden_rows())
def test_free_field_golden_eigenvalues(oracle, row):
    dims, k, mass, re_lam, im_lam = row
    U = c2r(np.broadcast_to(np.eye(3, dtype=np.complex128), (4,) + site_shape(dims) + (3, 3)).copy())
    rng = np.random.default_rng(7)
    p = [2 * np.pi * k[i] / dims[i] for i in range(4)]
    # spin matrix of the closed form for the reading of DESIGN.md S1: a + i sum gamma_mu sin p_mu
    a = mass + sum(1 - np.cos(pm) for pm in p)
    M = a * np.eye(4) + 1j * sum(np.sin(p[mu]) * G[mu] for mu in range(4))
    lam, vec = np.linalg.eig(M)
    # golden values are typed from the closed form by hand
    assert np.allclose(np.sort(lam.real), re_lam, atol=1e-12)
    assert np.allclose(np.sort(np.abs(lam.imag)), im_lam, atol=1e-12)
    for j in range(4):
        colour = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        u = np.outer(vec[:, j], colour)
        psi, _ = plane_wave(dims, k, u)
        out = apply_c(oracle, psi[None], r2c(U), dims, mass)[0]
        assert np.max(np.abs(out - lam[j] * psi)) < 1e-13 * max(1.0, abs(lam[j])) * np.max(np.abs(psi)) * 10
        assert abs(lam[j].real - re_lam) < 1e-12 and abs(abs(lam[j].imag) - im_lam) < 1e-12


@pytest.mark.parametrize("dims,k,mass", [((4, 6, 2, 3), (1, 5, 1, 2), -0.4), ((5, 3, 4, 2), (2, 1, 3, 1), 0.1),
                                         ((1, 2, 3, 4), (0, 1, 2, 3), 0.3)])
def test_free_field_general_spinor(oracle, dims, k, mass):
    rng = np.random.default_rng(11)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi, p = plane_wave(dims, k, u)
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), (4,) + site_shape(dims) + (3, 3)).copy()
    a = mass + sum(1 - np.cos(pm) for pm in p)
    slash = sum(np.sin(p[mu]) * G[mu] for mu in range(4))
    out = apply_c(oracle, psi[None], U, dims, mass)[0]
    expect = np.einsum("st,...tc->...sc", a * np.eye(4) + 1j * slash, psi)
    assert np.max(np.abs(out - expect)) < 1e-13 * 10
    # the other reading (sign=+1) is gamma5 D gamma5: a - i pslash
    out_p = apply_c(oracle, psi[None], U, dims, mass, sign=+1)[0]
    expect_p = np.einsum("st,...tc->...sc", a * np.eye(4) - 1j * slash, psi)
    assert np.max(np.abs(out_p - expect_p)) < 1e-13 * 10
    # convention-blind norm identity
    n2 = (a * a + sum(np.sin(pm) ** 2 for pm in p)) * np.sum(np.abs(psi) ** 2)
    assert abs(np.sum(np.abs(out) ** 2) - n2) < 1e-12 * n2


def test_constant_field_gives_mass(oracle):
    dims = (3, 4, 2, 5)
    rng = np.random.default_rng(3)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi = np.broadcast_to(u, site_shape(dims) + (4, 3)).copy()
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), (4,) + site_shape(dims) + (3, 3)).copy()
    out = apply_c(oracle, psi[None], U, dims, -0.37)[0]
    assert np.max(np.abs(out - (-0.37) * psi)) < 1e-14


@pytest.mark.parametrize("mu", [0, 1, 2, 3])
def test_s1_sign_single_direction_eigenspinor(oracle, mu):
    """gamma_mu u = +u and a single non-zero p_mu: lambda = a + i sin p_mu for the adopted reading."""
    dims = [4, 4, 4, 4]
    dims[mu] = 8
    k = [0, 0, 0, 0]
    k[mu] = 1
    w, v = np.linalg.eigh(G[mu])
    uplus = v[:, np.argmax(w)]
    assert np.allclose(G[mu] @ uplus, uplus)
    u = np.outer(uplus, np.array([1.0, 2.0 - 1j, 0.5j]))
    psi, p = plane_wave(tuple(dims), k, u)
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), (4,) + site_shape(dims) + (3, 3)).copy()
    mass = 0.2
    a = mass + (1 - np.cos(p[mu]))
    out = apply_c(oracle, psi[None], U, tuple(dims), mass)[0]
    assert np.max(np.abs(out - (a + 1j * np.sin(p[mu])) * psi)) < 1e-13


# ------------------------------------------------------------------ P2
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 2, 3), (3, 1, 5, 2)])
def test_gamma5_hermiticity(oracle, dims):
    U, psi = random_fields(dims, 21)
    _, phi = random_fields(dims, 22)
    mass = -0.4
    g5psi = np.einsum("st,...tc->...sc", G5, psi)
    D_g5psi = apply_c(oracle, g5psi, U, dims, mass)
    g5_D_g5psi = np.einsum("st,...tc->...sc", G5, D_g5psi)
    Dphi = apply_c(oracle, phi, U, dims, mass)
    lhs = np.vdot(phi, g5_D_g5psi)
    rhs = np.vdot(Dphi, psi)
    assert abs(lhs - rhs) < 1e-12 * abs(rhs) + 1e-10
    # and the sign=+1 operator IS gamma5 D gamma5
    Dp = apply_c(oracle, psi, U, dims, mass, sign=+1)
    assert np.max(np.abs(Dp - g5_D_g5psi)) < 1e-13


# ------------------------------------------------------------------ P3
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 3, 4, 5), (4, 2, 1, 3)])
def test_gauge_covariance(oracle, dims):
    U, psi = random_fields(dims, 31)
    rng = np.random.default_rng(32)
    g = rand_su3(rng, site_shape(dims))  # g(x)
    # U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dagger ; axes of the site grid are (t,z,y,x) -> mu=0 is axis 3
    Ug = np.empty_like(U)
    for mu in range(4):
        g_fwd = np.roll(g, -1, axis=3 - mu)  # g(x+mu)
        Ug[mu] = np.einsum("...ab,...bc,...dc->...ad", g, U[mu], g_fwd.conj())
    gpsi = np.einsum("...ab,...sb->...sa", g, psi[0])[None]
    lhs = apply_c(oracle, gpsi, Ug, dims, 0.1)[0]
    rhs = np.einsum("...ab,...sb->...sa", g, apply_c(oracle, psi, U, dims, 0.1)[0])
    assert np.max(np.abs(lhs - rhs)) < 1e-13


# ------------------------------------------------------------------ P4
def dense_matrix(U, dims, mass, sign=-1):
    """D as a dense (12V x 12V) matrix assembled from global operators:
    D = (4+m) 1 - 1/2 sum_mu [ (1+sign*gamma_mu) (x) H_mu + (1-sign*gamma_mu) (x) H_mu^dagger ],
    H_mu = blockdiag(U_mu(x)) . (T_mu (x) 1_3),  (T_mu f)(x) = f(x+mu) (periodic shift permutation).
    Index order (site, spin, colour), site lexicographic with x fastest."""
    Lx, Ly, Lz, Lt = dims
    V = Lx * Ly * Lz * Lt
    Usite = U.reshape(4, V, 3, 3)
    coords = np.array([(x, y, z, t) for t in range(Lt) for z in range(Lz) for y in range(Ly) for x in range(Lx)])
    lex = lambda c: c[0] + Lx * (c[1] + Ly * (c[2] + Lz * c[3]))
    D = np.zeros((V, 4, 3, V, 4, 3), dtype=np.complex128)
    for s in range(V):
        for sp in range(4):
            for a in range(3):
                D[s, sp, a, s, sp, a] += 4.0 + mass
    for mu in range(4):
        T = np.zeros((V, V))
        for s in range(V):
            c = coords[s].copy()
            c[mu] = (c[mu] + 1) % dims[mu]
            T[s, lex(c)] += 1.0
        H = np.einsum("xab,xy->xayb", Usite[mu], T)              # (V,3,V,3)
        Hd = np.conj(np.transpose(H, (2, 3, 0, 1)))              # H^dagger
        PF = np.eye(4) + sign * G[mu]
        PB = np.eye(4) - sign * G[mu]
        D += -0.5 * np.einsum("st,xayb->xsaytb", PF, H)
        D += -0.5 * np.einsum("st,xayb->xsaytb", PB, Hd)
    return D.reshape(12 * V, 12 * V)


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (3, 2, 1, 2), (1, 1, 1, 1), (4, 1, 2, 3)])
def test_brute_force_dense(oracle, dims):
    U, psi = random_fields(dims, 41)
    mass = 0.1
    M = dense_matrix(U, dims, mass)
    V = fields.volume(dims)
    out = apply_c(oracle, psi, U, dims, mass)[0]
    ref = (M @ psi[0].reshape(12 * V)).reshape(out.shape)
    assert np.max(np.abs(out - ref)) < 1e-13
    Gam5 = np.kron(np.eye(V), np.kron(G5, np.eye(3)))
    assert np.max(np.abs(Gam5 @ M @ Gam5 - M.conj().T)) < 1e-14
    # extent-2 directions: forward and backward neighbour coincide and both must count (S4)
    Mp = dense_matrix(U, dims, mass, sign=+1)
    outp = apply_c(oracle, psi, U, dims, mass, sign=+1)[0]
    assert np.max(np.abs(outp - (Mp @ psi[0].reshape(12 * V)).reshape(out.shape))) < 1e-13


# ------------------------------------------------------------------ P5
def test_point_source(oracle):
    dims = (4, 5, 3, 6)
    U, _ = random_fields(dims, 51)
    Lx, Ly, Lz, Lt = dims
    x0 = (1, 4, 0, 5)  # (x,y,z,t): touches wrap in y (4 -> 0), z (0 -> -1) and t (5 -> 0)
    sp, co = 2, 1
    psi = np.zeros(site_shape(dims) + (4, 3), dtype=np.complex128)
    psi[x0[3], x0[2], x0[1], x0[0], sp, co] = 1.0
    mass = -0.3
    out = apply_c(oracle, psi[None], U, dims, mass)[0]
    e = np.zeros((4, 3), dtype=np.complex128)
    e[sp, co] = 1.0
    expect = np.zeros_like(out)
    expect[x0[3], x0[2], x0[1], x0[0]] = (4 + mass) * e
    for mu in range(4):
        # site y = x0 - mu receives the FORWARD hop from x0: -1/2 (1 - gamma_mu) (x) U_mu(y) e
        y = list(x0)
        y[mu] = (y[mu] - 1) % dims[mu]
        Uy = U[mu, y[3], y[2], y[1], y[0]]
        expect[y[3], y[2], y[1], y[0]] += -0.5 * np.einsum("st,ab,tb->sa", np.eye(4) - G[mu], Uy, e)
        # site y = x0 + mu receives the BACKWARD hop from x0: -1/2 (1 + gamma_mu) (x) U_mu(x0)^dagger e
        y = list(x0)
        y[mu] = (y[mu] + 1) % dims[mu]
        Ux = U[mu, x0[3], x0[2], x0[1], x0[0]]
        expect[y[3], y[2], y[1], y[0]] += -0.5 * np.einsum("st,ba,tb->sa", np.eye(4) + G[mu], Ux.conj(), e)
    assert np.max(np.abs(out - expect)) < 1e-14
    nz = np.sum(np.any(np.abs(out) > 0, axis=(-1, -2)))
    assert nz == 9


# ------------------------------------------------------------------ P6
@pytest.mark.parametrize("mu", [0, 1, 2, 3])
def test_translation_covariance(oracle, mu):
    dims = (4, 3, 5, 2)
    U, psi = random_fields(dims, 61)
    ax = 3 - mu
    out = apply_c(oracle, psi, U, dims, 0.1)[0]
    Us = np.roll(U, 1, axis=1 + ax)
    ps = np.roll(psi, 1, axis=1 + ax)
    outs = apply_c(oracle, ps, Us, dims, 0.1)[0]
    assert np.array_equal(outs, np.roll(out, 1, axis=ax))


# ------------------------------------------------------------------ P7
def test_linearity_and_mass_derivative(oracle):
    dims = (3, 4, 2, 5)
    U, psi = random_fields(dims, 71)
    _, phi = random_fields(dims, 72)
    al, be = 0.7 - 0.2j, -1.3 + 0.4j
    lhs = apply_c(oracle, al * psi + be * phi, U, dims, 0.1)
    rhs = al * apply_c(oracle, psi, U, dims, 0.1) + be * apply_c(oracle, phi, U, dims, 0.1)
    assert np.max(np.abs(lhs - rhs)) < 1e-13
    d = apply_c(oracle, psi, U, dims, 0.25) - apply_c(oracle, psi, U, dims, -0.4)
    assert np.max(np.abs(d - 0.65 * psi)) < 1e-13


# ------------------------------------------------------------------ P9 / interface
def test_recon12_matches_full_links(oracle):
    dims = (4, 3, 2, 5)
    U, psi = random_fields(dims, 81, nrhs=2)
    full = oracle.apply(c2r(psi), c2r(U), dims, -0.4)
    r12 = oracle.apply(c2r(psi), c2r(U[..., 0:2, :]), dims, -0.4)
    assert np.max(np.abs(full - r12)) < 1e-14
    # a wrong reconstruction (e.g. missing conjugate) would not reproduce a generic SU(3) third row
    row2 = np.conj(np.cross(U[..., 0, :], U[..., 1, :]))
    assert np.max(np.abs(row2 - U[..., 2, :])) < 1e-14


def test_multi_rhs_and_range(oracle):
    dims = (4, 3, 2, 5)
    U, psi = random_fields(dims, 91, nrhs=3)
    full = oracle.apply(c2r(psi), c2r(U), dims, 0.1)
    for r in range(3):
        assert np.array_equal(full[r], oracle.apply(c2r(psi[r]), c2r(U), dims, 0.1))
    V = fields.volume(dims)
    part = oracle.apply_range(c2r(psi), c2r(U), dims, 0.1, 17, 61)
    assert np.array_equal(part, full.reshape(3, V, 4, 3, 2)[:, 17:61])


def test_oracle_rejects_bad_arguments(oracle):
    dims = (2, 2, 2, 2)
    U, psi = random_fields(dims, 5)
    with pytest.raises(ValueError):
        oracle.apply(c2r(psi), c2r(U), (2, 2, 2, 3), 0.1)
    with pytest.raises(RuntimeError):
        oracle.apply(c2r(psi), c2r(U), dims, 0.1, sign=0)
