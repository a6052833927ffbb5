"""Pins for oracle/wd_solvers.py (CGNR on the even-odd preconditioned operator).  CPU only.
  K1  the converged solution equals a dense solve with the brute-force Schur complement (test_oracle_pins.dense_matrix)
  K2  in exact arithmetic CGNR minimises |b - Mhat x| over the Krylov space: the residual history is non-increasing,
      and after n = dim iterations on a tiny system it has converged to rounding
  K3  the returned history is the true residual |b - Mhat x_k| / |b| (recomputed from x with the pinned operator)
"""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from oracle import wd_solvers
from test_oracle_pins import c2r, dense_matrix, r2c, random_fields
from test_oracle_pins_evenodd import parity_mask


@pytest.mark.parametrize("parity", [0, 1])
def test_k1_converged_solution_matches_dense_solve(oracle, parity):
    dims = (2, 2, 2, 2)
    U, b = random_fields(dims, 201)
    mass = 0.25
    V = fields.volume(dims)
    M = dense_matrix(U, dims, mass)
    par = np.repeat(parity_mask(dims).reshape(V), 12)
    ip, iq = np.where(par == parity)[0], np.where(par != parity)[0]
    S = M[np.ix_(ip, ip)] - M[np.ix_(ip, iq)] @ np.linalg.solve(M[np.ix_(iq, iq)], M[np.ix_(iq, ip)])
    x, hist = wd_solvers.cgnr_schur(c2r(b[0]), c2r(U), dims, mass, parity, niter=200, tol=1e-13)
    want = np.linalg.solve(S, b[0].reshape(12 * V)[ip])
    got = r2c(x).reshape(12 * V)
    assert hist[-1] <= 1e-13
    assert np.max(np.abs(got[ip] - want)) < 1e-11
    assert np.all(got[iq] == 0)


def test_k2_k3_residual_history(oracle):
    dims = (4, 2, 2, 4)
    U, b = random_fields(dims, 203)
    mass = -0.1
    x, hist = wd_solvers.cgnr_schur(c2r(b[0]), c2r(U), dims, mass, 0, niter=25)
    assert len(hist) == 26 and hist[0] == pytest.approx(1.0)
    assert np.all(np.diff(hist) <= 1e-14)                         # K2: monotone
    bm = np.where((parity_mask(dims) == 0)[..., None, None, None], c2r(b[0]), 0.0)
    true_r = bm - oracle.schur(x, c2r(U), dims, mass, 0)
    assert np.linalg.norm(true_r) / np.linalg.norm(bm) == pytest.approx(hist[-1], rel=1e-9)   # K3


@pytest.mark.parametrize("parity", [0, 1])
def test_k4_bicgstab_converged_solution_matches_dense_solve(oracle, parity):
    dims = (2, 2, 2, 2)
    U, b = random_fields(dims, 211)
    mass = 0.25
    V = fields.volume(dims)
    M = dense_matrix(U, dims, mass)
    par = np.repeat(parity_mask(dims).reshape(V), 12)
    ip, iq = np.where(par == parity)[0], np.where(par != parity)[0]
    S = M[np.ix_(ip, ip)] - M[np.ix_(ip, iq)] @ np.linalg.solve(M[np.ix_(iq, iq)], M[np.ix_(iq, ip)])
    x, hist = wd_solvers.bicgstab_schur(c2r(b[0]), c2r(U), dims, mass, parity, niter=200, tol=1e-13)
    want = np.linalg.solve(S, b[0].reshape(12 * V)[ip])
    got = r2c(x).reshape(12 * V)
    assert hist[-1] <= 1e-13
    assert np.max(np.abs(got[ip] - want)) < 1e-11
    assert np.all(got[iq] == 0)


def test_k5_bicgstab_history_is_the_true_residual(oracle):
    dims = (4, 2, 2, 4)
    U, b = random_fields(dims, 213)
    mass = -0.1
    x, hist = wd_solvers.bicgstab_schur(c2r(b[0]), c2r(U), dims, mass, 0, niter=12)
    bm = np.where((parity_mask(dims) == 0)[..., None, None, None], c2r(b[0]), 0.0)
    true_r = bm - oracle.schur(np.ascontiguousarray(x), c2r(U), dims, mass, 0)
    assert len(hist) == 13
    assert np.linalg.norm(true_r) / np.linalg.norm(bm) == pytest.approx(hist[-1], rel=1e-8)
    assert hist[-1] < 1e-2 * hist[0]   # it does converge on this well-conditioned system


@pytest.mark.parametrize("parity", [0, 1])
def test_k6_gcr_converged_solution_matches_dense_solve(oracle, parity):
    dims = (2, 2, 2, 2)
    U, b = random_fields(dims, 221)
    mass = 0.25
    V = fields.volume(dims)
    M = dense_matrix(U, dims, mass)
    par = np.repeat(parity_mask(dims).reshape(V), 12)
    ip, iq = np.where(par == parity)[0], np.where(par != parity)[0]
    S = M[np.ix_(ip, ip)] - M[np.ix_(ip, iq)] @ np.linalg.solve(M[np.ix_(iq, iq)], M[np.ix_(iq, ip)])
    x, hist = wd_solvers.gcr_schur(c2r(b[0]), c2r(U), dims, mass, parity, niter=400, restart=8, tol=1e-13)
    want = np.linalg.solve(S, b[0].reshape(12 * V)[ip])
    got = r2c(x).reshape(12 * V)
    assert hist[-1] <= 1e-13
    assert np.max(np.abs(got[ip] - want)) < 1e-11
    assert np.all(got[iq] == 0)


def test_k7_gcr_minimises_the_residual_and_reports_it(oracle):
    """GCR minimises |b - Mhat x| over the current cycle's search space: the history is non-increasing, within a cycle
    the q's are orthogonal so the first cycle equals the minimum-residual solution over span{q_0..q_7} (least squares),
    and the history is the true residual."""
    dims = (4, 2, 2, 4)
    U, b = random_fields(dims, 223)
    mass = -0.1
    x8, hist8 = wd_solvers.gcr_schur(c2r(b[0]), c2r(U), dims, mass, 0, niter=8, restart=8)
    x, hist = wd_solvers.gcr_schur(c2r(b[0]), c2r(U), dims, mass, 0, niter=20, restart=8)
    assert np.all(np.diff(hist) <= 1e-14)
    bm = np.where((parity_mask(dims) == 0)[..., None, None, None], c2r(b[0]), 0.0)
    Mop = lambda v: oracle.schur(np.ascontiguousarray(v), c2r(U), dims, mass, 0)
    assert np.linalg.norm(bm - Mop(x)) / np.linalg.norm(bm) == pytest.approx(hist[-1], rel=1e-8)
    # least squares over the Krylov space K_8(Mhat, b) = span{b, Mhat b, ..., Mhat^7 b}
    K = [bm]
    for _ in range(7):
        K.append(Mop(K[-1]))
    Kc = np.stack([r2c(v).ravel() for v in K], axis=1)
    AK = np.stack([r2c(Mop(v)).ravel() for v in K], axis=1)
    coef, *_ = np.linalg.lstsq(AK, r2c(bm).ravel(), rcond=None)
    best = np.linalg.norm(r2c(bm).ravel() - AK @ coef) / np.linalg.norm(bm)
    assert hist8[-1] == pytest.approx(best, rel=1e-6)


# ------------------------------------------------------------------------------------------------------------------
# Pins that bite on the RECURRENCES (round 2; VERDICT r01 "weak #1": the pins above only see convergence and the true
# residual, which steepest descent (beta = 0), a conjugated omega or a beta without alpha/omega also satisfy).
#   K8   CGNR iterate k is THE minimiser of |b - Mhat x| over K_k(Mhat^dag Mhat, Mhat^dag b) (Hestenes-Stiefel on the
#        normal equations; "CG on the normal equations"): compared with a least-squares solve over a
#        Krylov basis built here from the pinned operator, for every k
#   K9   finite termination: b = sum of k left singular vectors of the dense Schur complement => CGNR converges in
#        exactly k iterations (and not in k-1)
#   K10  BiCGstab per iteration: <rhat, s> = 0 (alpha), <t, r_new> = 0 and |r_new| = min_w |s - w t| (omega), and
#        x_new reproduces r_new = b - Mhat x_new
#   K11  finite termination of the BiCG part: b = sum of k eigenvectors of the dense Schur complement => BiCGstab
#        converges in exactly k iterations (needs beta = (rho'/rho)(alpha/omega))
# ------------------------------------------------------------------------------------------------------------------
def _dense_schur(dims, U, mass, parity):
    V = fields.volume(dims)
    M = dense_matrix(U, dims, mass)
    par = np.repeat(parity_mask(dims).reshape(V), 12)
    ip, iq = np.where(par == parity)[0], np.where(par != parity)[0]
    S = M[np.ix_(ip, ip)] - M[np.ix_(ip, iq)] @ np.linalg.solve(M[np.ix_(iq, iq)], M[np.ix_(iq, ip)])
    return S, ip


def _embed(vec_p, ip, dims):
    """parity-subspace complex vector -> full canonical real-pair field (zero on the other parity)"""
    V = fields.volume(dims)
    full = np.zeros(12 * V, dtype=np.complex128)
    full[ip] = vec_p
    return c2r(full.reshape(dims[3], dims[2], dims[1], dims[0], 4, 3))


def test_k8_cgnr_iterates_are_the_least_squares_minimisers(oracle):
    dims = (4, 2, 2, 4)
    U, b = random_fields(dims, 231)
    mass = -0.1
    Ur = c2r(U)
    bm = np.where((parity_mask(dims) == 0)[..., None, None, None], c2r(b[0]), 0.0)
    M = lambda v: oracle.schur(np.ascontiguousarray(v), Ur, dims, mass, 0, sign=-1)
    Md = lambda v: oracle.schur(np.ascontiguousarray(v), Ur, dims, mass, 0, sign=+1)
    kmax = 6
    trace = []
    x, hist = wd_solvers.cgnr_schur(c2r(b[0]), Ur, dims, mass, 0, niter=kmax, trace=trace)
    assert len(trace) == kmax
    K = [Md(bm)]                                       # Krylov basis of K_k(Mhat^dag Mhat, Mhat^dag b)
    for _ in range(kmax - 1):
        K.append(Md(M(K[-1])))
    bc = r2c(bm).ravel()
    for k in range(1, kmax + 1):
        Kc = np.stack([r2c(v).ravel() for v in K[:k]], axis=1)
        AK = np.stack([r2c(M(v)).ravel() for v in K[:k]], axis=1)
        Q, _ = np.linalg.qr(AK)                        # orthonormal basis of Mhat K_k: well conditioned projection
        best_r = bc - Q @ (Q.conj().T @ bc)
        assert hist[k] == pytest.approx(np.linalg.norm(best_r) / np.linalg.norm(bc), rel=1e-7)
        # the iterate itself: Mhat x_k is the projection of b onto Mhat K_k
        assert np.linalg.norm(r2c(M(trace[k - 1])).ravel() - (bc - best_r)) <= 1e-8 * np.linalg.norm(bc)


@pytest.mark.parametrize("k", [3, 5])
def test_k9_cgnr_terminates_in_k_steps_on_k_singular_vectors(oracle, k):
    dims = (2, 2, 2, 2)
    U, _ = random_fields(dims, 233)
    mass = 0.25
    S, ip = _dense_schur(dims, U, mass, 0)
    Us, sv, _ = np.linalg.svd(S)
    b_p = Us[:, [1, 17, 40, 63, 90][:k]] @ np.array([1.0, -0.7, 0.4 + 0.3j, 1.2j, -0.9][:k])
    x, hist = wd_solvers.cgnr_schur(_embed(b_p, ip, dims), c2r(U), dims, mass, 0, niter=k)
    assert len(hist) == k + 1
    assert hist[k] < 1e-10
    assert hist[k - 1] > 1e4 * max(hist[k], 1e-14)


def test_k10_bicgstab_step_orthogonalities(oracle):
    dims = (4, 2, 2, 4)
    U, b = random_fields(dims, 235)
    mass = -0.1
    Ur = c2r(U)
    bm = np.where((parity_mask(dims) == 0)[..., None, None, None], c2r(b[0]), 0.0)
    Mc = lambda v: r2c(oracle.schur(np.ascontiguousarray(c2r(v)), Ur, dims, mass, 0))
    trace = []
    wd_solvers.bicgstab_schur(c2r(b[0]), Ur, dims, mass, 0, niter=6, trace=trace)
    assert len(trace) == 6
    for rhat, s, t, r_new, x_new in trace:
        ns, nt = np.linalg.norm(s), np.linalg.norm(t)
        assert abs(np.vdot(rhat, s)) <= 1e-10 * np.linalg.norm(rhat) * ns          # alpha = rho' / <rhat, v>
        assert abs(np.vdot(t, r_new)) <= 1e-10 * nt * ns                            # omega = <t, s> / <t, t>
        w_best = np.vdot(t, s) / np.vdot(t, t)
        for dw in (1e-3, 1e-3j, -1e-3, -1e-3j):
            assert np.linalg.norm(r_new) <= np.linalg.norm(s - (w_best + dw) * t)   # the minimum over complex omega
        assert np.linalg.norm(r2c(bm) - Mc(x_new) - r_new) <= 1e-10 * np.linalg.norm(bm)


@pytest.mark.parametrize("k", [3, 4])
def test_k11_bicgstab_terminates_in_k_steps_on_k_eigenvectors(oracle, k):
    dims = (2, 2, 2, 2)
    U, _ = random_fields(dims, 237)
    mass = 0.25
    S, ip = _dense_schur(dims, U, mass, 0)
    _, W = np.linalg.eig(S)
    b_p = W[:, [2, 19, 47, 80][:k]] @ np.array([1.0, 0.8 - 0.2j, -0.6j, 1.1][:k])
    x, hist = wd_solvers.bicgstab_schur(_embed(b_p, ip, dims), c2r(U), dims, mass, 0, niter=k)
    assert len(hist) == k + 1
    assert hist[k] < 1e-9
    assert hist[k - 1] > 1e3 * max(hist[k], 1e-13)


def test_k12_preconditioned_gcr_minimises_over_the_preconditioned_krylov_space(oracle):
    """GCR with a fixed linear preconditioner K: x_k minimises |b - Mhat x| over K K_k(Mhat K, b) =
    span{K b, K Mhat K b, ...} (right preconditioning); K = 1 reproduces the unpreconditioned solver bit for bit."""
    dims = (4, 2, 2, 4)
    U, b = random_fields(dims, 241)
    mass = -0.1
    Ur = c2r(U)
    bm = np.where((parity_mask(dims) == 0)[..., None, None, None], c2r(b[0]), 0.0)
    Mc = lambda v: r2c(oracle.schur(np.ascontiguousarray(c2r(v)), Ur, dims, mass, 0))
    a0 = 4.0 + mass
    K = lambda r: (2.0 / a0) * r - Mc(r) / a0 ** 2           # two terms of the Neumann series of Mhat^-1
    x0, h0 = wd_solvers.gcr_schur(c2r(b[0]), Ur, dims, mass, 0, niter=6, restart=8)
    x1, h1 = wd_solvers.gcr_schur(c2r(b[0]), Ur, dims, mass, 0, niter=6, restart=8, precond=lambda r: r.copy())
    assert np.array_equal(x0, x1) and np.array_equal(h0, h1)
    k = 5
    xk, hk = wd_solvers.gcr_schur(c2r(b[0]), Ur, dims, mass, 0, niter=k, restart=8, precond=K)
    basis = [K(r2c(bm))]
    for _ in range(k - 1):
        basis.append(K(Mc(basis[-1])))
    AK = np.stack([Mc(v).ravel() for v in basis], axis=1)
    Q, _ = np.linalg.qr(AK)
    bc = r2c(bm).ravel()
    best = np.linalg.norm(bc - Q @ (Q.conj().T @ bc)) / np.linalg.norm(bc)
    assert hk[-1] == pytest.approx(best, rel=1e-7)
    assert hk[-1] < 0.5 * h0[k]                               # and the preconditioner helps
    assert np.linalg.norm(bc - Mc(r2c(xk)).ravel()) / np.linalg.norm(bc) == pytest.approx(hk[-1], rel=1e-8)
