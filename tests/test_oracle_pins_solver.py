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
