"""Pins for oracle/wd_storage.py (8-real links, half-precision storage).  CPU only.
  R1  8-real round trip on generic SU(3): reconstruct8(compress8(U)) = U for Haar-random and for smooth links, i.e.
      the rebuild formulas against matrices that were never built from them (the way P9 pins the 12-real rebuild)
  R2  any eight reals in range give a special-unitary matrix (U U^dag = 1, det U = 1): the rebuild itself is unitary
  R3  the rebuilt link carries exactly the stored numbers (a2, a3, b1, arg a1, arg c1 read back)
  R4  error amplification: perturbing the stored reals by eps moves the link by O(eps / N), N = |a2|^2 + |a3|^2
      (the bound DESIGN.md uses for the recon-8 tolerance)
  H1  half spinors: |value - psi| <= 2^-11 * site max, scale = site max exactly, zero sites stay zero
  H2  half links: |value - U| <= 2^-12 (reals in [-1, 1])
  H3  D on dequantised fields differs from D on the original ones by the quantisation level (a sanity bound used for
      the half-precision tolerance), through the pinned operator
"""
import numpy as np
import pytest

from oracle import wd_storage as ws
from paper_0912_2186_b200 import fields
from test_oracle_pins import c2r, r2c, random_fields


def _links(kind, dims=(4, 4, 4, 6)):
    return fields.haar_links(dims, 601) if kind == "haar" else fields.smooth_links(dims, 603, 0.3)


@pytest.mark.parametrize("kind,tol", [("haar", 1e-11), ("smooth", 1e-9)])
def test_r1_round_trip_on_generic_su3(kind, tol):
    U = _links(kind)
    back = ws.reconstruct8(ws.compress8(U))
    assert back.shape == U.shape
    assert np.max(np.abs(back - U)) < tol


def test_r2_rebuild_is_special_unitary_for_any_stored_reals():
    rng = np.random.default_rng(605)
    n = 2000
    v = rng.standard_normal((n, 6)) * 0.35
    keep = (v[:, :4] ** 2).sum(1) < 0.95
    v = v[keep]
    # b1 must fit the column: |b1|^2 <= 1 - |a1|^2 = N
    N = (v[:, :4] ** 2).sum(1)
    scale = np.minimum(1.0, 0.9 * np.sqrt(N / np.maximum((v[:, 4:6] ** 2).sum(1), 1e-30)))
    v[:, 4:6] *= scale[:, None]
    r = np.concatenate([v, rng.uniform(-1.0, 1.0, (len(v), 2))], axis=1)
    M = r2c(ws.reconstruct8(r))
    eye = np.eye(3)
    assert np.max(np.abs(M @ np.conj(np.swapaxes(M, -1, -2)) - eye)) < 1e-10
    assert np.max(np.abs(np.linalg.det(M) - 1.0)) < 1e-10


def test_r3_stored_numbers_are_carried():
    U = _links("haar")
    r = ws.compress8(U).astype(np.float32).astype(np.float64)
    M = r2c(ws.reconstruct8(r))
    assert np.array_equal(M[..., 0, 1].real, r[..., 0]) and np.array_equal(M[..., 0, 1].imag, r[..., 1])
    assert np.array_equal(M[..., 0, 2].real, r[..., 2]) and np.array_equal(M[..., 1, 0].imag, r[..., 5])
    wrap = lambda d: (d + 1.0) % 2.0 - 1.0                    # phases in units of pi, compared modulo 2
    assert np.max(np.abs(wrap(np.angle(M[..., 0, 0]) / np.pi - r[..., 6]))) < 1e-12
    assert np.max(np.abs(wrap(np.angle(M[..., 2, 0]) / np.pi - r[..., 7]))) < 1e-12


def test_r4_rounding_is_amplified_by_one_over_n():
    U = _links("smooth")
    r = ws.compress8(U)
    N = r[..., 0] ** 2 + r[..., 1] ** 2 + r[..., 2] ** 2 + r[..., 3] ** 2
    exact = ws.reconstruct8(r)
    rounded = ws.reconstruct8(r.astype(np.float32).astype(np.float64))
    err = np.max(np.abs(rounded - exact), axis=(-3, -2, -1))
    eps = 2.0 ** -24 * np.pi            # half an ulp of the largest stored number (a phase of 1, worth pi radians)
    assert np.all(err <= 40 * eps / np.minimum(N, 1.0))
    assert np.max(err * N) > 0.05 * eps  # (and the bound is not vacuous)


def test_h1_half_spinor_quantisation():
    psi = fields.gaussian_spinor((4, 4, 2, 6), 607, 2, 32)
    psi[0, 1, 0, 2, 3] = 0.0                                  # a zero site
    q, s = ws.quantise_half_spinor(psi)
    assert q.dtype == np.float16 and s.dtype == np.float32
    assert np.array_equal(s, np.max(np.abs(psi), axis=(-3, -2, -1)))
    val = ws.dequantise_half_spinor(q, s)
    assert np.all(np.abs(val - psi) <= 2.0 ** -11 * s[..., None, None, None] * (1 + 1e-6))
    assert np.all(val[0, 1, 0, 2, 3] == 0)
    assert np.max(np.abs(q.astype(np.float64))) == 1.0        # the largest component of a site is stored as +-1


def test_h2_half_links():
    U = _links("haar")
    assert np.max(np.abs(ws.quantise_half_links(U) - U)) <= 2.0 ** -12 * (1 + 1e-6) + 2.0 ** -25


def test_h3_operator_on_dequantised_fields(oracle):
    dims = (4, 4, 4, 4)
    U, psi = random_fields(dims, 609)
    q, s = ws.quantise_half_spinor(c2r(psi[0]))
    exact = oracle.apply(c2r(psi[0]), c2r(U), dims, -0.3)
    quant = oracle.apply(ws.dequantise_half_spinor(q, s), ws.quantise_half_links(c2r(U)), dims, -0.3)
    rel = np.linalg.norm(quant - exact) / np.linalg.norm(exact)
    assert 1e-5 < rel < 1e-3
