"""Seeded synthetic input generators shared by the oracle-side tests and the CUDA path.

This module holds NONE of the method's arithmetic (no gamma matrices, no hopping term, no link
reconstruction): it only draws random SU(3) links and Gaussian spinors in the canonical layouts
and lists the five BASELINE.json workloads.  Both the oracle (oracle/) and the CUDA library
consume exactly the arrays produced here (rounded ONCE to the working precision, S12).

The synthetic fields stand in for the paper's beta=5.5 gauge ensembles (16^3x64, 24^3x64,
32^3x96) and GPU volumes (24^3x48, 24^3xT), which are not
available; the kernel's cost is data independent, only shapes/word sizes/storage format matter.

Canonical layouts (S5/S6), numpy C-order:
  links   U[mu 0..3][t][z][y][x][row a][col b][re,im]
  spinor  psi[rhs][t][z][y][x][spin][colour][re,im]       dims = (Lx, Ly, Lz, Lt)
"""
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    dims: tuple          # (Lx, Ly, Lz, Lt)
    precision: int       # 32 or 64
    links: str           # "haar" | "smooth"
    recon: int           # 18 or 12
    mass: float
    nrhs: int
    seed: int
    eps: float = 0.3


# BASELINE.json:configs[0..4]; config 3 is quoted in both precisions.
CONFIGS = {
    "c0_4x4_fp64": Config("c0_4x4_fp64", (4, 4, 4, 4), 64, "haar", 18, 0.1, 1, 1),
    "c1_16x32_fp32": Config("c1_16x32_fp32", (16, 16, 16, 32), 32, "smooth", 18, -0.4, 1, 2),
    "c2_24x64_fp32_r12": Config("c2_24x64_fp32_r12", (24, 24, 24, 64), 32, "haar", 12, -0.4, 1, 3),
    "c3_32x64_fp32": Config("c3_32x64_fp32", (32, 32, 32, 64), 32, "smooth", 18, -0.42, 1, 4),
    "c3_32x64_fp64": Config("c3_32x64_fp64", (32, 32, 32, 64), 64, "smooth", 18, -0.42, 1, 4),
    "c4_32x64_fp32_24rhs": Config("c4_32x64_fp32_24rhs", (32, 32, 32, 64), 32, "smooth", 18, -0.42, 24, 5),
}


def volume(dims):
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def _site_shape(dims):
    Lx, Ly, Lz, Lt = (int(d) for d in dims)
    return (Lt, Lz, Ly, Lx)


def _complex_normal(rng, shape):
    """Re, Im ~ N(0,1) drawn in one standard_normal call in canonical order (..., [re,im])."""
    z = rng.standard_normal(shape + (2,))
    return z[..., 0] + 1j * z[..., 1]


# ---- batched 3x3 complex algebra in "component" form ------------------------------------------
# A stack of matrices is held as a list m[3*i+j] of nine contiguous complex vectors; numpy's
# stacked matmul / strided column slices are an order of magnitude slower for 3x3 blocks.
def _split9(z):
    """[n,3,3] complex -> list of nine contiguous [n] vectors."""
    return [np.ascontiguousarray(z[:, i, j]) for i in range(3) for j in range(3)]


def _join9(m, out):
    for i in range(3):
        for j in range(3):
            out[:, i, j] = m[3 * i + j]


def _mm9(a, b):
    return [a[3 * i] * b[j] + a[3 * i + 1] * b[3 + j] + a[3 * i + 2] * b[6 + j] for i in range(3) for j in range(3)]


def _unitarise9(m):
    """QR factorisation Z = Q R with R_ii > 0 (Gram-Schmidt on the columns of Z), then
    Q <- Q * exp(-i arg(det Q)/3) so that det Q = 1.

    For complex Gaussian Z this Q is Haar distributed on U(3) (BASELINE.json:configs[0]:
    "QR of complex Gaussian 3x3, phase-fixed to det=1")."""
    c = [[m[0 + j], m[3 + j], m[6 + j]] for j in range(3)]  # columns

    def dot(a, b):  # <a, b> = sum conj(a) b
        return np.conj(a[0]) * b[0] + np.conj(a[1]) * b[1] + np.conj(a[2]) * b[2]

    def normalise(v):
        n = 1.0 / np.sqrt(np.real(dot(v, v)))
        return [v[0] * n, v[1] * n, v[2] * n]

    def sub(v, w, s):
        return [v[0] - w[0] * s, v[1] - w[1] * s, v[2] - w[2] * s]

    for _ in range(2):  # two Gram-Schmidt passes: orthogonal to rounding level
        c[0] = normalise(c[0])
        c[1] = normalise(sub(c[1], c[0], dot(c[0], c[1])))
        c[2] = sub(c[2], c[0], dot(c[0], c[2]))
        c[2] = normalise(sub(c[2], c[1], dot(c[1], c[2])))
    q = [c[j][i] for i in range(3) for j in range(3)]
    det = (q[0] * (q[4] * q[8] - q[5] * q[7]) - q[1] * (q[3] * q[8] - q[5] * q[6])
           + q[2] * (q[3] * q[7] - q[4] * q[6]))
    phase = np.exp(-1j * np.angle(det) / 3.0)
    return [e * phase for e in q]


def _expm9(x):
    """exp(x) for |x| ~ 1: order-12 Taylor series of x/8 (Horner), squared three times."""
    y = [e / 8.0 for e in x]
    one = np.ones_like(y[0])
    zero = np.zeros_like(y[0])
    u = [one if i == j else zero for i in range(3) for j in range(3)]
    for k in range(12, 0, -1):
        yu = _mm9(y, u)
        u = [(one if i == j else zero) + yu[3 * i + j] / k for i in range(3) for j in range(3)]
    for _ in range(3):
        u = _mm9(u, u)
    return u


def _map_chunks(fn, z):
    """Apply fn (list-of-9 -> list-of-9) to a [..., 3, 3] complex array, chunked over a thread pool.
    Every matrix is processed independently, so the result does not depend on the thread count."""
    flat = z.reshape(-1, 3, 3)
    out = np.empty_like(flat)
    step = 1 << 15

    def work(s0):
        _join9(fn(_split9(flat[s0:s0 + step])), out[s0:s0 + step])

    with ThreadPoolExecutor(max_workers=min(32, os.cpu_count() or 1)) as pool:
        list(pool.map(work, range(0, flat.shape[0], step)))
    return out.reshape(z.shape)


def _to_real_pairs(c):
    out = np.empty(c.shape + (2,), dtype=np.float64)
    out[..., 0] = c.real
    out[..., 1] = c.imag
    return out


def haar_links(dims, seed):
    """Haar-random SU(3) links, float64 [4, Lt, Lz, Ly, Lx, 3, 3, 2]."""
    rng = np.random.default_rng(seed)
    z = _complex_normal(rng, (4,) + _site_shape(dims) + (3, 3))
    return _to_real_pairs(_map_chunks(_unitarise9, z))


def smooth_links(dims, seed, eps=0.3):
    """Links close to the identity: U = exp(i eps H), H traceless Hermitian Gaussian, each link
    independent, re-unitarised to SU(3) (BASELINE.json:configs[1]).  float64, same layout.

    H = (A + A^dagger)/2 - tr(.)/3, A complex Gaussian (Re, Im ~ N(0,1))."""
    rng = np.random.default_rng(seed)
    a = _complex_normal(rng, (4,) + _site_shape(dims) + (3, 3))

    def one_chunk(m):
        h = [0.5 * (m[3 * i + j] + np.conj(m[3 * j + i])) for i in range(3) for j in range(3)]
        tr = (h[0] + h[4] + h[8]) / 3.0
        for i in (0, 4, 8):
            h[i] = h[i] - tr
        return _unitarise9(_expm9([(1j * eps) * e for e in h]))

    return _to_real_pairs(_map_chunks(one_chunk, a))


def unit_links(dims):
    """U = identity everywhere (free field)."""
    u = np.zeros((4,) + _site_shape(dims) + (3, 3, 2), dtype=np.float64)
    for i in range(3):
        u[..., i, i, 0] = 1.0
    return u


def gaussian_spinor(dims, seed, nrhs=1, precision=64):
    """Complex Gaussian spinors (Re, Im ~ N(0,1)), [nrhs, Lt, Lz, Ly, Lx, 4, 3, 2].

    Drawn in canonical order from one generator, one right-hand side per standard_normal call
    (the stream is the same as a single call); each is rounded once to `precision` as it is drawn
    so that 24 right-hand sides of 32^3x64 never exist in float64 at the same time."""
    rng = np.random.default_rng(seed)
    shape = _site_shape(dims) + (4, 3, 2)
    out = np.empty((int(nrhs),) + shape, dtype=np.float32 if int(precision) == 32 else np.float64)
    for r in range(int(nrhs)):
        out[r] = rng.standard_normal(shape)
    return out


def round_to(a, precision):
    """Round ONCE to the working precision (S12).  The returned array is what the CUDA
    path receives as is; the oracle receives the same values widened back to float64."""
    return np.ascontiguousarray(a, dtype=np.float32 if int(precision) == 32 else np.float64)


def make_fields(cfg, nrhs=None, dims=None):
    """(U, psi) in working precision for a Config; links seeded with cfg.seed, spinors with seed+1000."""
    d = tuple(dims) if dims is not None else cfg.dims
    n = cfg.nrhs if nrhs is None else int(nrhs)
    if cfg.links == "haar":
        u = haar_links(d, cfg.seed)
    elif cfg.links == "smooth":
        u = smooth_links(d, cfg.seed, cfg.eps)
    else:
        raise ValueError(cfg.links)
    psi = gaussian_spinor(d, cfg.seed + 1000, n, cfg.precision)
    return round_to(u, cfg.precision), psi


def temporal_gauge(U, precision=64):
    """Gauge-transform canonical links U [4,Lt,Lz,Ly,Lx,3,3,2] to temporal gauge ("temporal gauge fixing"):
    g(x,0) = 1, g(x,t+1) = g(x,t) U_t(x,t), U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger, so that U'_t(x,t) = 1 (set exactly)
    for t < Lt-1 and the last slice carries the Polyakov lines.  Input preparation only: D(U')(g psi) = g D(U) psi is
    the same operator.  Returns (U' rounded to `precision`, g as complex [Lt,Lz,Ly,Lx,3,3])."""
    Uc = U[..., 0].astype(np.float64) + 1j * U[..., 1].astype(np.float64)        # [4,Lt,Lz,Ly,Lx,3,3]
    Lt = Uc.shape[1]
    g = np.empty(Uc.shape[1:], dtype=np.complex128)
    g[0] = np.eye(3)
    for t in range(Lt - 1):
        g[t + 1] = g[t] @ Uc[3, t]
    out = np.empty_like(Uc)
    for mu in range(4):
        g_fwd = np.roll(g, -1, axis=3 - mu)                                      # g(x + mu), site axes are [t,z,y,x]
        out[mu] = g @ Uc[mu] @ np.conj(np.swapaxes(g_fwd, -1, -2))
    out[3, :Lt - 1] = np.eye(3)
    return round_to(_to_real_pairs(out), precision), g
