"""CPU ORACLE for the Krylov shell around the Wilson-Dirac matvec (PAPER.md:116
"CG on the normal equations", PAPER.md:153-167 CG solvers built on the even-odd matvec).

TEST INFRASTRUCTURE ONLY (same rules as wd_oracle.py): plain numpy, fp64, textbook algorithm written out step by
step; every operator application goes through oracle/wd_oracle.c.  Nothing under paper_0912_2186_b200/ imports it.

cgnr_schur: conjugate gradients on the normal equations of the even-odd preconditioned operator
    Mhat^dagger Mhat x = Mhat^dagger b        (Mhat = (4+m) - H_pq H_qp/(4+m) on one parity; Mhat^dagger = sign=+1)
in the CGNR form (Hestenes-Stiefel CG applied to A = Mhat^dagger Mhat without ever forming A):

    x_0 = 0,  r_0 = b,  z_0 = Mhat^dagger r_0,  p_0 = z_0,  zz_0 = <z_0, z_0>
    for k = 0, 1, ...:
        w     = Mhat p_k
        alpha = zz_k / <w, w>
        x    += alpha p_k
        r    -= alpha w                         (r = b - Mhat x, the true-equation residual)
        z     = Mhat^dagger r
        zz'   = <z, z>
        beta  = zz' / zz_k
        p     = z + beta p_k

Fields are full-lattice canonical arrays that vanish off `parity` (as oracle.schur produces and ignores).
Returns x and the history of |r_k|_2 / |b|_2 (k = 0..niter).
"""
import numpy as np

from . import wd_oracle


def _mask(psi, dims, parity):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    on = ((x + y + z + t) % 2 == parity)[..., None, None, None]
    return np.where(on, psi, 0.0)


def cgnr_schur(b, U, dims, mass, parity, niter, tol=0.0):
    """niter iterations (or until |r|/|b| <= tol) of CGNR for Mhat x = b on `parity`.  b: [Lt,Lz,Ly,Lx,4,3,2] fp64."""
    b = _mask(np.ascontiguousarray(b, dtype=np.float64), dims, parity)
    U = np.ascontiguousarray(U, dtype=np.float64)
    M = lambda v: wd_oracle.schur(v, U, dims, mass, parity, sign=-1)
    Md = lambda v: wd_oracle.schur(v, U, dims, mass, parity, sign=+1)
    x = np.zeros_like(b)
    r = b.copy()
    z = Md(r)
    p = z.copy()
    zz = float(np.vdot(z, z))
    bnorm = float(np.sqrt(np.vdot(b, b)))
    hist = [float(np.sqrt(np.vdot(r, r))) / bnorm]
    for _ in range(niter):
        if hist[-1] <= tol:
            break
        w = M(p)
        alpha = zz / float(np.vdot(w, w))
        x += alpha * p
        r -= alpha * w
        z = Md(r)
        zz_new = float(np.vdot(z, z))
        beta = zz_new / zz
        p = z + beta * p
        zz = zz_new
        hist.append(float(np.sqrt(np.vdot(r, r))) / bnorm)
    return x, np.array(hist)
