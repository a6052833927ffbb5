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


def cgnr_schur(b, U, dims, mass, parity, niter, tol=0.0, trace=None):
    """niter iterations (or until |r|/|b| <= tol) of CGNR for Mhat x = b on `parity`.  b: [Lt,Lz,Ly,Lx,4,3,2] fp64.
    trace: optional list; a copy of the iterate x_k is appended after every iteration (for the pins only)."""
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
        if trace is not None:
            trace.append(x.copy())
    return x, np.array(hist)


def bicgstab_schur(b, U, dims, mass, parity, niter, tol=0.0, trace=None):
    """niter iterations (or until |r|/|b| <= tol) of BiCGstab (van der Vorst 1992, unpreconditioned) for
    Mhat x = b on `parity`, x_0 = 0 (the paper's other solver around the even-odd matvec):

        r = b, rhat = r, rho = alpha = omega = 1, v = p = 0
        loop:  rho' = <rhat, r>;  beta = (rho'/rho)(alpha/omega);  p = r + beta (p - omega v);  v = Mhat p
               alpha = rho' / <rhat, v>;  s = r - alpha v;  t = Mhat s;  omega = <t, s> / <t, t>
               x += alpha p + omega s;  r = s - omega t;  rho = rho'

    Complex inner products <a, b> = sum conj(a) b over (site, spin, colour).  Returns x (real-pair layout) and the
    history of |r_k| / |b|.  trace: optional list; the vectors (rhat, s, t, r_new, x_new) of every iteration are
    appended as complex arrays (for the pins only)."""
    b = _mask(np.ascontiguousarray(b, dtype=np.float64), dims, parity)
    U = np.ascontiguousarray(U, dtype=np.float64)
    c = lambda v: v[..., 0] + 1j * v[..., 1]
    rp = lambda v: np.stack([v.real, v.imag], axis=-1)
    M = lambda v: c(wd_oracle.schur(np.ascontiguousarray(rp(v)), U, dims, mass, parity))
    r = c(b)
    rhat = r.copy()
    x = np.zeros_like(r)
    v = np.zeros_like(r)
    p = np.zeros_like(r)
    rho = alpha = omega = 1.0 + 0.0j
    bnorm = float(np.sqrt(np.vdot(r, r).real))
    hist = [1.0]
    for _ in range(niter):
        if hist[-1] <= tol:
            break
        rho_new = np.vdot(rhat, r)
        beta = (rho_new / rho) * (alpha / omega)
        p = r + beta * (p - omega * v)
        v = M(p)
        alpha = rho_new / np.vdot(rhat, v)
        s = r - alpha * v
        t = M(s)
        omega = np.vdot(t, s) / np.vdot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho = rho_new
        hist.append(float(np.sqrt(np.vdot(r, r).real)) / bnorm)
        if trace is not None:
            trace.append((rhat.copy(), s.copy(), t.copy(), r.copy(), x.copy()))
    return rp(x), np.array(hist)


def gcr_schur(b, U, dims, mass, parity, niter, restart=8, tol=0.0, precond=None):
    """niter iterations of restarted GCR(restart) (Eisenstat-Elman-Schultz 1983; "GCR(8) outer Krylov
    solver") for Mhat x = b on `parity`, x_0 = 0.  precond: None, or a callable K on complex fields [Lt,Lz,Ly,Lx,4,3]
    (the multigrid cycle "is used as a preconditioner" for this solver): the search direction is K r.

        r = b
        loop k = 0, 1, ...   (j = k mod restart is the position inside the current cycle; a new cycle forgets all p's)
            p_j = K r  (K = 1 without a preconditioner);  q_j = Mhat p_j
            for i < j:  beta = <q_i, q_j> / <q_i, q_i>;  p_j -= beta p_i;  q_j -= beta q_i        (modified Gram-Schmidt)
            alpha = <q_j, r> / <q_j, q_j>;  x += alpha p_j;  r -= alpha q_j

    One operator application per iteration.  Returns x (real-pair layout) and the history of |r_k| / |b|."""
    b = _mask(np.ascontiguousarray(b, dtype=np.float64), dims, parity)
    U = np.ascontiguousarray(U, dtype=np.float64)
    c = lambda v: v[..., 0] + 1j * v[..., 1]
    rp = lambda v: np.stack([v.real, v.imag], axis=-1)
    M = lambda v: c(wd_oracle.schur(np.ascontiguousarray(rp(v)), U, dims, mass, parity))
    r = c(b)
    x = np.zeros_like(r)
    bnorm = float(np.sqrt(np.vdot(r, r).real))
    hist = [1.0]
    P, Q, QQ = [], [], []
    for k in range(niter):
        if hist[-1] <= tol:
            break
        if k % restart == 0:
            P, Q, QQ = [], [], []
        p = r.copy() if precond is None else precond(r)
        q = M(p)
        for pi, qi, qqi in zip(P, Q, QQ):
            beta = np.vdot(qi, q) / qqi
            p = p - beta * pi
            q = q - beta * qi
        qq = np.vdot(q, q).real
        alpha = np.vdot(q, r) / qq
        x = x + alpha * p
        r = r - alpha * q
        P.append(p)
        Q.append(q)
        QQ.append(qq)
        hist.append(float(np.sqrt(np.vdot(r, r).real)) / bnorm)
    return rp(x), np.array(hist)
