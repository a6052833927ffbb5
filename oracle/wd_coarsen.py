"""CPU ORACLE for the adaptive-multigrid transfer operators.

TEST INFRASTRUCTURE ONLY (same rules as wd_oracle.py).  Plain numpy, fp64, definitions written out.

Given N_v global vectors psi^(alpha) (the near-null vectors of eq. (2.6); how they are found is not specified by
the paper, PAPER.md:112 -- they are INPUTS here), eq. (2.7) defines the prolongator

    P_{x; xhat, alpha} = orthonormal basis for { theta_xhat(x) psi^(alpha)_x }

on 4^4 space-time blocks xhat, with every block split in two sub-blocks for gamma5 = +-1 (spin components 0,1
and 2,3 in the DeGrand-Rossi basis), labelled sigma3 = +-1, so that sigma3 P = P gamma5.
Reading (the paper does not say which orthonormal basis): modified Gram-Schmidt over alpha = 0..N_v-1 in the given
order, inside every (block, chirality) separately, complex inner product over the block's sites, the chirality's two
spin components and the three colours.  Coarse vectors: c[block (bt,bz,by,bx)][sigma 0..1][alpha 0..N_v-1].

    restrict   P^dagger psi :  c[b, s, a]   = sum_{x in b, spin in s, colour} conj(W_a(x)) psi(x)
    prolong    P c          :  psi(x)       = sum_a c[b(x), s(spin), a] W_a(x)
    coarse op  Dhat c       =  P^dagger D P c      (Galerkin, R = P^dagger), D through wd_oracle.c
"""
import numpy as np

from . import wd_oracle

BLOCK = (4, 4, 4, 4)  # (x, y, z, t) extents of a block


def _blocked(v, dims, block=BLOCK):
    """[..., Lt, Lz, Ly, Lx, 4, 3] -> [..., bt, bz, by, bx, chir, (t4, z4, y4, x4, spin-in-chirality, colour)]."""
    Lx, Ly, Lz, Lt = dims
    bx, by, bz, bt = block
    lead = v.shape[:-6]
    w = v.reshape(lead + (Lt // bt, bt, Lz // bz, bz, Ly // by, by, Lx // bx, bx, 2, 2, 3))
    n = len(lead)
    # axes: lead, Bt, t, Bz, z, By, y, Bx, x, chir, s, c  ->  lead, Bt, Bz, By, Bx, chir, t, z, y, x, s, c
    perm = tuple(range(n)) + tuple(n + i for i in (0, 2, 4, 6, 8, 1, 3, 5, 7, 9, 10))
    w = np.transpose(w, perm)
    return w.reshape(w.shape[:n + 5] + (-1,))


def _unblocked(w, dims, lead_shape, block=BLOCK):
    Lx, Ly, Lz, Lt = dims
    bx, by, bz, bt = block
    n = len(lead_shape)
    w = w.reshape(lead_shape + (Lt // bt, Lz // bz, Ly // by, Lx // bx, 2, bt, bz, by, bx, 2, 3))
    # inverse of the permutation above
    perm = tuple(range(n)) + tuple(n + i for i in (0, 5, 1, 6, 2, 7, 3, 8, 4, 9, 10))
    w = np.transpose(w, perm)
    return w.reshape(lead_shape + (Lt, Lz, Ly, Lx, 4, 3))


def check_dims(dims, block=BLOCK):
    for L, b in zip(dims, block):
        if L % b:
            raise ValueError(f"extent {L} is not a multiple of the block extent {b}")


def block_orthonormalise(psis, dims, block=BLOCK):
    """psis complex [Nv, Lt, Lz, Ly, Lx, 4, 3] -> W same shape: eq. (2.7), modified Gram-Schmidt per (block, chirality)."""
    check_dims(dims, block)
    v = _blocked(np.asarray(psis, dtype=np.complex128), dims, block).copy()   # [Nv, Bt,Bz,By,Bx, chir, n]
    nv = v.shape[0]
    for a in range(nv):
        for b in range(a):
            proj = np.sum(np.conj(v[b]) * v[a], axis=-1, keepdims=True)       # <w_b, v_a> per (block, chirality)
            v[a] = v[a] - proj * v[b]
        nrm = np.sqrt(np.sum(np.abs(v[a]) ** 2, axis=-1, keepdims=True))
        v[a] = v[a] / nrm
    return _unblocked(v, dims, (nv,), block)


def restrict(W, psi, dims, block=BLOCK):
    """P^dagger psi: W [Nv, sites.., 4, 3], psi [sites.., 4, 3] -> c [Bt, Bz, By, Bx, 2, Nv]."""
    wb = _blocked(np.asarray(W, dtype=np.complex128), dims, block)
    pb = _blocked(np.asarray(psi, dtype=np.complex128), dims, block)
    return np.moveaxis(np.sum(np.conj(wb) * pb[None], axis=-1), 0, -1)


def prolong(W, c, dims, block=BLOCK):
    """P c: c [Bt, Bz, By, Bx, 2, Nv] -> psi [sites.., 4, 3]."""
    wb = _blocked(np.asarray(W, dtype=np.complex128), dims, block)            # [Nv, B.., chir, n]
    out = np.sum(np.moveaxis(np.asarray(c, dtype=np.complex128), -1, 0)[..., None] * wb, axis=0)
    return _unblocked(out, dims, (), block)


def coarse_apply(W, c, U, dims, mass, block=BLOCK):
    """Dhat c = P^dagger D P c with D from wd_oracle.c (U real-pair canonical links)."""
    psi = prolong(W, c, dims, block)
    dpsi = wd_oracle.apply(np.ascontiguousarray(np.stack([psi.real, psi.imag], axis=-1)), U, dims, mass)
    return restrict(W, dpsi[..., 0] + 1j * dpsi[..., 1], dims, block)


# ----------------------------------------------------------------------------------------------------------------------
# The coarse operator as an explicit nearest-neighbour stencil (PAPER.md:82-88 Galerkin form Dhat = P^dagger D P;
# PAPER.md:116 4^4 blocks x chirality; "N_V x N_V complex matrix operations needed for the coarse
# operators").  D of eq. (2.2) couples nearest neighbours only, so Dhat couples a block to itself and to its 8
# neighbouring blocks.  With the coarse index i = sigma * N_v + alpha (n = 2 N_v per block) and W^sigma_alpha the basis
# vector restricted to chirality sigma, the definition written out is
#
#   S[b][0]       = A(b)     = sum_{x in b} W(x)^dag [ (4+m) W(x) + sum over the 8 hops whose source site is ALSO in b ]
#   S[b][1 + mu]  = F_mu(b)  = sum_{x in b, x+mu in b+mu}  W(x)^dag [ -1/2 (1 - gamma_mu) U_mu(x)          W(x+mu) ]
#   S[b][5 + mu]  = B_mu(b)  = sum_{x in b, x-mu in b-mu}  W(x)^dag [ -1/2 (1 + gamma_mu) U_mu(x-mu)^dag   W(x-mu) ]
#
#   (Dhat c)(b) = A(b) c(b) + sum_mu [ F_mu(b) c(b+mu) + B_mu(b) c(b-mu) ]          (periodic coarse lattice)
#
# "x+mu in b+mu" means the hop leaves the block through its +mu face (x_mu mod 4 == 3), whatever block it lands in: with
# coarse extent 1 or 2 the block b+mu coincides with b or with b-mu and the terms simply add (reading S4 carried over).
# Explicit dense gamma matrices (wd_oracle.gamma), np.roll for the periodic shifts; no blocking or fusion.
# ----------------------------------------------------------------------------------------------------------------------
def _site_axis(mu):
    """axis of direction mu (0..3 = x,y,z,t) in a [Lt, Lz, Ly, Lx, ...] array"""
    return 3 - mu


def coarse_stencil(W, U, dims, mass, block=BLOCK):
    """W complex [Nv, Lt,Lz,Ly,Lx, 4,3] (the columns of P, eq. (2.7)); U real-pair canonical links [4, Lt,Lz,Ly,Lx,3,3,2].
    Returns S complex [Bt,Bz,By,Bx, 9, n, n], n = 2 Nv, row/column index sigma * Nv + alpha, matrices ordered
    (A, F_x, F_y, F_z, F_t, B_x, B_y, B_z, B_t)."""
    check_dims(dims, block)
    W = np.asarray(W, dtype=np.complex128)
    nv = W.shape[0]
    Uc = np.asarray(U, dtype=np.float64)
    Uc = Uc[..., 0] + 1j * Uc[..., 1]                                   # [4, Lt,Lz,Ly,Lx, 3,3]
    Lx, Ly, Lz, Lt = dims
    coords = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")   # t, z, y, x
    nb = (Lt // block[3], Lz // block[2], Ly // block[1], Lx // block[0])
    S = np.zeros(nb + (9, 2, nv, 2, nv), dtype=np.complex128)          # [.., k, sigma, alpha, sigma', alpha']
    Wb = _blocked(W, dims, block)                                      # [Nv, B.., sigma, sites x spin-in-chirality x colour]

    def accumulate(k, H, sp, mask):
        """S[.., k, sigma, alpha, sp, alpha'] += sum over the masked sites of conj(W_alpha) . H_alpha' (rows in sigma)"""
        Hb = _blocked(H * mask[None, ..., None, None], dims, block)    # [Nv', B.., sigma, n]
        S[..., k, :, :, sp, :] += np.einsum("aBCDEsn,cBCDEsn->BCDEsac", np.conj(Wb), Hb)

    one = np.ones((Lt, Lz, Ly, Lx))
    for sp in range(2):                                                # chirality sigma' of the source vectors
        Wsp = np.zeros_like(W)
        Wsp[..., 2 * sp:2 * sp + 2, :] = W[..., 2 * sp:2 * sp + 2, :]
        accumulate(0, (4.0 + mass) * Wsp, sp, one)                     # diagonal term of eq. (2.2)
        for mu in range(4):
            ax = _site_axis(mu)
            g = wd_oracle.gamma(mu)
            xm = coords[ax] % block[mu]
            # forward hop: -1/2 (1 - gamma_mu) U_mu(x) W(x + mu)
            Wf = np.roll(Wsp, -1, axis=1 + ax)
            H = np.einsum("...ab,n...sb->n...sa", Uc[mu], Wf)
            H = -0.5 * np.einsum("st,n...ta->n...sa", np.eye(4) - g, H)
            leaves = (xm == block[mu] - 1).astype(np.float64)
            accumulate(1 + mu, H, sp, leaves)
            accumulate(0, H, sp, 1.0 - leaves)
            # backward hop: -1/2 (1 + gamma_mu) U_mu(x - mu)^dag W(x - mu)
            Wbk = np.roll(Wsp, +1, axis=1 + ax)
            Ub = np.roll(Uc[mu], +1, axis=ax)
            H = np.einsum("...ba,n...sb->n...sa", np.conj(Ub), Wbk)
            H = -0.5 * np.einsum("st,n...ta->n...sa", np.eye(4) + g, H)
            leaves = (xm == 0).astype(np.float64)
            accumulate(5 + mu, H, sp, leaves)
            accumulate(0, H, sp, 1.0 - leaves)
    return S.reshape(nb + (9, 2 * nv, 2 * nv))


def coarse_apply_stencil(S, c):
    """(Dhat c)(b) = A(b) c(b) + sum_mu [ F_mu(b) c(b+mu) + B_mu(b) c(b-mu) ];  c [Bt,Bz,By,Bx, 2, Nv] -> same shape."""
    c = np.asarray(c, dtype=np.complex128)
    shp = c.shape
    v = c.reshape(shp[:4] + (-1,))
    out = np.einsum("...ij,...j->...i", S[..., 0, :, :], v)
    for mu in range(4):
        ax = _site_axis(mu)
        out += np.einsum("...ij,...j->...i", S[..., 1 + mu, :, :], np.roll(v, -1, axis=ax))
        out += np.einsum("...ij,...j->...i", S[..., 5 + mu, :, :], np.roll(v, +1, axis=ax))
    return out.reshape(shp)
