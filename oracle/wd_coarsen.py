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
