"""ctypes wrapper around oracle/wd_oracle.c -- the CPU ORACLE for D*psi (eq. (2.2)).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Nothing under paper_0912_2186_b200/ imports this module
and this module imports nothing from there.  All arithmetic is in wd_oracle.c (fp64); this file
only builds the shared object with gcc and marshals numpy arrays.

Canonical layouts (S5/S6):
  psi  float64 [nrhs, Lt, Lz, Ly, Lx, 4, 3, 2]      (or without the leading nrhs axis)
  U    float64 [4, Lt, Lz, Ly, Lx, 3, 3, 2]         recon 18
  U12  float64 [4, Lt, Lz, Ly, Lx, 2, 3, 2]         recon 12 (rows 0,1 of each link)
  dims = (Lx, Ly, Lz, Lt)
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wd_oracle.c")
_LIB = os.path.join(_HERE, "libwd_oracle.so")
_lib = None


def build(force=False):
    """Compile wd_oracle.c with gcc (plain -O2, OpenMP over sites). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.wdo_apply.argtypes = [dp, dp, dp, ip, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.wdo_apply.restype = ctypes.c_int
        lib.wdo_apply_range.argtypes = [dp, dp, dp, ip, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                        ctypes.c_int, ctypes.c_long, ctypes.c_long]
        lib.wdo_apply_range.restype = ctypes.c_int
        lib.wdo_hop_parity.argtypes = [dp, dp, dp, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.wdo_hop_parity.restype = ctypes.c_int
        lib.wdo_schur.argtypes = [dp, dp, dp, ip, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.wdo_schur.restype = ctypes.c_int
        lib.wdo_gamma.argtypes = [ctypes.c_int, dp]
        lib.wdo_gamma.restype = None
        lib.wdo_num_threads.restype = ctypes.c_int
        lib.wdo_set_num_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def num_threads():
    """OpenMP threads the oracle will use (omp_get_max_threads)."""
    return int(_load().wdo_num_threads())


def set_num_threads(n):
    _load().wdo_set_num_threads(int(n))


def gamma(mu):
    """The oracle's own gamma_mu (mu = 0..3 = x,y,z,t) as a complex 4x4 array."""
    buf = np.zeros(32, dtype=np.float64)
    _load().wdo_gamma(int(mu), _dptr(buf))
    g = buf.reshape(4, 4, 2)
    return g[..., 0] + 1j * g[..., 1]


def _check(psi, U, dims):
    Lx, Ly, Lz, Lt = (int(d) for d in dims)
    psi = np.ascontiguousarray(psi, dtype=np.float64)
    U = np.ascontiguousarray(U, dtype=np.float64)
    squeeze = False
    if psi.ndim == 7:
        psi = psi[None]
        squeeze = True
    if psi.shape[1:] != (Lt, Lz, Ly, Lx, 4, 3, 2):
        raise ValueError(f"psi shape {psi.shape} does not match dims {dims}")
    if U.shape == (4, Lt, Lz, Ly, Lx, 3, 3, 2):
        recon = 18
    elif U.shape == (4, Lt, Lz, Ly, Lx, 2, 3, 2):
        recon = 12
    else:
        raise ValueError(f"U shape {U.shape} does not match dims {dims}")
    return psi, U, recon, squeeze, (Lx, Ly, Lz, Lt)


def apply(psi, U, dims, mass, sign=-1):
    """out = D(U; mass) psi in fp64.  sign=-1: the operator of the build; sign=+1: gamma5 D gamma5."""
    psi, U, recon, squeeze, d = _check(psi, U, dims)
    out = np.empty_like(psi)
    cd = (ctypes.c_int * 4)(*d)
    rc = _load().wdo_apply(_dptr(out), _dptr(psi), _dptr(U), cd, float(mass), psi.shape[0], recon, int(sign))
    if rc != 0:
        raise RuntimeError(f"wdo_apply failed rc={rc}")
    return out[0] if squeeze else out


def apply_range(psi, U, dims, mass, site_begin, site_end, sign=-1):
    """Like apply() but only lexicographic sites [site_begin, site_end) are computed.

    Returns float64 [nrhs, site_end-site_begin, 4, 3, 2] (or without nrhs axis)."""
    psi, U, recon, squeeze, d = _check(psi, U, dims)
    out = np.zeros_like(psi)
    cd = (ctypes.c_int * 4)(*d)
    rc = _load().wdo_apply_range(_dptr(out), _dptr(psi), _dptr(U), cd, float(mass), psi.shape[0], recon,
                                 int(sign), int(site_begin), int(site_end))
    if rc != 0:
        raise RuntimeError(f"wdo_apply_range failed rc={rc}")
    res = out.reshape(psi.shape[0], -1, 4, 3, 2)[:, site_begin:site_end].copy()
    return res[0] if squeeze else res


def hop_parity(psi, U, dims, parity, sign=-1):
    """Red/black hopping block: on the sites of `parity`,
    out = -1/2 sum_mu [(1+sign g_mu) U psi(x+mu) + (1-sign g_mu) U^dag psi(x-mu)] read from the
    opposite parity; 0 on the other sites.  Full-lattice canonical arrays; extents must be even."""
    psi, U, recon, squeeze, d = _check(psi, U, dims)
    out = np.empty_like(psi)
    cd = (ctypes.c_int * 4)(*d)
    rc = _load().wdo_hop_parity(_dptr(out), _dptr(psi), _dptr(U), cd, psi.shape[0], recon, int(sign), int(parity))
    if rc != 0:
        raise RuntimeError(f"wdo_hop_parity failed rc={rc}")
    return out[0] if squeeze else out


def schur(psi, U, dims, mass, parity, sign=-1):
    """Even-odd preconditioned operator on `parity`: (4+m) psi_p - H_pq H_qp psi_p / (4+m); 0 elsewhere."""
    psi, U, recon, squeeze, d = _check(psi, U, dims)
    out = np.empty_like(psi)
    cd = (ctypes.c_int * 4)(*d)
    rc = _load().wdo_schur(_dptr(out), _dptr(psi), _dptr(U), cd, float(mass), psi.shape[0], recon, int(sign),
                           int(parity))
    if rc != 0:
        raise RuntimeError(f"wdo_schur failed rc={rc}")
    return out[0] if squeeze else out
