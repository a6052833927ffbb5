"""CPU ORACLE for the storage variants of the fields (Table 2: gauge field
"stored as 12 or 8 ... floats", kernel rows "Half", "SP", "DP").

TEST INFRASTRUCTURE ONLY (same rules as wd_oracle.py): plain numpy, fp64 arithmetic, definitions written out.
The paper names the variants but prints neither parametrisation nor number format (its ref. [8] is not available);
the readings taken are recorded in DESIGN.md section 2 (R8, RH) and restated here.

8 reals per link (reading R8).  For a link with rows a, b, c (c = conj(a x b)):
    stored   r = (Re a2, Im a2, Re a3, Im a3, Re b1, Im b1, arg(a1)/pi, arg(c1)/pi)      (phases in units of pi, in [-1, 1])
    rebuild  N = |a2|^2 + |a3|^2;  a1 = sqrt(1 - N) e^{i pi r6};  c1 = sqrt(1 - |a1|^2 - |b1|^2) e^{i pi r7}
             (row 0 and column 0 of a unitary matrix have unit length), and from  <a, b> = 0,  c1 = conj(a2 b3 - a3 b2):
                 conj(a2) b2 + conj(a3) b3 = -conj(a1) b1
                      -a3 b2 +      a2 b3 =  conj(c1)
             solved by Cramer's rule (determinant N);  then c2 = conj(a3 b1 - a1 b3), c3 = conj(a1 b2 - a2 b1).
    The stored numbers are rounded ONCE to the working precision; the oracle rebuilds the link from those rounded
    numbers in fp64.

Half precision (reading RH).  IEEE binary16 storage, fp32 arithmetic:
    links    every stored real (|.| <= 1) rounded to binary16;
    spinors  per site a float32 scale s = max_k |psi_k| over the 24 reals of the site, and the 24 ratios psi_k / s
             (formed in float32, IEEE division) rounded to binary16; a site with s = 0 stores zeros.  value = s * q.
"""
import numpy as np


def compress8(U):
    """U real-pair canonical [..., 3, 3, 2] -> the eight stored reals [..., 8] (fp64, not yet rounded)."""
    U = np.asarray(U, dtype=np.float64)
    a1 = U[..., 0, 0, 0] + 1j * U[..., 0, 0, 1]
    c1 = U[..., 2, 0, 0] + 1j * U[..., 2, 0, 1]
    return np.stack([U[..., 0, 1, 0], U[..., 0, 1, 1], U[..., 0, 2, 0], U[..., 0, 2, 1], U[..., 1, 0, 0], U[..., 1, 0, 1],
                     np.arctan2(a1.imag, a1.real) / np.pi, np.arctan2(c1.imag, c1.real) / np.pi], axis=-1)


def reconstruct8(r):
    """[..., 8] stored reals -> full links, real-pair canonical [..., 3, 3, 2], fp64."""
    r = np.asarray(r, dtype=np.float64)
    a2 = r[..., 0] + 1j * r[..., 1]
    a3 = r[..., 2] + 1j * r[..., 3]
    b1 = r[..., 4] + 1j * r[..., 5]
    N = np.abs(a2) ** 2 + np.abs(a3) ** 2
    a1 = np.sqrt(np.maximum(0.0, 1.0 - N)) * np.exp(1j * np.pi * r[..., 6])
    c1 = np.sqrt(np.maximum(0.0, 1.0 - np.abs(a1) ** 2 - np.abs(b1) ** 2)) * np.exp(1j * np.pi * r[..., 7])
    rhs1 = -np.conj(a1) * b1
    rhs2 = np.conj(c1)
    b2 = (rhs1 * a2 - np.conj(a3) * rhs2) / N          # Cramer, matrix [[conj a2, conj a3], [-a3, a2]]
    b3 = (np.conj(a2) * rhs2 + a3 * rhs1) / N
    c2 = np.conj(a3 * b1 - a1 * b3)
    c3 = np.conj(a1 * b2 - a2 * b1)
    M = np.stack([np.stack([a1, a2, a3], axis=-1), np.stack([b1, b2, b3], axis=-1), np.stack([c1, c2, c3], axis=-1)], axis=-2)
    return np.stack([M.real, M.imag], axis=-1)


def links_from_8(U, precision):
    """What a gauge field loaded with 8 reals per link IS: compress, round once to the working precision, rebuild (fp64)."""
    dt = {16: np.float16, 32: np.float32, 64: np.float64}[int(precision)]
    return reconstruct8(compress8(U).astype(dt).astype(np.float64))


def quantise_half_links(U):
    """Every real of the (18- or 12-real) link array rounded to binary16, returned widened to fp64."""
    return np.asarray(U, dtype=np.float32).astype(np.float16).astype(np.float64)


def quantise_half_spinor(psi):
    """psi [..., 4, 3, 2] (any float type; taken as float32) -> (q binary16 [..., 4, 3, 2], s float32 [...])."""
    p = np.asarray(psi, dtype=np.float32)
    s = np.max(np.abs(p), axis=(-3, -2, -1)).astype(np.float32)
    safe = np.where(s > 0, s, np.float32(1.0)).astype(np.float32)
    q = (p / safe[..., None, None, None]).astype(np.float32).astype(np.float16)
    q = np.where((s > 0)[..., None, None, None], q, np.float16(0))
    return q, s


def dequantise_half_spinor(q, s):
    """value = s * q in fp64."""
    return np.asarray(q, dtype=np.float64) * np.asarray(s, dtype=np.float64)[..., None, None, None]
