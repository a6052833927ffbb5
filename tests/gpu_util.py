"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI on numpy inputs and
compare with the oracle.  torch is used only to hold device memory."""
import numpy as np

TOL = {64: 1e-13, 32: 2e-6}  # BASELINE.json:north_star: relative L2 error bounds


def rel_l2(a, b):
    """||a-b||_2 / ||b||_2 in float64 over the whole field."""
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def np_dtype(precision):
    return np.float32 if int(precision) == 32 else np.float64


class GpuOp:
    """One gauge field on cuda:0 behind the C ABI."""

    def __init__(self, U, dims, precision, recon=18, kernel=0):
        import torch
        from paper_0912_2186_b200 import binding
        self.torch = torch
        self.binding = binding
        self.dims = tuple(dims)
        self.precision = precision
        U = np.ascontiguousarray(U, dtype=np_dtype(precision))
        assert U.shape[-3:] == (3, 3, 2)
        u_dev = torch.from_numpy(U).cuda()
        self.op = binding.WilsonDirac(self.dims, u_dev, precision, recon, kernel=kernel)
        torch.cuda.synchronize()
        del u_dev

    def apply(self, psi, mass, return_native=False):
        """psi: numpy canonical [nrhs, Lt,Lz,Ly,Lx,4,3,2] in working precision -> D psi, same layout."""
        torch = self.torch
        psi = np.ascontiguousarray(psi, dtype=np_dtype(self.precision))
        nrhs = psi.shape[0]
        canon = torch.from_numpy(psi).cuda()
        n = self.op.native_numel(nrhs)  # >= canon.numel(): the native volume is padded to 32-site blocks
        native_in = torch.full((n,), float("nan"), dtype=canon.dtype, device=canon.device)
        native_out = torch.full((n,), float("nan"), dtype=canon.dtype, device=canon.device)
        self.op.pack(native_in, canon, nrhs)
        self.op.apply(native_out, native_in, mass, nrhs)
        if return_native:
            torch.cuda.synchronize()
            return native_out
        canon_out = torch.full_like(canon, float("nan"))
        self.op.unpack(canon_out, native_out, nrhs)
        torch.cuda.synchronize()
        return canon_out.cpu().numpy()

    def close(self):
        self.op.close()


def oracle_apply(oracle, psi, U, dims, mass):
    """Oracle on the same (already rounded) inputs, widened to float64, one RHS at a time."""
    U64 = np.ascontiguousarray(U, dtype=np.float64)
    out = np.empty(psi.shape, dtype=np.float64)
    for r in range(psi.shape[0]):
        out[r] = oracle.apply(np.ascontiguousarray(psi[r], dtype=np.float64), U64, dims, mass)
    return out
