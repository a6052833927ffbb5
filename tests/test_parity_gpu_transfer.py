"""-m gpu parity tests of the multigrid transfer operators (wd_block_orthonormalise, wd_restrict, wd_prolong) against
oracle/wd_coarsen.py (pinned in tests/test_oracle_pins_coarsen.py), through the C ABI.  SURVEY.md 8(f) row f3.

Tolerances: restrict / prolong are sums of <= 1536 / N_v products: north-star bounds 1e-13 / 2e-6 (relative L2).
Gram-Schmidt amplifies rounding by the conditioning of the block vectors; for the random Gaussian vectors used here
(condition number of a 1536 x N_v Gaussian block ~ 1.2) 1e-12 / 2e-5 on the basis -- derived, written here."""
import numpy as np
import pytest

from paper_0912_2186_b200 import binding, fields
from oracle import wd_coarsen as wc
from gpu_util import np_dtype, rel_l2

pytestmark = pytest.mark.gpu
TOL_BASIS = {64: 1e-12, 32: 2e-5}
TOL_XFER = {64: 1e-13, 32: 2e-6}


def to_c(r):
    return r[..., 0].astype(np.float64) + 1j * r[..., 1].astype(np.float64)


def rv(c):
    """complex array -> contiguous float64 view (re, im interleaved) for rel_l2."""
    return np.ascontiguousarray(c).view(np.float64)


class Xfer:
    def __init__(self, dims, precision):
        import torch
        self.torch, self.dims, self.precision = torch, dims, precision
        self.lat = binding.wd_create_lattice(dims)
        self.tdt = torch.float32 if precision == 32 else torch.float64

    def native(self, canon_np, nrhs):
        t = self.torch
        canon = t.from_numpy(np.ascontiguousarray(canon_np)).cuda()
        n = binding.wd_spinor_bytes(self.lat, nrhs, self.precision) // (self.precision // 8)
        nat = t.full((n,), float("nan"), dtype=self.tdt, device="cuda")
        binding.wd_pack_spinor(self.lat, nat, canon, nrhs, self.precision)
        return nat

    def canonical(self, nat, nrhs):
        t = self.torch
        V = fields.volume(self.dims)
        out = t.empty((nrhs,) + (self.dims[3], self.dims[2], self.dims[1], self.dims[0], 4, 3, 2), dtype=self.tdt, device="cuda")
        binding.wd_unpack_spinor(self.lat, out, nat, nrhs, self.precision)
        t.cuda.synchronize()
        return out.cpu().numpy()

    def close(self):
        binding.wd_destroy(self.lat)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 4, 8), (16, 8, 4, 4), (32, 8, 8, 4)])
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("nv", [1, 4, 20])
def test_transfer_operators_match_the_oracle(dims, precision, nv):
    import torch
    psis = fields.gaussian_spinor(dims, 401, nv, precision)           # [nv, sites.., 4, 3, 2] in working precision
    phi = fields.gaussian_spinor(dims, 403, 1, precision)
    x = Xfer(dims, precision)
    basis = x.native(psis, nv)
    binding.wd_block_orthonormalise(x.lat, basis, nv, precision)
    W = x.canonical(basis, nv)
    W_want = wc.block_orthonormalise(to_c(psis), dims)
    for a in range(nv):
        assert rel_l2(rv(to_c(W[a])), rv(W_want[a])) <= TOL_BASIS[precision], a
    # restrict / prolong with the GPU's own basis (so that only the transfer arithmetic is compared)
    Wc = to_c(W)
    ncr = binding.wd_coarse_reals(x.lat, nv)
    assert ncr == fields.volume(dims) // 256 * 2 * nv * 2
    coarse = torch.full((ncr,), float("nan"), dtype=x.tdt, device="cuda")
    phin = x.native(phi, 1)
    binding.wd_restrict(x.lat, coarse, basis, phin, nv, precision)
    torch.cuda.synchronize()
    c = coarse.cpu().numpy().astype(np.float64).reshape(dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 2, nv, 2)
    c_want = wc.restrict(Wc, to_c(phi[0]), dims)
    assert rel_l2(rv(to_c(c)), rv(c_want)) <= TOL_XFER[precision] * 10   # relative to |c| << |phi|
    out = torch.full_like(phin, float("nan"))
    binding.wd_prolong(x.lat, out, basis, coarse, nv, precision)
    back = x.canonical(out, 1)[0]
    back_want = wc.prolong(Wc, to_c(c), dims)
    assert rel_l2(rv(to_c(back)), rv(back_want)) <= TOL_XFER[precision]
    # P^dagger P = 1 on the device: restrict(prolong(c)) = c
    coarse2 = torch.full_like(coarse, float("nan"))
    binding.wd_restrict(x.lat, coarse2, basis, out, nv, precision)
    torch.cuda.synchronize()
    assert rel_l2(coarse2.cpu().numpy(), coarse.cpu().numpy()) <= TOL_BASIS[precision] * 10
    x.close()


def test_transfer_rejects_bad_extents():
    lat = binding.wd_create_lattice((6, 4, 4, 4))
    assert binding.wd_coarse_reals(lat, 4) == -1
    import torch
    buf = torch.zeros(6 * 4 * 4 * 4 * 24 * 4, device="cuda")
    with pytest.raises(binding.WdError) as e:
        binding.wd_block_orthonormalise(lat, buf, 4, 32)
    assert e.value.code == -2
    binding.wd_destroy(lat)


@pytest.mark.parametrize("precision,tol", [(64, 1e-12), (32, 5e-6)])
def test_galerkin_coarse_operator_by_composition(oracle, precision, tol):
    """Dhat c = P^dagger D P c with every factor on the GPU (wd_prolong -> wd_apply -> wd_restrict)
    against oracle/wd_coarsen.py:coarse_apply with the same basis."""
    import torch
    from gpu_util import GpuOp
    dims, nv = (8, 8, 4, 8), 6
    cfg = fields.Config("gal", dims, precision, "smooth", 18, -0.3, nv, 405)
    U, psis = fields.make_fields(cfg)
    x = Xfer(dims, precision)
    basis = x.native(psis, nv)
    binding.wd_block_orthonormalise(x.lat, basis, nv, precision)
    Wc = to_c(x.canonical(basis, nv))
    rng = np.random.default_rng(407)
    shape = (dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 2, nv)
    c = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    c_dev = torch.from_numpy(np.ascontiguousarray(np.stack([c.real, c.imag], axis=-1)).astype(np_dtype(precision))).cuda()
    op = GpuOp(U, dims, precision, 18)
    n1 = op.op.native_numel(1)
    fine = torch.full((n1,), float("nan"), dtype=x.tdt, device="cuda")
    dfine = torch.full_like(fine, float("nan"))
    out = torch.full_like(c_dev, float("nan"))
    binding.wd_prolong(x.lat, fine, basis, c_dev, nv, precision)
    op.op.apply(dfine, fine, cfg.mass, 1)
    binding.wd_restrict(x.lat, out, basis, dfine, nv, precision)
    torch.cuda.synchronize()
    got = to_c(out.cpu().numpy().astype(np.float64))
    cq = to_c(c_dev.cpu().numpy().astype(np.float64))       # the coarse vector as rounded to the working precision
    want = wc.coarse_apply(Wc, cq, U.astype(np.float64), dims, cfg.mass)
    op.close()
    x.close()
    assert rel_l2(rv(got), rv(want)) <= tol
