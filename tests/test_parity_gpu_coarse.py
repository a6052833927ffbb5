"""-m gpu parity tests of the explicit coarse operator (wd_build_coarse, wd_apply_coarse) against
oracle/wd_coarsen.py:coarse_stencil / coarse_apply_stencil (pinned C7-C9), through the C ABI.  SURVEY.md 8(f) row f3;
PAPER.md:82-88, 116, 149.

Both sides get the same basis W (the GPU's own block-orthonormalised vectors, read back) and the same links.
Tolerances (relative L2 over all nine matrices / over the coarse vector): every stencil entry is a sum of <= 256 x 6
products formed in the working precision (6-term dots) and accumulated in fp64, so the north-star bounds 1e-13 / 2e-6
apply to the build; the apply is a sum of 9 n <= 360 products: same bounds."""
import numpy as np
import pytest

from paper_0912_2186_b200 import binding, fields
from oracle import wd_coarsen as wc
from gpu_util import GpuOp, np_dtype, rel_l2
from test_parity_gpu_transfer import Xfer, rv, to_c

pytestmark = pytest.mark.gpu
TOL = {64: 1e-13, 32: 2e-6}


def gpu_stencil(dims, precision, recon, nv, mass, seed, links="haar"):
    """(S_gpu [B.., 9, n, n] complex, W complex as the GPU holds it, U as rounded, handles)"""
    import torch
    cfg = fields.Config("coarse", dims, precision, links, recon, mass, nv, seed)
    U, psis = fields.make_fields(cfg)
    x = Xfer(dims, precision)
    basis = x.native(psis, nv)
    binding.wd_block_orthonormalise(x.lat, basis, nv, precision)
    Wc = to_c(x.canonical(basis, nv))
    op = GpuOp(U, dims, precision, recon)
    ns = binding.wd_coarse_stencil_reals(x.lat, nv)
    n = 2 * nv
    nb = fields.volume(dims) // 256
    assert ns == nb * 9 * n * n * 2
    S = torch.full((ns,), float("nan"), dtype=x.tdt, device="cuda")
    scratch = torch.empty_like(S)
    binding.wd_build_coarse(op.op.gauge, S, scratch, basis, mass, dims, nv, precision)
    torch.cuda.synchronize()
    # device layout [block][k][column][row][re, im] -> [Bt, Bz, By, Bx, 9, row, column]
    Sg = to_c(S.cpu().numpy().astype(np.float64).reshape(dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 9, n, n, 2))
    Sg = np.swapaxes(Sg, -1, -2)
    return Sg, S, Wc, U, x, op


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 4, 8, 4), (4, 4, 4, 4), (16, 8, 4, 8)])
@pytest.mark.parametrize("precision,recon", [(64, 18), (32, 18), (32, 12), (64, 12)])
@pytest.mark.parametrize("nv", [4, 20])
def test_build_and_apply_match_the_oracle(oracle, dims, precision, recon, nv):
    import torch
    mass = -0.3
    Sg, S_dev, Wc, U, x, op = gpu_stencil(dims, precision, recon, nv, mass, 501)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    if recon == 12:   # the oracle of the stencil takes 18-real links: rebuild row 2 the way P9 pins it
        Uc = to_c(Uo)
        row2 = np.conj(np.cross(Uc[..., 0, :], Uc[..., 1, :]))
        Uc = np.concatenate([Uc, row2[..., None, :]], axis=-2)
        Uo = np.stack([Uc.real, Uc.imag], axis=-1)
    S_want = wc.coarse_stencil(Wc, Uo, dims, mass)
    assert rel_l2(rv(Sg), rv(S_want)) <= TOL[precision]
    for k in range(9):   # every matrix separately too (the diagonal block dominates the norm)
        assert rel_l2(rv(Sg[..., k, :, :]), rv(S_want[..., k, :, :])) <= 5 * TOL[precision], k
    # apply: 1 and 5 right-hand sides against the oracle's apply of the GPU's own stencil (rounded once)
    rng = np.random.default_rng(503)
    shape = (5, dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 2, nv)
    c = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    c_dev = torch.from_numpy(np.ascontiguousarray(np.stack([c.real, c.imag], axis=-1)).astype(np_dtype(precision))).cuda()
    cq = to_c(c_dev.cpu().numpy().astype(np.float64))
    for nrhs in (1, 5):
        out = torch.full_like(c_dev[:nrhs], float("nan")).contiguous()
        binding.wd_apply_coarse(x.lat, out, c_dev[:nrhs].contiguous(), S_dev, nv, nrhs, precision)
        torch.cuda.synchronize()
        got = to_c(out.cpu().numpy().astype(np.float64))
        for r in range(nrhs):
            want = wc.coarse_apply_stencil(Sg, cq[r])
            assert rel_l2(rv(got[r]), rv(want)) <= TOL[precision], (nrhs, r)
    op.close()
    x.close()


def test_coarse_apply_equals_the_galerkin_composition_on_the_gpu(oracle):
    """Dhat c from the stencil = P^dagger D P c with every factor on the GPU (wd_prolong -> wd_apply -> wd_restrict)."""
    import torch
    dims, nv, precision, mass = (8, 8, 4, 8), 6, 64, -0.3
    Sg, S_dev, Wc, U, x, op = gpu_stencil(dims, precision, 18, nv, mass, 505, links="smooth")
    basis = x.native(np.stack([Wc.real, Wc.imag], axis=-1), nv)
    rng = np.random.default_rng(507)
    shape = (dims[3] // 4, dims[2] // 4, dims[1] // 4, dims[0] // 4, 2, nv, 2)
    c_dev = torch.from_numpy(rng.standard_normal(shape)).cuda()
    fine = torch.empty(op.op.native_numel(1), dtype=torch.float64, device="cuda")
    dfine = torch.empty_like(fine)
    comp = torch.empty_like(c_dev)
    binding.wd_prolong(x.lat, fine, basis, c_dev, nv, precision)
    op.op.apply(dfine, fine, mass, 1)
    binding.wd_restrict(x.lat, comp, basis, dfine, nv, precision)
    out = torch.empty_like(c_dev)
    binding.wd_apply_coarse(x.lat, out, c_dev, S_dev, nv, 1, precision)
    torch.cuda.synchronize()
    assert rel_l2(out.cpu().numpy(), comp.cpu().numpy()) <= 1e-12
    op.close()
    x.close()


def test_coarse_entry_points_validate_their_arguments():
    import torch
    lat = binding.wd_create_lattice((6, 4, 4, 4))
    assert binding.wd_coarse_stencil_reals(lat, 4) == -1
    binding.wd_destroy(lat)
    lat = binding.wd_create_lattice((4, 4, 4, 4))
    buf = torch.zeros(64, device="cuda")
    with pytest.raises(binding.WdError) as e:
        binding.wd_apply_coarse(lat, buf, buf, buf, 2, 1, 32)
    assert e.value.code == -6
    binding.wd_destroy(lat)
