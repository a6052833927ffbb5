"""-m gpu: temporal gauge (wd_set_temporal_gauge; Table 2 "GF").  The operator is
unchanged -- the oracle applies eq. (2.2) to the gauge-fixed links like to any others -- so parity is the ordinary
element-wise comparison; what is new is that the staged kernel skips the unit links."""
import numpy as np
import pytest

from paper_0912_2186_b200 import binding, fields
from gpu_util import TOL, GpuOp, rel_l2

pytestmark = pytest.mark.gpu
KERNELS = {"auto": 0, "site": 1, "stage": 3}


def test_generator_fixes_the_gauge_and_keeps_the_operator(oracle):
    """CPU part: U_t = 1 below the last slice, and D(U^g)(g psi) = g D(U) psi through the oracle."""
    cfg = fields.Config("tg", (4, 4, 4, 6), 64, "haar", 18, -0.2, 1, 5)
    U, psi = fields.make_fields(cfg)
    Ug, g = fields.temporal_gauge(U)
    assert np.all(Ug[3, :-1, ..., 0] == np.eye(3)) and np.all(Ug[3, :-1, ..., 1] == 0)
    pc = psi[0][..., 0] + 1j * psi[0][..., 1]
    gp = np.einsum("...ab,...sb->...sa", g, pc)
    lhs = oracle.apply(np.ascontiguousarray(np.stack([gp.real, gp.imag], -1)), Ug, cfg.dims, cfg.mass)
    rhs = oracle.apply(psi[0], U, cfg.dims, cfg.mass)
    grhs = np.einsum("...ab,...sb->...sa", g, rhs[..., 0] + 1j * rhs[..., 1])
    assert np.max(np.abs(lhs[..., 0] + 1j * lhs[..., 1] - grhs)) < 1e-13


@pytest.mark.parametrize("dims", [(32, 4, 4, 4), (16, 8, 8, 6), (8, 4, 4, 12), (24, 4, 4, 5), (32, 8, 8, 2), (16, 4, 4, 1)])
@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (64, 18), (64, 12)])
def test_staged_kernel_in_temporal_gauge_matches_the_oracle(oracle, dims, precision, recon):
    cfg = fields.Config("tg", dims, precision, "haar", recon, -0.3, 3, 81)
    U, psi = fields.make_fields(cfg)
    Ug, _ = fields.temporal_gauge(U, precision)
    Uo = (Ug if recon == 18 else np.ascontiguousarray(Ug[..., :2, :, :])).astype(np.float64)
    op = GpuOp(Ug, dims, precision, recon, KERNELS["stage"])
    plain = op.apply(psi, cfg.mass)
    op.op.set_temporal_gauge(True)
    fixed = op.apply(psi, cfg.mass)
    one = op.apply(psi[:1], cfg.mass)       # single-RHS member as well as the multi-RHS path taken for 3 RHS
    op.close()
    for r in range(3):
        want = oracle.apply(psi[r].astype(np.float64), Uo, dims, cfg.mass)
        assert rel_l2(fixed[r], want) <= TOL[precision]
        assert rel_l2(fixed[r], plain[r]) <= TOL[precision]
    assert rel_l2(one[0], oracle.apply(psi[0].astype(np.float64), Uo, dims, cfg.mass)) <= TOL[precision]


@pytest.mark.parametrize("dims", [(8, 4, 4, 6), (16, 8, 2, 2), (4, 4, 4, 4)])
@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (64, 18), (64, 12)])
@pytest.mark.parametrize("parity", [0, 1])
def test_even_odd_blocks_in_temporal_gauge(oracle, dims, precision, recon, parity):
    """The red/black kernel skips the unit t-links too (the paper's Fig. 4 "GF" curves are this kernel):
    M-hat, M-hat^dagger and a CGNR solve with the flag set against the oracle on the same gauge-fixed links, and against
    the same calls with the flag off."""
    import torch
    nrhs = 2
    cfg = fields.Config("tgeo", dims, precision, "haar", recon, 0.25, nrhs, 85)
    U, psi = fields.make_fields(cfg)
    Ug, _ = fields.temporal_gauge(U, precision)
    Uo = (Ug if recon == 18 else np.ascontiguousarray(Ug[..., :2, :, :])).astype(np.float64)
    op = GpuOp(Ug, dims, precision, recon)
    w = op.op
    canon = torch.from_numpy(psi).cuda()
    n = w.half_numel(nrhs)
    hi, tmp = (torch.empty(n, dtype=canon.dtype, device="cuda") for _ in range(2))
    w.pack_parity(hi, canon, nrhs, parity)
    res = {}
    for flag in (False, True):
        w.set_temporal_gauge(flag)
        for name, fn in (("schur", w.apply_schur), ("dagger", w.apply_schur_dagger)):
            ho = torch.empty_like(hi)
            fn(ho, hi, tmp, cfg.mass, parity, nrhs)
            full = torch.zeros_like(canon)
            w.unpack_parity(full, ho, nrhs, parity)
            res[name, flag] = full.cpu().numpy()
    op.close()
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    mine = ((x + y + z + t) % 2 == parity)
    for r in range(nrhs):
        src = np.where(mine[..., None, None, None], psi[r].astype(np.float64), 0.0)
        for name, sign in (("schur", -1), ("dagger", +1)):
            want = oracle.schur(src, Uo, dims, cfg.mass, parity, sign=sign)
            assert rel_l2(res[name, True][r][mine], want[mine]) <= TOL[precision]
            assert rel_l2(res[name, True][r][mine], res[name, False][r][mine]) <= TOL[precision]


def test_full_size_temporal_gauge_32x64(oracle):
    cfg = fields.CONFIGS["c3_32x64_fp32"]
    U, psi = fields.make_fields(cfg)
    Ug, _ = fields.temporal_gauge(U, 32)
    op = GpuOp(Ug, cfg.dims, 32, 18)
    op.op.set_temporal_gauge(True)
    got = op.apply(psi, cfg.mass)
    op.close()
    assert rel_l2(got[0], oracle.apply(psi[0].astype(np.float64), Ug.astype(np.float64), cfg.dims, cfg.mass)) <= TOL[32]


def test_links_not_in_temporal_gauge_are_refused():
    cfg = fields.Config("ntg", (8, 4, 4, 4), 32, "haar", 18, 0.1, 1, 83)
    U, _ = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    with pytest.raises(binding.WdError) as e:
        op.op.set_temporal_gauge(True)
    assert e.value.code == -7
    op.op.set_temporal_gauge(False)   # switching it off is always allowed
    op.close()
