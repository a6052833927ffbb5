"""-m gpu parity tests of the red/black (even-odd) blocks (wd_apply_hop, wd_apply_schur) against the oracle
(oracle.hop_parity / oracle.schur, pinned in tests/test_oracle_pins_evenodd.py), through the C ABI.
SURVEY.md 8(f) row f1.  Same tolerances as the full operator."""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from gpu_util import TOL, GpuOp, np_dtype, rel_l2

pytestmark = pytest.mark.gpu

SHAPES = [(4, 4, 4, 4), (2, 2, 2, 2), (8, 4, 6, 2), (16, 8, 8, 6), (32, 4, 4, 8), (6, 10, 4, 8), (24, 12, 4, 2), (2, 4, 2, 16)]


def parity_mask(dims):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return ((x + y + z + t) % 2)[None, ..., None, None, None]


def run_eo(op, psi, mass, parity, what):
    """psi canonical full-lattice [nrhs,...]; returns the canonical full-lattice result (zeros where nothing is written)."""
    import torch
    nrhs = psi.shape[0]
    w = op.op
    canon = torch.from_numpy(np.ascontiguousarray(psi)).cuda()
    n = w.half_numel(nrhs)
    a = torch.full((n,), float("nan"), dtype=canon.dtype, device="cuda")
    b = torch.full((n,), float("nan"), dtype=canon.dtype, device="cuda")
    out = torch.zeros_like(canon)
    if what == "hop":     # out_p = H_pq in_q
        w.pack_parity(a, canon, nrhs, 1 - parity)
        w.apply_hop(b, a, parity, nrhs)
    else:                 # out_p = Mhat in_p
        tmp = torch.full((n,), float("nan"), dtype=canon.dtype, device="cuda")
        w.pack_parity(a, canon, nrhs, parity)
        w.apply_schur(b, a, tmp, mass, parity, nrhs)
    w.unpack_parity(out, b, nrhs, parity)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("precision,recon", [(64, 18), (32, 18), (32, 12), (64, 12)])
def test_hop_and_schur_match_the_oracle(oracle, dims, precision, recon):
    cfg = fields.Config("eo", dims, precision, "haar", recon, -0.31, 3, 61)
    U, psi = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    p64 = psi.astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    try:
        for parity in (0, 1):
            got = run_eo(op, psi, cfg.mass, parity, "hop")
            want = oracle.hop_parity(p64, Uo, dims, parity)
            assert np.all(got[np.broadcast_to(parity_mask(dims) != parity, got.shape)] == 0)
            for r in range(3):
                assert rel_l2(got[r], want[r]) <= TOL[precision], (dims, parity, "hop")
            got = run_eo(op, psi, cfg.mass, parity, "schur")
            want = oracle.schur(p64, Uo, dims, cfg.mass, parity)
            for r in range(3):
                assert rel_l2(got[r], want[r]) <= TOL[precision], (dims, parity, "schur")
    finally:
        op.close()


def test_hop_blocks_rebuild_the_full_operator(oracle):
    """D psi = (4+m) psi + H_eo psi_o + H_oe psi_e with every piece from the CUDA path (16^3 x 32, config 1)."""
    cfg = fields.CONFIGS["c1_16x32_fp32"]
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    full = op.apply(psi, cfg.mass)
    rebuilt = (4.0 + cfg.mass) * psi.astype(np.float64)
    for parity in (0, 1):
        rebuilt += run_eo(op, psi, cfg.mass, parity, "hop")
    op.close()
    assert rel_l2(rebuilt, full) <= 1e-6


def test_full_size_schur_32x64(oracle):
    cfg = fields.CONFIGS["c3_32x64_fp32"]
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    got = run_eo(op, psi, cfg.mass, 0, "schur")
    op.close()
    want = oracle.schur(psi.astype(np.float64), U.astype(np.float64), cfg.dims, cfg.mass, 0)
    assert rel_l2(got[0], want[0]) <= TOL[32]


def test_odd_extents_and_bad_parity_are_refused():
    import torch
    from paper_0912_2186_b200 import binding
    cfg = fields.Config("odd", (4, 3, 4, 4), 32, "haar", 18, 0.1, 1, 3)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    assert op.op.half_numel(1) == 0
    a = torch.zeros(4 * 3 * 4 * 4 * 24, device="cuda")
    b = torch.zeros_like(a)
    with pytest.raises(binding.WdError) as e:
        op.op.apply_hop(b, a, 0, 1)
    assert e.value.code == -2
    op.close()
    cfg = fields.Config("even", (4, 4, 4, 4), 32, "haar", 18, 0.1, 1, 3)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    a = torch.zeros(op.op.half_numel(1), device="cuda")
    b = torch.zeros_like(a)
    for fn, code in ((lambda: op.op.apply_hop(b, a, 2, 1), -7), (lambda: op.op.apply_hop(a, a, 0, 1), -6),
                     (lambda: op.op.apply_schur(b, a, a, 0.1, 0, 1), -6), (lambda: op.op.apply_schur(b, a, None, 0.1, 0, 1), -1)):
        with pytest.raises(binding.WdError) as e:
            fn()
        assert e.value.code == code
    op.close()
