"""-m gpu parity tests of the bulk-copy member of the staged kernel (csrc/wd_dslash_stage_bulk.cu; Lx = 32, tile 32 x 2 x 2:
every staged piece is one cp.async.bulk per warp instead of 16-byte cp.async per thread).  Selected with the tuning variable
stage_bulk (WD_STAGE_BULK, read at wd_load_gauge); every case goes through the C ABI against the oracle, element by element.
Tolerances: BASELINE.json:north_star (1e-13 fp64, 2e-6 fp32); 8-real links: reading R8 of DESIGN.md (1e-5 / 1e-10)."""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from oracle import wd_storage as ws
from gpu_util import TOL, GpuOp, rel_l2

pytestmark = pytest.mark.gpu
STAGE = 3
TOL8 = {32: 1e-5, 64: 1e-10}


def oracle_links(U, recon, precision):
    if recon == 8:
        return ws.links_from_8(U, precision)
    return (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)


def run(oracle, cfg, dagger=False):
    import torch
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, cfg.precision, cfg.recon, STAGE)
    try:
        if dagger:
            w = op.op
            canon = torch.from_numpy(psi).cuda()
            a = torch.full((w.native_numel(cfg.nrhs),), float("nan"), dtype=canon.dtype, device="cuda")
            b = torch.full_like(a, float("nan"))
            out = torch.full_like(canon, float("nan"))
            w.pack(a, canon, cfg.nrhs)
            w.apply_dagger(b, a, cfg.mass, cfg.nrhs)
            w.unpack(out, b, cfg.nrhs)
            torch.cuda.synchronize()
            got = out.cpu().numpy()
        else:
            got = op.apply(psi, cfg.mass)
    finally:
        op.close()
    assert np.isfinite(got).all()
    Uo = oracle_links(U, cfg.recon, cfg.precision)
    bound = TOL8[cfg.precision] if cfg.recon == 8 else TOL[cfg.precision]
    for r in range(cfg.nrhs):
        want = oracle.apply(psi[r].astype(np.float64), Uo, cfg.dims, cfg.mass, sign=+1 if dagger else -1)
        assert rel_l2(got[r], want) <= bound, (cfg.dims, cfg.precision, cfg.recon, r)


@pytest.mark.parametrize("dims", [(32, 4, 4, 4), (32, 8, 8, 3), (32, 2, 2, 2), (32, 6, 10, 4), (32, 4, 2, 1), (32, 2, 4, 7)])
@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (32, 8), (64, 18), (64, 12), (64, 8)])
def test_bulk_shapes(oracle, monkeypatch, dims, precision, recon):
    monkeypatch.setenv("WD_STAGE_BULK", "1")
    run(oracle, fields.Config("bulk", dims, precision, "haar", recon, -0.3, 1, 91))


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("tc", ["1", "2", "5", "100"])
@pytest.mark.parametrize("patch", ["0", "2"])
def test_bulk_chunks_and_multi_rhs_block_orders(oracle, monkeypatch, precision, tc, patch):
    """Marches of 1 .. Lt slices; several right-hand sides through this member (fp64, or fp32 with the multi-RHS kernels off)
    in both block orders."""
    monkeypatch.setenv("WD_STAGE_BULK", "1")
    monkeypatch.setenv("WD_STAGE_NO_MRHS", "1")
    monkeypatch.setenv("WD_TILE_TC", tc)
    monkeypatch.setenv("WD_MRHS_PATCH", patch)
    run(oracle, fields.Config("bulkc", (32, 4, 8, 5), precision, "smooth", 18, -0.42, 3, 93))


@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (64, 18), (32, 8)])
def test_bulk_dagger(oracle, monkeypatch, precision, recon):
    monkeypatch.setenv("WD_STAGE_BULK", "1")
    run(oracle, fields.Config("bulkd", (32, 4, 4, 6), precision, "haar", recon, -0.2, 1, 95), dagger=True)


@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (64, 18)])
def test_bulk_temporal_gauge(oracle, monkeypatch, precision, recon):
    """Unit t-links are neither copied nor multiplied: the z,t piece of the link record shrinks to the z vectors."""
    monkeypatch.setenv("WD_STAGE_BULK", "1")
    dims = (32, 4, 4, 5)
    cfg = fields.Config("bulktg", dims, precision, "haar", recon, -0.3, 1, 97)
    U, psi = fields.make_fields(cfg)
    Ug, _ = fields.temporal_gauge(U, precision)
    Uo = (Ug if recon == 18 else np.ascontiguousarray(Ug[..., :2, :, :])).astype(np.float64)
    op = GpuOp(Ug, dims, precision, recon, STAGE)
    op.op.set_temporal_gauge(True)
    got = op.apply(psi, cfg.mass)
    op.close()
    assert rel_l2(got[0], oracle.apply(psi[0].astype(np.float64), Uo, dims, cfg.mass)) <= TOL[precision]


@pytest.mark.parametrize("name", ["c3_32x64_fp32", "c3_32x64_fp64"])
def test_bulk_config3_full_size(oracle, monkeypatch, name):
    """BASELINE.json:configs[3] in the launch configuration bench.py times."""
    monkeypatch.setenv("WD_STAGE_BULK", "1")
    run(oracle, fields.CONFIGS[name])


def test_bulk_is_bit_identical_to_the_per_thread_member(monkeypatch):
    """Same arithmetic in the same order: the two members of the staged kernel agree bit for bit, repeatedly."""
    import torch
    cfg = fields.Config("bulkdet", (32, 8, 8, 16), 32, "smooth", 18, -0.42, 1, 99)
    U, psi = fields.make_fields(cfg)
    monkeypatch.setenv("WD_STAGE_BULK", "0")
    op = GpuOp(U, cfg.dims, 32, 18, STAGE)
    ref = op.apply(psi, cfg.mass, return_native=True).clone()
    op.close()
    monkeypatch.setenv("WD_STAGE_BULK", "1")
    op = GpuOp(U, cfg.dims, 32, 18, STAGE)
    for _ in range(10):
        b = op.apply(psi, cfg.mass, return_native=True)
        assert torch.equal(ref, b)
    op.close()
