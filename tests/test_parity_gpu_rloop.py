"""-m gpu parity tests of the multi-right-hand-side member with the links in registers (csrc/wd_dslash_rloop.cu;
SURVEY.md 8(a) step a'): a thread owns a site and loops over the right-hand sides of its group.
Selected with the tuning variable mrhs_reg (WD_MRHS_REG, read at wd_load_gauge); every case runs through the C ABI against
the oracle, per right-hand side.  Tolerances: BASELINE.json:north_star (2e-6 fp32); 8-real links: reading R8 (1e-5).
"""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from oracle import wd_storage as ws
from gpu_util import TOL, GpuOp, oracle_apply, rel_l2

pytestmark = pytest.mark.gpu
STAGE = 3


def oracle_links(U, recon):
    if recon == 8:
        return ws.links_from_8(U, 32)
    return (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)


def run(oracle, cfg, dagger=False, tol=None):
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, cfg.recon, STAGE)
    try:
        if dagger:
            import torch
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
    Uo = oracle_links(U, cfg.recon)
    bound = tol if tol is not None else (1e-5 if cfg.recon == 8 else TOL[32])
    for r in range(cfg.nrhs):
        want = oracle.apply(psi[r].astype(np.float64), Uo, cfg.dims, cfg.mass, sign=+1 if dagger else -1)
        assert rel_l2(got[r], want) <= bound, (cfg.dims, cfg.recon, r)


SHAPES = [(32, 4, 4, 4), (16, 8, 8, 6), (8, 4, 4, 12), (4, 8, 16, 5), (32, 8, 8, 3), (32, 2, 2, 2), (16, 2, 4, 1), (32, 6, 10, 4)]


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_rloop_shapes(oracle, monkeypatch, dims, recon):
    monkeypatch.setenv("WD_MRHS_REG", "1")
    for nrhs in (2, 5):
        run(oracle, fields.Config("rloop", dims, 32, "haar", recon, -0.3, nrhs, 41))


@pytest.mark.parametrize("nrhs", [2, 3, 7, 12, 20, 24, 29])
@pytest.mark.parametrize("rgrp", [None, "1", "3", "8", "1000"])
def test_rloop_groups_and_partial_groups(oracle, monkeypatch, nrhs, rgrp):
    """Group sizes that do and do not divide nrhs (a partial last group simply loops over fewer right-hand sides)."""
    monkeypatch.setenv("WD_MRHS_REG", "1")
    if rgrp:
        monkeypatch.setenv("WD_MRHS_RGRP", rgrp)
    run(oracle, fields.Config("rloopg", (16, 4, 8, 6), 32, "smooth", 18, -0.42, nrhs, 43))


@pytest.mark.parametrize("shape", ["2,2", "4,2", "2,4", "4,4", "8,2"])
@pytest.mark.parametrize("tc", ["1", "2", "5", "100"])
@pytest.mark.parametrize("patch", ["0", "2"])
def test_rloop_tile_shapes_chunks_and_block_orders(oracle, monkeypatch, shape, tc, patch):
    """Tile extents 2 (folded exchange arrays) and > 2 (interior sites send and receive both ways), marches of 1 .. Lt slices,
    both block orders."""
    monkeypatch.setenv("WD_MRHS_REG", "1")
    monkeypatch.setenv("WD_TILE_SHAPE", shape)
    monkeypatch.setenv("WD_TILE_TC", tc)
    monkeypatch.setenv("WD_MRHS_PATCH", patch)
    Lx = 8 if shape in ("4,4", "8,2") else 16
    run(oracle, fields.Config("rloopt", (Lx, 8, 8, 5), 32, "smooth", 18, -0.42, 3, 47))


@pytest.mark.parametrize("recon", [18, 12, 8])
def test_rloop_dagger(oracle, monkeypatch, recon):
    monkeypatch.setenv("WD_MRHS_REG", "1")
    run(oracle, fields.Config("rloopd", (32, 4, 4, 6), 32, "haar", recon, -0.2, 4, 53), dagger=True)


@pytest.fixture(scope="module")
def config4_reference():
    """configs[4] inputs (seeded, fields.make_fields) packed on the device once for the three full-size tests below, and the
    result of the default multi-RHS member on them (tests/test_parity_gpu.py checks that member against the oracle on all 24
    right-hand sides)."""
    import os
    import torch
    cfg = fields.CONFIGS["c4_32x64_fp32_24rhs"]
    U, psi = fields.make_fields(cfg)
    old = os.environ.get("WD_MRHS_REG")
    os.environ["WD_MRHS_REG"] = "0"
    try:
        op = GpuOp(U, cfg.dims, 32, cfg.recon, STAGE)
    finally:
        if old is None:
            del os.environ["WD_MRHS_REG"]
        else:
            os.environ["WD_MRHS_REG"] = old
    w = op.op
    canon = torch.from_numpy(psi).cuda()
    native_in = torch.full((w.native_numel(cfg.nrhs),), float("nan"), dtype=canon.dtype, device="cuda")
    ref = torch.full_like(native_in, float("nan"))
    w.pack(native_in, canon, cfg.nrhs)
    w.apply(ref, native_in, cfg.mass, cfg.nrhs)
    torch.cuda.synchronize()
    del canon
    op.close()
    yield cfg, U, psi, native_in, ref
    del native_in, ref
    torch.cuda.empty_cache()


def full_size_config4(oracle, monkeypatch, reg, reference):
    """BASELINE.json:configs[4] (32^3 x 64, 24 right-hand sides) in the launch configuration bench.py times: all 24 right-hand
    sides against the default multi-RHS member (compared on the device, in the native layout), and right-hand sides 0, 5, 11,
    12, 23 (first / last of a group for every group size in use) element by element against the oracle."""
    import torch
    cfg, U, psi, native_in, ref = reference
    monkeypatch.setenv("WD_MRHS_REG", reg)
    op = GpuOp(U, cfg.dims, 32, cfg.recon, STAGE)
    w = op.op
    got = torch.full_like(native_in, float("nan"))
    w.apply(got, native_in, cfg.mass, cfg.nrhs)
    n1 = w.native_numel(1)
    for r in range(cfg.nrhs):
        g, f = got[r * n1:(r + 1) * n1].double(), ref[r * n1:(r + 1) * n1].double()
        live = torch.isfinite(f)                       # pad sites of the native layout are never written
        assert bool(torch.isfinite(g[live]).all())
        assert float(torch.linalg.vector_norm(g[live] - f[live]) / torch.linalg.vector_norm(f[live])) <= TOL[32], r
    Lx, Ly, Lz, Lt = cfg.dims
    canon = torch.full((cfg.nrhs, Lt, Lz, Ly, Lx, 4, 3, 2), float("nan"), dtype=got.dtype, device="cuda")
    w.unpack(canon, got, cfg.nrhs)
    torch.cuda.synchronize()
    op.close()
    U64 = U.astype(np.float64)
    for r in (0, 5, 11, 12, 23):
        assert rel_l2(canon[r].cpu().numpy(), oracle.apply(psi[r].astype(np.float64), U64, cfg.dims, cfg.mass)) <= TOL[32], r


def test_rloop_config4_full_size(oracle, monkeypatch, config4_reference):
    full_size_config4(oracle, monkeypatch, "1", config4_reference)


def test_rloop_nv20_on_the_paper_volume_shape(oracle, monkeypatch):
    """N_v = 20 test vectors: two groups of 10."""
    monkeypatch.setenv("WD_MRHS_REG", "1")
    run(oracle, fields.Config("rloop20", (16, 16, 16, 16), 32, "smooth", 18, -0.42, 20, 59))


def test_rloop_deterministic(monkeypatch):
    import torch
    monkeypatch.setenv("WD_MRHS_REG", "1")
    cfg = fields.Config("rloopdet", (32, 8, 8, 8), 32, "smooth", 18, -0.42, 6, 61)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18, STAGE)
    a = op.apply(psi, cfg.mass, return_native=True).clone()
    for _ in range(10):
        b = op.apply(psi, cfg.mass, return_native=True)
    assert torch.equal(a, b)
    op.close()


# ---------------------------------------------------------------- the ring member (Lx = 32: warp-private cp.async.bulk row slots)
# reg = "2": in-tile backward products formed at the source site; "3": uniform roles (every thread holds the links below it)
@pytest.mark.parametrize("dims", [(32, 4, 4, 4), (32, 8, 8, 3), (32, 2, 2, 2), (32, 6, 10, 4), (32, 4, 2, 1)])
@pytest.mark.parametrize("recon", [18, 12, 8])
@pytest.mark.parametrize("reg", ["2", "3"])
def test_ring_shapes(oracle, monkeypatch, dims, recon, reg):
    monkeypatch.setenv("WD_MRHS_REG", reg)
    for nrhs in (2, 7):
        run(oracle, fields.Config("ring", dims, 32, "haar", recon, -0.3, nrhs, 67))


@pytest.mark.parametrize("rgrp", [None, "1", "3", "5", "1000"])
@pytest.mark.parametrize("tc", ["1", "2", "5", "100"])
@pytest.mark.parametrize("patch", ["0", "2"])
@pytest.mark.parametrize("reg", ["2", "3"])
def test_ring_groups_chunks_and_block_orders(oracle, monkeypatch, rgrp, tc, patch, reg):
    monkeypatch.setenv("WD_MRHS_REG", reg)
    monkeypatch.setenv("WD_TILE_TC", tc)
    monkeypatch.setenv("WD_MRHS_PATCH", patch)
    if rgrp:
        monkeypatch.setenv("WD_MRHS_RGRP", rgrp)
    run(oracle, fields.Config("ringg", (32, 4, 8, 5), 32, "smooth", 18, -0.42, 11, 71))


@pytest.mark.parametrize("recon", [18, 12, 8])
@pytest.mark.parametrize("reg", ["2", "3"])
def test_ring_dagger(oracle, monkeypatch, recon, reg):
    monkeypatch.setenv("WD_MRHS_REG", reg)
    run(oracle, fields.Config("ringd", (32, 4, 4, 6), 32, "haar", recon, -0.2, 4, 73), dagger=True)


@pytest.mark.parametrize("reg", ["2", "3"])
def test_ring_config4_full_size(oracle, monkeypatch, config4_reference, reg):
    full_size_config4(oracle, monkeypatch, reg, config4_reference)


@pytest.mark.parametrize("reg", ["2", "3"])
def test_ring_deterministic(monkeypatch, reg):
    import torch
    monkeypatch.setenv("WD_MRHS_REG", reg)
    cfg = fields.Config("ringdet", (32, 8, 8, 8), 32, "smooth", 18, -0.42, 6, 79)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18, STAGE)
    a = op.apply(psi, cfg.mass, return_native=True).clone()
    for _ in range(10):
        b = op.apply(psi, cfg.mass, return_native=True)
    assert torch.equal(a, b)
    op.close()
