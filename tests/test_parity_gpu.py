"""-m gpu parity tests: the CUDA path, called through the C ABI (libwd.so), against the CPU oracle
on the same seeded inputs, element by element (relative L2 over the whole field, per RHS).

Tolerances (BASELINE.json:north_star): <= 1e-13 in fp64, <= 2e-6 in fp32.  The inputs are rounded
once to the working precision and the oracle consumes those same bits widened to fp64 (S12).
For recon 12 the oracle consumes the same 12 stored reals per link (rows 0,1; S7).
"""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from gpu_util import TOL, GpuOp, np_dtype, oracle_apply, rel_l2

pytestmark = pytest.mark.gpu

KERNELS = {"auto": 0, "site": 1, "stage": 3}


def oracle_links(U, recon):
    return U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])


def check_config(oracle, cfg, kernel="auto", nrhs=None, dims=None):
    U, psi = fields.make_fields(cfg, nrhs=nrhs, dims=dims)
    d = tuple(dims) if dims is not None else cfg.dims
    op = GpuOp(U, d, cfg.precision, cfg.recon, KERNELS[kernel])
    try:
        got = op.apply(psi, cfg.mass)
    finally:
        op.close()
    assert np.isfinite(got).all()
    Uo = oracle_links(U, cfg.recon)
    worst = 0.0
    for r in range(psi.shape[0]):
        want = oracle.apply(psi[r].astype(np.float64), Uo.astype(np.float64), d, cfg.mass)
        worst = max(worst, rel_l2(got[r], want))
    assert worst <= TOL[cfg.precision], (cfg.name, kernel, worst)
    return worst


# ---------------------------------------------------------------- the five BASELINE configs
@pytest.mark.parametrize("name", ["c0_4x4_fp64", "c1_16x32_fp32", "c2_24x64_fp32_r12"])
@pytest.mark.parametrize("kernel", ["auto", "site"])
def test_baseline_configs_small(oracle, name, kernel):
    check_config(oracle, fields.CONFIGS[name], kernel)


@pytest.mark.parametrize("name", ["c3_32x64_fp32", "c3_32x64_fp64"])
def test_baseline_config3_full_size(oracle, name):
    check_config(oracle, fields.CONFIGS[name], "auto")


def test_baseline_config4_24rhs_full_size(oracle):
    check_config(oracle, fields.CONFIGS["c4_32x64_fp32_24rhs"], "auto")


def test_paper_nv20_rhs(oracle):
    """N_v = 20 test vectors on a smaller lattice: nrhs is a runtime value."""
    check_config(oracle, fields.CONFIGS["c4_32x64_fp32_24rhs"], "auto", nrhs=20, dims=(16, 16, 16, 16))


# ---------------------------------------------------------------- shapes, tails, degenerate extents
SHAPES = [(4, 8, 12, 16), (8, 4, 4, 12), (6, 10, 4, 8), (3, 5, 2, 7), (2, 2, 2, 2), (1, 1, 1, 1), (1, 4, 1, 3),
          (5, 1, 2, 9), (32, 4, 4, 4), (16, 8, 8, 6), (24, 12, 4, 5), (12, 12, 12, 12), (32, 8, 8, 3)]


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("precision,recon", [(64, 18), (32, 18), (32, 12), (64, 12)])
def test_shapes(oracle, dims, precision, recon):
    cfg = fields.Config("shape", dims, precision, "haar", recon, -0.3, 1, 11)
    for nrhs in (1, 3):
        check_config(oracle, cfg, "auto", nrhs=nrhs)
    check_config(oracle, cfg, "site", nrhs=2)


@pytest.mark.parametrize("nrhs", [1, 2, 3, 4, 5, 7, 8, 12, 20, 24])
def test_nrhs_sweep(oracle, nrhs):
    cfg = fields.Config("nrhs", (8, 8, 8, 8), 32, "smooth", 18, -0.42, nrhs, 21)
    check_config(oracle, cfg, "auto")


# ---------------------------------------------------------------- the cp.async-staged t-marching kernels (fp32, fp64)
STAGE_SHAPES = [(32, 4, 4, 4), (16, 8, 8, 6), (8, 4, 4, 12), (4, 8, 16, 5), (32, 8, 8, 3), (32, 2, 2, 2), (16, 2, 4, 1),
                (32, 6, 10, 4), (8, 12, 4, 7),
                # Lx not a power of two: x hops through shared memory instead of warp shuffles
                (24, 4, 4, 6), (24, 6, 2, 3), (12, 8, 4, 5), (6, 8, 8, 4), (24, 2, 2, 2)]


@pytest.mark.parametrize("dims", STAGE_SHAPES)
@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (64, 18), (64, 12)])
def test_stage_kernel_shapes(oracle, dims, precision, recon):
    cfg = fields.Config("stage", dims, precision, "haar", recon, -0.3, 1, 15)
    check_config(oracle, cfg, "stage", nrhs=1)
    check_config(oracle, cfg, "stage", nrhs=3)


@pytest.mark.parametrize("shape", ["2,2", "4,2", "2,4", "4,4", "8,1"])
@pytest.mark.parametrize("tc", ["1", "2", "5", "100"])
def test_stage_kernel_forced_tile_shapes_and_chunks(oracle, monkeypatch, shape, tc):
    monkeypatch.setenv("WD_TILE_SHAPE", shape)
    monkeypatch.setenv("WD_TILE_TC", tc)
    cfg = fields.Config("stageshape", (32, 8, 8, 5), 32, "smooth", 18, -0.42, 2, 23)
    check_config(oracle, cfg, "stage")


@pytest.mark.parametrize("name", ["c1_16x32_fp32", "c2_24x64_fp32_r12", "c3_32x64_fp32", "c3_32x64_fp64"])
def test_stage_kernel_baseline_configs(oracle, name):
    check_config(oracle, fields.CONFIGS[name], "stage")


@pytest.mark.parametrize("nrb", ["1", "2", "3"])
@pytest.mark.parametrize("nrhs", [2, 3, 4, 5, 7, 24])
@pytest.mark.parametrize("recon", [18, 12])
def test_stage_kernel_multi_rhs_groups(oracle, monkeypatch, nrb, nrhs, recon):
    """The multi-RHS staged kernel (links shared in smem by WD_TILE_NRB right-hand sides per CTA),
    including partial last groups."""
    monkeypatch.setenv("WD_TILE_NRB", nrb)
    cfg = fields.Config("mrhs", (16, 4, 8, 6), 32, "haar", recon, -0.42, nrhs, 29)
    check_config(oracle, cfg, "stage")


def test_stage_kernel_nv20_and_batched_consistency(oracle):
    """N_v = 20 through the multi-RHS kernel; each RHS equals its single-RHS apply bit for bit
    is not required (S10), 1e-6 is."""
    cfg = fields.Config("nv20", (32, 4, 4, 8), 32, "smooth", 18, -0.42, 20, 33)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18, KERNELS["stage"])
    batched = op.apply(psi, cfg.mass)
    for r in (0, 7, 19):
        single = op.apply(psi[r:r + 1], cfg.mass)
        assert rel_l2(batched[r], single[0]) <= 1e-6
    want = oracle_apply(oracle, psi, U, cfg.dims, cfg.mass)
    for r in range(20):
        assert rel_l2(batched[r], want[r]) <= TOL[32]
    op.close()


def test_stage_kernel_rejects_lattices_it_cannot_tile():
    from paper_0912_2186_b200 import binding
    for dims, precision in (((20, 4, 4, 4), 64), ((36, 4, 4, 4), 32), ((32, 3, 4, 4), 32), ((4, 2, 2, 4), 32)):
        cfg = fields.Config("bad", dims, precision, "haar", 18, 0.1, 1, 3)
        U, _ = fields.make_fields(cfg)
        op = GpuOp(U, cfg.dims, precision, 18)
        with pytest.raises(binding.WdError) as e:
            binding.wd_set_kernel(op.op.gauge, KERNELS["stage"])
        assert e.value.code == -7
        op.close()


def test_stage_kernel_deterministic():
    import torch
    cfg = fields.Config("det", (32, 8, 8, 16), 32, "smooth", 18, -0.42, 1, 19)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18, KERNELS["stage"])
    a = op.apply(psi, cfg.mass, return_native=True).clone()
    for _ in range(20):
        b = op.apply(psi, cfg.mass, return_native=True)
    assert torch.equal(a, b)
    op.close()


# ---------------------------------------------------------------- invariants of the CUDA path itself
def test_deterministic_and_repeatable():
    """No atomics: launch #100 on input A is bit-identical to launch #1 on input A (S9)."""
    import torch
    cfg = fields.CONFIGS["c1_16x32_fp32"]
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, cfg.precision, cfg.recon)
    canon = torch.from_numpy(psi).cuda()
    a = torch.empty_like(canon)
    op.op.pack(a, canon, 1)
    outs = [torch.empty_like(canon) for _ in range(3)]
    op.op.apply(outs[0], a, cfg.mass, 1)
    first = outs[0].clone()
    for i in range(1, 100):
        op.op.apply(outs[i % 3], a, cfg.mass, 1)
    torch.cuda.synchronize()
    assert torch.equal(outs[99 % 3], first)
    op.close()


def test_batched_matches_single(oracle):
    """out[r] of one 6-RHS apply agrees with six single applies (S10) to fp32 rounding."""
    cfg = fields.Config("b", (8, 8, 8, 16), 32, "smooth", 18, -0.42, 6, 31)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    batched = op.apply(psi, cfg.mass)
    for r in range(6):
        single = op.apply(psi[r:r + 1], cfg.mass)
        assert rel_l2(batched[r], single[0]) <= 1e-6
    op.close()


def test_translation_covariance_through_native_layout():
    """P6 on the CUDA path: shifting U and psi by one site in direction mu shifts the output."""
    dims = (8, 4, 12, 6)
    cfg = fields.Config("t", dims, 64, "haar", 18, 0.05, 1, 41)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, dims, 64, 18)
    base = op.apply(psi, cfg.mass)
    op.close()
    for mu in range(4):
        ax = 3 - mu  # site axes are [t, z, y, x]
        Us = np.roll(U, 1, axis=1 + ax)
        ps = np.roll(psi, 1, axis=1 + ax)
        op = GpuOp(Us, dims, 64, 18)
        got = op.apply(ps, cfg.mass)
        op.close()
        assert rel_l2(got, np.roll(base, 1, axis=1 + ax)) <= 1e-14


def test_pack_unpack_roundtrip_and_native_layout():
    """Native layout is [rhs][block of 32 sites][16-byte vector][lane] (include/wd.h), the volume
    padded to a multiple of 32 sites; pure data movement, pad sites untouched."""
    import torch
    from paper_0912_2186_b200 import binding
    for dims in ((6, 4, 2, 5), (3, 5, 2, 7), (8, 4, 4, 4)):
        V = int(np.prod(dims))
        Vp = (V + 31) // 32 * 32
        for precision, cr in ((32, 4), (64, 2)):
            psi = fields.gaussian_spinor(dims, 5, 3, precision)
            lat = binding.wd_create_lattice(dims)
            assert binding.wd_spinor_bytes(lat, 3, precision) == 3 * Vp * 24 * (precision // 8)
            canon = torch.from_numpy(psi).cuda()
            native = torch.full((3 * Vp * 24,), -7.0, dtype=canon.dtype, device="cuda")
            back = torch.empty_like(canon)
            binding.wd_pack_spinor(lat, native, canon, 3, precision)
            binding.wd_unpack_spinor(lat, back, native, 3, precision)
            torch.cuda.synchronize()
            assert torch.equal(back, canon)
            nvec = 24 // cr
            padded = np.full((3, Vp, nvec, cr), -7.0, dtype=psi.dtype)
            padded[:, :V] = psi.reshape(3, V, nvec, cr)
            want = padded.reshape(3, Vp // 32, 32, nvec, cr).transpose(0, 1, 3, 2, 4)
            assert np.array_equal(native.cpu().numpy().reshape(3, Vp // 32, nvec, 32, cr), want)
            binding.wd_destroy(lat)


def test_apply_host_matches_device_path(oracle):
    cfg = fields.Config("h", (8, 8, 4, 6), 32, "haar", 18, -0.4, 2, 51)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    dev = op.apply(psi, cfg.mass)
    out = np.full_like(psi, np.nan)
    op.op.apply_host(out, psi, cfg.mass, 2)
    assert np.array_equal(out, dev)
    want = oracle_apply(oracle, psi, U, cfg.dims, cfg.mass)
    assert rel_l2(out, want) <= TOL[32]
    op.close()


def test_argument_errors_on_device():
    import torch
    from paper_0912_2186_b200 import binding
    cfg = fields.Config("e", (4, 4, 4, 4), 32, "haar", 18, 0.1, 1, 61)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    a = torch.from_numpy(psi).cuda()
    b = torch.empty_like(a)
    c = torch.empty(a.numel() + 64, dtype=a.dtype, device=a.device)
    cases = [
        (lambda: binding.wd_apply(a, a, op.op.gauge, 0.1, cfg.dims, 1, 32), -6),
        (lambda: binding.wd_apply(b, a, op.op.gauge, 0.1, (4, 4, 4, 8), 1, 32), -2),
        (lambda: binding.wd_apply(b, a, op.op.gauge, 0.1, cfg.dims, 1, 64), -3),
        (lambda: binding.wd_apply(b, a, op.op.gauge, 0.1, cfg.dims, 0, 32), -5),
        (lambda: binding.wd_apply(c.data_ptr() + 4, a, op.op.gauge, 0.1, cfg.dims, 1, 32), -7),
        (lambda: binding.wd_set_kernel(op.op.gauge, 99), -7),
    ]
    for fn, code in cases:
        with pytest.raises(binding.WdError) as e:
            fn()
        assert e.value.code == code
    op.close()


@pytest.mark.parametrize("dims,precision,recon,nrhs,nslab", [
    ((16, 16, 16, 16), 32, 18, 2, None), ((32, 16, 16, 5), 64, 12, 2, None), ((32, 8, 16, 3), 32, 18, 8, None),
    ((16, 16, 8, 24), 32, 12, 3, None),
    # Lt >= 4 nslab: thin slabs at either end of the pipeline (default 16 slabs, then 8, 9, 3 and 32 by the tuning variable)
    ((16, 16, 8, 64), 32, 18, 1, None), ((16, 16, 8, 64), 32, 12, 2, 8), ((16, 8, 8, 72), 64, 18, 1, 9),
    ((16, 16, 8, 64), 32, 18, 1, 3), ((16, 16, 8, 64), 32, 18, 1, 32), ((16, 8, 8, 33), 64, 18, 2, 8)])
def test_apply_host_pipelined_path(oracle, monkeypatch, dims, precision, recon, nrhs, nslab):
    """wd_apply_host on fields large enough for its slab pipeline (H2D / apply / D2H overlapped on three
    streams): same bits as the one-stream host path, and the oracle's result."""
    cfg = fields.Config("hp", dims, precision, "haar", recon, -0.4, nrhs, 53)
    U, psi = fields.make_fields(cfg)
    assert psi.nbytes >= 8 << 20
    op = GpuOp(U, dims, precision, recon, KERNELS["site"])
    if nslab:
        op.op.set_tuning("host_nslab", nslab)
    out = np.full_like(psi, np.nan)
    op.op.apply_host(out, psi, cfg.mass, nrhs)
    again = np.full_like(psi, np.nan)
    op.op.apply_host(again, psi, cfg.mass, nrhs)
    assert np.array_equal(out, again)
    op.op.set_tuning("host_no_pipeline", 1)
    plain = np.full_like(psi, np.nan)
    op.op.apply_host(plain, psi, cfg.mass, nrhs)
    op.close()
    assert np.array_equal(out, plain)
    Uo = oracle_links(U, recon)
    want = oracle_apply(oracle, psi, Uo, dims, cfg.mass)
    for r in range(nrhs):
        assert rel_l2(out[r], want[r]) <= TOL[precision]


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 12, 6), (3, 5, 2, 7), (2, 2, 2, 2), (16, 8, 8, 6)])
@pytest.mark.parametrize("precision,recon", [(64, 18), (32, 18), (32, 12), (64, 12)])
def test_apply_dagger_matches_the_oracle_and_gamma5_hermiticity(oracle, dims, precision, recon):
    """wd_apply_dagger = D^dagger = gamma5 D gamma5: against the oracle's sign=+1 operator, and
    <phi, D^dagger psi> = <D phi, psi> with both sides from the CUDA path."""
    import torch
    cfg = fields.Config("dag", dims, precision, "haar", recon, -0.3, 2, 91)
    U, psi = fields.make_fields(cfg)
    Uo = oracle_links(U, recon).astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    w = op.op
    canon = torch.from_numpy(psi).cuda()
    n = w.native_numel(2)
    a = torch.empty(n, dtype=canon.dtype, device="cuda")
    b = torch.empty_like(a)
    c = torch.empty_like(a)
    out = torch.empty_like(canon)
    w.pack(a, canon, 2)
    w.apply_dagger(b, a, cfg.mass, 2)
    w.unpack(out, b, 2)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    for r in range(2):
        want = oracle.apply(psi[r].astype(np.float64), Uo, dims, cfg.mass, sign=+1)
        assert rel_l2(got[r], want) <= TOL[precision]
    w.apply(c, a, cfg.mass, 2)                      # D psi_0, D psi_1
    dout = torch.empty_like(canon)
    w.unpack(dout, c, 2)
    torch.cuda.synchronize()
    d = dout.cpu().numpy().astype(np.float64)
    cplx = lambda v: v[..., 0] + 1j * v[..., 1]
    phi, ps = cplx(psi[0].astype(np.float64)), cplx(psi[1].astype(np.float64))
    lhs = np.vdot(phi, cplx(got[1].astype(np.float64)))        # <phi, D^dagger psi>
    rhs = np.vdot(cplx(d[0]), ps)                              # <D phi, psi>
    assert abs(lhs - rhs) <= (1e-11 if precision == 64 else 2e-4) * abs(rhs) + (1e-9 if precision == 64 else 1e-2)
    op.close()


# ---------------------------------------------------------------- round 2: dagger / Lx = 24 / fp64 members of the staged family
@pytest.mark.parametrize("dims", [(32, 4, 4, 5), (16, 8, 8, 6), (8, 4, 12, 6), (4, 4, 4, 4), (24, 4, 4, 6), (12, 8, 4, 3)])
@pytest.mark.parametrize("precision,recon", [(64, 18), (32, 18), (32, 12), (64, 12)])
@pytest.mark.parametrize("nrhs", [1, 3, 4, 8])
def test_staged_dagger_matches_the_oracle(oracle, dims, precision, recon, nrhs):
    """wd_apply_dagger through the STAGED kernel (templated on the projector sign): D^dagger = gamma5 D gamma5
     against the oracle's sign=+1 operator; several right-hand sides go through the sign-swapped member of
    the multi-RHS kernel (fp32, 128-site tiles of a power-of-two Lx; 4 = a full group + a single-RHS launch, 8 = two groups
    + a pair) and otherwise through the single-RHS member in the (patch, column, right-hand side) block order."""
    import torch
    cfg = fields.Config("sdag", dims, precision, "haar", recon, -0.3, nrhs, 93)
    U, psi = fields.make_fields(cfg)
    Uo = oracle_links(U, recon).astype(np.float64)
    op = GpuOp(U, dims, precision, recon, KERNELS["stage"])
    w = op.op
    canon = torch.from_numpy(psi).cuda()
    a = torch.empty(w.native_numel(nrhs), dtype=canon.dtype, device="cuda")
    b = torch.full_like(a, float("nan"))
    out = torch.empty_like(canon)
    w.pack(a, canon, nrhs)
    w.apply_dagger(b, a, cfg.mass, nrhs)
    w.unpack(out, b, nrhs)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    op.close()
    for r in range(nrhs):
        want = oracle.apply(psi[r].astype(np.float64), Uo, dims, cfg.mass, sign=+1)
        assert rel_l2(got[r], want) <= TOL[precision]


@pytest.mark.parametrize("dims,nrhs", [((24, 8, 4, 6), 20), ((24, 4, 4, 5), 7), ((12, 8, 8, 4), 4), ((24, 2, 2, 3), 3)])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("force_mrhs", [False, True])
def test_multi_rhs_when_lx_is_not_a_power_of_two(oracle, monkeypatch, dims, nrhs, recon, force_mrhs):
    """The paper's volumes have Lx = 24 and N_v = 20.  Default: the single-RHS staged member
    in the (patch, column, right-hand side) order (links shared through L2, the faster choice there); WD_STAGE_NO_MRHS=0
    forces the multi-RHS member (links shared in shared memory, x hops through the slice buffer)."""
    if force_mrhs:
        monkeypatch.setenv("WD_STAGE_NO_MRHS", "0")
    cfg = fields.Config("mrhs24", dims, 32, "haar", recon, -0.41, nrhs, 95)
    check_config(oracle, cfg, "stage")


@pytest.mark.parametrize("dims,nrhs", [((32, 8, 8, 4), 5), ((16, 4, 8, 6), 24), ((24, 4, 4, 3), 4)])
@pytest.mark.parametrize("recon", [18, 12])
def test_fp64_multi_rhs_shares_links_through_l2(oracle, dims, nrhs, recon):
    """fp64, several right-hand sides: the single-RHS staged kernel in the (patch of columns, right-hand side fastest)
    block order; every right-hand side against the oracle at the fp64 bound."""
    cfg = fields.Config("mrhs64", dims, 64, "haar", recon, -0.41, nrhs, 97)
    check_config(oracle, cfg, "stage")


@pytest.mark.parametrize("recon,tgauge", [(18, False), (12, False), (18, True)])
def test_multi_rhs_bulk_copy_variant_is_bit_identical(oracle, recon, tgauge):
    """WD_MRHS_BULK: the link halves staged by cp.async.bulk + mbarrier instead of per-thread cp.async (the A/B variant of
    profiles/r02_ncu.md section 6): same bits as the default staging, and the oracle's result."""
    import torch
    cfg = fields.Config("bulk", (32, 8, 8, 6), 32, "smooth", recon, -0.42, 7, 101)
    U, psi = fields.make_fields(cfg)
    if tgauge:
        U, _ = fields.temporal_gauge(U, 32)
    op = GpuOp(U, cfg.dims, 32, recon, KERNELS["stage"])
    if tgauge:
        op.op.set_temporal_gauge(True)
    a = op.apply(psi, cfg.mass, return_native=True).clone()
    op.op.set_tuning("mrhs_bulk", 1)
    b = op.apply(psi, cfg.mass, return_native=True).clone()
    got = op.apply(psi, cfg.mass)
    op.close()
    assert torch.equal(a, b)
    want = oracle_apply(oracle, psi, oracle_links(U, recon), cfg.dims, cfg.mass)
    for r in range(7):
        assert rel_l2(got[r], want[r]) <= TOL[32]


def test_multi_rhs_tail_wave_split_is_bit_identical(oracle):
    """A launch of more work items than SMs whose last wave is partial cuts that wave's items into shorter marches
    (wd_dslash_mrhs.cu); the result is bit-identical to the uncut launch and matches the oracle."""
    import torch
    cfg = fields.Config("tail", (32, 16, 16, 16), 32, "smooth", 18, -0.42, 24, 99)   # 64 columns x 8 groups = 512 items
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18, KERNELS["stage"])
    a = op.apply(psi, cfg.mass, return_native=True).clone()
    op.op.set_tuning("mrhs_no_tail", 1)
    b = op.apply(psi, cfg.mass, return_native=True).clone()
    op.op.set_tuning("mrhs_no_tail", -1)
    got = op.apply(psi, cfg.mass)
    op.close()
    assert torch.equal(a, b)
    want = oracle_apply(oracle, psi[:3], U, cfg.dims, cfg.mass)
    for r in range(3):
        assert rel_l2(got[r], want[r]) <= TOL[32]


def test_auto_kernel_selection():
    """WD_KERNEL_AUTO resolves by lattice, precision and nrhs; a forced kernel is reported."""
    from paper_0912_2186_b200 import binding
    cases = [((32, 16, 16, 32), 32, 1, "stage"), ((32, 16, 16, 32), 32, 24, "stage"), ((32, 16, 16, 32), 64, 1, "stage"),
             ((32, 16, 16, 32), 64, 4, "stage"), ((24, 24, 24, 32), 32, 1, "stage"), ((24, 24, 24, 32), 32, 3, "stage"), ((20, 20, 20, 40), 32, 1, "site"), ((8, 8, 8, 8), 32, 1, "site")]
    for dims, precision, nrhs, want in cases:
        cfg = fields.Config("sel", dims, precision, "haar", 18, 0.1, 1, 5)
        U, _ = fields.make_fields(cfg)
        op = GpuOp(U, dims, precision, 18)
        assert op.op.selected_kernel(nrhs) == want, (dims, precision, nrhs)
        op.op.set_kernel(KERNELS["site"])
        assert op.op.selected_kernel(nrhs) == "site"
        op.close()


def test_launch_counter_counts_kernels():
    from paper_0912_2186_b200 import binding
    cfg = fields.Config("l", (4, 4, 4, 4), 32, "haar", 18, 0.1, 1, 71)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, cfg.dims, 32, 18)
    n0 = binding.wd_launch_count()
    op.apply(psi, cfg.mass)  # pack + apply + unpack
    assert binding.wd_launch_count() - n0 == 3
    op.close()


# ---------------------------------------------------------------- guard bands (compute-sanitizer is closed on this pool)
@pytest.mark.parametrize("dims,precision,recon,nrhs,kernel", [
    ((16, 16, 16, 32), 32, 18, 1, "stage"), ((16, 16, 16, 32), 32, 18, 1, "site"), ((4, 4, 4, 4), 64, 18, 1, "auto"),
    ((16, 8, 8, 6), 32, 12, 5, "stage"), ((24, 4, 4, 6), 32, 18, 4, "stage"), ((16, 8, 8, 6), 64, 18, 3, "stage"),
    ((32, 4, 4, 5), 32, 8, 2, "stage"), ((6, 10, 4, 9), 32, 18, 3, "site"), ((16, 8, 8, 6), 16, 12, 2, "stage"),
    ((6, 10, 4, 9), 16, 18, 2, "site")])
def test_kernels_write_only_their_output(dims, precision, recon, nrhs, kernel):
    """The output buffer sits between two 64 KB guard bands filled with a bit pattern, the input likewise: after wd_apply
    and wd_apply_dagger every guard byte is unchanged and every real site of the output has been written.  (Stands in
    for a memcheck run: compute-sanitizer answers "closed on this pool".)"""
    import torch
    from paper_0912_2186_b200 import binding
    cprec = 32 if precision == 16 else precision
    cfg = fields.Config("guard", dims, cprec, "haar", recon, -0.3, nrhs, 121)
    U, psi = fields.make_fields(cfg)
    op = binding.WilsonDirac(dims, torch.from_numpy(U).cuda(), precision, recon, kernel=KERNELS[kernel])
    nbytes = binding.wd_spinor_bytes(op.lat, nrhs, precision)
    G = 65536
    bufs = []
    for _ in range(2):
        raw = torch.full((nbytes + 2 * G,), 0x5A, dtype=torch.uint8, device="cuda")
        bufs.append(raw)
    src, dst = bufs[0][G:G + nbytes], bufs[1][G:G + nbytes]
    canon = torch.from_numpy(psi).cuda()
    op.pack(src, canon, nrhs)
    for fn in (op.apply, op.apply_dagger):
        dst.fill_(0x5A)
        fn(dst, src, cfg.mass, nrhs)
        torch.cuda.synchronize()
        for raw in bufs:
            assert bool(torch.all(raw[:G] == 0x5A)) and bool(torch.all(raw[G + nbytes:] == 0x5A))
        out = torch.full_like(canon, float("nan"))
        op.unpack(out, dst, nrhs)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(out).all())
        assert not bool((out.view(torch.uint8) == 0x5A).all(dim=-1).any())   # no site left at the fill pattern
    op.close()


@pytest.mark.parametrize("env,dims,precision,recon,nrhs", [
    ({"WD_MRHS_REG": "1"}, (16, 8, 8, 6), 32, 18, 5), ({"WD_MRHS_REG": "1"}, (32, 4, 4, 5), 32, 12, 4),
    ({"WD_MRHS_REG": "2"}, (32, 4, 4, 5), 32, 18, 7), ({"WD_MRHS_REG": "2"}, (32, 8, 4, 3), 32, 8, 3),
    ({"WD_STAGE_BULK": "1"}, (32, 4, 4, 5), 32, 18, 1), ({"WD_STAGE_BULK": "1"}, (32, 4, 8, 4), 64, 12, 1),
    ({"WD_STAGE_BULK": "1", "WD_STAGE_NO_MRHS": "1"}, (32, 4, 4, 3), 32, 18, 3)])
def test_round2_late_members_write_only_their_output(monkeypatch, env, dims, precision, recon, nrhs):
    """Guard bands around the buffers of the members added late in round 2: the links-in-registers multi-RHS kernels (plain
    loads, ring of cp.async.bulk row copies) and the bulk-copy member of the single-RHS staged kernel.  A bulk copy that ran
    past its row, or a prefetch-distance bug turned into a store, would show up here."""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    test_kernels_write_only_their_output(dims, precision, recon, nrhs, "stage")


# ---------------------------------------------------------------- a lattice beyond 2^31 bytes per field: sampled outputs
def test_large_lattice_sampled_against_the_oracle(oracle):
    """32 x 48 x 72 x 64 (7.1 M sites: the link field is 2.0 GB, byte offsets beyond 2^31; 864 tile columns):
    the staged kernel on analytic SU(3) links (cheap to generate: a colour rotation with site-dependent angle and phases)
    and Gaussian spinors, compared with the oracle on runs of consecutive sites taken at the start, the middle, around a
    time-slice boundary and at the very end of the lattice."""
    import torch
    dims = (32, 48, 72, 64)
    Lx, Ly, Lz, Lt = dims
    V = fields.volume(dims)
    t, z, y, x = np.meshgrid(np.arange(Lt, dtype=np.float32), np.arange(Lz, dtype=np.float32), np.arange(Ly, dtype=np.float32),
                             np.arange(Lx, dtype=np.float32), indexing="ij", sparse=True)
    U = np.zeros((4, Lt, Lz, Ly, Lx, 3, 3, 2), dtype=np.float32)
    for mu in range(4):
        phi = 0.37 * x + 0.11 * y * (mu + 1) + 0.23 * z + 0.05 * t + 0.7 * mu
        al = 0.19 * x * y + 0.31 * t + mu
        be = 0.13 * z * x + 0.29 * y - mu
        c, s = np.cos(phi), np.sin(phi)
        U[mu, ..., 0, 0, 0], U[mu, ..., 0, 0, 1] = c * np.cos(al), c * np.sin(al)
        U[mu, ..., 0, 1, 0], U[mu, ..., 0, 1, 1] = s * np.cos(be), s * np.sin(be)
        U[mu, ..., 1, 0, 0], U[mu, ..., 1, 0, 1] = -s * np.cos(be), s * np.sin(be)
        U[mu, ..., 1, 1, 0], U[mu, ..., 1, 1, 1] = c * np.cos(al), -c * np.sin(al)
        U[mu, ..., 2, 2, 0] = 1.0
    rng = np.random.default_rng(131)
    psi = rng.standard_normal((1, Lt, Lz, Ly, Lx, 4, 3, 2), dtype=np.float32)
    mass = -0.4
    op = GpuOp(U, dims, 32, 18, KERNELS["auto"])
    assert op.op.selected_kernel(1) == "stage"
    got = op.apply(psi, mass)[0].reshape(V, 4, 3, 2)
    op.close()
    U64 = U.astype(np.float64)
    p64 = psi[0].astype(np.float64)
    S3 = Lx * Ly * Lz
    for begin in (0, V // 2 - 777, 17 * S3 - 300, V - 600):
        end = begin + 600
        want = oracle.apply_range(p64, U64, dims, mass, begin, end)
        assert rel_l2(got[begin:end], want) <= TOL[32], begin
