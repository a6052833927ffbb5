"""-m gpu parity tests of the Krylov shell (wd_apply_schur_dagger, wd_cgnr_schur) against the oracle
(oracle.schur sign=+1, oracle/wd_solvers.py:cgnr_schur), through the C ABI.  SURVEY.md 8(f) row f2.

Tolerances: the operator keeps the north-star bounds (1e-13 / 2e-6).  CG is an iteration: after K steps in
working precision eps the iterates of two correct implementations differ by O(K * kappa * eps); with the masses
used here (well conditioned, kappa ~ 10) and K = 12: 1e-10 in fp64, 2e-4 in fp32 on x and on the residual history
-- derived bounds, written here, far below any plausible algorithmic mistake (a wrong alpha/beta gives O(1))."""
import numpy as np
import pytest

from paper_0912_2186_b200 import fields
from oracle import wd_solvers
from gpu_util import TOL, GpuOp, rel_l2
from test_parity_gpu_evenodd import parity_mask

pytestmark = pytest.mark.gpu


def to_half(op, canon_np, parity):
    import torch
    w = op.op
    canon = torch.from_numpy(np.ascontiguousarray(canon_np)).cuda()
    h = torch.full((w.half_numel(1),), float("nan"), dtype=canon.dtype, device="cuda")
    w.pack_parity(h, canon, 1, parity)
    return h


def from_half(op, h, shape, parity):
    import torch
    out = torch.zeros(shape, dtype=h.dtype, device="cuda")
    op.op.unpack_parity(out, h, 1, parity)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 6, 2), (16, 8, 8, 6)])
@pytest.mark.parametrize("precision,recon", [(64, 18), (32, 18), (32, 12)])
def test_schur_dagger_matches_the_oracle(oracle, dims, precision, recon):
    import torch
    cfg = fields.Config("sd", dims, precision, "haar", recon, -0.31, 1, 63)
    U, psi = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    for parity in (0, 1):
        a = to_half(op, psi, parity)
        b, tmp = torch.empty_like(a), torch.empty_like(a)
        op.op.apply_schur_dagger(b, a, tmp, cfg.mass, parity, 1)
        got = from_half(op, b, psi.shape, parity)
        want = oracle.schur(psi.astype(np.float64), Uo, dims, cfg.mass, parity, sign=+1)
        assert rel_l2(got[0], want[0]) <= TOL[precision]
    op.close()


@pytest.mark.parametrize("dims,parity", [((4, 4, 4, 4), 0), ((8, 4, 6, 2), 1), ((16, 8, 8, 8), 0), ((2, 6, 4, 2), 1)])
@pytest.mark.parametrize("precision,recon,tol_x", [(64, 18, 1e-10), (64, 12, 1e-10), (32, 18, 2e-4), (32, 12, 2e-4)])
def test_cgnr_fixed_iterations_match_the_oracle(oracle, dims, parity, precision, recon, tol_x):
    import torch
    K = 12
    cfg = fields.Config("cg", dims, precision, "smooth", recon, 0.2, 1, 65)
    U, b = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    bh = to_half(op, b, parity)
    xh = torch.full_like(bh, float("nan"))
    iters, hist = op.op.cgnr_schur(xh, bh, cfg.mass, parity, K)
    x = from_half(op, xh, b.shape, parity)[0]
    # determinism: a second solve gives the same bits
    xh2 = torch.full_like(bh, float("nan"))
    op.op.cgnr_schur(xh2, bh, cfg.mass, parity, K)
    x2 = from_half(op, xh2, b.shape, parity)[0]
    op.close()
    want_x, want_hist = wd_solvers.cgnr_schur(b[0].astype(np.float64), Uo, dims, cfg.mass, parity, K)
    assert iters == K and len(hist) == K + 1
    assert np.array_equal(x, x2)
    assert np.all(x[np.broadcast_to(parity_mask(dims)[0] != parity, x.shape)] == 0)
    assert rel_l2(x, want_x) <= tol_x
    assert np.max(np.abs(np.array(hist) / want_hist - 1.0)) <= tol_x * 10


def test_cgnr_converges_to_the_solution(oracle):
    import torch
    dims, parity = (8, 8, 8, 8), 0
    cfg = fields.Config("cgc", dims, 64, "smooth", 18, 0.1, 1, 67)
    U, b = fields.make_fields(cfg)
    op = GpuOp(U, dims, 64, 18)
    bh = to_half(op, b, parity)
    xh = torch.empty_like(bh)
    iters, hist = op.op.cgnr_schur(xh, bh, cfg.mass, parity, 500, tol=1e-11)
    x = from_half(op, xh, b.shape, parity)
    op.close()
    assert iters < 500 and hist[-1] <= 1e-11 and hist[0] == pytest.approx(1.0)
    bm = np.where(parity_mask(dims) == parity, b, 0.0)
    res = bm - oracle.schur(x.astype(np.float64), U.astype(np.float64), dims, cfg.mass, parity)
    assert np.linalg.norm(res) / np.linalg.norm(bm) <= 2e-11   # true residual, recomputed by the oracle


@pytest.mark.parametrize("dims,parity", [((4, 4, 4, 4), 0), ((8, 4, 6, 2), 1), ((16, 8, 8, 8), 0), ((2, 6, 4, 2), 1)])
@pytest.mark.parametrize("precision,recon,tol_x", [(64, 18, 1e-9), (64, 12, 1e-9), (32, 18, 1e-3), (32, 12, 1e-3)])
def test_bicgstab_fixed_iterations_match_the_oracle(oracle, dims, parity, precision, recon, tol_x):
    """K = 8 BiCGstab iterations (16 matvecs).  BiCGstab's scalars are ratios of inner products that shrink with the
    residual, so rounding differences grow faster than in CG: 1e-9 (fp64) / 1e-3 (fp32) on x, ten times that on the
    residual history -- derived bounds; a wrong alpha, omega or beta changes x at O(1)."""
    import torch
    K = 8
    cfg = fields.Config("bi", dims, precision, "smooth", recon, 0.2, 1, 69)
    U, b = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    bh = to_half(op, b, parity)
    xh = torch.full_like(bh, float("nan"))
    iters, hist = op.op.bicgstab_schur(xh, bh, cfg.mass, parity, K)
    x = from_half(op, xh, b.shape, parity)[0]
    xh2 = torch.full_like(bh, float("nan"))
    op.op.bicgstab_schur(xh2, bh, cfg.mass, parity, K)
    x2 = from_half(op, xh2, b.shape, parity)[0]
    op.close()
    want_x, want_hist = wd_solvers.bicgstab_schur(b[0].astype(np.float64), Uo, dims, cfg.mass, parity, K)
    assert iters == K and len(hist) == K + 1
    assert np.array_equal(x, x2)                                   # deterministic reductions
    assert rel_l2(x, want_x) <= tol_x
    assert np.max(np.abs(np.array(hist) / want_hist - 1.0)) <= tol_x * 10


def test_bicgstab_converges_to_the_solution(oracle):
    import torch
    dims, parity = (8, 8, 8, 8), 1
    cfg = fields.Config("bic", dims, 64, "smooth", 18, 0.1, 1, 71)
    U, b = fields.make_fields(cfg)
    op = GpuOp(U, dims, 64, 18)
    bh = to_half(op, b, parity)
    xh = torch.empty_like(bh)
    iters, hist = op.op.bicgstab_schur(xh, bh, cfg.mass, parity, 300, tol=1e-11)
    x = from_half(op, xh, b.shape, parity)
    op.close()
    assert iters < 300 and hist[-1] <= 1e-11
    bm = np.where(parity_mask(dims) == parity, b, 0.0)
    res = bm - oracle.schur(x.astype(np.float64), U.astype(np.float64), dims, cfg.mass, parity)
    assert np.linalg.norm(res) / np.linalg.norm(bm) <= 5e-11


@pytest.mark.parametrize("dims,parity", [((4, 4, 4, 4), 0), ((8, 4, 6, 2), 1), ((16, 8, 8, 8), 0)])
@pytest.mark.parametrize("precision,recon,tol_x", [(64, 18, 1e-10), (64, 12, 1e-10), (32, 18, 2e-4), (32, 12, 2e-4)])
@pytest.mark.parametrize("restart", [8, 3, 11])  # 11: two groups of the grouped Gram-Schmidt (8 + up to 2)
def test_gcr_fixed_iterations_match_the_oracle(oracle, dims, parity, precision, recon, tol_x, restart):
    """K = 13 iterations of GCR(restart): more than one restart cycle.  Same derived bounds as CGNR (orthogonal
    projections, well-conditioned system)."""
    import torch
    K = 13
    cfg = fields.Config("gcr", dims, precision, "smooth", recon, 0.2, 1, 73)
    U, b = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    bh = to_half(op, b, parity)
    xh = torch.full_like(bh, float("nan"))
    iters, hist = op.op.gcr_schur(xh, bh, cfg.mass, parity, K, restart)
    x = from_half(op, xh, b.shape, parity)[0]
    xh2 = torch.full_like(bh, float("nan"))
    op.op.gcr_schur(xh2, bh, cfg.mass, parity, K, restart)
    x2 = from_half(op, xh2, b.shape, parity)[0]
    op.close()
    want_x, want_hist = wd_solvers.gcr_schur(b[0].astype(np.float64), Uo, dims, cfg.mass, parity, K, restart=restart)
    assert iters == K and len(hist) == K + 1
    assert np.array_equal(x, x2)
    assert rel_l2(x, want_x) <= tol_x
    assert np.max(np.abs(np.array(hist) / want_hist - 1.0)) <= tol_x * 10


def test_gcr8_converges_to_the_solution(oracle):
    import torch
    dims, parity = (8, 8, 8, 8), 0
    cfg = fields.Config("gcrc", dims, 64, "smooth", 18, 0.1, 1, 75)
    U, b = fields.make_fields(cfg)
    op = GpuOp(U, dims, 64, 18)
    bh = to_half(op, b, parity)
    xh = torch.empty_like(bh)
    iters, hist = op.op.gcr_schur(xh, bh, cfg.mass, parity, 400, 8, tol=1e-11)
    x = from_half(op, xh, b.shape, parity)
    op.close()
    assert iters < 400 and hist[-1] <= 1e-11
    bm = np.where(parity_mask(dims) == parity, b, 0.0)
    res = bm - oracle.schur(x.astype(np.float64), U.astype(np.float64), dims, cfg.mass, parity)
    assert np.linalg.norm(res) / np.linalg.norm(bm) <= 5e-11


# ---------------------------------------------------------------- round 2: preconditioner slot, true-residual control, guards
@pytest.mark.parametrize("precision,tol_x", [(64, 1e-9), (32, 5e-4)])
def test_gcr_preconditioner_slot(oracle, precision, tol_x):
    """wd_gcr_schur_precond with K = Mhat^dagger supplied through the callback (the slot the paper fills with the
    multigrid cycle) against the oracle's preconditioned GCR; K = NULL stays wd_gcr_schur."""
    import torch
    dims, parity, K = (8, 4, 8, 4), 0, 6
    cfg = fields.Config("gp", dims, precision, "smooth", 18, 0.1, 1, 81)
    U, b = fields.make_fields(cfg)
    op = GpuOp(U, dims, precision, 18)
    w = op.op
    bh = to_half(op, b, parity)
    xh = torch.full_like(bh, float("nan"))
    tmp = torch.empty_like(bh)
    calls = []

    def precond(z_ptr, r_ptr, stream_ptr):
        calls.append(stream_ptr)
        w.apply_schur_dagger(z_ptr, r_ptr, tmp, cfg.mass, parity, 1)       # z = Mhat^dagger r on the gauge's stream
        return 0

    iters, hist = w.gcr_schur_precond(xh, bh, cfg.mass, parity, K, 8, 0.0, precond)
    x = from_half(op, xh, b.shape, parity)[0]
    op.close()
    assert iters == K and len(calls) == K
    Uo = U.astype(np.float64)
    c = lambda v: v[..., 0] + 1j * v[..., 1]
    rp = lambda v: np.stack([v.real, v.imag], axis=-1)
    Md = lambda r: c(oracle.schur(np.ascontiguousarray(rp(r)), Uo, dims, cfg.mass, parity, sign=+1))
    want_x, want_hist = wd_solvers.gcr_schur(b[0].astype(np.float64), Uo, dims, cfg.mass, parity, K, restart=8, precond=Md)
    assert rel_l2(x, want_x) <= tol_x
    assert np.max(np.abs(np.array(hist) / want_hist - 1.0)) <= tol_x * 10


@pytest.mark.parametrize("solver", ["cgnr", "bicgstab", "gcr"])
def test_fp32_tolerance_is_checked_on_the_true_residual(oracle, solver):
    """In fp32 the recursively updated residual falls below what |b - Mhat x| can reach.  With tol > 0 the last history
    entry is the TRUE residual (recomputed by the library, checked here by the oracle), in the negative-mass regime of
    the paper (m = -0.3 on smooth links); a reachable tolerance is reached, an unreachable one is reported honestly."""
    import torch
    dims, parity = (8, 8, 8, 8), 0
    cfg = fields.Config("tr", dims, 32, "smooth", 18, -0.3, 1, 83)
    U, b = fields.make_fields(cfg)
    op = GpuOp(U, dims, 32, 18)
    w = op.op
    bh = to_half(op, b, parity)
    solve = {"cgnr": lambda x, it, tol: w.cgnr_schur(x, bh, cfg.mass, parity, it, tol=tol),
             "bicgstab": lambda x, it, tol: w.bicgstab_schur(x, bh, cfg.mass, parity, it, tol=tol),
             "gcr": lambda x, it, tol: w.gcr_schur(x, bh, cfg.mass, parity, it, 8, tol=tol)}[solver]
    bm = np.where(parity_mask(dims) == parity, b, 0.0).astype(np.float64)

    def true_rel(xh):
        x = from_half(op, xh, b.shape, parity).astype(np.float64)
        return np.linalg.norm(bm - oracle.schur(x, U.astype(np.float64), dims, cfg.mass, parity)) / np.linalg.norm(bm)

    xh = torch.full_like(bh, float("nan"))
    iters, hist = solve(xh, 400, 1e-5)
    t = true_rel(xh)
    assert hist[-1] <= 1e-5 and iters < 400
    assert t == pytest.approx(hist[-1], rel=0.05, abs=2e-7)
    xh2 = torch.full_like(bh, float("nan"))
    iters2, hist2 = solve(xh2, 400, 1e-9)                      # below the reach of fp32
    t2 = true_rel(xh2)
    assert t2 == pytest.approx(hist2[-1], rel=0.05, abs=2e-7)  # whatever was reached is what is reported
    assert hist2[-1] < 2e-6 and iters2 <= 400
    op.close()


@pytest.mark.parametrize("solver", ["cgnr", "bicgstab", "gcr"])
@pytest.mark.parametrize("tol", [0.0, 1e-8])
def test_zero_right_hand_side_gives_zero_not_nan(solver, tol):
    import torch
    dims = (4, 4, 4, 4)
    cfg = fields.Config("z", dims, 64, "haar", 18, 0.1, 1, 85)
    U, b = fields.make_fields(cfg)
    op = GpuOp(U, dims, 64, 18)
    w = op.op
    bh = torch.zeros(w.half_numel(1), dtype=torch.float64, device="cuda")
    xh = torch.full_like(bh, float("nan"))
    if solver == "cgnr":
        w.cgnr_schur(xh, bh, cfg.mass, 0, 5, tol=tol)
    elif solver == "bicgstab":
        w.bicgstab_schur(xh, bh, cfg.mass, 0, 5, tol=tol)
    else:
        w.gcr_schur(xh, bh, cfg.mass, 0, 5, 4, tol=tol)
    torch.cuda.synchronize()
    assert torch.all(xh == 0)
    op.close()


@pytest.mark.parametrize("precision,recon,tol_x", [(64, 18, 1e-10), (32, 12, 2e-4)])
def test_block_cgnr_is_the_single_solve_per_right_hand_side(oracle, precision, recon, tol_x):
    """wd_cgnr_schur_block: nrhs right-hand sides in lock step with batched operator applications.  Each right-hand side's
    iterate and history are bit-identical to wd_cgnr_schur on it alone, and match the oracle's CGNR."""
    import torch
    dims, parity, K, nrhs = (8, 8, 4, 8), 1, 10, 3
    cfg = fields.Config("blk", dims, precision, "smooth", recon, 0.2, nrhs, 87)
    U, b = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    op = GpuOp(U, dims, precision, recon)
    w = op.op
    canon = torch.from_numpy(b).cuda()
    n1 = w.half_numel(1)
    bh = torch.zeros(nrhs * n1, dtype=canon.dtype, device="cuda")
    w.pack_parity(bh, canon, nrhs, parity)
    xh = torch.full_like(bh, float("nan"))
    iters, hists = w.cgnr_schur_block(xh, bh, cfg.mass, parity, nrhs, K)
    assert iters == K and len(hists) == nrhs
    for r in range(nrhs):
        xs = torch.full((n1,), float("nan"), dtype=canon.dtype, device="cuda")
        it1, h1 = w.cgnr_schur(xs, bh[r * n1:(r + 1) * n1], cfg.mass, parity, K)
        torch.cuda.synchronize()
        assert torch.equal(xs, xh[r * n1:(r + 1) * n1])
        assert h1 == hists[r]
        x = from_half(op, xs, b[r:r + 1].shape, parity)[0]
        want_x, want_hist = wd_solvers.cgnr_schur(b[r].astype(np.float64), Uo, dims, cfg.mass, parity, K)
        assert rel_l2(x, want_x) <= tol_x
        assert np.max(np.abs(np.array(hists[r]) / want_hist - 1.0)) <= tol_x * 10
    # tolerance mode: stops when every right-hand side has converged
    it2, h2 = w.cgnr_schur_block(xh, bh, cfg.mass, parity, nrhs, 300, tol=1e-5 if precision == 32 else 1e-10)
    assert it2 < 300 and all(h[-1] <= (1e-5 if precision == 32 else 1e-10) for h in h2)
    op.close()
