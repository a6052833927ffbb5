"""-m gpu: wd_apply_schur_static, the entry point that allocates nothing (include/wd.h; csrc/wd_noalloc.cu): the even-odd
preconditioned operator with its intermediate half field in a static device array of WD_STATIC_SCRATCH_BYTES.  Checked
against the existing path (wd_apply_schur with a caller-owned intermediate field) at the north-star tolerances, on two
calls in a row with different inputs -- the array keeps the previous call's contents, which must not matter -- and
against the oracle.  This file is collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_0912_2186_b200 import binding, fields
from gpu_util import TOL, GpuOp, rel_l2

pytestmark = pytest.mark.gpu


def _parity_mask(dims, parity):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (x + y + z + t) % 2 == parity


@pytest.mark.parametrize("dims,precision,recon,nrhs,parity", [
    ((16, 16, 16, 32), 32, 18, 2, 0),   # config 1's lattice, two right-hand sides: 12.6 of the 16.8 MB
    ((16, 16, 16, 32), 64, 12, 1, 1),
    ((8, 4, 6, 2), 32, 12, 3, 1),
    ((6, 4, 2, 2), 64, 18, 1, 0),       # Vh = 48 sites: a ragged last layout block
    ((8, 8, 4, 4), 32, 8, 1, 0),
])
def test_schur_static_matches_the_existing_path_twice_in_a_row(oracle, dims, precision, recon, nrhs, parity):
    import torch
    cfg = fields.Config("noalloc", dims, precision, "haar", recon, -0.3, 2 * nrhs, 901)
    U, psi = fields.make_fields(cfg)
    op = GpuOp(U, dims, precision, recon)
    w = op.op
    n = w.half_numel(nrhs)
    assert n * (4 if precision == 32 else 8) <= binding.WD_STATIC_SCRATCH_BYTES
    canon = [torch.from_numpy(np.ascontiguousarray(psi[i * nrhs:(i + 1) * nrhs])).cuda() for i in range(2)]
    hin = [torch.empty(n, dtype=canon[0].dtype, device="cuda") for _ in range(2)]
    got = [torch.full((n,), float("nan"), dtype=canon[0].dtype, device="cuda") for _ in range(2)]
    ref = [torch.full((n,), float("nan"), dtype=canon[0].dtype, device="cuda") for _ in range(2)]
    tmp = torch.empty(n, dtype=canon[0].dtype, device="cuda")
    full = [torch.zeros_like(canon[0]) for _ in range(4)]
    for i in range(2):
        w.pack_parity(hin[i], canon[i], nrhs, parity)
    torch.cuda.synchronize()
    # the static entry point first: before any other red/black call on this handle (it needs no parity-ordered link copy)
    w.apply_schur_static(got[0], hin[0], cfg.mass, parity, nrhs)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    w.apply_schur_static(got[1], hin[1], cfg.mass, parity, nrhs)      # second call in a row, other input, stale scratch
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after >= free_before - (1 << 20), "a call of wd_apply_schur_static took device memory"
    for i in range(2):
        w.apply_schur(ref[i], hin[i], tmp, cfg.mass, parity, nrhs)     # existing path, caller-owned intermediate field
    for i in range(2):
        w.unpack_parity(full[i], got[i], nrhs, parity)
        w.unpack_parity(full[2 + i], ref[i], nrhs, parity)
    torch.cuda.synchronize()
    op.close()
    mine = _parity_mask(dims, parity)
    Uo = (U if recon != 12 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    if recon == 8:
        from oracle import wd_storage
        Uo = wd_storage.links_from_8(U, precision)
    tol = TOL[precision] if recon != 8 else {32: 1e-5, 64: 1e-10}[precision]   # reading R8
    for i in range(2):
        g, r = full[i].cpu().numpy(), full[2 + i].cpu().numpy()
        assert np.isfinite(g).all()
        assert not g[:, ~mine].any()
        for k in range(nrhs):
            assert rel_l2(g[k][mine], r[k][mine]) <= tol, (i, k)
            src = np.where(mine[..., None, None, None], psi[i * nrhs + k].astype(np.float64), 0.0)
            want = oracle.schur(src, Uo, dims, cfg.mass, parity)
            assert rel_l2(g[k][mine], want[mine]) <= tol, (i, k)


def test_schur_static_rejects_what_does_not_fit_and_bad_arguments():
    import torch
    dims = (16, 16, 16, 32)
    cfg = fields.Config("noalloc2", dims, 32, "haar", 18, 0.1, 1, 903)
    U, _ = fields.make_fields(cfg)
    op = GpuOp(U, dims, 32, 18)
    w = op.op
    # 3 right-hand sides: 3 * 65536 * 96 B = 18.9 MB > 16.8 MB
    n3 = w.half_numel(3)
    assert n3 * 4 > binding.WD_STATIC_SCRATCH_BYTES
    a = torch.zeros(n3, dtype=torch.float32, device="cuda")
    b = torch.zeros(n3, dtype=torch.float32, device="cuda")
    with pytest.raises(binding.WdError) as e:
        w.apply_schur_static(b, a, 0.1, 0, 3)
    assert e.value.code == -2 and "static scratch" in str(e.value)
    with pytest.raises(binding.WdError) as e:                       # 4 + m = 0
        w.apply_schur_static(b, a, -4.0, 0, 1)
    assert e.value.code == -7
    with pytest.raises(binding.WdError) as e:                       # in place
        w.apply_schur_static(a, a, 0.1, 0, 1)
    assert e.value.code == -6
    with pytest.raises(binding.WdError) as e:
        w.apply_schur_static(b, a, 0.1, 2, 1)
    assert e.value.code == -7
    with pytest.raises(binding.WdError) as e:                       # precision of the handle
        binding.wd_apply_schur_static(b, a, w.gauge, 0.1, dims, 1, 64, 0)
    assert e.value.code == -3
    op.close()
