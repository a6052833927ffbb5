"""-m gpu parity tests of the storage variants: 8-real links and half-precision
storage, through the C ABI, against the oracle fed with what the storage format actually holds
(oracle/wd_storage.py, pinned in tests/test_oracle_pins_storage.py).

Tolerances (readings R8 / RH):
  8 reals   both sides rebuild the link from the SAME eight rounded numbers; the CUDA path does it in the working
            precision, and rounding in the rebuilt rows is amplified by 1/N, N = |a2|^2 + |a3|^2.  Over a field of
            Haar or smooth (eps = 0.3) links the rms of 1/N is ~10^2, so the bound is 1e-5 (fp32) / 1e-10 (fp64).
  half      inputs are the dequantised fields on both sides; the CUDA result is rounded once more to binary16 relative
            to the site maximum: |error| <= 2^-11 max_site, i.e. <= 2^-11 * sqrt(24) relative L2 in the worst case; 1e-3.
"""
import numpy as np
import pytest

from paper_0912_2186_b200 import binding, fields
from oracle import wd_storage as ws
from gpu_util import GpuOp, rel_l2

pytestmark = pytest.mark.gpu
TOL8 = {32: 1e-5, 64: 1e-10}
KERNELS = {"auto": 0, "site": 1, "stage": 3}


@pytest.mark.parametrize("dims", [(32, 4, 4, 5), (16, 8, 8, 6), (24, 4, 4, 6), (6, 10, 4, 8), (3, 5, 2, 7)])
@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("links", ["haar", "smooth"])
def test_recon8_matches_the_oracle(oracle, dims, precision, links):
    cfg = fields.Config("r8", dims, precision, links, 8, -0.35, 3, 701)
    U, psi = fields.make_fields(cfg)
    U8 = ws.links_from_8(U, precision)                       # what the 8 stored reals say, rebuilt in fp64
    for kernel in ("site", "stage"):
        try:
            op = GpuOp(U, dims, precision, 8, KERNELS[kernel])
        except binding.WdError as e:
            assert e.code == -7 and kernel == "stage"        # lattices the staged kernel cannot tile
            continue
        for nrhs in (1, 3):
            got = op.apply(psi[:nrhs], cfg.mass)
            for r in range(nrhs):
                want = oracle.apply(psi[r].astype(np.float64), U8, dims, cfg.mass)
                assert rel_l2(got[r], want) <= TOL8[precision], (kernel, nrhs, r)
        op.close()


@pytest.mark.parametrize("precision", [32, 64])
def test_recon8_dagger_and_even_odd(oracle, precision):
    import torch
    dims = (16, 4, 8, 6)
    cfg = fields.Config("r8b", dims, precision, "haar", 8, -0.2, 1, 703)
    U, psi = fields.make_fields(cfg)
    U8 = ws.links_from_8(U, precision)
    op = GpuOp(U, dims, precision, 8, KERNELS["stage"])
    w = op.op
    canon = torch.from_numpy(psi).cuda()
    a = torch.empty(w.native_numel(1), dtype=canon.dtype, device="cuda")
    b = torch.empty_like(a)
    out = torch.empty_like(canon)
    w.pack(a, canon, 1)
    w.apply_dagger(b, a, cfg.mass, 1)
    w.unpack(out, b, 1)
    torch.cuda.synchronize()
    want = oracle.apply(psi[0].astype(np.float64), U8, dims, cfg.mass, sign=+1)
    assert rel_l2(out.cpu().numpy()[0], want) <= TOL8[precision]
    # even-odd preconditioned operator with 8-real links
    n = w.half_numel(1)
    hi, ho, tmp = (torch.empty(n, dtype=canon.dtype, device="cuda") for _ in range(3))
    w.pack_parity(hi, canon, 1, 0)
    w.apply_schur(ho, hi, tmp, cfg.mass, 0, 1)
    full = torch.zeros_like(canon)
    w.unpack_parity(full, ho, 1, 0)
    torch.cuda.synchronize()
    want = oracle.schur(psi[0].astype(np.float64), U8, dims, cfg.mass, 0)
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    even = ((x + y + z + t) % 2 == 0)
    assert rel_l2(full.cpu().numpy()[0][even], want[even]) <= TOL8[precision]
    op.close()


def test_recon8_refuses_links_it_cannot_hold():
    dims = (4, 4, 4, 4)
    U = fields.unit_links(dims).astype(np.float32)
    with pytest.raises(binding.WdError) as e:
        GpuOp(U, dims, 32, 8)
    assert e.value.code == -4
    cfg = fields.Config("r8c", dims, 32, "haar", 8, 0.1, 1, 705)
    Uh, _ = fields.make_fields(cfg)
    op = GpuOp(Uh, dims, 32, 8)
    with pytest.raises(binding.WdError) as e:
        op.op.set_temporal_gauge(True)
    assert e.value.code == -4
    op.close()


# ---------------------------------------------------------------- half-precision storage
def _half_case(oracle, dims, recon, links, nrhs, dagger=False, seed=711, kernel=0):
    import torch
    cfg = fields.Config("half", dims, 32, links, 18, -0.35, nrhs, seed)
    U, psi = fields.make_fields(cfg)                                    # float32 canonical fields
    op = binding.WilsonDirac(dims, torch.from_numpy(U).cuda(), 16, recon, kernel=kernel)
    assert op.selected_kernel(nrhs) == ("stage" if kernel == 3 else "site")
    canon = torch.from_numpy(psi).cuda()
    n = op.native_numel(nrhs)
    assert n == nrhs * (-(-fields.volume(dims) // 32) * 32) * 26
    a = torch.zeros(n, dtype=torch.float16, device="cuda")
    b = torch.zeros(n, dtype=torch.float16, device="cuda")
    back = torch.full_like(canon, float("nan"))
    out = torch.full_like(canon, float("nan"))
    op.pack(a, canon, nrhs)
    op.unpack(back, a, nrhs)                                            # what the half field holds
    (op.apply_dagger if dagger else op.apply)(b, a, cfg.mass, nrhs)
    op.unpack(out, b, nrhs)
    torch.cuda.synchronize()
    op.close()
    # the stored input is exactly the oracle's quantisation of the same float32 field
    q, s = ws.quantise_half_spinor(psi)
    held = ws.dequantise_half_spinor(q, s)
    assert np.max(np.abs(back.cpu().numpy().astype(np.float64) - held)) <= 1e-6 * np.max(np.abs(held))
    if recon == 8:
        Uo = ws.links_from_8(U, 16)
    else:
        Uo = ws.quantise_half_links(U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :]))
    got = out.cpu().numpy().astype(np.float64)
    for r in range(nrhs):
        want = oracle.apply(held[r], Uo, dims, cfg.mass, sign=+1 if dagger else -1)
        assert rel_l2(got[r], want) <= 1e-3, (recon, r, rel_l2(got[r], want))
        # and it is not the fp32 result in disguise: the error is at the binary16 level
        assert rel_l2(got[r], want) >= 1e-5


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (16, 4, 6, 5), (3, 5, 2, 7)])
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_half_storage_matches_the_oracle_on_the_dequantised_fields(oracle, dims, recon):
    _half_case(oracle, dims, recon, "haar", 2)


def test_half_storage_dagger_and_smooth_links(oracle):
    _half_case(oracle, (8, 4, 8, 6), 12, "smooth", 1, dagger=True)


@pytest.mark.parametrize("dims", [(32, 4, 4, 5), (16, 8, 8, 6), (8, 4, 12, 7), (4, 8, 8, 3), (32, 6, 10, 4)])
@pytest.mark.parametrize("recon", [18, 12, 8])
@pytest.mark.parametrize("dagger", [False, True])
def test_half_storage_staged_kernel(oracle, dims, recon, dagger):
    """The staged (cp.async, t-marching) member of the half-precision family: raw binary16 data staged in shared memory,
    converted at the LDS, result requantised in the epilogue; chunk boundaries and faces as in the fp32 kernel."""
    _half_case(oracle, dims, recon, "haar", 2, dagger=dagger, kernel=3)


def test_half_storage_staged_kernel_is_deterministic(monkeypatch):
    """Same launch twice: same bits.  Other t-chunk lengths (march restarts at other slices): the same field up to the
    binary16 rounding of the result (the restart computes the first backward t hop from global memory, a different
    instruction sequence, so bit equality across chunkings is not promised)."""
    import torch
    dims = (16, 8, 8, 12)
    cfg = fields.Config("halfdet", dims, 32, "smooth", 18, -0.42, 1, 715)
    U, psi = fields.make_fields(cfg)
    outs = []
    for tc in ("16", "16", "1", "5"):
        monkeypatch.setenv("WD_TILE_TC", tc)
        op = binding.WilsonDirac(dims, torch.from_numpy(U).cuda(), 16, 12, kernel=3)
        a = torch.zeros(op.native_numel(1), dtype=torch.float16, device="cuda")
        b = torch.zeros_like(a)
        canon = torch.from_numpy(psi).cuda()
        op.pack(a, canon, 1)
        op.apply(b, a, cfg.mass, 1)
        out = torch.empty_like(canon)
        op.unpack(out, b, 1)
        torch.cuda.synchronize()
        outs.append((b.clone(), out.cpu().numpy().astype(np.float64)))
        op.close()
    assert torch.equal(outs[0][0].view(torch.int16), outs[1][0].view(torch.int16))
    for k in (2, 3):
        assert rel_l2(outs[k][1], outs[0][1]) <= 5e-4


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (16, 4, 6, 2), (4, 2, 2, 6)])
@pytest.mark.parametrize("recon", [18, 12, 8])
@pytest.mark.parametrize("parity", [0, 1])
def test_half_storage_even_odd_blocks(oracle, dims, recon, parity):
    """wd_apply_hop / wd_apply_schur / wd_apply_schur_dagger on half-storage fields of one parity (the operator of the paper's
    fastest kernel row): inputs are the dequantised fields on both sides, the result (and, for the Schur
    operator, the intermediate field) is rounded to binary16 relative to the site maximum -- the bounds of reading RH."""
    import torch
    nrhs = 2
    cfg = fields.Config("halfeo", dims, 32, "haar", 18, 0.3, nrhs, 721)
    U, psi = fields.make_fields(cfg)
    w = binding.WilsonDirac(dims, torch.from_numpy(U).cuda(), 16, recon)
    canon = torch.from_numpy(psi).cuda()
    n = w.half_numel(nrhs)
    assert n == nrhs * (-(-(fields.volume(dims) // 2) // 32) * 32) * 26
    hi, ho, hd, hop, tmp = (torch.zeros(n, dtype=torch.float16, device="cuda") for _ in range(5))
    w.pack_parity(hi, canon, nrhs, parity)
    back = torch.zeros_like(canon)
    w.unpack_parity(back, hi, nrhs, parity)
    w.apply_schur(ho, hi, tmp, cfg.mass, parity, nrhs)
    w.apply_schur_dagger(hd, hi, tmp, cfg.mass, parity, nrhs)
    binding.wd_apply_hop(hop, hi, w.gauge, dims, nrhs, 16, 1 - parity)
    outs = []
    for h, par in ((ho, parity), (hd, parity), (hop, 1 - parity)):
        full = torch.zeros_like(canon)
        w.unpack_parity(full, h, nrhs, par)
        outs.append(full.cpu().numpy().astype(np.float64))
    torch.cuda.synchronize()
    w.close()
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    mine = ((x + y + z + t) % 2 == parity)
    q, s = ws.quantise_half_spinor(psi)
    held = ws.dequantise_half_spinor(q, s)
    got_in = back.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got_in[:, mine] - held[:, mine])) <= 1e-6 * np.max(np.abs(held))
    assert not got_in[:, ~mine].any()
    if recon == 8:
        Uo = ws.links_from_8(U, 16)
    else:
        Uo = ws.quantise_half_links(U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :]))
    for r in range(nrhs):
        src = np.where(mine[..., None, None, None], held[r], 0.0)
        for got, want, m in ((outs[0][r], oracle.schur(src, Uo, dims, cfg.mass, parity), mine),
                             (outs[1][r], oracle.schur(src, Uo, dims, cfg.mass, parity, sign=+1), mine),
                             (outs[2][r], oracle.hop_parity(src, Uo, dims, 1 - parity), ~mine)):
            err = rel_l2(got[m], want[m])
            assert 1e-5 <= err <= 1e-3, (recon, r, err)
            assert not got[~m].any()


def test_half_storage_is_refused_where_it_is_not_implemented():
    import torch
    dims = (4, 4, 4, 4)
    cfg = fields.Config("halfno", dims, 32, "haar", 18, 0.1, 1, 713)
    U, psi = fields.make_fields(cfg)
    op = binding.WilsonDirac(dims, torch.from_numpy(U).cuda(), 16, 12)
    buf = torch.zeros(op.half_numel(1), dtype=torch.float16, device="cuda")
    buf2 = torch.zeros_like(buf)
    with pytest.raises(binding.WdError) as e:                                  # the solvers run in fp32 / fp64
        binding.wd_cgnr_schur(buf2, buf, op.gauge, 0.1, dims, 16, 0, 3)
    assert e.value.code == -3
    op.set_kernel(3)                                    # 4^4 can be tiled by the staged half kernel
    with pytest.raises(binding.WdError) as e:
        op.set_temporal_gauge(True)
    assert e.value.code == -3
    op.close()
