"""-m gpu: seeded sweep over anisotropic lattices x precision x link storage x kernel x tuning variables, a random number
of right-hand sides and a random mass per case, every result against the oracle (north-star tolerances).  Catches
dimension-order, face, chunk-boundary and partial-group mistakes that the cubic configs hide."""
import numpy as np
import pytest

from paper_0912_2186_b200 import binding, fields
from gpu_util import TOL, GpuOp, rel_l2

pytestmark = pytest.mark.gpu

SHAPES = [(32, 6, 4, 3), (32, 10, 2, 2), (16, 12, 6, 5), (8, 16, 4, 9), (4, 8, 24, 2), (32, 4, 12, 7), (24, 8, 2, 4),
          (12, 8, 4, 6), (16, 2, 2, 17), (32, 2, 6, 1), (32, 12, 12, 3)]
ENVS = [{}, {"WD_TILE_TC": "1"}, {"WD_TILE_TC": "3", "WD_TILE_NRB": "2"}, {"WD_MRHS_PATCH": "0", "WD_TILE_SHAPE": "2,2"},
        # the members added late in round 2 (they apply where Lx is a power of two / Lx = 32 and fall through elsewhere)
        {"WD_MRHS_REG": "1", "WD_MRHS_RGRP": "3"}, {"WD_MRHS_REG": "2", "WD_TILE_TC": "2"}, {"WD_STAGE_BULK": "1"},
        {"WD_STAGE_BULK": "1", "WD_STAGE_NO_MRHS": "1", "WD_TILE_TC": "3"}]


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("precision,recon", [(32, 18), (32, 12), (64, 18), (64, 12)])
def test_every_kernel_on_anisotropic_lattices(oracle, monkeypatch, dims, precision, recon):
    rng = np.random.default_rng(abs(hash((dims, precision, recon))) % (2 ** 31))
    nrhs = int(rng.integers(1, 8))
    cfg = fields.Config("soak", dims, precision, "haar", recon, float(rng.uniform(-0.45, 0.3)), nrhs, int(rng.integers(1, 10 ** 6)))
    U, psi = fields.make_fields(cfg)
    Uo = (U if recon == 18 else np.ascontiguousarray(U[..., :2, :, :])).astype(np.float64)
    want = [oracle.apply(psi[r].astype(np.float64), Uo, dims, cfg.mass) for r in range(nrhs)]
    ran = 0
    for kernel in (1, 3):
        for env in ENVS:
            with monkeypatch.context() as m:
                for k, v in env.items():
                    m.setenv(k, v)
                try:
                    op = GpuOp(U, dims, precision, recon, kernel)
                except binding.WdError as e:
                    assert e.code == -7 and kernel != 1   # a tiled kernel may refuse a lattice it cannot tile; never the site kernel
                    continue
                got = op.apply(psi, cfg.mass)
                op.close()
            ran += 1
            for r in range(nrhs):
                assert rel_l2(got[r], want[r]) <= TOL[precision], (dims, precision, recon, nrhs, kernel, env, r)
    assert ran >= len(ENVS)
