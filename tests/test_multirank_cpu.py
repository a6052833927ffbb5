"""N > 1 host logic of bench.py on CPU (no GPU): world-size-2 gloo process group for the max-over-ranks
timing and the rank-shifted replica seeds, and the reference arm under torchrun (rank 0 alone prints).
The data path has no collective: ranks run independent replicas."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _gloo_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    from paper_0912_2186_b200 import fields
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg = fields.CONFIGS["c0_4x4_fp64"]
    cfg_r = bench.rank_config(cfg, cfg.recon, cfg.nrhs, rank)
    ms = bench.max_over_ranks(10.0 * (rank + 1), world)  # rank 1 is the slow one
    value = bench.whole_job_gflops(world, 7, 1368 * 256, ms)
    dist.barrier()
    with open(os.path.join(out, f"r{rank}.json"), "w") as f:
        json.dump({"seed": cfg_r.seed, "dims": list(cfg_r.dims), "ms": ms, "value": value}, f)
    dist.destroy_process_group()


def test_gloo_world2_max_over_ranks_and_replica_seeds(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_gloo_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"r{i}.json")) for i in range(2)]
    assert r[0]["ms"] == r[1]["ms"] == 20.0  # the slowest rank decides
    assert r[0]["seed"] != r[1]["seed"] and r[0]["dims"] == r[1]["dims"]  # independent replicas, same shape
    want = 2 * 7 * 1368 * 256 / 20e-3 / 1e9  # whole-job aggregate over both ranks
    assert r[0]["value"] == pytest.approx(want) and r[1]["value"] == pytest.approx(want)


def test_single_rank_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5


def test_reference_arm_under_torchrun_two_ranks():
    """bench.py --impl reference launched as the driver does for N = 2: rank 0 alone runs the oracle and
    prints the JSON line, the other rank exits 0 without output."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference",
           "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "c0_4x4_fp64"]
    p = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [json.loads(l) for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["value"] > 0
