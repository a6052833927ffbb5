#!/usr/bin/env python
"""bench.py -- throughput of the Wilson-Dirac matvec D*psi (eq. (2.2)) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--kernel auto|site|stage]
                    [--recon 18|12] [--impl wd|reference]

One JSON line on stdout (rank 0).  Definitions:
  * workload   default c3_32x64_fp32 = BASELINE.json:configs[3], the configuration the metric is
               quoted on: 32^3x64, fp32, smooth links, m=-0.42, single RHS, 18-real links.
  * step       the Krylov-loop batch of configs[3]: APPLIES_PER_STEP (=100) wd_apply calls back to
               back on one stream with no host sync, rotating through NBUF distinct input and
               output fields (reading S9: not a chain D^100 psi, which overflows fp32).
  * value      Gflop/s at 1368 flops/site/RHS (1320 hopping + 48 diagonal), all ranks together,
               inputs resident in HBM, timed with CUDA events on the launching stream, max over ranks.
  * L2         gauge (604 MB) + rotating spinors exceed the 126 MB L2, so no flush is needed
               ("inputs larger than L2" in config.l2).
  * e2e        the same metric through wd_apply_host: pinned HOST buffers in canonical layout,
               H2D copy + pack + apply + unpack + D2H copy + sync inside the timed region.
  * roofline   HBM: algorithmic (compulsory) bytes per launch / mean launch duration, against
               MEASURED_PEAKS.json:hbm_gbs.
  * secondary  (default run only) two short legs after the headline timing, same launch path, own clocks record:
               configs[4] = 24 right-hand sides (2 steps x 10 applies; roofline.frac against the HBM peak, plus
               frac_of_own_peak against min(HBM bound, FMA-pipe bound at the observed clock)) and configs[3] in fp64
               (2 steps x 25 applies), then the same two with 12-real links and the storage variants of the paper's
               Table 2 on the headline lattice (12-real, 8-real, half storage).  The headline's metric, config and value
               are unchanged.
  * next_rows  (default run only) short legs of the rows built after the hot path, on the headline's lattice and links:
               the even-odd preconditioned operator (f1), CGNR / BiCGstab / GCR(8) on it (f2; 48 iterations each) and the
               block CGNR on 12 right-hand sides, restrict + prolong and the coarse operator apply at N_v = 20 (f3); each
               with its own byte model, roofline fraction and clocks record.
  * cpu_baseline  the oracle (oracle/wd_oracle.c, fp64, OpenMP) on this box's host cores, on a
               bounded sample of the same workload.
Multi-GPU (torchrun): the path has no exchange step on one GPU per lattice; ranks run independent
replicas of the workload (different seeds), no data-path collective; scaling "weak".
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_0912_2186_b200 import fields  # noqa: E402  (seeded generators only; no arithmetic of the method)

APPLIES_PER_STEP = 100
NBUF = 4
FLOPS_PER_SITE = 1368
METRIC = "wilson_dslash_gflops"
UNIT = "Gflop/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def compulsory_bytes_per_site(precision, recon, nrhs):
    """Algorithmic HBM bytes per site per launch: every spinor read once and
    written once, every link read once."""
    if precision == 16:  # half-precision storage: 24 binary16 ratios + one float32 scale per site; links binary16
        return nrhs * 2 * 52 + 4 * recon * 2
    w = 4 if precision == 32 else 8
    return nrhs * 2 * 24 * w + 4 * recon * w


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json:hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload, recon):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    try:
        return json.load(open(p)).get(f"{workload}_r{recon}", {}).get("dram_bytes_per_launch")
    except Exception:
        return None


class ClockSampler:
    """Samples SM clock and clock-event (throttle) reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
             0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
             0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.NAMES.items():
                    if mask & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        return {"sm_mhz": (float(np.median(self.samples)) if self.samples else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    return rank, local, world


def rank_config(cfg, recon, nrhs, rank):
    """Replica of the workload for one rank: same shape, seeds shifted by rank (no data-path collective)."""
    return fields.Config(cfg.name, cfg.dims, cfg.precision, cfg.links, recon, cfg.mass, nrhs, cfg.seed + 100 * rank, cfg.eps)


def max_over_ranks(value, world, device=None):
    """Slowest rank decides: all-reduce MAX of a host float over the default process group."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gflops(world, applies, flops_per_apply, ms):
    """Aggregate throughput of `world` replicas that each did `applies` applies in `ms` (max over ranks)."""
    return world * applies * flops_per_apply / (ms * 1e-3) / 1e9


def oracle_rate(cfg, U, psi, budget_s=12.0):
    """Time the oracle as it stands on a bounded sample: whole-lattice applies of RHS 0, repeated
    until ~budget_s of CPU work (at least 1, at most 8).  Returns the cpu_baseline object."""
    from oracle import wd_oracle
    U64 = np.ascontiguousarray(U if cfg.recon == 18 else U[..., :2, :, :], dtype=np.float64)
    p64 = np.ascontiguousarray(psi[0], dtype=np.float64)
    V = fields.volume(cfg.dims)
    # calibrate on a slab so a slow box cannot run away
    n0 = max(1, V // 16)
    t0 = time.perf_counter()
    wd_oracle.apply_range(p64, U64, cfg.dims, cfg.mass, 0, n0)
    rate = n0 / (time.perf_counter() - t0)
    n = int(min(V, max(n0, rate * budget_s / 3)))
    best = None
    reps = 0
    t_all = time.perf_counter()
    while reps < 8 and (reps < 1 or time.perf_counter() - t_all < budget_s):
        t0 = time.perf_counter()
        wd_oracle.apply_range(p64, U64, cfg.dims, cfg.mass, 0, n)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
        reps += 1
    return {"value": n * FLOPS_PER_SITE / best / 1e9, "unit": UNIT, "cores": wd_oracle.num_threads(),
            "kind": "oracle", "sites_per_s": n / best,
            "sample": f"fp64 oracle, first {n} of {V} sites of {cfg.name} (1 RHS), best of {reps} passes"}


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only), same metric/config/unit."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import wd_oracle
    cfg = fields.CONFIGS[args.workload]
    U, psi = fields.make_fields(cfg, nrhs=1)
    U64 = np.ascontiguousarray(U if args.recon == 18 else U[..., :2, :, :], dtype=np.float64)
    p64 = np.ascontiguousarray(psi[0], dtype=np.float64)
    V = fields.volume(cfg.dims)
    n0 = max(1, V // 32)
    t0 = time.perf_counter()
    wd_oracle.apply_range(p64, U64, cfg.dims, cfg.mass, 0, n0)
    rate = n0 / (time.perf_counter() - t0)
    # each step: a bounded sample of ~1 s so that steps+warmup end within a few minutes
    n = int(min(V, max(1024, rate * min(1.0, 120.0 / max(1, args.steps + args.warmup)))))
    for _ in range(args.warmup):
        wd_oracle.apply_range(p64, U64, cfg.dims, cfg.mass, 0, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        wd_oracle.apply_range(p64, U64, cfg.dims, cfg.mass, 0, n)
    dt = time.perf_counter() - t0
    value = args.steps * n * FLOPS_PER_SITE / dt / 1e9
    sample = f"fp64 oracle, first {n} of {V} sites of {cfg.name} (1 RHS) per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "dims": list(cfg.dims), "recon": args.recon, "nrhs": 1,
                   "flops_per_site": FLOPS_PER_SITE, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": wd_oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def issue_bound_gbs(precision, recon, nrhs, sm_mhz):
    """FP32/FP64-pipe ceiling of a multi-RHS apply expressed in the roofline's unit (algorithmic GB/s): the SASS of
    the staged kernels spends ~912 FMA-pipe cycles per 32 (site, rhs) (profiles/r02_ubench.md: FFMA2 2 clk, scalar
    FADD/FMUL 1 clk per warp instruction and SMSP), i.e. 148 SMs x 4 SMSPs x 32 / 912 (site, rhs) per clock."""
    if sm_mhz is None:
        return None
    per_clk = 148 * 4 * 32 / (912.0 if precision == 32 else 2 * 912.0)
    site_rhs_per_s = per_clk * sm_mhz * 1e6
    return site_rhs_per_s / nrhs * compulsory_bytes_per_site(precision, recon, nrhs) / 1e9


def secondary_leg(binding, torch, dev, stream, local, name, U, recon, nrhs, steps, aps, storage=None):
    """One short timed leg of another BASELINE workload (north_star: "the batched 24-RHS apply reported in Gflop/s
    and as a fraction of its own roofline"; configs[3] is "fp64 and fp32").  Links: the array handed in (same recipe
    and shape as the workload's); spinors: complex Gaussian drawn on the device (seeded torch generator) straight into
    the native buffers -- the native layout is a permutation of the canonical one, so the distribution is the same."""
    cfg = fields.CONFIGS[name]
    V = fields.volume(cfg.dims)
    prec = storage or cfg.precision        # storage = 16: half-precision storage, float32 canonical side
    tdt = {16: torch.float16, 32: torch.float32, 64: torch.float64}[prec]
    nbuf = 2 if nrhs > 1 else NBUF
    with torch.cuda.stream(stream):
        u_dev = torch.from_numpy(fields.round_to(U, 32 if prec == 16 else prec)).to(dev)
        op = binding.WilsonDirac(cfg.dims, u_dev, prec, recon, stream=stream.cuda_stream)
        g = torch.Generator(device=dev).manual_seed(cfg.seed + 1000)
        if prec == 16:   # pack float32 Gaussian fields (the native half field is ratios + scales, not plain numbers)
            ins = [torch.empty(op.native_numel(nrhs), dtype=tdt, device=dev) for _ in range(nbuf)]
            Lx, Ly, Lz, Lt = cfg.dims
            for b in ins:
                c = torch.randn((nrhs, Lt, Lz, Ly, Lx, 4, 3, 2), dtype=torch.float32, device=dev, generator=g)
                op.pack(b, c, nrhs)
            del c
        else:
            ins = [torch.randn(op.native_numel(nrhs), dtype=tdt, device=dev, generator=g) for _ in range(nbuf)]
        outs = [torch.empty(op.native_numel(nrhs), dtype=tdt, device=dev) for _ in range(nbuf)]
    stream.synchronize()
    del u_dev

    def step():
        for i in range(aps):
            op.apply(outs[i % nbuf], ins[i % nbuf], cfg.mass, nrhs)

    for _ in range(3):
        step()
    torch.cuda.synchronize()
    n0 = binding.wd_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        ev0.record(stream)
        for _ in range(steps):
            step()
        ev1.record(stream)
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / (steps * aps)
    launches = binding.wd_launch_count() - n0
    kern = op.selected_kernel(nrhs)
    op.close()
    del ins, outs
    torch.cuda.empty_cache()
    bytes_per_launch = compulsory_bytes_per_site(prec, recon, nrhs) * V
    peak, peak_src = measured_peak()
    achieved = bytes_per_launch / (ms * 1e-3) / 1e9
    ck = clocks.summary()
    roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": None if storage else ncu_traffic(name, recon), "peak_source": peak_src, "bytes_per_launch": bytes_per_launch,
            "kernel": "wd dslash, " + kern + " kernel" + (" (multi-RHS member)" if nrhs > 1 and kern == "stage" else "")}
    if nrhs > 1:  # its own roofline = min(HBM bound, FMA-pipe bound at the observed clock); both printed
        ib = issue_bound_gbs(cfg.precision, recon, nrhs, ck["sm_mhz"])
        roof["fma_pipe_bound_gbs"] = ib
        roof["own_peak"] = min(peak, ib) if ib else peak
        roof["frac_of_own_peak"] = achieved / roof["own_peak"]
    return {"workload": name, "value": FLOPS_PER_SITE * V * nrhs / (ms * 1e-3) / 1e9, "unit": UNIT, "nrhs": nrhs,
            "recon": recon, "dtype": {16: "f32 arithmetic on f16 storage", 32: "f32", 64: "f64"}[prec],
            "bytes_per_site": compulsory_bytes_per_site(prec, recon, nrhs), "us_per_apply": ms * 1e3,
            "steps": steps, "applies_per_step": aps, "gpu_launches": int(launches),
            "data": "synthetic: " + ("headline links recipe (smooth, eps=0.3)" if cfg.links == "smooth" else "the workload's links recipe (" + cfg.links + ")") + ", device-drawn Gaussian spinors",
            "roofline": roof, "clocks": ck}


SOLVER_MODEL = {"cgnr": (288, 8, 2), "bicgstab": (672, 15, 2), "gcr": (1150, 22.25, 1)}  # BLAS-1 flops, spinor passes, matvecs


def next_rows_legs(binding, torch, dev, stream, local, name, U, recon):
    """Short timed legs of the "next" rows on the headline's lattice and links (the operator and the
    solvers of the paper's Table 2): the even-odd preconditioned operator Mhat, CGNR, BiCGstab and GCR(8)
    on it, and the 12-right-hand-side block CGNR.  Same byte and flop models as --op schur / cgnr / bicgstab / gcr."""
    cfg = fields.CONFIGS[name]
    V, w = fields.volume(cfg.dims), 4
    peak, peak_src = measured_peak()
    out = []
    with torch.cuda.stream(stream):
        u_dev = torch.from_numpy(fields.round_to(U, 32)).to(dev)
        op = binding.WilsonDirac(cfg.dims, u_dev, 32, recon, stream=stream.cuda_stream)
        g = torch.Generator(device=dev).manual_seed(cfg.seed + 2000)
        n = op.half_numel(1)
        b = torch.randn(12 * n, dtype=torch.float32, device=dev, generator=g)  # native half fields: any values are vectors
        x = torch.empty_like(b)
        tmp = torch.empty(n, dtype=torch.float32, device=dev)
    stream.synchronize()
    del u_dev

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        n0 = binding.wd_launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(local) as clocks:
            ev0.record(stream)
            for _ in range(reps):
                fn()
            ev1.record(stream)
            torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / reps, int(binding.wd_launch_count() - n0), clocks.summary()

    def entry(row, what, units, unit_name, ms, flops, nbytes, launches, ck, nrhs=1):
        achieved = nbytes * units / (ms * 1e-3) / 1e9
        return {"row": row, "op": what, "workload": name, "recon": recon, "nrhs": nrhs, "dtype": "f32",
                "value": units * flops / (ms * 1e-3) / 1e9, "unit": UNIT, "us_per_" + unit_name: ms / units * 1e3,
                "gpu_launches": launches, "clocks": ck,
                "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                             "peak_source": peak_src, "bytes_per_" + unit_name: nbytes}}

    aps = 20

    def schur():
        for i in range(aps):
            op.apply_schur(x[(i % 4) * n:(i % 4 + 1) * n], b[(i % 4) * n:(i % 4 + 1) * n], tmp, cfg.mass, 0, 1)

    ms, nl, ck = timed(schur, 2)
    out.append(entry("f1", "even-odd preconditioned operator Mhat (2 launches)", aps, "apply", ms,
                     (2 * 1320 + 48) * (V // 2), (V // 2) * (2 * 2 * 4 * recon * w + 5 * 24 * w), nl, ck))
    iters = 48
    for key, label, solve in (("cgnr", "CGNR on Mhat", op.cgnr_schur), ("bicgstab", "BiCGstab on Mhat", op.bicgstab_schur),
                              ("gcr", "GCR(8) on Mhat", op.gcr_schur)):
        bf, bp, nmv = SOLVER_MODEL[key]
        ms, nl, ck = timed(lambda: solve(x[:n], b[:n], cfg.mass, 0, iters), 1)
        out.append(entry("f2", label, iters, "iteration", ms, (nmv * (2 * 1320 + 48) + bf) * (V // 2),
                         (V // 2) * (nmv * (2 * 2 * 4 * recon * w + 5 * 24 * w) + bp * 24 * w), nl, ck))
    bf, bp, nmv = SOLVER_MODEL["cgnr"]
    ms, nl, ck = timed(lambda: op.cgnr_schur_block(x, b, cfg.mass, 0, 12, 10), 1)
    out.append(entry("f2 + a'", "block CGNR on Mhat, 12 right-hand sides in lock step", 10, "iteration", ms,
                     (nmv * (2 * 1320 + 48) + bf) * (V // 2) * 12,
                     (V // 2) * (nmv * (2 * 2 * 4 * recon * w + 12 * 5 * 24 * w) + 12 * bp * 24 * w), nl, ck, nrhs=12))
    del b, x, tmp
    torch.cuda.empty_cache()
    # ---- row f3 (N_v = 20): restrict + prolong, coarse operator build and apply ----
    nv, nc = 20, 40
    nb = V // 256
    with torch.cuda.stream(stream):
        basis = torch.randn(op.native_numel(nv), dtype=torch.float32, device=dev, generator=g)
        psi = torch.randn(op.native_numel(1), dtype=torch.float32, device=dev, generator=g)
        res = torch.empty_like(psi)
        coarse = torch.empty(binding.wd_coarse_reals(op.lat, nv), dtype=torch.float32, device=dev)
        binding.wd_block_orthonormalise(op.lat, basis, nv, 32, stream.cuda_stream)

    def transfer():
        binding.wd_restrict(op.lat, coarse, basis, psi, nv, 32, stream.cuda_stream)
        binding.wd_prolong(op.lat, res, basis, coarse, nv, 32, stream.cuda_stream)

    ms, nl, ck = timed(transfer, 5)
    out.append(entry("f3", "restrict + prolong, N_v = 20, 4^4 blocks x 2 chiralities", 1, "step", ms, 2 * nv * V * 12 * 8,
                     (2 * nv + 2) * V * 24 * w, nl, ck))
    ns = binding.wd_coarse_stencil_reals(op.lat, nv)
    with torch.cuda.stream(stream):
        S = torch.empty(ns, dtype=torch.float32, device=dev)
        scratch = torch.empty(ns, dtype=torch.float32, device=dev)
        cin = [torch.randn(nb * nc * 2, dtype=torch.float32, device=dev, generator=g) for _ in range(2)]
        cout = [torch.empty_like(cin[0]) for _ in range(2)]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    binding.wd_build_coarse(op.gauge, S, scratch, basis, cfg.mass, cfg.dims, nv, 32)
    ev1.record(stream)
    torch.cuda.synchronize()
    build_ms = ev0.elapsed_time(ev1)
    del scratch, basis, psi, res

    def coarse_apply():
        for i in range(20):
            binding.wd_apply_coarse(op.lat, cout[i % 2], cin[i % 2], S, nv, 1, 32, stream.cuda_stream)

    ms, nl, ck = timed(coarse_apply, 3)
    e = entry("f3", "coarse operator apply, 9-point stencil of (2 N_v)^2 complex blocks, N_v = 20", 20, "apply", ms,
              nb * 9 * nc * nc * 8, nb * (9 * nc * nc * 2 * w + 2 * nc * 2 * w), nl, ck)
    e["build_ms_first_call"] = build_ms
    out.append(e)
    op.close()
    del S, cin, cout, coarse
    torch.cuda.empty_cache()
    return out


def pcie_peaks(torch, dev, h_in, h_out):
    """Measured copy rates of THIS box for the e2e roofline: one large cudaMemcpyAsync per direction from / to the pinned
    buffers the e2e leg uses, alone (h2d, d2h) and both at once on two streams (duplex, rate per direction), best of 3,
    CUDA events.  GB/s."""
    nbytes = h_in.numel() * h_in.element_size()
    d_a = torch.empty_like(h_in, device=dev)
    d_b = torch.empty_like(h_in, device=dev)
    s1, s2 = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)

    def timed(fn):
        best = None
        for _ in range(3):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(s1)
            s2.wait_event(e0)
            fn()
            e2 = torch.cuda.Event()
            e2.record(s2)
            s1.wait_event(e2)
            e1.record(s1)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        return nbytes / (best * 1e-3) / 1e9

    def h2d():
        with torch.cuda.stream(s1):
            d_a.copy_(h_in, non_blocking=True)

    def d2h():
        with torch.cuda.stream(s1):
            h_out.copy_(d_b, non_blocking=True)

    def both():
        with torch.cuda.stream(s1):
            d_a.copy_(h_in, non_blocking=True)
        with torch.cuda.stream(s2):
            h_out.copy_(d_b, non_blocking=True)

    d_b.zero_()
    out = {"h2d_gbs": timed(h2d), "d2h_gbs": timed(d2h), "duplex_gbs_per_direction": timed(both)}
    del d_a, d_b
    return out


def run_wd_device_inputs(args, torch, binding, cfg, recon, nrhs, dev, local, kernel):
    """--device-inputs: a quick timing-only run for kernel work (sweeps, ncu captures): links and spinors are
    N(0,1)/2 numbers drawn on the device (the kernels' cost is data independent), no e2e leg, no oracle leg.
    Its line says data = "device-random (timing only)" and is never a bench record."""
    V = fields.volume(cfg.dims)
    prec = 16 if args.half else cfg.precision
    tdt = {16: torch.float16, 32: torch.float32, 64: torch.float64}[prec]
    cdt = torch.float64 if prec == 64 else torch.float32
    stream = torch.cuda.Stream(device=dev)
    nbuf = 2 if nrhs > 1 else NBUF
    with torch.cuda.stream(stream):
        g = torch.Generator(device=dev).manual_seed(cfg.seed)
        Lx, Ly, Lz, Lt = cfg.dims
        u_dev = torch.randn((4, Lt, Lz, Ly, Lx, 3, 3, 2), dtype=cdt, device=dev, generator=g) * 0.5
        if recon == 8:  # the 8-real format needs |a2|^2 + |a3|^2 <= 1: scale the random numbers down
            u_dev *= 0.5
        op = binding.WilsonDirac(cfg.dims, u_dev, prec, recon, stream=stream.cuda_stream, kernel=kernel)
        if prec == 16:
            ins = [torch.empty(op.native_numel(nrhs), dtype=tdt, device=dev) for _ in range(nbuf)]
            for b in ins:
                c = torch.randn((nrhs, Lt, Lz, Ly, Lx, 4, 3, 2), dtype=torch.float32, device=dev, generator=g)
                op.pack(b, c, nrhs)
            del c
        else:
            ins = [torch.randn(op.native_numel(nrhs), dtype=tdt, device=dev, generator=g) for _ in range(nbuf)]
        outs = [torch.empty(op.native_numel(nrhs), dtype=tdt, device=dev) for _ in range(nbuf)]
    stream.synchronize()
    del u_dev
    aps = args.applies_per_step
    for _ in range(max(args.warmup, 3) * aps):
        op.apply(outs[0], ins[0], cfg.mass, nrhs)
    torch.cuda.synchronize()
    graph = None
    if args.graph:  # the step captured once in a CUDA graph and replayed: takes the host's launch rate out of the number
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            for i in range(aps):
                op.apply(outs[i % nbuf], ins[i % nbuf], cfg.mass, nrhs)
        with torch.cuda.stream(stream):
            graph.replay()
        torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        ev0.record(stream)
        if graph is not None:
            with torch.cuda.stream(stream):
                for _ in range(args.steps):
                    graph.replay()
        else:
            for i in range(args.steps * aps):
                op.apply(outs[i % nbuf], ins[i % nbuf], cfg.mass, nrhs)
        ev1.record(stream)
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / (args.steps * aps)
    bytes_per_launch = compulsory_bytes_per_site(prec, recon, nrhs) * V
    peak, peak_src = measured_peak()
    achieved = bytes_per_launch / (ms * 1e-3) / 1e9
    line = {"metric": METRIC, "value": FLOPS_PER_SITE * V * nrhs / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "data": "device-random (timing only)",
            "config": {"workload": cfg.name, "recon": recon, "nrhs": nrhs, "kernel": args.kernel, "applies_per_step": aps},
            "us_per_apply": ms * 1e3, "clocks": clocks.summary(),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "peak_source": peak_src, "kernel": op.selected_kernel(nrhs)}}
    print(json.dumps(line), flush=True)
    op.close()
    return line

def run_wd(args):
    import torch
    from paper_0912_2186_b200 import binding, build

    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    build.build()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = fields.CONFIGS[args.workload]
    recon = args.recon
    nrhs = args.nrhs if args.nrhs else cfg.nrhs
    V = fields.volume(cfg.dims)
    tdt = torch.float32 if cfg.precision == 32 else torch.float64
    kernel = {"auto": binding.WD_KERNEL_AUTO, "site": binding.WD_KERNEL_SITE,
              "stage": binding.WD_KERNEL_STAGE}[args.kernel]

    # ---- synthetic inputs (each rank its own replica: seeds shifted by rank) -------------------
    cfg_r = rank_config(cfg, recon, nrhs, rank)
    if args.device_inputs:
        return run_wd_device_inputs(args, torch, binding, cfg, recon, nrhs, dev, local, kernel)
    U, psi = fields.make_fields(cfg_r)
    want_secondary = (world == 1 and args.workload == "c3_32x64_fp32" and not args.no_secondary and args.nrhs is None
                      and not args.temporal_gauge and args.kernel == "auto")
    if args.temporal_gauge:
        U, _ = fields.temporal_gauge(U, cfg.precision)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        u_dev = torch.from_numpy(U).to(dev)
        op = binding.WilsonDirac(cfg.dims, u_dev, cfg.precision, recon, stream=stream.cuda_stream, kernel=kernel)
        if args.temporal_gauge:
            op.set_temporal_gauge(True)
        canon = torch.from_numpy(psi).to(dev)
        ins = [torch.empty(op.native_numel(nrhs), dtype=tdt, device=dev) for _ in range(NBUF)]
        outs = [torch.empty(op.native_numel(nrhs), dtype=tdt, device=dev) for _ in range(NBUF)]
        op.pack(ins[0], canon, nrhs)
        for b in range(1, NBUF):  # distinct inputs: scaled copies of the packed field
            torch.mul(ins[0], 1.0 + 0.25 * b, out=ins[b])
    stream.synchronize()
    del u_dev, canon

    aps = args.applies_per_step

    def step():
        for i in range(aps):
            op.apply(outs[i % NBUF], ins[i % NBUF], cfg.mass, nrhs)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ---------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    n0 = binding.wd_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        ev0.record(stream)
        for _ in range(args.steps):
            step()
        ev1.record(stream)
        barrier()
    launches = binding.wd_launch_count() - n0
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
    applies = args.steps * aps
    flops_per_apply = FLOPS_PER_SITE * V * nrhs
    value = whole_job_gflops(world, applies, flops_per_apply, ms)
    launch_ms = ms / applies
    bytes_per_launch = compulsory_bytes_per_site(cfg.precision, recon, nrhs) * V
    if args.temporal_gauge:  # unit t-links are not read except on the last time slice
        bytes_per_launch -= recon * (4 if cfg.precision == 32 else 8) * (V - V // cfg.dims[3])
    peak, peak_src = measured_peak()
    achieved = bytes_per_launch / (launch_ms * 1e-3) / 1e9

    # ---- end to end through wd_apply_host (pinned host buffers, copies inside the timed region) -
    e2e_applies = max(2, min(args.steps, 5))
    h_in = torch.from_numpy(psi).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    for _ in range(2):
        op.apply_host(h_out, h_in, cfg.mass, nrhs)
    barrier()
    t0 = time.perf_counter()  # wd_apply_host synchronises its stream before returning: wall clock is exact
    for _ in range(e2e_applies):
        op.apply_host(h_out, h_in, cfg.mass, nrhs)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms = max_over_ranks(e2e_ms, world, dev)
    e2e_value = whole_job_gflops(world, e2e_applies, flops_per_apply, e2e_ms)
    field_bytes = nrhs * V * 24 * (4 if cfg.precision == 32 else 8)
    # the e2e roofline: the field must cross PCIe once in each direction; with both directions busy the bound is
    # field_bytes / (duplex rate per direction), measured here with plain copies of the same pinned buffers
    pcie = pcie_peaks(torch, dev, h_in, h_out) if world == 1 else None

    secondary = None
    next_rows = None
    if want_secondary:
        # free the headline's device buffers first (24 RHS need 2 x 2 x 4.8 GB)
        del ins, outs, h_in, h_out
        torch.cuda.empty_cache()
        secondary = [
            secondary_leg(binding, torch, dev, stream, local, "c4_32x64_fp32_24rhs", U, 18, 24, 2, 10),
            secondary_leg(binding, torch, dev, stream, local, "c3_32x64_fp64", U, 18, 1, 2, 25),
            # configs 3 and 4 "18 (primary; also report 12)"
            secondary_leg(binding, torch, dev, stream, local, "c4_32x64_fp32_24rhs", U, 12, 24, 2, 10),
            secondary_leg(binding, torch, dev, stream, local, "c3_32x64_fp64", U, 12, 1, 2, 25),
            # storage variants of the paper's Table 2: 12 and 8 reals per link, half-precision storage
            secondary_leg(binding, torch, dev, stream, local, "c3_32x64_fp32", U, 12, 1, 2, 50),
            secondary_leg(binding, torch, dev, stream, local, "c3_32x64_fp32", U, 8, 1, 2, 50),
            secondary_leg(binding, torch, dev, stream, local, "c3_32x64_fp32", U, 12, 1, 2, 50, storage=16),
        ]
        # configs[2] (24^3 x 64, 12-real links: Lx not a power of two) and the paper's own set-up shape on it: N_v = 20
        # right-hand sides on a 24^3 x 64 volume
        U2, _ = fields.make_fields(fields.CONFIGS["c2_24x64_fp32_r12"], nrhs=1)
        secondary += [
            secondary_leg(binding, torch, dev, stream, local, "c2_24x64_fp32_r12", U2, 12, 1, 2, 50),
            secondary_leg(binding, torch, dev, stream, local, "c2_24x64_fp32_r12", U2, 12, 20, 2, 10),
        ]
        del U2
        next_rows = next_rows_legs(binding, torch, dev, stream, local, "c3_32x64_fp32", U, 18)

    line = None
    if rank == 0:
        cpu = oracle_rate(cfg_r, U, psi) if (world == 1 and not args.no_cpu_baseline) else None
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if cfg.precision == 32 else "f64",
            "data": "synthetic",
            "config": {"workload": cfg.name, "dims": list(cfg.dims), "links": cfg.links, "recon": recon, "nrhs": nrhs,
                       "mass": cfg.mass, "kernel": args.kernel, "temporal_gauge": bool(args.temporal_gauge), "applies_per_step": aps,
                       "rotating_buffers": NBUF, "flops_per_site": FLOPS_PER_SITE,
                       "gflops_at_1320_per_site": value * 1320.0 / FLOPS_PER_SITE,
                       "l2": "inputs larger than L2 (gauge + rotating spinor fields), no flush",
                       "parallelism": "independent replicas, no collective" if world > 1 else "single GPU"},
            "us_per_apply": launch_ms * 1e3,
            "clocks": clocks.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": field_bytes * aps,
                    "d2h_bytes_per_step": field_bytes * aps, "applies_timed": e2e_applies,
                    "ms_per_apply": e2e_ms / e2e_applies,
                    "pcie": pcie,
                    "roofline": None if pcie is None else {
                        "bound": "pcie", "unit": "GB/s per direction", "peak": pcie["duplex_gbs_per_direction"],
                        "achieved": field_bytes / (e2e_ms / e2e_applies * 1e-3) / 1e9,
                        "frac": field_bytes / (e2e_ms / e2e_applies * 1e-3) / 1e9 / pcie["duplex_gbs_per_direction"],
                        "frac_of_one_direction_alone": field_bytes / (e2e_ms / e2e_applies * 1e-3) / 1e9 / min(pcie["h2d_gbs"], pcie["d2h_gbs"])},
                    "note": "wd_apply_host per apply: H2D + pack + apply + unpack + D2H + sync; bytes are per "
                            "100-apply step"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": ncu_traffic(cfg.name, recon), "peak_source": peak_src,
                         "bytes_per_launch": bytes_per_launch,
                         "kernel": "wd dslash, " + op.selected_kernel(nrhs) + " kernel" + (" (multi-RHS member)" if nrhs > 1 and op.selected_kernel(nrhs) == "stage" else "")},
        }
        if cpu is not None:
            line["cpu_baseline"] = cpu
        if secondary is not None:
            line["secondary"] = secondary
            line["next_rows"] = next_rows
        print(json.dumps(line), flush=True)
    op.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return line


def run_schur(args):
    """--op schur: the even-odd preconditioned operator on the same
    lattice: a step = APPLIES wd_apply_schur calls (two kernel launches each) on half fields resident in HBM.
    Flops per even site: 2 x 1320 (two hopping blocks) + 48; algorithmic bytes per even site: both launches
    read every link once (2 x 4*recon*w x 2 sites); spinors: in, tmp written, tmp read, in again, out = 5 x 24*w."""
    import torch
    from paper_0912_2186_b200 import binding, build
    rank, local, world = dist_env()
    if world > 1:
        raise SystemExit("bench.py --op schur: single GPU only")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    build.build()
    dev = torch.device("cuda", local)
    torch.cuda.set_device(local)
    cfg = fields.CONFIGS[args.workload]
    recon, nrhs = args.recon, (args.nrhs or cfg.nrhs)  # --nrhs N: N right-hand sides per batched launch
    V = fields.volume(cfg.dims)
    if args.half and cfg.precision != 32:
        raise SystemExit("bench.py --op schur --half: half storage has float32 canonical fields; use an fp32 workload")
    prec = 16 if args.half else cfg.precision  # --half: binary16 storage, fp32 arithmetic (row f4 on the operator of row f1)
    w = {16: 2, 32: 4, 64: 8}[prec]
    tdt = {16: torch.float16, 32: torch.float32, 64: torch.float64}[prec]
    U, psi = fields.make_fields(rank_config(cfg, recon, nrhs, rank))
    if args.temporal_gauge:  # Fig. 4 "GF": unit t-links below the last slice, skipped by the kernel
        if prec == 16 or recon == 8:
            raise SystemExit("bench.py --op schur --temporal-gauge: 18- or 12-real links in fp32 / fp64")
        U, _ = fields.temporal_gauge(U, cfg.precision)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        u_dev = torch.from_numpy(U).to(dev)
        op = binding.WilsonDirac(cfg.dims, u_dev, prec, recon, stream=stream.cuda_stream)
        if args.temporal_gauge:
            op.set_temporal_gauge(True)
        canon = torch.from_numpy(psi).to(dev)
        n = op.half_numel(nrhs)
        ins = [torch.empty(n, dtype=tdt, device=dev) for _ in range(NBUF)]
        outs = [torch.empty(n, dtype=tdt, device=dev) for _ in range(NBUF)]
        tmp = torch.empty(n, dtype=tdt, device=dev)
        for b in range(NBUF):  # (half storage holds ratios and scales: every input is packed, not scaled in place)
            op.pack_parity(ins[b], canon * (1.0 + 0.25 * b), nrhs, 0)
    stream.synchronize()
    aps = args.applies_per_step

    def step():
        for i in range(aps):
            op.apply_schur(outs[i % NBUF], ins[i % NBUF], tmp, cfg.mass, 0, nrhs)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    n0 = binding.wd_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        ev0.record(stream)
        for _ in range(args.steps):
            step()
        ev1.record(stream)
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1)
    applies = args.steps * aps
    flops = (2 * 1320 + 48) * (V // 2) * nrhs
    spinor_b = 52 if prec == 16 else 24 * w  # half storage: 24 binary16 ratios + a float32 scale per site
    bytes_per_apply = (V // 2) * (2 * 2 * 4 * recon * w + nrhs * 5 * spinor_b)
    if args.temporal_gauge:  # the t-links are read on one slice of Lt only (forward on the last, backward on the first)
        bytes_per_apply -= (V // 2) * 2 * 2 * recon * w * (cfg.dims[3] - 1) // cfg.dims[3]
    peak, peak_src = measured_peak()
    achieved = bytes_per_apply * applies / (ms * 1e-3) / 1e9
    line = {"metric": "wilson_schur_gflops", "value": applies * flops / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": {16: "f32 arithmetic on f16 storage", 32: "f32", 64: "f64"}[prec], "data": "synthetic",
            "config": {"workload": cfg.name, "op": "even-odd preconditioned operator (2 launches per apply)",
                       "dims": list(cfg.dims), "recon": recon, "nrhs": nrhs, "mass": cfg.mass, "applies_per_step": aps,
                       "temporal_gauge": bool(args.temporal_gauge), "flops_per_even_site": 2 * 1320 + 48,
                       "l2": "inputs larger than L2 (gauge + rotating half fields), no flush"},
            "us_per_apply": ms / applies * 1e3, "clocks": clocks.summary(),
            "gpu_launches": int(binding.wd_launch_count() - n0),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src, "bytes_per_launch": bytes_per_apply // 2,
                         "kernel": "wd dslash_eo (site-style half-lattice kernel)"}}
    print(json.dumps(line), flush=True)
    op.close()


def run_cgnr(args):
    """--op cgnr | bicgstab: the Krylov solvers on the even-odd preconditioned operator (
    PAPER.md:116, Table 2): a step = one solver call of ITER iterations (tol = 0: no host synchronisation inside).
    Per iteration and even site: two operator applications (2 x (2 x 1320 + 48) flops, 2 x Schur-apply bytes) plus
    the BLAS-1 kernels: CGNR 288 flops / 8 spinor passes (the two norms come out of the matvec epilogue; x += alpha p rides
    on the p update), BiCGstab
    672 flops / 15 spinor passes (<rhat, v>, <t, s>, |t|^2 come out of the matvec epilogues, <rhat, r> out of the x / r update), GCR(8) ~1150 flops / 22.25 passes averaged over a cycle
    (direction j of a cycle: j + 1 passes for its inner products with the earlier q_i, 2j + 5 for the orthogonalisation that
    also takes <q_j, r> and |q_j|^2, 6 for the x / r update)."""
    import torch
    from paper_0912_2186_b200 import binding, build
    rank, local, world = dist_env()
    if world > 1:
        raise SystemExit("bench.py --op cgnr: single GPU only")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    build.build()
    dev = torch.device("cuda", local)
    torch.cuda.set_device(local)
    cfg = fields.CONFIGS[args.workload]
    recon = args.recon
    V = fields.volume(cfg.dims)
    w = 4 if cfg.precision == 32 else 8
    tdt = torch.float32 if cfg.precision == 32 else torch.float64
    U, psi = fields.make_fields(rank_config(cfg, recon, 1, rank), nrhs=1)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        u_dev = torch.from_numpy(U).to(dev)
        op = binding.WilsonDirac(cfg.dims, u_dev, cfg.precision, recon, stream=stream.cuda_stream)
        canon = torch.from_numpy(psi).to(dev)
        n = op.half_numel(1)
        b = torch.empty(n, dtype=tdt, device=dev)
        x = torch.empty(n, dtype=tdt, device=dev)
        op.pack_parity(b, canon, 1, 0)
    stream.synchronize()
    iters = args.applies_per_step
    nblk = args.nrhs or 1   # --op cgnr --nrhs N: the block solve (N right-hand sides in lock step, batched operator applies)
    if nblk > 1:
        if args.op != "cgnr":
            raise SystemExit("bench.py: --nrhs with --op is the block CGNR only")
        with torch.cuda.stream(stream):
            g = torch.Generator(device=dev).manual_seed(cfg.seed + 1000)
            b = torch.randn(n * nblk, dtype=tdt, device=dev, generator=g)   # native half fields: any values are valid vectors
            x = torch.empty_like(b)
        stream.synchronize()
    solve = {"cgnr": op.cgnr_schur, "bicgstab": op.bicgstab_schur, "gcr": op.gcr_schur}[args.op]
    if nblk > 1:
        solve = lambda xx, bb, mass, parity, it: op.cgnr_schur_block(xx, bb, mass, parity, nblk, it)
    # BLAS-1 flops / spinor passes per iteration and even site; matvecs per iteration.  GCR(8): averages over a cycle
    # (direction j: 3j + 12 passes for j >= 1, 10 for j = 0)
    blas_flops, blas_passes, nmv = {"cgnr": (288, 8, 2), "bicgstab": (672, 15, 2), "gcr": (1150, 22.25, 1)}[args.op]
    for _ in range(max(args.warmup, 3)):
        solve(x, b, cfg.mass, 0, iters)
    torch.cuda.synchronize()
    n0 = binding.wd_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        ev0.record(stream)
        for _ in range(args.steps):
            done, hist = solve(x, b, cfg.mass, 0, iters)
        ev1.record(stream)
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1)
    total_iters = args.steps * iters
    flops_it = (nmv * (2 * 1320 + 48) + blas_flops) * (V // 2) * nblk
    # (block solve: the links are read once per batched launch, the spinor passes scale with the right-hand sides)
    bytes_it = (V // 2) * (nmv * (2 * 2 * 4 * recon * w + nblk * 5 * 24 * w) + nblk * blas_passes * 24 * w)
    if nblk > 1:
        hist = hist[0]
    peak, peak_src = measured_peak()
    achieved = bytes_it * total_iters / (ms * 1e-3) / 1e9
    line = {"metric": "wilson_%s_gflops" % args.op, "value": total_iters * flops_it / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if cfg.precision == 32 else "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "op": {"cgnr": "CGNR", "bicgstab": "BiCGstab", "gcr": "GCR(8)"}[args.op] + " on the even-odd preconditioned operator", "dims": list(cfg.dims),
                       "recon": recon, "mass": cfg.mass, "iterations_per_step": iters, "nrhs": nblk,
                       "relative_residual_after_step": hist[-1],
                       "l2": "inputs larger than L2 (gauge + five half fields), no flush"},
            "us_per_iteration": ms / total_iters * 1e3, "clocks": clocks.summary(),
            "gpu_launches": int(binding.wd_launch_count() - n0),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src, "bytes_per_iteration": bytes_it,
                         "kernel": "wd dslash_eo + fused BLAS-1"}}
    print(json.dumps(line), flush=True)
    op.close()


def run_transfer(args):
    """--op transfer: the multigrid transfer operators (eq. (2.7)) with N_v = 20 vectors
     on the workload's lattice: a step = one wd_restrict + one wd_prolong; the block Gram-Schmidt is
    timed once.  Algorithmic bytes: restrict reads N_v + 1 fields, prolong reads N_v and writes 1."""
    import torch
    from paper_0912_2186_b200 import binding, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    build.build()
    cfg = fields.CONFIGS[args.workload]
    nv = 20
    V = fields.volume(cfg.dims)
    w = 4 if cfg.precision == 32 else 8
    tdt = torch.float32 if cfg.precision == 32 else torch.float64
    lat = binding.wd_create_lattice(cfg.dims)
    n = binding.wd_spinor_bytes(lat, 1, cfg.precision) // w
    g = torch.Generator(device="cuda").manual_seed(cfg.seed)
    basis = torch.randn(nv * n, dtype=tdt, device="cuda", generator=g)   # native layout: any values are valid vectors
    psi = torch.randn(n, dtype=tdt, device="cuda", generator=g)
    out = torch.empty_like(psi)
    coarse = torch.empty(binding.wd_coarse_reals(lat, nv), dtype=tdt, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    ev[0].record()
    binding.wd_block_orthonormalise(lat, basis, nv, cfg.precision)
    ev[1].record()
    for _ in range(max(args.warmup, 3)):
        binding.wd_restrict(lat, coarse, basis, psi, nv, cfg.precision)
        binding.wd_prolong(lat, out, basis, coarse, nv, cfg.precision)
    torch.cuda.synchronize()
    n0 = binding.wd_launch_count()
    with ClockSampler(0) as clocks:
        ev[2].record()
        for _ in range(args.steps):
            binding.wd_restrict(lat, coarse, basis, psi, nv, cfg.precision)
            binding.wd_prolong(lat, out, basis, coarse, nv, cfg.precision)
        ev[3].record()
        torch.cuda.synchronize()
    ms = ev[2].elapsed_time(ev[3]) / args.steps
    bytes_step = (2 * nv + 2) * V * 24 * w
    flops_step = 2 * nv * V * 12 * 8   # one complex multiply-add per component, vector and direction
    peak, peak_src = measured_peak()
    achieved = bytes_step / (ms * 1e-3) / 1e9
    line = {"metric": "mg_transfer_gflops", "value": flops_step / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if cfg.precision == 32 else "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "op": "restrict + prolong, N_v = 20, 4^4 blocks x 2 chiralities",
                       "dims": list(cfg.dims), "block_gram_schmidt_ms": ev[0].elapsed_time(ev[1]),
                       "l2": "basis (20 fields) larger than L2, no flush"},
            "clocks": clocks.summary(), "gpu_launches": int(binding.wd_launch_count() - n0),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src, "bytes_per_step": bytes_step,
                         "kernel": "wd restrict_kernel + prolong_kernel"}}
    print(json.dumps(line), flush=True)
    binding.wd_destroy(lat)


def run_coarse(args):
    """--op coarse: the explicit coarse operator Dhat = P^dagger D P (row f3) with N_v = 20 on the
    workload's lattice: wd_build_coarse timed once, then a step = APPLIES wd_apply_coarse calls.  Per coarse site the apply
    streams nine (2 N_v)^2 complex matrices once: algorithmic bytes = 9 n^2 2w + (nrhs) (1 + 1) n 2w, flops = 9 n^2 8 nrhs."""
    import torch
    from paper_0912_2186_b200 import binding, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    build.build()
    cfg = fields.CONFIGS[args.workload]
    nv, nrhs = 20, (args.nrhs or 1)
    n = 2 * nv
    V = fields.volume(cfg.dims)
    nb = V // 256
    w = 4 if cfg.precision == 32 else 8
    tdt = torch.float32 if cfg.precision == 32 else torch.float64
    g = torch.Generator(device="cuda").manual_seed(cfg.seed)
    Lx, Ly, Lz, Lt = cfg.dims
    stream = torch.cuda.current_stream()
    u_dev = torch.randn((4, Lt, Lz, Ly, Lx, 3, 3, 2), dtype=tdt, device="cuda", generator=g) * 0.5   # cost is data independent
    op = binding.WilsonDirac(cfg.dims, u_dev, cfg.precision, 18, stream=stream.cuda_stream)
    del u_dev
    basis = torch.randn(op.native_numel(nv), dtype=tdt, device="cuda", generator=g)
    binding.wd_block_orthonormalise(op.lat, basis, nv, cfg.precision, stream.cuda_stream)
    ns = binding.wd_coarse_stencil_reals(op.lat, nv)
    S = torch.empty(ns, dtype=tdt, device="cuda")
    scratch = torch.empty(ns, dtype=tdt, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    binding.wd_build_coarse(op.gauge, S, scratch, basis, cfg.mass, cfg.dims, nv, cfg.precision)   # warm-up
    ev[0].record()
    binding.wd_build_coarse(op.gauge, S, scratch, basis, cfg.mass, cfg.dims, nv, cfg.precision)
    ev[1].record()
    del scratch
    cin = [torch.randn(nrhs * nb * n * 2, dtype=tdt, device="cuda", generator=g) for _ in range(2)]
    cout = [torch.empty_like(cin[0]) for _ in range(2)]
    aps = args.applies_per_step
    for i in range(max(args.warmup, 3) * 3):
        binding.wd_apply_coarse(op.lat, cout[i % 2], cin[i % 2], S, nv, nrhs, cfg.precision, stream.cuda_stream)
    torch.cuda.synchronize()
    n0 = binding.wd_launch_count()
    with ClockSampler(0) as clocks:
        ev[2].record()
        for i in range(args.steps * aps):
            binding.wd_apply_coarse(op.lat, cout[i % 2], cin[i % 2], S, nv, nrhs, cfg.precision, stream.cuda_stream)
        ev[3].record()
        torch.cuda.synchronize()
    ms = ev[2].elapsed_time(ev[3]) / (args.steps * aps)
    bytes_apply = nb * (9 * n * n * 2 * w + nrhs * 2 * n * 2 * w)
    flops_apply = nb * 9 * n * n * 8 * nrhs
    peak, peak_src = measured_peak()
    achieved = bytes_apply / (ms * 1e-3) / 1e9
    build_ms = ev[0].elapsed_time(ev[1])
    build_flops = V * 9 * nv * nv * 4 * 6 * 8   # the W^dag H contractions only (96 complex multiply-adds per site, pair, term)
    line = {"metric": "mg_coarse_apply_gflops", "value": flops_apply / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms * aps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if cfg.precision == 32 else "f64",
            "data": "device-random links and vectors (cost is data independent)",
            "config": {"workload": cfg.name, "op": "coarse operator apply, 9-point stencil of (2 N_v)^2 complex blocks",
                       "dims": list(cfg.dims), "coarse_dims": [d // 4 for d in cfg.dims], "nv": nv, "nrhs": nrhs,
                       "applies_per_step": aps, "build_ms": build_ms, "build_gflops": build_flops / (build_ms * 1e-3) / 1e9,
                       "stencil_MB": ns * w / 1e6, "l2": "stencil larger than L2, no flush"},
            "us_per_apply": ms * 1e3, "clocks": clocks.summary(), "gpu_launches": int(binding.wd_launch_count() - n0),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "peak_source": peak_src, "bytes_per_launch": bytes_apply,
                         "kernel": "wd coarse_apply_kernel"}}
    print(json.dumps(line), flush=True)
    op.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c3_32x64_fp32", choices=sorted(fields.CONFIGS))
    ap.add_argument("--kernel", default="auto", choices=["auto", "site", "stage"])
    ap.add_argument("--recon", type=int, default=None, choices=[18, 12, 8])
    ap.add_argument("--impl", default="wd", choices=["wd", "reference"])
    ap.add_argument("--op", default="full", choices=["full", "schur", "cgnr", "bicgstab", "gcr", "transfer", "coarse"],
                    help="full = D of eq. (2.2) (the headline); schur = even-odd preconditioned operator (row f1); cgnr = CG on its normal equations (row f2, --applies-per-step = iterations)")
    ap.add_argument("--nrhs", type=int, default=None,
                    help="override the workload's number of right-hand sides (e.g. 20 = the paper's N_v, PAPER.md:124)")
    ap.add_argument("--temporal-gauge", action="store_true",
                    help="gauge-fix the synthetic links to temporal gauge and let the kernel skip the unit t-links "
                         "(PAPER.md:157; row f4); algorithmic bytes then count 3 links + the last slice's t-links")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--device-inputs", action="store_true",
                    help="timing-only quick mode for kernel work: device-drawn random links and spinors, no e2e/oracle legs")
    ap.add_argument("--graph", action="store_true",
                    help="(with --device-inputs) capture the step of APPLIES wd_apply launches in a CUDA graph and time its replays")
    ap.add_argument("--half", action="store_true", help="(with --device-inputs) half-precision storage, fp32 arithmetic")
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the short legs for configs[4] (24 RHS) and configs[3] in fp64 that the default run adds")
    ap.add_argument("--applies-per-step", type=int, default=APPLIES_PER_STEP,
                    help="wd_apply calls per step (default 100 = configs[3]; lower it only for profiling)")
    args = ap.parse_args()
    if args.recon is None:
        args.recon = fields.CONFIGS[args.workload].recon
    if args.impl == "reference":
        run_reference(args)
    elif args.op == "schur":
        run_schur(args)
    elif args.op == "transfer":
        run_transfer(args)
    elif args.op == "coarse":
        run_coarse(args)
    elif args.op in ("cgnr", "bicgstab", "gcr"):
        run_cgnr(args)
    else:
        run_wd(args)


if __name__ == "__main__":
    main()
