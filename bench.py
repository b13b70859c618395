#!/usr/bin/env python
"""bench.py -- wall-RPY mobility matvec throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 1..5] [--prec f32|f64] [--variant wall|free] [--no-extra]

A "step" is one pass of the whole hot path (prepack -> all-pairs -> finalise, i.e. one call of
rpy_wall_matvec) over one synthetic workload.  Default workload: BASELINE.json configs[2]
("config 3": 4,096 rigid 42-blob shells = 172,032 blobs, wall-corrected, fp32 path with fp64
accumulation) -- the configuration north_star quotes its target on ("N >= 1.7e5 blobs").
Prints ONE JSON line on stdout (rank 0); progress goes to stderr.

Metric: G blob-pairs/s = N^2 / t / 1e9 (ordered pairs, i = j included; for k right-hand sides the
pair-RHS products N^2 k / t are in "pair_rhs_gps").

  value     device-resident inputs, CUDA-event time of K steps (L2 flushed between steps)
  e2e       same metric through the C-ABI host-buffer call (pinned host tensors; H2D of
            positions+forces and D2H of velocities inside the timed region)
  roofline  ALU bound: algorithmic flops of the all-pairs kernel / its CUDA-event duration,
            against 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (fp64: 64 lanes), DESIGN.md
  cpu_baseline  the float64 oracle (oracle/) on this box's host cores, on a bounded row sample
  parity    rel-L2 and per-blob maximum error of the timed step's result against that oracle sample
            (exit status 3 when outside north_star's tolerance)
  value_f64, roofline_f64, parity_f64   the fp64 path on the same workload (the paper's precision)

N > 1 (torchrun): the work is sharded across ranks -- one right-hand side: each rank takes 1/N of the
unordered tile pairs of the symmetric kernel and one NCCL all-reduce adds the partial u; several
right-hand sides: each rank takes a slice of target rows and one all-gather collects u.  No
collective inside the kernels; strong scaling.
--impl reference: times the oracle (this tier has no reference implementation to install).
"""
from __future__ import annotations

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

METRIC = "wall_rpy_matvec_blob_pairs_per_s"
UNIT = "G blob-pairs/s"

# Work of the all-pairs kernel per ordered pair: FP-pipe lane operations
# (one per FFMA/FMUL/FADD lane; a packed FFMA2 counts two) and flops (FMA = 2, MUL/ADD = 1) that the
# kernel EXECUTES on the every-pair path, measured with ncu (per-opcode "Thread Instructions
# Executed" of the source page / N^2, profiles/*_allpairs_*.md) and equal to the count of the
# expression tree in csrc/rpy_math.cuh.  k right-hand sides: geometry part + per-RHS apply part.
# The fp64 path executes the same tree plus five DFMA-pipe operations per reciprocal square root
# (MUFU.RSQ64H seed + one cubic Newton step): two roots for the wall tensor, one for free space.
WORK = {
    # (prec, variant): (lane_ops_geom, lane_ops_per_rhs, flop_geom, flop_per_rhs)
    ("f32", "wall"): (44, 10, 70, 18),
    ("f32", "free"): (12, 10, 19, 18),
    ("f64", "wall"): (52, 10, 82, 18),
    ("f64", "free"): (17, 10, 24, 18),
}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel come from the committed
# `ncu --set full` captures: profiles/dram_traffic.csv lists (config, prec, variant, kernel, bytes read,
# bytes written, the summary file the row was copied from).  Algorithmic bytes of the cfg-3 launch:
# 172,032 x 24 B of records read + 16 partial slices x 172,032 x 24 B written/accumulated = 70 MB (mostly
# L2-resident); the point of the figure is that DRAM traffic is ~1e-3 of what an HBM-bound kernel of this
# duration would move.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "dram_traffic.csv")
TOL = {"f64": 1e-12, "f32": 1e-5}            # north_star: rel-L2 vs the oracle
PARITY_ROWS = 2048                           # seeded target rows for configs 3-5 (all rows for 1-2)


def ncu_traffic(config: int, prec: str, variant: str):
    """(bytes per launch, source file) of the latest committed capture for this case, else (None, None)."""
    try:
        import csv
        with open(TRAFFIC_CSV) as f:
            rows = [r for r in csv.DictReader(f)
                    if int(r["config"]) == config and r["prec"] == prec and r["variant"] == variant]
        if not rows:
            return None, None
        r = rows[-1]
        return float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]), r["source"]
    except Exception:
        return None, None
SM_COUNT = 148
LANES = {"f32": 128, "f64": 64}
SM_MAX_GHZ = 1.965


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def work_per_pair(prec: str, variant: str, k: int, symmetric: bool = False):
    """(FP-pipe lane operations, flops) per ORDERED pair.  The symmetric kernel builds the geometry
    and the coefficients once per unordered pair and applies them twice (M_ij and M_ij^T)."""
    ig, ir, fg, fr = WORK[(prec, variant)]
    if symmetric:
        return (ig + 2 * ir * k) / 2, (fg + 2 * fr * k) / 2
    return ig + ir * k, fg + fr * k


def peak_tflops(prec: str) -> float:
    return SM_COUNT * LANES[prec] * 2 * SM_MAX_GHZ * 1e9 / 1e12


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock, power and throttle reasons during the timed region (NVML)."""

    def __init__(self, index: int, period: float = 0.1):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.sm_max, self.power = None, []
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # pragma: no cover
            log(f"[bench] NVML unavailable: {e}")
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self) -> dict:
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unsampled"]}
        s = sorted(self.samples)
        load = [x for x in s if x >= 0.5 * s[-1]] or s
        return {"sm_mhz": float(load[len(load) // 2]), "sm_max_mhz": float(self.sm_max or 0),
                "reasons": sorted(self.reasons), "samples": len(s),
                "power_w_max": max(self.power) if self.power else None}


# ------------------------------------------------------------------------------- oracle leg
def oracle_sample(wl, variant: str, prec: str, budget_s: float, max_rows: int = 1 << 16):
    """Times the oracle, as it stands, on a row sample sized for ~budget_s of CPU work.
    Returns (G pairs/s, cores, description, seconds)."""
    import oracle
    from paper_1602_02170_b200 import workloads
    ov = oracle.WALL if variant == "wall" else oracle.FREE
    npdt = np.float32 if prec == "f32" else np.float64
    pos = wl.pos.astype(npdt).astype(np.float64)
    force = wl.force.astype(npdt).astype(np.float64)
    n, k = wl.n_blobs, wl.n_rhs
    cores = oracle.num_threads()
    probe_rows = workloads.sample_rows(n, min(n, 4 * cores), seed=7)
    t0 = time.perf_counter()
    oracle.matvec(ov, pos, force, wl.a, wl.eta, rows=probe_rows)
    t_probe = time.perf_counter() - t0
    per_row = t_probe / len(probe_rows)
    n_rows = int(max(cores, min(max_rows, n, budget_s / max(per_row, 1e-9))))
    rows = workloads.sample_rows(n, n_rows, seed=12345)
    t0 = time.perf_counter()
    ref = oracle.matvec(ov, pos, force, wl.a, wl.eta, rows=rows)
    t = time.perf_counter() - t0
    gps = len(rows) * n / t / 1e9
    desc = f"{len(rows)} seeded target rows x all {n} sources, k={k}, {variant}, float64"
    return gps, cores, desc, t, len(rows), rows, ref


def parity_of(u_gpu, ref, rows, prec: str) -> dict:
    """rel-L2 over all sampled components and the per-blob maximum max_i |du_i| / |u_i| of the CUDA result
    `u_gpu` [k, N, 3] against the oracle's `ref` [k, len(rows), 3] (north_star's two figures)."""
    u = u_gpu.detach().cpu().numpy().astype(np.float64)
    u = u.reshape(-1, u.shape[-2], 3)[:, rows, :]
    ref = ref.reshape(u.shape)
    rel = float(np.linalg.norm((u - ref).ravel()) / np.linalg.norm(ref.ravel()))
    num = np.linalg.norm(u - ref, axis=-1); den = np.linalg.norm(ref, axis=-1)
    pb = float((num / np.maximum(den, 1e-300)).max())
    return {"rel_l2": rel, "per_blob_max": pb, "rows": int(len(rows)), "tol": TOL[prec],
            "ok": bool(np.isfinite(u).all() and rel <= TOL[prec])}


def oracle_parity(wl, variant: str, prec: str, u_gpu, n_rows: int = PARITY_ROWS) -> dict:
    """The oracle on a seeded row sample (all rows when N <= 20,000) against the CUDA result of the timed step."""
    import oracle
    from paper_1602_02170_b200 import workloads
    ov = oracle.WALL if variant == "wall" else oracle.FREE
    npdt = np.float32 if prec == "f32" else np.float64
    pos = wl.pos.astype(npdt).astype(np.float64)          # the values that cross the boundary (reading A8)
    force = wl.force.astype(npdt).astype(np.float64)
    n = wl.n_blobs
    rows = np.arange(n, dtype=np.int64) if n <= 20000 else workloads.sample_rows(n, n_rows, seed=2024)
    ref = oracle.matvec(ov, pos, force, wl.a, wl.eta, rows=rows)
    return parity_of(u_gpu, ref, rows, prec)


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1602_02170_b200 import workloads
    wl = workloads.make(args.config)
    k = wl.n_rhs
    budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    times, rows_used, cores, desc = [], 0, 1, ""
    for it in range(args.warmup + args.steps):
        gps, cores, desc, t, nr, _, _ = oracle_sample(wl, args.variant, args.prec, budget)
        log(f"[reference] step {it}: {gps:.4f} {UNIT} ({t:.2f} s)")
        if it >= args.warmup:
            times.append(t); rows_used = nr
    t_mean = float(np.mean(times))
    value = rows_used * wl.n_blobs / t_mean / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_mean * 1e3,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": wl.name, "config_index": args.config, "n_blobs": wl.n_blobs, "n_rhs": k,
                   "variant": args.variant, "step": "oracle on a bounded row sample: " + desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------- GPU leg
def time_config(torch, binding, wl, prec, variant, steps, warmup, flush_buf, rank=0, world=1, dist=None):
    """Device-resident timing of `steps` calls; returns dict with ms per step (max over ranks)."""
    from paper_1602_02170_b200 import sharding
    dt = torch.float32 if prec == "f32" else torch.float64
    dev = torch.device("cuda", torch.cuda.current_device())
    pos = torch.from_numpy(wl.pos).to(dt).to(dev)
    force = torch.from_numpy(wl.force).to(dt).to(dev)
    n, k = wl.n_blobs, wl.n_rhs
    fn = binding.rpy_wall_matvec if variant == "wall" else binding.rpy_free_matvec
    fn_shard = binding.rpy_wall_matvec_shard if variant == "wall" else binding.rpy_free_matvec_shard
    # N > 1: one right-hand side -> work shards of the symmetric kernel + all-reduce (sum) of u;
    #        several -> row shards of the plain kernel + all-gather of u
    work_shards = world > 1 and k == 1
    rows = None if (world == 1 or work_shards) else sharding.shard_rows(n, rank, world)
    ws = torch.empty(binding.rpy_matvec_workspace_bytes(prec, n, k), dtype=torch.uint8, device=dev)
    # the partial products of a work shard are float64 on both paths (fp64 accumulation across ranks)
    out = torch.empty((k, n if rows is None else rows[1], 3), dtype=torch.float64 if work_shards else dt, device=dev)
    gathered = sharding.gather_buffers(n, k, world, dt, dev) if (world > 1 and not work_shards) else None

    def step():
        if work_shards:
            fn_shard(pos, force, rank, world, wl.a, wl.eta, out=out, workspace=ws)
            sharding.reduce_velocities(out)
            return
        fn(pos, force, wl.a, wl.eta, out=out, workspace=ws, rows=rows)
        if world > 1:
            sharding.gather_velocities(out, n, buffers=gathered, concatenate=False)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    evs = []
    for _ in range(steps):
        if flush_buf is not None:
            flush_buf.zero_()                      # > L2 size: evicts the previous step's lines
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(); step(); e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in evs]
    total = torch.tensor([sum(ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total, op=dist.ReduceOp.MAX)
    ms_per_step = total.item() / steps
    return {"ms_per_step": ms_per_step, "ms_min": min(ms), "gps": n * n / (ms_per_step * 1e-3) / 1e9,
            "pos": pos, "force": force, "ws": ws,
            # the full u: single GPU, or after the all-reduce of the work shards (every rank holds it)
            "out": out if (world == 1 or work_shards) else None}


def time_allpairs_kernel(torch, binding, res, wl, variant, steps, flush_buf):
    """CUDA events recorded by the library on its launch stream around the all-pairs kernel."""
    import bench_aids
    times, pre, fin = [], [], []
    for _ in range(steps):
        if flush_buf is not None:
            flush_buf.zero_()
        _, ev = bench_aids.matvec_phases(variant, res["pos"], res["force"], wl.a, wl.eta, out=res["out"],
                                         workspace=res["ws"])
        torch.cuda.synchronize()
        pre.append(ev[0].elapsed_time(ev[1])); times.append(ev[1].elapsed_time(ev[2])); fin.append(ev[2].elapsed_time(ev[3]))
    return float(np.mean(times)), float(np.mean(pre)), float(np.mean(fin))


def time_e2e(torch, binding, wl, prec, variant, steps, warmup):
    dt = torch.float32 if prec == "f32" else torch.float64
    pos = torch.from_numpy(wl.pos).to(dt).pin_memory()
    force = torch.from_numpy(wl.force).to(dt).pin_memory()
    out = torch.empty(force.shape, dtype=dt).pin_memory()
    n, k = wl.n_blobs, wl.n_rhs
    dev = torch.device("cuda", torch.cuda.current_device())
    scratch = torch.empty(binding.rpy_matvec_host_scratch_bytes(prec, n, k), dtype=torch.uint8, device=dev)
    fn = binding.rpy_wall_matvec_host if variant == "wall" else binding.rpy_free_matvec_host
    for _ in range(warmup):
        fn(pos, force, wl.a, wl.eta, out=out, scratch=scratch)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        fn(pos, force, wl.a, wl.eta, out=out, scratch=scratch)      # synchronises before returning
    t = (time.perf_counter() - t0) / steps
    checksum = float(out.double().abs().sum())
    es = 4 if prec == "f32" else 8
    return {"value": n * n / t / 1e9, "unit": UNIT, "h2d_bytes_per_step": int((pos.numel() + force.numel()) * es),
            "d2h_bytes_per_step": int(out.numel() * es), "ms_per_step": t * 1e3, "checksum_abs_u": checksum}


def time_solve(torch, cfg: int, matvec_prec: str, tol: float, restart: int = 60):
    """The rigid-multiblob mobility solve (SURVEY 8(f) N1+N2) on a rigid-body workload: preconditioner
    build, GMRES on Eq. (11) to `tol`, and the per-application cost of its pieces (CUDA events)."""
    from paper_1602_02170_b200 import rigid, workloads
    wl = workloads.make(cfg, k=1) if cfg != 5 else workloads.make(3)
    hb = workloads.bodies_of(wl)
    dev = torch.device("cuda", torch.cuda.current_device())
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).to(dev)
    b = rigid.bodies(t(wl.pos), t(hb.q), hb.offsets)
    F = t(hb.F)
    slip = t(0.1 * np.random.default_rng(8).standard_normal(wl.pos.shape))

    def timed(fn, reps=3):
        fn(); torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            out = fn()
        e1.record(); torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps, out

    pbuf = torch.empty(rigid.rpy_rigid_precond_bytes(hb.offsets), dtype=torch.uint8, device=dev)
    build_ms, pc = timed(lambda: rigid.rpy_rigid_precond_build(b, "wall", wl.a, wl.eta, check=False, buf=pbuf), reps=5)
    rigid.rpy_rigid_precond_info(pc)
    vec = torch.randn(b.n, dtype=torch.float64, device=dev)
    out = torch.empty_like(vec)
    apply_ms, _ = timed(lambda: rigid.rpy_rigid_precond_apply(pc, vec, out=out), reps=10)
    inner = "f32" if matvec_prec == "mixed" else matvec_prec
    saddle_ms, _ = timed(lambda: rigid.rpy_rigid_saddle_apply(b, vec, "wall", wl.a, wl.eta, inner), reps=3)
    ws = torch.empty(rigid.rpy_rigid_solve_workspace_bytes(matvec_prec, b.n_blobs, b.n_bodies, restart),
                     dtype=torch.uint8, device=dev)
    solve = lambda: rigid.rpy_rigid_mobility_solve(b, pc, F, slip, "wall", wl.a, wl.eta, tol=tol, restart=restart,
                                                   matvec_prec=matvec_prec, workspace=ws)
    solve(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    r = solve()
    wall_ms = (time.perf_counter() - t0) * 1e3
    it = max(1, r["n_iter"])
    return {"workload": wl.name, "n_blobs": b.n_blobs, "n_bodies": b.n_bodies, "matvec_prec": matvec_prec,
            "tol": tol, "restart": restart, "n_iter": r["n_iter"], "rel_resid": r["rel_resid"],
            "solve_ms": wall_ms, "ms_per_iter": wall_ms / it, "precond_build_ms": build_ms,
            "precond_apply_ms": apply_ms, "saddle_apply_ms": saddle_ms,
            "krylov_ms_per_iter": wall_ms / it - apply_ms - saddle_ms,
            "matvec_share": saddle_ms / (wall_ms / it)}


def time_solve_batch(torch, cfg: int, matvec_prec: str, tol: float, k: int = 8, restart: int = 40):
    """k right-hand sides (random force/torque on every body) solved at once by lockstep GMRES with one
    k-right-hand-side product per iteration, against k single solves' cost per right-hand side."""
    from paper_1602_02170_b200 import rigid, workloads
    wl = workloads.make(cfg, k=1)
    hb = workloads.bodies_of(wl)
    dev = torch.device("cuda", torch.cuda.current_device())
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).to(dev)
    b = rigid.bodies(t(wl.pos), t(hb.q), hb.offsets)
    F = t(np.random.default_rng(9).standard_normal((k, b.n_bodies, 6)))
    pc = rigid.rpy_rigid_precond_build(b, "wall", wl.a, wl.eta)
    ws = torch.empty(rigid.rpy_rigid_solve_batch_workspace_bytes(matvec_prec, b.n_blobs, b.n_bodies, restart, k),
                     dtype=torch.uint8, device=dev)
    run = lambda: rigid.rpy_rigid_mobility_solve_batch(b, pc, F, None, "wall", wl.a, wl.eta, tol=tol, restart=restart,
                                                       matvec_prec=matvec_prec, workspace=ws)
    run(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    r = run()
    ms = (time.perf_counter() - t0) * 1e3
    return {"workload": wl.name, "n_blobs": b.n_blobs, "n_bodies": b.n_bodies, "n_rhs": k, "matvec_prec": matvec_prec,
            "tol": tol, "restart": restart, "n_iter": r["n_iter"], "rel_resid_max": max(r["rel_resid"]),
            "solve_ms": ms, "ms_per_iter": ms / max(1, r["n_iter"]), "ms_per_rhs": ms / k}


def size_sweep(torch):
    """Kernel time, product time and FP-pipe fraction of the wall product against N (config-1 recipe at
    growing N, k = 1): the evidence behind the kernel / tile-size selection."""
    import bench_aids
    from paper_1602_02170_b200 import binding, workloads
    lane = {"f32": SM_COUNT * LANES["f32"] * SM_MAX_GHZ * 1e9, "f64": SM_COUNT * LANES["f64"] * SM_MAX_GHZ * 1e9}
    rows = []
    for n in (1000, 1152, 1500, 2000, 3000, 3584, 4000, 6144, 8000, 10000, 15000, 20000, 30000, 50000, 100000, 172032):
        w = workloads.config1(seed=0, n=n)
        for prec, dt in (("f32", torch.float32), ("f64", torch.float64)):
            pos = torch.from_numpy(w.pos).to(dt).cuda(); lam = torch.from_numpy(w.force).to(dt).cuda()
            plan = binding.rpy_matvec_launch_plan(prec, n, 1, n)
            ts, ts_all = [], []
            for _ in range(8):
                _, ev = bench_aids.matvec_phases("wall", pos, lam)
                torch.cuda.synchronize()
                ts.append(ev[1].elapsed_time(ev[2])); ts_all.append(ev[0].elapsed_time(ev[3]))
            k_ms = min(ts[2:])
            ph_ms = min(t for t in ts_all[2:])               # prepack .. finalise with events between the kernels (as in r1g)
            # the product as the device sees it: ten back-to-back products captured in a CUDA graph (no host work,
            # no events between its kernels -- they would undo the programmatic dependent launch), replayed
            ws = torch.empty(binding.rpy_matvec_workspace_bytes(prec, n, 1), dtype=torch.uint8, device=pos.device)
            out = torch.empty_like(lam)
            g = torch.cuda.CUDAGraph(); side = torch.cuda.Stream()
            torch.cuda.synchronize()
            with torch.cuda.stream(side):
                with torch.cuda.graph(g, stream=side):
                    for _ in range(10):
                        binding.rpy_wall_matvec(pos, lam, out=out, workspace=ws)
            tot = 1e9
            for _ in range(4):
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(); g.replay(); e1.record(); torch.cuda.synchronize()
                tot = min(tot, e0.elapsed_time(e1) / 10)
            del g
            ops, _ = work_per_pair(prec, "wall", 1, plan["symmetric"])
            rows.append({"n": n, "prec": prec, "symmetric": plan["symmetric"], "tile": plan["tile_sources"],
                         "n_ctas": plan["n_ctas"], "kernel_us": k_ms * 1e3, "product_us": tot * 1e3, "product_phases_us": ph_ms * 1e3,
                         "gps_kernel": n * n / k_ms / 1e6, "pipe_frac": n * n * ops / (k_ms * 1e-3) / lane[prec]})
            log(f"[sweep] {rows[-1]}")
    return rows


def time_table3(torch, n_rods: int, matvec_prec: str, paper_iters: int, paper_seconds: float):
    """Table III (right): the paper's 21-blob rods at phi = 0.1, H/D = 0.75, GMRES to 1e-8
    with the wall-corrected preconditioner; the paper's iteration count and its Tesla K20 wall-clock time
    are quoted as context (another machine, another packing)."""
    from paper_1602_02170_b200 import rigid, workloads
    pos, hb = workloads.rods_near_wall(n_rods, 0.1, 0.75, seed=0)
    dev = torch.device("cuda", torch.cuda.current_device())
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).to(dev)
    b = rigid.bodies(t(pos), t(hb.q), hb.offsets)
    slip = t(0.1 * np.random.default_rng(8).standard_normal(pos.shape))
    F = t(hb.F)
    torch.cuda.synchronize(); t0 = time.perf_counter()
    pc = rigid.rpy_rigid_precond_build(b, "wall")
    torch.cuda.synchronize(); build_ms = (time.perf_counter() - t0) * 1e3
    run = lambda: rigid.rpy_rigid_mobility_solve(b, pc, F, slip, "wall", tol=1e-8, matvec_prec=matvec_prec)
    run(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    r = run()
    ms = (time.perf_counter() - t0) * 1e3
    return {"workload": f"table3_rods{n_rods}x21_phi0.1_HD0.75", "n_blobs": b.n_blobs, "n_bodies": n_rods,
            "matvec_prec": matvec_prec, "n_iter": r["n_iter"], "rel_resid": r["rel_resid"], "solve_ms": ms,
            "precond_build_ms": build_ms, "paper_iterations": paper_iters, "paper_seconds_tesla_k20": paper_seconds}


def run_ours(args):
    import torch
    from paper_1602_02170_b200 import binding, workloads
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local % torch.cuda.device_count())
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", torch.cuda.current_device()))
    binding.load_library()
    dev = torch.device("cuda", torch.cuda.current_device())
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # 256 MiB > 126 MB L2

    wl = workloads.make(args.config)
    prec, variant = args.prec, args.variant
    n, k = wl.n_blobs, wl.n_rhs
    if rank == 0:
        log(f"[bench] {wl.name}: N={n} k={k} {variant} {prec}, steps={args.steps} warmup={args.warmup} world={world}")

    with ClockSampler(torch.cuda.current_device()) as clk:
        res = time_config(torch, binding, wl, prec, variant, args.steps, args.warmup, flush, rank, world, dist)
    clocks = clk.summary()
    ms = res["ms_per_step"]
    value = n * n / (ms * 1e-3) / 1e9
    plan = binding.rpy_matvec_launch_plan(prec, n, k, n // world if (world > 1 and k > 1) else n)
    instr, flops = work_per_pair(prec, variant, k, plan["symmetric"])

    line = None
    parity_failed = False
    if rank == 0:
        import bench_aids
        # measured FMA-chain rates on this GPU, same run (context for the derived peak)
        probe = {}
        try:
            for kind, name in ((0, "ffma"), (1, "ffma2"), (2, "dfma"), (3, "mufu_rsq"), (4, "ffma2_three_reg"), (5, "ffma_three_reg")):
                probe[name + "_g_per_s"] = round(bench_aids.pipe_probe(kind, 8192)["gfma_per_s"], 1)
            # what an FFMA2 / DFMA costs by operand form (T lane-ops/s at 4 CTAs x 128 threads per SM): the all-pairs
            # kernels are bound by register-operand delivery, DESIGN.md section 6
            probe["operand_forms_tlaneops_per_s"] = {
                bench_aids.OPERAND_FORMS[kind]: round(bench_aids.operand_probe(kind, 4, 8192)["tlaneops_per_s"], 2)
                for kind in range(8)}
        except Exception as e:  # pragma: no cover
            probe = {"error": str(e)}

        def roofline_of(cfg, p, v, w, r, plan_, kernel_steps):
            """Roofline object of the dominant kernel of one configuration (single-GPU geometry): the kernel is
            timed on its own launch stream by CUDA events recorded inside the library call."""
            ops, fl = work_per_pair(p, v, w.n_rhs, plan_["symmetric"])
            if world == 1:
                k_ms, pre_ms, fin_ms = time_allpairs_kernel(torch, binding, r, w, v, kernel_steps, flush)
            else:
                k_ms, pre_ms, fin_ms = r["ms_per_step"], 0.0, 0.0
            pairs_launch = w.n_blobs * w.n_blobs // world
            achieved = pairs_launch * fl / (k_ms * 1e-3) / 1e12
            peak = peak_tflops(p)
            lane_peak = SM_COUNT * LANES[p] * SM_MAX_GHZ * 1e9
            traffic, src = ncu_traffic(cfg, p, v) if w.n_rhs == 1 else (None, None)   # captures exist for k = 1
            return {
                "bound": "alu", "kernel": "allpairs_sym_kernel" if plan_["symmetric"] else "allpairs_kernel",
                "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": src,
                "peak_source": f"derived: {SM_COUNT} SM x {LANES[p]} lanes x 2 flop x {SM_MAX_GHZ} GHz (DESIGN.md)",
                "flop_per_pair": fl, "lane_ops_per_pair": ops,
                "pipe_frac": pairs_launch * ops / (k_ms * 1e-3) / lane_peak,
                "kernel_ms": k_ms, "prepack_ms": pre_ms, "finalise_ms": fin_ms,
                "kernel_share_of_step": k_ms / (k_ms + pre_ms + fin_ms) if world == 1 else None,
            }

        roofline = roofline_of(args.config, prec, variant, wl, res, plan, max(3, min(args.steps, 10)))
        roofline["measured_chain_rates"] = probe
        # --- end to end through the host-buffer C-ABI call
        e2e = time_e2e(torch, binding, wl, prec, variant, max(2, min(args.steps, 5)), 1) if world == 1 else \
            {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
             "note": "host-buffer call is single-GPU; run with --gpus 1"}
        # --- the oracle on the host cores, bounded sample; its velocities give the parity of the timed step
        cpu, parity = None, None
        if world == 1 and not args.no_cpu:
            gps, cores, desc, t, _, orows, oref = oracle_sample(wl, variant, prec, 15.0)
            cpu = {"value": gps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": t}
            parity = parity_of(res["out"], oref, orows, prec)
        elif world > 1 and res["out"] is not None and not args.no_cpu:
            parity = oracle_parity(wl, variant, prec, res["out"])      # the all-reduced sum of the ranks' shards
        if parity is not None:
            parity_failed = parity_failed or not parity["ok"]
            log(f"[bench] parity vs oracle: {parity}")
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None,
            "dtype": "f32 pair arithmetic, f64 accumulation" if prec == "f32" else "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "config_index": args.config, "n_blobs": n, "n_rhs": k,
                       "variant": variant, "a": wl.a, "eta": wl.eta, "seed": wl.meta.get("seed"),
                       "l2": "flushed between steps (256 MiB write)",
                       "parallelism": "single GPU" if world == 1 else (
                           f"unordered tile pairs of the symmetric kernel sharded over {world} ranks + all-reduce of u" if k == 1
                           else f"target rows sharded over {world} ranks + all-gather of u"),
                       "launch_plan": plan},
            "pair_rhs_gps": value * k,
            "clocks": clocks, "e2e": e2e, "gpu_launches": 3 * args.steps * (1 if k <= 8 else -(-k // 8)),
            "roofline": roofline, "cpu_baseline": cpu, "parity": parity,
        }
        # --- the paper's own precision ("in double precision"): the fp64 path on the same workload,
        # in fields of its own so that it is not only a context line
        if world == 1 and prec == "f32" and not args.no_f64:
            st64 = max(3, min(args.steps, 5))
            r64 = time_config(torch, binding, wl, "f64", variant, st64, 3, flush)
            pl64 = binding.rpy_matvec_launch_plan("f64", n, k, n)
            line["value_f64"] = r64["gps"]
            line["ms_per_step_f64"] = r64["ms_per_step"]
            line["roofline_f64"] = roofline_of(args.config, "f64", variant, wl, r64, pl64, 3)
            if not args.no_cpu:
                line["parity_f64"] = oracle_parity(wl, variant, "f64", r64["out"])
                parity_failed = parity_failed or not line["parity_f64"]["ok"]
                log(f"[bench] f64: {r64['gps']:.1f} {UNIT}, parity {line['parity_f64']}")
            del r64
        # --- the other BASELINE.json configurations, fewer steps (context; not the headline)
        if world == 1 and not args.no_extra:
            extra = []
            for cfg, p, v, st in ((3, "f32", "free", 3), (3, "f64", "free", 3), (5, "f32", "wall", 3), (5, "f32", "free", 3),
                                  (2, "f64", "wall", 10), (2, "f32", "wall", 10), (1, "f64", "wall", 10),
                                  (4, "f32", "wall", 1), (3, "f64", "wall", 3)):
                if (cfg, p, v) == (args.config, prec, variant) or ((cfg, v) == (args.config, variant) and "value_f64" in line and p == "f64"):
                    continue
                w2 = workloads.make(cfg)
                r2 = time_config(torch, binding, w2, p, v, st, 3 if cfg != 4 else 1, flush)
                km, _, _ = time_allpairs_kernel(torch, binding, r2, w2, v, 2 if cfg != 4 else 1, flush)
                pl2 = binding.rpy_matvec_launch_plan(p, w2.n_blobs, w2.n_rhs, w2.n_blobs)
                i2, f2 = work_per_pair(p, v, w2.n_rhs, pl2["symmetric"])
                lane2 = SM_COUNT * LANES[p] * SM_MAX_GHZ * 1e9
                par2 = None
                if not args.no_cpu:
                    par2 = oracle_parity(w2, v, p, r2["out"])
                    parity_failed = parity_failed or not par2["ok"]
                extra.append({"workload": w2.name, "prec": p, "variant": v, "n_blobs": w2.n_blobs, "n_rhs": w2.n_rhs,
                              "ms_per_step": r2["ms_per_step"], "gps": r2["gps"], "pair_rhs_gps": r2["gps"] * w2.n_rhs,
                              "kernel_ms": km, "symmetric": pl2["symmetric"],
                              "pipe_frac": w2.n_blobs ** 2 * i2 / (km * 1e-3) / lane2,
                              "flop_frac": w2.n_blobs ** 2 * f2 / (km * 1e-3) / 1e12 / peak_tflops(p),
                              "parity": par2})
                log(f"[bench] extra {extra[-1]}")
                del r2
            line["other_configs"] = extra
            # --- next rows of SURVEY 8(f): the preconditioned GMRES mobility solve around the matvec
            solves = []
            for cfg, p, tol in ((2, "f64", 1e-8), (2, "mixed", 1e-8), (3, "f64", 1e-8), (3, "mixed", 1e-8), (3, "f32", 1e-5)):
                try:
                    solves.append(time_solve(torch, cfg, p, tol))
                    log(f"[bench] solve {solves[-1]}")
                except Exception as e:  # pragma: no cover
                    solves.append({"config": cfg, "matvec_prec": p, "error": repr(e)})
            line["rigid_solve"] = solves
            batch = []
            for cfg, p, tol in ((2, "mixed", 1e-8), (3, "mixed", 1e-8)):
                try:
                    batch.append(time_solve_batch(torch, cfg, p, tol))
                    log(f"[bench] batch solve {batch[-1]}")
                except Exception as e:  # pragma: no cover
                    batch.append({"config": cfg, "matvec_prec": p, "error": repr(e)})
            line["rigid_solve_batch"] = batch
            t3 = []
            for nr, p, it, sec in ((1000, "f64", 19, 32.7), (1000, "mixed", 19, 32.7), (10000, "mixed", 20, 2050.0)):
                try:
                    t3.append(time_table3(torch, nr, p, it, sec))
                    log(f"[bench] table III {t3[-1]}")
                except Exception as e:  # pragma: no cover
                    t3.append({"n_rods": nr, "matvec_prec": p, "error": repr(e)})
            line["table3_rods"] = t3
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)
        if parity_failed:
            log("[bench] PARITY FAILURE: a CUDA result is outside north_star's tolerance of the oracle (see 'parity' fields)")
            return 3
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--prec", choices=["f32", "f64"], default="f32")
    ap.add_argument("--variant", choices=["wall", "free"], default="wall")
    ap.add_argument("--no-extra", action="store_true", help="skip the other configurations")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle timing and the parity figures")
    ap.add_argument("--no-f64", action="store_true", help="skip the fp64 path of the headline workload (value_f64, roofline_f64)")
    ap.add_argument("--rigid-solve", type=int, default=0, choices=[0, 2, 3],
                    help="only time the preconditioned GMRES mobility solve on this rigid-body config "
                         "(--prec f64|f32, or --solve-prec mixed) and print its JSON (profiling aid)")
    ap.add_argument("--solve-prec", choices=["f64", "f32", "mixed"], default="f64")
    ap.add_argument("--size-sweep", action="store_true",
                    help="only print kernel/product time and pipe fraction of the wall product against N (profiling aid)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        log("[bench] note: fewer than 3 warm-up steps requested")
    if args.impl == "reference":
        return run_reference(args)
    if args.size_sweep:
        import torch
        torch.cuda.set_device(0)
        print(json.dumps(size_sweep(torch)), flush=True)
        return 0
    if args.rigid_solve:
        import torch
        torch.cuda.set_device(0)
        tol = 1e-5 if args.solve_prec == "f32" else 1e-8
        print(json.dumps(time_solve(torch, args.rigid_solve, args.solve_prec, tol)), flush=True)
        return 0
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
