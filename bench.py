#!/usr/bin/env python
"""Benchmark of the B200 spectral Ewald hot path (one JSON line on stdout, rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl b200|reference]

A step = one pass of the whole hot path (K1 sort, K2 P2P, K3 P2G, cuFFT R2C, K4 scale, cuFFT C2R,
K5 G2P, K6 sum: SURVEY.md §8(a)) over one synthetic batch.  Default workload: BASELINE.json
configs[2] (N = 1,048,576 uniform, fp64, 9 digits), the configuration SURVEY.md §8(d) names as the
fp64 headline that fits one GPU comfortably; `--config` selects another (1..5).
Multi-GPU (`--gpus N` under torchrun): N independent replicas, no data-path collective
(replicas only); value = particles all ranks processed / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "particles/s, full Stokes SE sum"
UNIT = "particles/s"
# FP64 / FP32 FMA peak of one B200 from unit counts and clocks:
# 148 SMs x 64 (128) FMA lanes x 2 flop x 1.965 GHz.  A register-only DFMA/FFMA chain measured
# 36.7 / 72.0 TFLOP/s on this pool (profiles/r01b_mma_ws.md).
ALU_PEAK_TFLOPS = {"fp64": 148 * 64 * 2 * 1.965e9 / 1e12, "fp32": 148 * 128 * 2 * 1.965e9 / 1e12}
SAMPLE_CFG = 2          # the oracle's bounded sample: config 2 in full


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id: str):
        self.proc = None
        self.lines = []
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={gpu_id}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.perf_counter(), ln.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        inside = [l for (t, l) in self.lines if t0 <= t <= t1] or [l for (_, l) in self.lines]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in inside:
            p = [q.strip() for q in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for nm, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def stage_flops_bytes(c, stage):
    """Algorithmic work of one launch of a stage (per-unit figure x units)."""
    B = 8 if c.precision == "fp64" else 4
    N, M, P = c.N, c.M, c.P
    nk = M * M * (M // 2 + 1)
    if stage in ("p2g", "g2p"):
        return {"bound": "alu", "work": 2.0 * 3 * P ** 3 * N, "unit": "TFLOP/s"}
    if stage == "scale":
        return {"bound": "hbm", "work": 12.0 * B * nk, "unit": "GB/s"}
    if stage in ("fft", "ifft"):
        return {"bound": "hbm", "work": 3.0 * (B * M ** 3 + 2 * B * nk), "unit": "GB/s"}
    if stage == "sort":
        return {"bound": "hbm", "work": N * (6.0 * B * 3 + 3 * P * B + 40), "unit": "GB/s"}
    if stage == "sum":
        return {"bound": "hbm", "work": N * (12.0 * B + 8), "unit": "GB/s"}
    return None


def oracle_sample():
    """The bounded sample the CPU oracle is timed on (same dimensionless parameters as the workload)."""
    from paper_2606_19059_b200 import workloads as W
    c, x, f = W.make(SAMPLE_CFG)
    desc = (f"config {SAMPLE_CFG} in full (N={c.N}, M={c.M}, P={c.P}: same xi*rc, pi*M/(2 xi L), P and "
            f"neighbours per particle as config 3, 1/16 of its particles)")
    return c, x, f, desc


def time_oracle_once(c, x, f):
    import oracle
    t = time.perf_counter()
    oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P)
    return time.perf_counter() - t


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if env_int("RANK", 0) != 0:
        return 0
    import oracle
    from paper_2606_19059_b200 import workloads as W
    oracle.build()
    c, x, f, desc = oracle_sample()
    wl = W.CONFIGS[args.config]
    for _ in range(args.warmup):
        time_oracle_once(c, x, f)
    ts = [time_oracle_once(c, x, f) for _ in range(args.steps)]
    total = sum(ts)
    val = c.N * args.steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.label, "timed_on": desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_2606_19059_b200 as se
    from paper_2606_19059_b200 import replicas, workloads as W

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    se.lib()                                          # fail loudly if libse_b200.so is missing
    torch.cuda.set_device(local)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    c, x, f = W.make(args.config)
    if rank > 0 and c.kind == "uniform":              # replicas: every rank its own seeded batch
        x, f = (a.astype(W.np_dtype(c.precision))
                for a in W.uniform_cloud(replicas.replica_seed(W.SEED_BASE + args.config, rank), c.N, c.L))
    dt = torch.float64 if c.precision == "fp64" else torch.float32
    xh = torch.as_tensor(np.ascontiguousarray(x), dtype=dt).pin_memory()
    fh = torch.as_tensor(np.ascontiguousarray(f), dtype=dt).pin_memory()
    uh = torch.empty_like(xh).pin_memory()
    xd, fd = xh.cuda(), fh.cuda()
    ud = torch.empty_like(xd)
    stream = torch.cuda.current_stream()

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(v):
        return replicas.aggregate(0.0, v, device="cuda")[1]

    plan = se.Plan(c.N, c.L, c.xi, c.rc, c.M, c.P, c.precision)
    info = plan.info()
    plan.set_profiling(True)                          # CUDA events around each stage, no host sync
    for _ in range(max(args.warmup, 3)):
        plan.eval(xd, fd, ud)
    barrier()

    props = torch.cuda.get_device_properties(local)
    sampler = ClockSampler("GPU-" + str(props.uuid)) if rank == 0 else None
    time.sleep(0.3 if rank == 0 else 0.0)
    barrier()

    # ---- device-resident timed region: exactly K steps ---------------------------------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_acc = {k: 0.0 for k in se.STAGES}
    launches = 0
    t_wall0 = time.perf_counter()
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        plan.eval(xd, fd, ud)
    e1.record(stream)
    barrier()
    ms_dev = max_over_ranks(e0.elapsed_time(e1))
    # stage times of the LAST timed step come from the events se_eval recorded on the same stream;
    # re-run K profiled steps to average them (outside the headline timing, same launches).
    for _ in range(args.steps):
        plan.eval(xd, fd, ud)
        sm = plan.stage_ms()
        for k, v in sm.items():
            stage_acc[k] += v
    launches = plan.launch_count() * args.steps
    stage_ms = {k: v / args.steps for k, v in stage_acc.items()}

    # ---- end to end through the host-buffer entry point ------------------------------------
    for _ in range(2):
        plan.eval_host(xh, fh, uh)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        plan.eval_host(xh, fh, uh)
    e1.record(stream)
    barrier()
    t_wall1 = time.perf_counter()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None

    ok = bool(torch.isfinite(ud).all().item()) and bool(torch.isfinite(uh).all().item())
    if distributed:
        dist.barrier()
    if rank != 0:
        plan.destroy()
        if distributed:
            dist.destroy_process_group()
        return 0

    B = 8 if c.precision == "fp64" else 4
    value = world * c.N * args.steps / (ms_dev * 1e-3)
    e2e = world * c.N * args.steps / (ms_e2e * 1e-3)

    # ---- roofline of every stage; the headline object is the dominant kernel of ours -------
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh_:
            peaks = json.load(fh_)
    except OSError:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"
    traffic = {}
    try:
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as fh_:
            for ln in fh_:
                p = ln.strip().split(",")
                if len(p) >= 3 and p[0] == str(args.config):
                    traffic[p[1]] = float(p[2])
    except OSError:
        pass
    per_stage = {}
    for st, ms in stage_ms.items():
        w = stage_flops_bytes(c, st)
        if w is None or ms <= 0:
            continue
        if w["bound"] == "alu":
            ach = w["work"] / (ms * 1e-3) / 1e12
            # fp32 plans grid on the FP64 tensor path too (double records and accumulators, float grid)
            peak = ALU_PEAK_TFLOPS["fp64" if info.grid_mode == 2 else c.precision]
        else:
            ach = w["work"] / (ms * 1e-3) / 1e9
            peak = hbm_peak
        per_stage[st] = {"bound": w["bound"], "achieved": ach, "peak": peak, "unit": w["unit"],
                         "frac": ach / peak, "ms": ms, "traffic": traffic.get(st)}
    own = [s for s in ("p2g", "g2p", "scale", "sort", "sum") if s in per_stage]
    dom = max(own, key=lambda s: stage_ms[s])
    roof = dict(per_stage[dom])
    roof["kernel"] = {"p2g": "k_p2g (K3)", "g2p": "k_g2p (K5)", "scale": "k_scale (K4)", "sort": "K1", "sum": "K6"}[dom]
    roof["peak_source"] = ("unit counts x clock: 148 SM x %d FMA/clk x 2 x 1.965 GHz (DESIGN.md)" %
                           (64 if (c.precision == "fp64" or info.grid_mode == 2) else 128)) if roof["bound"] == "alu" else hbm_src
    # P2P: plain-ALU kernel whose work is data dependent -- reported as in-range pairs/s
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_dev / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if c.precision == "fp64" else "f32",
        "data": "synthetic",
        "config": {"workload": c.label, "N": c.N, "L": c.L, "xi": c.xi, "rc": c.rc, "M": c.M, "P": c.P,
                   "precision": c.precision, "eta": info.eta, "ncell": info.ncell,
                   "gridding": ("FP64 tensor-core sweep (double records and accumulators%s)" %
                                (", float grid" if c.precision == "fp32" else "")) if info.grid_mode == 2
                   else "generic tile kernel in the plan's precision",
                   "parallelism": "replicas x%d" % world,
                   "l2": "no explicit flush: every step streams the %.2f GB plan workspace (grid %.2f GB + "
                         "spectrum %.2f GB), far larger than the 126 MB L2" %
                         (info.workspace_bytes / 1e9, 3 * B * c.M ** 3 / 1e9, 6 * B * info.nmodes / 1e9)},
        "e2e": {"value": e2e, "unit": UNIT, "ms_per_step": ms_e2e / args.steps,
                "h2d_bytes_per_step": 2 * 3 * c.N * B, "d2h_bytes_per_step": 3 * c.N * B},
        "gpu_launches": launches,
        "clocks": clocks,
        "roofline": roof,
        "stages_ms": {k: round(v, 4) for k, v in stage_ms.items()},
        "stages_roofline": {k: {"bound": v["bound"], "frac": round(v["frac"], 4), "achieved": round(v["achieved"], 2),
                                "unit": v["unit"]} for k, v in per_stage.items()},
        "value_excluding_fft": world * c.N / ((sum(stage_ms.values()) - stage_ms["fft"] - stage_ms["ifft"]) * 1e-3),
        "finite": ok,
    }
    plan.destroy()
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        sc, sx, sf, desc = oracle_sample()
        t = time_oracle_once(sc, sx, sf)
        reps = 1
        while t < 8.0 and reps < 8:                    # aim at ~10-30 s of CPU work in total
            t += time_oracle_once(sc, sx, sf)
            reps += 1
        line["cpu_baseline"] = {"value": sc.N * reps / t, "unit": UNIT, "cores": oracle.n_threads(),
                                "kind": "oracle", "sample": desc + f", {reps} run(s), {t:.1f} s"}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    if distributed:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    world = env_int("WORLD_SIZE", 1)
    if world != args.gpus:
        if args.gpus == 1 and world > 1:
            pass
        elif world == 1 and args.gpus > 1:
            raise SystemExit("bench.py: --gpus %d needs torchrun with --nproc-per-node %d" % (args.gpus, args.gpus))
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
