#!/usr/bin/env python
"""Benchmark of the B200 spectral Ewald hot path (one JSON line on stdout, rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl b200|reference]

A step = one pass of the whole hot path (K1 sort, K2 P2P, K3 P2G, cuFFT R2C, K4 scale, cuFFT C2R,
K5 G2P, K6 sum: SURVEY.md §8(a)) over one synthetic batch; on plans with fft_fused (se.h) the transforms over x
run inside the K4 kernel and the 2-D transforms of the x-planes are the library's own kernels (fft_planes_own) or cuFFT's.  Default workload: BASELINE.json
configs[2] (N = 1,048,576 uniform, fp64, 9 digits), the configuration SURVEY.md §8(d) names as the
fp64 headline that fits one GPU comfortably; `--config` selects another (1..5).
Multi-GPU (`--gpus N` under torchrun): N independent replicas, no data-path collective
(replicas only); value = particles all ranks processed / max-over-ranks time.
The default run (config 3, one GPU) also carries `configs`: sub-results for config 5, config 4 and the same workloads with
the paper's Kaiser-Bessel window, each with its own stage times and rooflines, and `peaks`: the FP64 / FP32 / HBM
figures se_measure_peak measured on this device before the timed region.
`--impl reference` times the CPU oracle (oracle/, as it stands) on the bench workload itself, one evaluation per step.
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
# Nominal FP64 / FP32 FMA peaks of one B200 from unit counts and clocks (148 SMs x 64 / 128 FMA lanes x 2 flop x
# 1.965 GHz) and the fallback HBM figure of /opt/skills/guides/B200_PROFILING.md; used only when the measured ones
# (se_measure_peak: register-only DFMA / DMMA / FFMA chains, run before the timed region) are unavailable.
NOMINAL_TFLOPS = {"fp64": 148 * 64 * 2 * 1.965e9 / 1e12, "fp32": 148 * 128 * 2 * 1.965e9 / 1e12}
# FP64 (FP32) arithmetic instructions K2 spends per in-range pair (DESIGN.md section 6 "K2"): the "alu" work of P2P.
# fp64: 60 DFMA + 10.5 DMUL + 7 DADD + 3 DSETP per pair in the SASS of the evaluation round (profiles/r02r_final.md);
# fp32: the same algorithm with the degree-6 rational and expf, counted from the source
P2P_INSTR_PER_PAIR = {"fp64": 80, "fp32": 50}
# sub-results of the default run (world size 1): (key, config, steps, plan overrides)
SUB_RESULTS = [("cfg5", 5, 3, {}), ("cfg4", 4, 5, {}),
               ("cfg3_kb_P12", 3, 5, {"window": "kb", "P": 12}), ("cfg5_kb_P12", 5, 3, {"window": "kb", "P": 12}),
               ("cfg4_kb_P8", 4, 5, {"window": "kb", "P": 8}),
               # the headline workload with cuFFT's batched 3-D transforms and the stand-alone K4 kernel (SE_FFT_MODE=3d at plan
               # creation): what north_star's "the 3-D FFTs use cuFFT" prescribes, next to the library's own transforms
               ("cfg3_cufft3d", 3, 5, {"env": {"SE_FFT_MODE": "3d"}})]


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


def stage_work(c, P, stage, pairs):
    """Algorithmic work of one launch of a stage (per-unit figure x units)."""
    B = 8 if c.precision == "fp64" else 4
    N, M = c.N, c.M
    nk = M * M * (M // 2 + 1)
    if stage in ("p2g", "g2p"):
        return {"bound": "alu", "work": 2.0 * 3 * P ** 3 * N, "unit": "TFLOP/s"}
    if stage == "p2p" and pairs:
        return {"bound": "alu", "work": 2.0 * P2P_INSTR_PER_PAIR[c.precision] * pairs, "unit": "TFLOP/s"}
    if stage == "scale":
        return {"bound": "hbm", "work": 12.0 * B * nk, "unit": "GB/s"}
    if stage in ("fft", "ifft"):
        return {"bound": "hbm", "work": 3.0 * (B * M ** 3 + 2 * B * nk), "unit": "GB/s"}
    if stage == "sort":
        # x, f read twice (binning; gather), two sorted copies and the FP32 filter copy written, index arrays,
        # and the per-particle window records of the tensor-core sweep (8 bytes per entry in every precision)
        return {"bound": "hbm", "work": N * (4.0 * 3 * B + 6.0 * B + 16 + 3 * B + 40 + 8.0 * (8 * P + 8)), "unit": "GB/s"}
    if stage == "sum":
        return {"bound": "hbm", "work": N * (12.0 * B + 8), "unit": "GB/s"}
    return None


def gridding_hbm_bytes(c, P):
    """Compulsory DRAM bytes of one gridding launch: the grid once plus the particles' records once."""
    B = 8 if c.precision == "fp64" else 4
    return 3.0 * B * c.M ** 3 + c.N * 8.0 * (4 * P + 4)


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh_:
            return json.load(fh_)
    except (OSError, ValueError):
        return {}


def load_traffic():
    """profiles/dram_traffic.csv: cfg, stage, dram bytes per launch (ncu --set full), source."""
    out = {}
    try:
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as fh_:
            for ln in fh_:
                p = ln.strip().split(",")
                if len(p) >= 3 and not p[0].startswith("#"):
                    try:
                        out[(p[0], p[1])] = float(p[2])
                    except ValueError:
                        pass
    except OSError:
        pass
    return out


def measure_peaks(se):
    """Register-only chains and a read+write stream on this device (se_measure_peak), before any timed region."""
    out = {}
    for key, which in (("fp64_tflops_measured", "fp64"), ("fp64_tensor_tflops_measured", "fp64_tensor"),
                       ("fp32_tflops_measured", "fp32"), ("hbm_stream_tbs_measured", "hbm")):
        try:
            out[key] = se.measure_peak(which, 5)
        except Exception as ex:                          # reported, never fatal
            out[key] = None
            out.setdefault("errors", []).append(f"{which}: {ex}")
    return out


def oracle_step(c, x, f):
    """One evaluation of the CPU oracle, as it stands, on the workload itself; seconds and per-step timings."""
    import oracle
    tm = {}
    t = time.perf_counter()
    oracle.se_eval(x, f, c.L, c.xi, c.rc, c.M, c.P, timings=tm)
    return time.perf_counter() - t, tm


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, one full evaluation of the bench workload per step
    (rank 0 only).  At most one warm-up evaluation is made (an evaluation of config 3 takes ~12 s on 16 cores)."""
    if env_int("RANK", 0) != 0:
        return 0
    import oracle
    from paper_2606_19059_b200 import workloads as W
    oracle.build()
    c, x, f = W.make(args.config)
    warm = min(args.warmup, 1)
    for _ in range(warm):
        oracle_step(c, x, f)
    ts = [oracle_step(c, x, f)[0] for _ in range(args.steps)]
    total = sum(ts)
    val = c.N * args.steps / total
    desc = (f"the bench workload itself, in full ({c.label}: every step is one oracle.se_eval over all N = {c.N} "
            f"particles; {warm} warm-up evaluation(s) instead of {args.warmup})")
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": warm, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": c.label, "N": c.N, "L": c.L, "xi": c.xi, "rc": c.rc, "M": c.M, "P": c.P,
                   "precision": c.precision},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


class Ctx:
    """Process-wide state of one bench run: torch, ranks, peaks."""
    pass


def bench_plan(ctx, cfg, steps, warmup, over, headline):
    """Time one plan on config `cfg` (plan overrides `over`: window, P).  Returns the result dict; for the headline
    also samples clocks around the timed regions."""
    torch, se, W, replicas = ctx.torch, ctx.se, ctx.W, ctx.replicas
    c, x, f = W.make(cfg)
    if ctx.rank > 0 and c.kind == "uniform":              # replicas: every rank its own seeded batch
        x, f = (a.astype(W.np_dtype(c.precision))
                for a in W.uniform_cloud(replicas.replica_seed(W.SEED_BASE + cfg, ctx.rank), c.N, c.L))
    window, P = over.get("window", "gaussian"), over.get("P", c.P)
    dt = torch.float64 if c.precision == "fp64" else torch.float32
    xh = torch.as_tensor(np.ascontiguousarray(x), dtype=dt).pin_memory()
    fh = torch.as_tensor(np.ascontiguousarray(f), dtype=dt).pin_memory()
    uh = torch.empty_like(xh).pin_memory()
    xd, fd = xh.cuda(), fh.cuda()
    ud = torch.empty_like(xd)
    stream = torch.cuda.current_stream()

    plan = se.Plan(c.N, c.L, c.xi, c.rc, c.M, P, c.precision, window=window)
    info = plan.info()
    plan.set_profiling(True)                          # CUDA events around each stage, no host sync
    for _ in range(max(warmup, 3)):
        plan.eval(xd, fd, ud)
    ctx.barrier()
    cand, pairs = plan.count_pairs()                  # K2's work, counted once outside every timed region

    sampler = None
    if headline and ctx.rank == 0:
        props = torch.cuda.get_device_properties(ctx.local)
        sampler = ClockSampler("GPU-" + str(props.uuid))
        time.sleep(0.3)
    ctx.barrier()

    # ---- device-resident timed region: exactly `steps` evaluations ----------------------------------------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.perf_counter()
    ctx.barrier()
    e0.record(stream)
    for _ in range(steps):
        plan.eval(xd, fd, ud)
    e1.record(stream)
    ctx.barrier()
    ms_dev = ctx.max_over_ranks(e0.elapsed_time(e1))
    # stage times: the events se_eval records on the same stream, averaged over `steps` more evaluations (outside the
    # headline timing, same launches)
    stage_acc = {k: 0.0 for k in se.STAGES}
    for _ in range(steps):
        plan.eval(xd, fd, ud)
        for k, v in plan.stage_ms().items():
            stage_acc[k] += v
    launches = plan.launch_count() * steps
    stage_ms = {k: v / steps for k, v in stage_acc.items()}

    # ---- end to end through the host-buffer entry point ------------------------------------------------------
    for _ in range(2):
        plan.eval_host(xh, fh, uh)
    ctx.barrier()
    e0.record(stream)
    for _ in range(steps):
        plan.eval_host(xh, fh, uh)
    e1.record(stream)
    ctx.barrier()
    t_wall1 = time.perf_counter()
    ms_e2e = ctx.max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ok = bool(torch.isfinite(ud).all().item()) and bool(torch.isfinite(uh).all().item())
    plan.destroy()
    del xd, fd, ud, xh, fh, uh
    torch.cuda.empty_cache()

    B = 8 if c.precision == "fp64" else 4
    world = ctx.world
    pk = ctx.peaks
    hbm_peak = float(ctx.file_peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (copy)" if "hbm_gbs" in ctx.file_peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    # the FP64 datapath serves DFMA and DMMA alike: the measured peak is the better of the two chains
    f64 = max([v for v in (pk.get("fp64_tflops_measured"), pk.get("fp64_tensor_tflops_measured")) if v] or [0.0])
    f32 = pk.get("fp32_tflops_measured") or 0.0
    alu = {"fp64": (f64, "measured: register-only DFMA / DMMA chain (se_measure_peak)") if f64 else
           (NOMINAL_TFLOPS["fp64"], "nominal: 148 SM x 64 FMA/clk x 2 x 1.965 GHz"),
           "fp32": (f32, "measured: register-only FFMA chain (se_measure_peak)") if f32 else
           (NOMINAL_TFLOPS["fp32"], "nominal: 148 SM x 128 FMA/clk x 2 x 1.965 GHz")}
    tag = "%d%s" % (cfg, "" if not over else "_" + window + str(P))
    per_stage = {}
    for st, ms in stage_ms.items():
        w = stage_work(c, P, st, pairs)
        if w is None or ms <= 0:
            continue
        r = {"bound": w["bound"], "unit": w["unit"], "ms": ms}
        if w["bound"] == "alu":
            r["achieved"] = w["work"] / (ms * 1e-3) / 1e12
            # the survey's bound for a plan is the ALU pipe of its own precision; fp32 plans grid on
            # the FP64 datapath (double records and accumulators), so that figure is given beside it
            r["peak"], r["peak_source"] = alu[c.precision]
            if st in ("p2g", "g2p"):
                if c.precision == "fp32" and info.grid_mode == 2:
                    r["frac_of_fp64_datapath"] = r["achieved"] / alu["fp64"][0]
                r["hbm_gbs_on_compulsory_bytes"] = gridding_hbm_bytes(c, P) / (ms * 1e-3) / 1e9
                r["hbm_frac_on_compulsory_bytes"] = r["hbm_gbs_on_compulsory_bytes"] / hbm_peak
        else:
            r["achieved"] = w["work"] / (ms * 1e-3) / 1e9
            r["peak"], r["peak_source"] = hbm_peak, hbm_src
        r["frac"] = r["achieved"] / r["peak"]
        if r["bound"] == "hbm" and r["frac"] > 1.0:
            r["note"] = ("above the copy figure of MEASURED_PEAKS.json; this device's read+write stream measured "
                         "%.0f GB/s (se_measure_peak)" % (1e3 * (pk.get("hbm_stream_tbs_measured") or 0.0)))
        r["traffic"] = ctx.traffic.get((tag, st))
        per_stage[st] = r
    own = [s_ for s_ in ("p2p", "p2g", "g2p", "scale", "sort", "sum") if s_ in per_stage]
    dom = max(own, key=lambda s_: stage_ms[s_])
    roof = dict(per_stage[dom])
    roof["kernel"] = {"p2p": "k_p2p (K2)", "p2g": "k_mma<spread> (K3)", "g2p": "k_mma<gather> (K5)",
                      "scale": "k_xfft_scale (K4x)" if info.fft_fused else "k_scale (K4)", "sort": "K1", "sum": "K6"}[dom]
    total_stage = sum(stage_ms.values())
    res = {
        "workload": c.label + ("" if not over else f" [{window} window, P={P}]"),
        "value": world * c.N * steps / (ms_dev * 1e-3), "unit": UNIT, "steps": steps,
        "ms_per_step": ms_dev / steps,
        "e2e": {"value": world * c.N * steps / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e / steps,
                "h2d_bytes_per_step": 2 * 3 * c.N * B, "d2h_bytes_per_step": 3 * c.N * B},
        "gpu_launches": launches, "roofline": roof,
        "stages_ms": {k: round(v, 4) for k, v in stage_ms.items()},
        "stages_roofline": {k: {kk: (round(vv, 4) if isinstance(vv, float) else vv) for kk, vv in v.items()
                                if kk not in ("ms", "peak_source")} for k, v in per_stage.items()},
        "p2p_pairs": {"in_range": pairs, "candidates": cand, "in_range_per_s": pairs / (stage_ms["p2p"] * 1e-3)
                      if stage_ms["p2p"] > 0 else None},
        "value_excluding_fft": world * c.N / ((total_stage - stage_ms["fft"] - stage_ms["ifft"]) * 1e-3),
        "finite": ok,
    }
    cfgd = {"workload": res["workload"], "N": c.N, "L": c.L, "xi": c.xi, "rc": c.rc, "M": c.M, "P": P,
            "precision": c.precision, "window": window, "eta": info.eta, "ncell": info.ncell,
            "gridding": ("FP64 tensor-core sweep (double records and accumulators%s)" %
                         (", float grid" if c.precision == "fp32" else "")) if info.grid_mode == 2
            else "generic tile kernel in the plan's precision",
            "transforms": ("fft / ifft = %s 2-D over (y, z) of every x-plane, scale = k_xfft_scale: transform over x + K4 + "
                           "inverse transform over x in one kernel (se.h, fft_fused), %d threads per block"
                           % ("own (k_zr2c + k_yfft / k_yfft + k_zc2r)" if info.fft_planes_own else "cuFFT", info.fft_threads)) if info.fft_fused
            else "fft / ifft = cuFFT 3-D, scale = k_scale (K4)",
            "parallelism": "replicas x%d" % world,
            "l2": "no explicit flush: every step streams the %.2f GB plan workspace (grid %.2f GB + spectrum %.2f GB), "
                  "far larger than the 126 MB L2" % (info.workspace_bytes / 1e9, 3 * B * c.M ** 3 / 1e9,
                                                      6 * B * info.nmodes / 1e9)}
    return res, cfgd, clocks, c


def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_2606_19059_b200 as se
    from paper_2606_19059_b200 import replicas, workloads as W

    ctx = Ctx()
    ctx.torch, ctx.se, ctx.W, ctx.replicas = torch, se, W, replicas
    ctx.rank, ctx.world, ctx.local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    se.lib()                                          # fail loudly if libse_b200.so is missing
    torch.cuda.set_device(ctx.local)
    distributed = ctx.world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", ctx.local))

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    ctx.barrier = barrier
    ctx.max_over_ranks = lambda v: replicas.aggregate(0.0, v, device="cuda")[1]
    ctx.file_peaks, ctx.traffic = load_peaks(), load_traffic()
    ctx.peaks = measure_peaks(se)
    barrier()

    steps, warmup = args.steps, max(args.warmup, 3)
    res, cfgd, clocks, c = bench_plan(ctx, args.config, steps, warmup, {}, headline=True)
    subs = {}
    if ctx.world == 1 and not args.no_sub and args.config == 3:
        for key, cfg, k, over in SUB_RESULTS:
            try:
                saved = {kk: os.environ.get(kk) for kk in over.get("env", {})}
                os.environ.update(over.get("env", {}))
                try:
                    r, cd, _, _ = bench_plan(ctx, cfg, k, 3, over, headline=False)
                finally:
                    for kk, vv in saved.items():
                        if vv is None:
                            os.environ.pop(kk, None)
                        else:
                            os.environ[kk] = vv
                r["config"] = {kk: cd[kk] for kk in ("N", "xi", "rc", "M", "P", "precision", "window", "gridding", "transforms")}
                subs[key] = r
            except Exception as ex:                      # a sub-result must never cost the headline
                subs[key] = {"error": repr(ex)}
    if distributed:
        dist.barrier()
    if ctx.rank != 0:
        if distributed:
            dist.destroy_process_group()
        return 0

    line = {
        "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": ctx.world, "steps": steps,
        "warmup": warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if c.precision == "fp64" else "f32",
        "data": "synthetic", "config": cfgd, "e2e": res["e2e"], "gpu_launches": res["gpu_launches"],
        "clocks": clocks, "roofline": res["roofline"], "stages_ms": res["stages_ms"],
        "stages_roofline": res["stages_roofline"], "p2p_pairs": res["p2p_pairs"],
        "value_excluding_fft": res["value_excluding_fft"], "finite": res["finite"],
        "peaks": dict(ctx.peaks, hbm_gbs_file=ctx.file_peaks.get("hbm_gbs"),
                      fp64_tflops_nominal=NOMINAL_TFLOPS["fp64"], fp32_tflops_nominal=NOMINAL_TFLOPS["fp32"]),
        "configs": subs,
    }
    if ctx.world == 1 and not args.no_cpu_baseline:
        import oracle
        from paper_2606_19059_b200 import workloads as W2
        oracle.build()
        oc, ox, of = W2.make(args.config)
        t, tm = oracle_step(oc, ox, of)
        line["cpu_baseline"] = {"value": oc.N / t, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle",
                                "sample": f"the bench workload itself, in full ({oc.label}), one evaluation, {t:.1f} s",
                                "stages_s": {k: round(v, 2) for k, v in tm.items()}}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    if distributed:
        dist.destroy_process_group()
    return 0


def run_slabs(args):
    """--mode slabs: ONE evaluation of the config cut into x-slabs, one per rank (paper_2606_19059_b200/
    slabs.py): strong scaling, value = N / time of one evaluation.  Needs torchrun with >= 2 ranks (NCCL).  Not the default
    multi-GPU arm (that is the replica arm, `north_star`: "everything runs on one GPU"): the boxes of this build have one
    GPU, so this arm has only been run through its single-GPU emulation (tests/test_gpu_slabs.py) and under gloo on CPU
    (tests/test_slabs_host.py)."""
    import torch
    import torch.distributed as dist
    import paper_2606_19059_b200 as se
    from paper_2606_19059_b200 import slabs, workloads as W
    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if world < 2:
        raise SystemExit("bench.py --mode slabs needs torchrun with at least 2 ranks")
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c, x, f = W.make(args.config)
    lay = slabs.SlabLayout(c.L, c.M, c.P, c.rc, world)
    mine = np.nonzero(lay.owner(x[:, 0].astype(np.float64)) == rank)[0]
    xd, fd = torch.as_tensor(x[mine], device="cuda"), torch.as_tensor(f[mine], device="cuda")
    ev = slabs.SlabEval(lay, rank, c.xi, precision=c.precision)
    for _ in range(max(args.warmup, 3)):
        u = slabs.evaluate_distributed(ev, xd, fd)
    torch.cuda.synchronize(); dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        u = slabs.evaluate_distributed(ev, xd, fd)
    e1.record()
    torch.cuda.synchronize(); dist.barrier()
    t = torch.tensor([e0.elapsed_time(e1)], device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    fin = torch.tensor([float(torch.isfinite(u).all())], device="cuda")
    dist.all_reduce(fin, op=dist.ReduceOp.MIN)
    ms = float(t[0]) / args.steps
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": c.N / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64" if c.precision == "fp64" else "f32", "data": "synthetic",
            "config": {"workload": c.label, "N": c.N, "xi": c.xi, "rc": c.rc, "M": c.M, "P": c.P, "precision": c.precision,
                       "parallelism": f"x-slabs{world}: ghost sources, ghost planes, slab-decomposed FFT",
                       "planes_per_rank": lay.Ml, "points_rank0": int(len(mine))},
            "finite": bool(fin[0] > 0)}), flush=True)
    ev.destroy()
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
    ap.add_argument("--no-sub", action="store_true", help="skip the sub-results (configs 4, 5, Kaiser-Bessel variants)")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "slabs"],
                    help="multi-GPU arm: independent replicas (default, weak scaling) or one evaluation cut into x-slabs")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.mode == "slabs":
        return run_slabs(args)
    world = env_int("WORLD_SIZE", 1)
    if world == 1 and args.gpus > 1:
        raise SystemExit("bench.py: --gpus %d needs torchrun with --nproc-per-node %d" % (args.gpus, args.gpus))
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
