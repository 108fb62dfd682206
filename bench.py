#!/usr/bin/env python
"""bench.py -- likelihood evaluations per second of the batched BANG likelihood on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4|5] [--precision fp32|fp64]
                    [--impl ours|reference] [--scaling weak|strong] [--no-sweep] [--no-cpu]

A "step" is one pass of the whole hot path (decode -> radial table -> fine cells -> PSF + rebin -> masked chi-square)
over one batch of synthetic theta: one bang_loglike call.  Default workload: BASELINE.json configs[2], the live-point
batch (B = 16384 theta, 128 x 128 map, 30 % mask, x3 supersampling, four-component model, fp32 compute with fp64 logL
accumulation) -- the largest batch of the single-GPU configs; configs 2, 3 (fp64), 4 (four variants) and 5 follow as
`sweep` rows, each with its own steps, clocks, end-to-end figure and roofline.  Prints ONE JSON line.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload instead.
`--scaling strong` (N > 1) shards ONE config batch over the ranks and all-gathers logL (dist.loglike_sharded).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2205_06819_b200 import dist as D          # noqa: E402
from paper_2205_06819_b200 import roofline as R      # noqa: E402
from paper_2205_06819_b200 import workloads as W     # noqa: E402

METRIC = "likelihood evals/sec (batched theta)"
UNIT = "evals/s"


def workload_name(idx, prec):
    return f"{W.CONFIGS[idx]['name']}_{prec}"


def fine_cells(cfg):
    s = cfg["supersample"]
    rk = int(np.ceil(cfg.get("trunc_nsigma", 3.0) * cfg["sigma_pix"] * s - 1e-9))
    return (cfg["nx"] * s + 2 * rk) * (cfg["ny"] * s + 2 * rk), rk


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.01):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        self._period = period
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:                                   # no NVML: say so in the JSON
            self.err = repr(e)

    def _once(self):
        nv = self.nv
        self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        try:
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "app_clocks", 0x10: "sync_boost"}
        for bit, name in names.items():
            if r & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            time.sleep(self._period)

    def __enter__(self):
        if self.ok:
            self._once()
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        return self

    def __exit__(self, *a):
        if self.ok:
            self._stop.set()
            self.t.join()
            self._once()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML unavailable"}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ CPU oracle legs
class OracleLeg:
    """The oracle, as it stands, on bounded samples of the workload's theta (all host cores through its OpenMP loop)."""

    def __init__(self, idx, variant=None):
        from oracle import bang_oracle as bo                # the ONLY place bench.py touches oracle/
        self.bo, self.idx = bo, idx
        self.cfg = W.config(idx, variant)
        self.theta = W.theta_batch(idx)
        mtrue = bo.model_maps(W.theta_true(idx), W.config(idx))[0]
        self.data, self.err, self.mask = W.make_data(idx, mtrue)
        self.run(np.arange(1))                               # first call: library load, thread pool
        npilot = min(8, self.theta.shape[0])
        self.t1 = self.run(np.arange(npilot)) / npilot       # seconds per theta, for sizing the samples

    def run(self, sub):
        t0 = time.perf_counter()
        ll = self.bo.loglike(self.theta[sub], self.cfg, self.data, self.err, self.mask)
        dt = time.perf_counter() - t0
        assert np.isfinite(ll).all()
        return dt

    def single_thread(self):
        """one theta, one thread."""
        n0 = self.bo.get_threads()
        self.bo.set_threads(1)
        try:
            dt = self.run(np.arange(1))
        finally:
            self.bo.set_threads(n0)
        return {"value": 1.0 / dt, "unit": UNIT, "cores": 1, "sample": f"1 theta, 1 thread, {dt:.2f} s wall"}

    def sample(self, budget_s, offset=0, max_n=4096):
        n = int(max(1, min(max_n, budget_s / max(self.t1, 1e-3))))
        B = self.theta.shape[0]
        sub = (offset + np.arange(n)) % B
        dt = self.run(sub)
        return {"value": n / dt, "unit": UNIT, "cores": self.bo.get_threads(), "kind": "oracle",
                "sample": f"{n} of {B} theta of {W.CONFIGS[self.idx]['name']}, fp64, {dt:.1f} s wall", "seconds": dt, "n": n}


def run_reference(args):
    rank, world, _ = D.env_rank_world()
    if rank != 0:
        return
    idx = args.config
    leg = OracleLeg(idx)
    budget = min(15.0, 150.0 / max(1, args.steps + args.warmup))     # the whole run ends within a few minutes
    per_step, last = [], None
    for i in range(args.warmup + args.steps):
        last = leg.sample(budget, offset=i * 64)
        if i >= args.warmup:
            per_step.append(last)
    tot_n = sum(p["n"] for p in per_step)
    tot_t = sum(p["seconds"] for p in per_step)
    value = tot_n / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, len(per_step)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(idx, args.precision), "theta_per_step": last["n"],
                       "note": "CPU oracle (fp64) on a bounded sample of the workload's theta per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ GPU legs
COMP_NAMES = {1: "bulge", 2: "disc1", 4: "disc2", 8: "nfw"}


def comp_string(comps):
    return "+".join(n for b, n in COMP_NAMES.items() if comps & b)


def make_context(bang, idx, prec, device, variant=None, extra=None):
    """Context with synthetic data of the config: model(theta_true) from the library's own fp64 mode + seeded noise.
    extra: overrides of the config (bulge_profile, psf_weighting: the widened variants of SURVEY.md sec. 8f)."""
    cfg = W.config(idx, variant)
    cfg.update(extra or {})
    c64 = bang.Context(dict(W.config(idx), **(extra or {})), precision="fp64", device=device)
    mtrue = c64.model_maps(W.theta_true(idx)).cpu().numpy()[0]
    c64.close()
    data, err, mask = W.make_data(idx, mtrue)
    ctx = bang.Context(cfg, precision=prec, device=device)
    ctx.set_data(data, err, mask)
    return ctx, cfg


def time_steps(torch, ctx, theta_dev, out, steps, warmup, flush):
    """CUDA events on the context's stream (the stream the kernels are launched on) around each bang_loglike call."""
    assert theta_dev.device == ctx.device == out.device == flush.device
    stream = ctx.stream
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            ctx.loglike(theta_dev, out)
        stream.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        n0 = ctx.launches
        for e0, e1 in ev:
            flush.add_(1.0)                                    # L2 flush: rewrite a 256 MiB buffer (untimed)
            e0.record(stream)
            ctx.loglike(theta_dev, out)
            e1.record(stream)
        stream.synchronize()
    return [e0.elapsed_time(e1) * 1e-3 for e0, e1 in ev], ctx.launches - n0


def time_e2e(torch, ctx, theta_np, steps, warmup, flush):
    """HOST theta -> bang_loglike_host -> HOST logL (pinned staging, H2D, kernels, D2H inside the call): host wall
    clock per call; the L2 flush between calls is not timed."""
    host_out = np.empty(theta_np.shape[0])
    for _ in range(warmup):
        ctx.loglike_host(theta_np, host_out)
    total = 0.0
    for _ in range(steps):
        flush.add_(1.0)
        torch.cuda.synchronize(ctx.device)
        t0 = time.perf_counter()
        ctx.loglike_host(theta_np, host_out)
        total += time.perf_counter() - t0
    assert np.isfinite(host_out).all()
    return total


def profile_numbers(name):
    """DRAM bytes per k_fused launch and FMA-pipe utilisation from the committed ncu captures (profiles/traffic.csv)."""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["workload"] == name:
                fma = row.get("fma_pipe_pct")
                return float(row["dram_bytes_per_launch"]), (float(fma) if fma not in (None, "") else None)
    return None, None


def measure(torch, bang, idx, prec, device, flush, steps, warmup, variant=None, extra=None, world=1, tag=None):
    """One workload: device-timed steps (+ clocks), the end-to-end leg and the roofline object."""
    ctx, cfg = make_context(bang, idx, prec, device, variant, extra)
    ncell, rk = fine_cells(cfg)
    theta_np = W.theta_batch(idx)
    B = theta_np.shape[0]
    theta_dev = torch.as_tensor(theta_np, device=ctx.device)
    out = torch.empty(B, dtype=torch.float64, device=ctx.device)
    e2e_t = D.max_over_ranks(time_e2e(torch, ctx, theta_np, steps, max(3, warmup), flush), device="cuda" if world > 1 else None)
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize(ctx.device)
    with ClockSampler(index=device) as clk:
        times, launches = time_steps(torch, ctx, theta_dev, out, steps, max(3, warmup), flush)
    torch.cuda.synchronize(ctx.device)
    if world > 1:
        torch.distributed.barrier()
    assert torch.isfinite(out).all()
    total = D.max_over_ranks(sum(times), device="cuda" if world > 1 else None)
    name = workload_name(idx, prec) + (f"_{tag or variant}" if (tag or variant) else "")
    clocks = clk.summary()
    res = {"workload": name, "B": B, "steps": steps, "ms_per_step": 1e3 * total / steps,
           "value": world * B * steps / total, "ncell": ncell, "rk": rk, "cfg": cfg, "launches": launches,
           "e2e": {"value": world * B * steps / e2e_t, "unit": UNIT, "h2d_bytes_per_step": B * W.NTHETA * 8,
                   "d2h_bytes_per_step": B * 8},
           "clocks": clocks}
    traffic, fma = profile_numbers(name)
    mean_t = total / steps
    roof = R.roofline(B * ncell, mean_t, cfg["supersample"], rk, prec, clocks.get("sm_mhz"), traffic,
                      comps=cfg["components"], fma_pipe_pct=fma)
    roof["kernel"] = "k_fused"
    roof["kernel_ms_best"] = 1e3 * min(times)
    roof["kernel_ms_median"] = 1e3 * statistics.median(times)
    res["roofline"] = roof
    res["ctx"] = ctx
    return res


SWEEP = [  # (config, precision, config-4 variant, overrides, tag)
    (2, "fp32", None, None, None), (2, "fp64", None, None, None), (3, "fp64", None, None, None),
    (4, "fp32", "B+D", None, None), (4, "fp32", "B+2D", None, None), (4, "fp32", "2D+H", None, None),
    (4, "fp32", "B+2D+H", None, None), (5, "fp32", None, None, None),
    (2, "fp32", None, {"bulge_profile": 1}, "jaffe"), (2, "fp32", None, {"psf_weighting": 1}, "fluxpsf"),
    (2, "fp32", None, {"bulge_potential": 1}, "totalpot"),
]


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start the N ranks ourselves (same contract as the driver's launch)."""
    import subprocess
    port = 29500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def run_ours(args):
    import torch
    rank, world, local = D.env_rank_world()
    if args.gpus > 1 and world == 1:
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {torch.cuda.device_count()} CUDA device(s) visible")
        spawn_ranks(args)
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = local if world > 1 else torch.cuda.current_device()
    from paper_2205_06819_b200 import bang                     # raises if libbang.so is missing: no fallback

    idx, prec = args.config, args.precision
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device=torch.device("cuda", dev))

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        leg = OracleLeg(idx)
        s = leg.sample(15.0)
        cpu = {k: s[k] for k in ("value", "unit", "cores", "kind", "sample")}
        cpu["single_thread"] = leg.single_thread()
        cpu["note"] = ("the oracle as it stands: direct evaluation per fine cell (N_J-node quadrature and 8 Bessel calls per "
                       "cell, no tables), not an optimised CPU implementation")

    if args.scaling == "strong" and world > 1:
        line = run_strong(torch, bang, args, idx, prec, dev, flush, rank, world)
    else:
        m = measure(torch, bang, idx, prec, dev, flush, args.steps, args.warmup, world=world,
                    variant="B+2D+H" if idx == 4 else None)
        cfg, ctx = m["cfg"], m["ctx"]
        roof = m["roofline"]
        # measured counterparts of the derived peaks (dependency-free FFMA / MUFU / DFMA chains, bang_probe_peaks)
        pk = ctx.probe_peaks()
        cen = R.census(cfg["supersample"], m["rk"], prec, cfg["components"])
        t_meas = m["B"] * m["ncell"] * (cen["fp64"] / pk["fp64_fma"] if prec == "fp64"
                                        else max(cen["fp32"] / pk["fp32_fma"], cen["mufu"] / pk["mufu"]))
        roof["peaks_measured_Tinstr"] = {k: v / 1e12 for k, v in pk.items()}
        roof["frac_of_measured_peaks"] = t_meas / (1e-3 * m["ms_per_step"])
        ctx.close()
        line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": m["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32" if prec == "fp32" else "f64", "data": "synthetic",
                "config": {"workload": m["workload"], "B_per_gpu": m["B"], "nx": cfg["nx"], "ny": cfg["ny"],
                           "supersample": cfg["supersample"], "sigma_pix": cfg["sigma_pix"], "r_k": m["rk"],
                           "jeans_nodes": cfg["jeans_nodes"], "fine_cells_per_theta": m["ncell"],
                           "components": comp_string(cfg["components"]), "logL_accumulation": "f64",
                           "mask_frac": cfg.get("mask_frac", 0.0), "seed": W.SEED0 + idx,
                           "l2": "flushed between timed iterations (256 MiB rewrite)",
                           "parallelism": f"theta-sharded x{world}, every rank runs the config batch, no data-path collective"},
                "fine_cell_evals_per_s": m["value"] * m["ncell"], "e2e": m["e2e"], "gpu_launches": m["launches"],
                "clocks": m["clocks"], "roofline": roof}
    if cpu is not None:
        line["cpu_baseline"] = cpu

    if rank == 0 and world == 1 and not args.no_sweep:
        sweep = []
        for (i2, p2, var, extra, tag) in SWEEP:
            if (i2, p2) == (idx, prec) and var is None and extra is None:
                continue
            r = measure(torch, bang, i2, p2, dev, flush, max(20, min(args.steps, 50)), 3, var, extra, tag=tag)
            r.pop("ctx").close()
            r.pop("cfg")
            row = {"workload": r["workload"], "B": r["B"], "steps": r["steps"], "ms_per_step": r["ms_per_step"],
                   "evals_per_s": r["value"], "e2e": r["e2e"], "clocks": r["clocks"], "gpu_launches": r["launches"]}
            row["roofline"] = r["roofline"]
            row["roofline_frac"] = r["roofline"]["frac"]
            if extra:
                row["note"] = "widened variant (SURVEY.md sec. 8f): the census is the paper's path's, so frac understates the work done"
            sweep.append(row)
        line["sweep"] = sweep
    if rank == 0:
        print(json.dumps(line))
    if torch.distributed.is_available() and torch.distributed.is_initialized():
        torch.distributed.destroy_process_group()


def run_strong(torch, bang, args, idx, prec, dev, flush, rank, world):
    """SURVEY.md sec. 8(e) as one call: shard theta[B] over the ranks, evaluate, all-gather logL (strong scaling)."""
    ctx, cfg = make_context(bang, idx, prec, dev, "B+2D+H" if idx == 4 else None)
    ncell, rk = fine_cells(cfg)
    theta_np = W.theta_batch(idx)
    B = theta_np.shape[0]
    theta_dev = torch.as_tensor(theta_np, device=ctx.device)
    for _ in range(max(3, args.warmup)):
        full = D.loglike_sharded(ctx, theta_dev)
    torch.cuda.synchronize(ctx.device)
    torch.distributed.barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    with ClockSampler(index=dev) as clk:
        for e0, e1 in ev:
            flush.add_(1.0)
            e0.record()
            full = D.loglike_sharded(ctx, theta_dev)
            e1.record()
        torch.cuda.synchronize(ctx.device)
    torch.distributed.barrier()
    assert full.shape == (B,) and torch.isfinite(full).all()
    total = D.max_over_ranks(sum(e0.elapsed_time(e1) * 1e-3 for e0, e1 in ev), device="cuda")
    lo, hi = D.shard_bounds(B, rank, world)
    roof = R.roofline(B * ncell / world, total / args.steps, cfg["supersample"], rk, prec, clk.summary().get("sm_mhz"),
                      None, comps=cfg["components"])
    roof["kernel"] = "k_fused"
    ctx.close()
    return {"metric": METRIC, "value": B * args.steps / total, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32" if prec == "fp32" else "f64", "data": "synthetic",
            "config": {"workload": workload_name(idx, prec), "B_total": B, "B_per_gpu": hi - lo, "nx": cfg["nx"], "ny": cfg["ny"],
                       "supersample": cfg["supersample"], "fine_cells_per_theta": ncell,
                       "l2": "flushed between timed iterations (256 MiB rewrite)",
                       "parallelism": f"ONE batch sharded x{world} (dist.loglike_sharded), all-gather of logL inside the timed region"},
            "fine_cell_evals_per_s": B * args.steps / total * ncell,
            "e2e": {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                    "note": "not measured in the strong-scaling mode"},
            "gpu_launches": 2 * args.steps, "clocks": clk.summary(), "roofline": roof}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[2, 3, 4, 5])
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
