#!/usr/bin/env python
"""bench.py -- likelihood evaluations per second of the batched BANG likelihood on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4|5] [--precision fp32|fp64]
                    [--impl ours|reference] [--no-sweep]

A "step" is one pass of the whole hot path (decode -> radial table -> fine cells -> PSF + rebin -> masked chi-square)
over one batch of synthetic theta: one bang_loglike call.  Default workload: BASELINE.json configs[1] (B = 1024 theta,
64 x 64 map, x3 supersampling, four-component model, fp32 compute with fp64 logL accumulation).  Prints ONE JSON line.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload instead.
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
def make_context(bang, idx, prec, variant=None, extra=None):
    """Context with synthetic data of the config: model(theta_true) from the library's own fp64 mode + seeded noise.
    extra: overrides of the config (bulge_profile, psf_weighting: the widened variants of SURVEY.md sec. 8f)."""
    cfg = W.config(idx, variant)
    cfg.update(extra or {})
    c64 = bang.Context(dict(W.config(idx), **(extra or {})), precision="fp64")
    mtrue = c64.model_maps(W.theta_true(idx)).cpu().numpy()[0]
    c64.close()
    data, err, mask = W.make_data(idx, mtrue)
    ctx = bang.Context(cfg, precision=prec)
    ctx.set_data(data, err, mask)
    return ctx, cfg


def time_steps(torch, ctx, theta_dev, out, steps, warmup, flush):
    for _ in range(warmup):
        ctx.loglike(theta_dev, out)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    n0 = ctx.launches
    for e0, e1 in ev:
        flush.add_(1.0)                                        # L2 flush: rewrite a 256 MiB buffer (untimed)
        e0.record()
        ctx.loglike(theta_dev, out)
        e1.record()
    torch.cuda.synchronize()
    return [e0.elapsed_time(e1) * 1e-3 for e0, e1 in ev], ctx.launches - n0


def run_ours(args):
    import torch
    rank, world, local = D.env_rank_world()
    if args.gpus > 1 or world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.cuda.current_device()
    from paper_2205_06819_b200 import bang                     # raises if libbang.so is missing: no fallback

    idx, prec = args.config, args.precision
    ctx, cfg = make_context(bang, idx, prec)
    ncell, rk = fine_cells(cfg)
    theta_np = W.theta_batch(idx)                              # weak scaling: every rank runs the full config batch
    B = theta_np.shape[0]
    theta_dev = torch.as_tensor(theta_np, device="cuda")
    out = torch.empty(B, dtype=torch.float64, device="cuda")
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = OracleLeg(idx).sample(15.0)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}

    # end-to-end leg: HOST theta -> bang_loglike_host -> HOST logL (pinned staging, H2D, kernel, D2H inside the call)
    host_out = np.empty(B)
    for _ in range(max(3, args.warmup)):
        ctx.loglike_host(theta_np, host_out)
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    e2e_local = 0.0
    for _ in range(args.steps):
        flush.add_(1.0)                                        # L2 flush between steps, outside the timed call
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.loglike_host(theta_np, host_out)                   # returns after the D2H copy: host wall clock is the cost
        e2e_local += time.perf_counter() - t0
    e2e_t = D.max_over_ranks(e2e_local, device="cuda" if world > 1 else None)

    # device-timed leg
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    with ClockSampler(index=dev) as clk:
        times, launches = time_steps(torch, ctx, theta_dev, out, args.steps, max(3, args.warmup), flush)
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    total = D.max_over_ranks(sum(times), device="cuda" if world > 1 else None)
    ms_step = 1e3 * total / args.steps
    value = world * B * args.steps / total
    clocks = clk.summary()
    assert torch.isfinite(out).all()

    traffic = None                                             # DRAM bytes per k_fused launch from the ncu capture
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["workload"] == workload_name(idx, prec):
                traffic = float(row["dram_bytes_per_launch"])
    roof = R.roofline(B * ncell, statistics.mean(times), cfg["supersample"], rk, prec, clocks.get("sm_mhz"), traffic)
    roof["kernel"] = "k_fused"
    roof["kernel_ms_best"] = 1e3 * min(times)
    # measured counterparts of the derived peaks (dependency-free FFMA / MUFU / DFMA chains, bang_probe_peaks)
    pk = ctx.probe_peaks()
    cen = R.census(cfg["supersample"], rk, prec)
    t_meas = B * ncell * (cen["fp64"] / pk["fp64_fma"] if prec == "fp64"
                          else max(cen["fp32"] / pk["fp32_fma"], cen["mufu"] / pk["mufu"]))
    roof["peaks_measured_Tinstr"] = {k: v / 1e12 for k, v in pk.items()}
    roof["frac_of_measured_peaks"] = t_meas / statistics.mean(times)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if prec == "fp32" else "f64", "data": "synthetic",
            "config": {"workload": workload_name(idx, prec), "B_per_gpu": B, "nx": cfg["nx"], "ny": cfg["ny"],
                       "supersample": cfg["supersample"], "sigma_pix": cfg["sigma_pix"], "r_k": rk,
                       "jeans_nodes": cfg["jeans_nodes"], "fine_cells_per_theta": ncell,
                       "components": "bulge+disc1+disc2+nfw", "logL_accumulation": "f64",
                       "l2": "flushed between timed iterations (256 MiB rewrite)",
                       "parallelism": f"theta-sharded x{world}, no data-path collective"},
            "fine_cell_evals_per_s": value * ncell,
            "e2e": {"value": world * B * args.steps / e2e_t, "unit": UNIT, "h2d_bytes_per_step": B * W.NTHETA * 8,
                    "d2h_bytes_per_step": B * 8},
            "gpu_launches": launches, "clocks": clocks, "roofline": roof}
    if cpu is not None:
        line["cpu_baseline"] = cpu
    ctx.close()

    if rank == 0 and world == 1 and not args.no_sweep:
        sweep = []
        for (i2, p2, var, extra) in [(2, "fp32", None, None), (2, "fp64", None, None), (3, "fp32", None, None),
                                     (3, "fp64", None, None), (4, "fp32", "B+D", None), (4, "fp32", "B+2D", None),
                                     (4, "fp32", "2D+H", None), (4, "fp32", "B+2D+H", None), (5, "fp32", None, None),
                                     (2, "fp32", "jaffe", {"bulge_profile": 1}), (2, "fp32", "fluxpsf", {"psf_weighting": 1})]:
            c2, cf2 = make_context(bang, i2, p2, var if extra is None else None, extra)
            n2, rk2 = fine_cells(cf2)
            th2 = torch.as_tensor(W.theta_batch(i2), device="cuda")
            o2 = torch.empty(th2.shape[0], dtype=torch.float64, device="cuda")
            ts, _ = time_steps(torch, c2, th2, o2, 5, 3, flush)
            r2 = R.roofline(th2.shape[0] * n2, statistics.mean(ts), cf2["supersample"], rk2, p2)
            sweep.append({"workload": workload_name(i2, p2) + (f"_{var}" if var else ""), "B": th2.shape[0],
                          "ms_per_step": 1e3 * statistics.mean(ts), "evals_per_s": th2.shape[0] / statistics.mean(ts),
                          "roofline_frac": r2["frac"], "clk_per_cell": r2["clk_per_cell_measured"]})
            if extra and extra.get("psf_weighting"):
                sweep[-1]["note"] = "side variant, run UNFUSED through HBM scratch (DESIGN.md sec. 11): not the tuned path"
            c2.close()
        line["sweep"] = sweep
    if rank == 0:
        print(json.dumps(line))
    if torch.distributed.is_available() and torch.distributed.is_initialized():
        torch.distributed.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4, 5])
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64"])
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
