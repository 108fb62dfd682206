"""Roofline arithmetic for the fused likelihood kernel.

The path is bound by the plain fp32 ALUs and the special-function unit, not by HBM or the tensor cores.  The unit of
work is one fine cell (one supersampled grid point of one theta, PSF halo included).  The ALGORITHMIC work per cell is
SURVEY.md sec. 8(d)'s census of what the method must compute -- not the instructions the kernel happens to execute:

    part                               fp32 instr (FMA = 1)        MUFU
    a2 geometry                        14                          2  (rsqrt)
    a2 discs                            6                          2  (ex2)
    a2 table look-ups                  30                          2  (lg2)
    a3 combine                         25                          4  (2 sqrt, 2 rcp)
    a4+a5 PSF fused with rebin         4 (s+1)(2 r_k+s)/s^2        0
    a6 chi-square                      24/s^2                      0

A B200 SM issues 128 fp32 lanes, 16 MUFU results and 64 fp64 lanes per clock; 148 SMs at clocks.max.sm = 1965 MHz
(MEASURED_PEAKS.json "sm_max_mhz") give the peaks below.  fp64 mode: the same census on the fp64 pipe, with each of the
10 transcendentals expanded to 16 fp64 instructions ("~250-300 DP instr/cell").
"""
from __future__ import annotations

import json
import os

N_SM = 148
FP32_LANES, MUFU_LANES, FP64_LANES = 128, 16, 64
SM_MAX_MHZ_FALLBACK = 1965.0

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def sm_max_mhz() -> float:
    try:
        with open(os.path.join(_ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"])
    except Exception:
        return SM_MAX_MHZ_FALLBACK


def census(s: int, r_k: int, precision: str = "fp32") -> dict:
    """Algorithmic instructions per fine cell."""
    base = 14 + 6 + 30 + 25
    psf = 4.0 * (s + 1) * (2 * r_k + s) / (s * s)
    chi = 24.0 / (s * s)
    fp32 = base + psf + chi
    mufu = 10.0
    if precision == "fp64":
        return {"fp64": fp32 + 16.0 * mufu, "fp32": 0.0, "mufu": 0.0}
    return {"fp32": fp32, "mufu": mufu, "fp64": 0.0}


def clocks_per_cell(s: int, r_k: int, precision: str = "fp32") -> float:
    c = census(s, r_k, precision)
    return max(c["fp32"] / FP32_LANES, c["mufu"] / MUFU_LANES, c["fp64"] / FP64_LANES)


def roofline(cells_per_launch: float, seconds_per_launch: float, s: int, r_k: int, precision: str = "fp32",
             sm_mhz_measured: float | None = None, traffic=None) -> dict:
    """The `roofline` object of bench.py's JSON line.  achieved and peak count thread-level instructions of the
    binding pipe per second (fp32 ALU lanes, or fp64 lanes in fp64 mode); frac = roofline time / measured time."""
    c = census(s, r_k, precision)
    pipe = "fp64" if precision == "fp64" else "fp32"
    lanes = FP64_LANES if precision == "fp64" else FP32_LANES
    fmax = sm_max_mhz() * 1e6
    peak = N_SM * lanes * fmax                               # instr/s of the binding pipe
    t_roof = cells_per_launch * clocks_per_cell(s, r_k, precision) / (N_SM * fmax)
    achieved = cells_per_launch * c[pipe] / seconds_per_launch
    # when MUFU binds harder than the ALU pipe, frac is the time ratio (achieved/peak would overstate the headroom)
    frac = t_roof / seconds_per_launch
    out = {"bound": "alu", "pipe": pipe, "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "Tinstr/s",
           "frac": frac, "traffic": traffic,
           "peak_source": f"derived: {N_SM} SMs x {lanes} {pipe} lanes x {sm_max_mhz():.0f} MHz (clocks.max.sm, MEASURED_PEAKS.json)",
           "instr_per_cell": c[pipe], "mufu_per_cell": c["mufu"], "clk_per_cell_roof": clocks_per_cell(s, r_k, precision),
           "clk_per_cell_measured": seconds_per_launch * N_SM * fmax / cells_per_launch,
           "cells_per_launch": cells_per_launch}
    if sm_mhz_measured:
        out["frac_at_measured_clock"] = frac * sm_max_mhz() / sm_mhz_measured
    return out
