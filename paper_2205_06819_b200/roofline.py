"""Roofline arithmetic for the fused likelihood kernel.

The path is bound by the plain fp32 ALUs and the special-function unit, not by HBM or the tensor cores.  The unit of
work is one fine cell (one supersampled grid point of one theta, PSF halo included).  Two counts of the ALGORITHMIC
work per cell are kept -- neither is the number of instructions the kernel happens to execute:

  "survey": SURVEY.md sec. 8(d)'s estimate of what the method must compute (the figure `roofline.frac` is quoted on, so
            that rounds stay comparable), made to depend on the components of the model variant:

    part                               fp32 instr (FMA = 1)                MUFU
    a2 geometry                        14                                  2  (rsqrt)
    a2 discs                            3 per disc                         1 per disc (ex2)
    a2 table look-ups                  10 per table: v_c always,           1 per argument (lg2): r always, R with a bulge
                                       Sigma_b and Sigma_b sigma_b^2 with a bulge
    a3 combine                         25                                  4  (2 sqrt, 2 rcp)
    a4+a5 PSF fused with rebin         4 (s+1)(2 r_k+s)/s^2                0
    a6 chi-square                      24/s^2                              0

  "tight":  the exact census of the method AS TABULATED: what one fine cell needs once the radial
            functions are piecewise cubics addressed by the bits of their argument (no logarithm), counted operation
            by operation from the formulas -- geometry 8 + 2/3 (the column's rotation is shared by its s cells: 2/s
            here taken at s = 3), 1 rsqrt; bulge 10 (argument, position in the interval, two cubics, two amplitudes);
            discs 1 + 1 ex2 each; v_c 4; combine 16 + 2 rcp + 1 sqrt with a bulge; without a bulge the common factor
            of the exponentials costs 4 more and 1 ex2.  Four components: 40 + 2/3 fp32 and 6 MUFU.
            PSF and chi-square as above.  `roofline.frac_tight` is quoted on it.

A B200 SM issues 128 fp32 lanes, 16 MUFU results and 64 fp64 lanes per clock; 148 SMs at clocks.max.sm = 1965 MHz
(MEASURED_PEAKS.json "sm_max_mhz") give the peaks below.  fp64 mode: the same census on the fp64 pipe, with each
transcendental expanded to FP64_PER_TRANSCENDENTAL fp64 instructions -- an ASSUMPTION ("~250-300 DP
instr/cell"), flagged as such in the JSON.
"""
from __future__ import annotations

import json
import os

N_SM = 148
FP32_LANES, MUFU_LANES, FP64_LANES = 128, 16, 64
SM_MAX_MHZ_FALLBACK = 1965.0
FP64_PER_TRANSCENDENTAL = 16.0
BULGE, DISC1, DISC2, HALO = 1, 2, 4, 8

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def sm_max_mhz() -> float:
    try:
        with open(os.path.join(_ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"])
    except Exception:
        return SM_MAX_MHZ_FALLBACK


def model_census(comps: int = 15, kind: str = "survey") -> tuple[float, float]:
    """(fp32 instructions, MUFU results) of steps a2 + a3 for one fine cell of a model with the given components."""
    bulge = bool(comps & BULGE)
    ndisc = bool(comps & DISC1) + bool(comps & DISC2)
    if kind == "survey":
        fp32 = 14 + 3 * ndisc + 10 * (1 + 2 * bulge) + 25
        mufu = 2 + ndisc + (1 + bulge) + 4
        return float(fp32), float(mufu)
    if kind == "tight":
        fp32 = (8 + 2.0 / 3.0) + 10 * bulge + ndisc + 4 + 16 + (0 if bulge else 4)
        mufu = 1 + ndisc + 3 + (0 if bulge else 1)
        return float(fp32), float(mufu)
    raise ValueError(kind)


def census(s: int, r_k: int, precision: str = "fp32", comps: int = 15, kind: str = "survey") -> dict:
    """Algorithmic instructions per fine cell."""
    base, mufu = model_census(comps, kind)
    psf = 4.0 * (s + 1) * (2 * r_k + s) / (s * s)
    chi = 24.0 / (s * s)
    fp32 = base + psf + chi
    if precision == "fp64":
        return {"fp64": fp32 + FP64_PER_TRANSCENDENTAL * mufu, "fp32": 0.0, "mufu": 0.0}
    return {"fp32": fp32, "mufu": mufu, "fp64": 0.0}


def clocks_per_cell(s: int, r_k: int, precision: str = "fp32", comps: int = 15, kind: str = "survey") -> float:
    c = census(s, r_k, precision, comps, kind)
    return max(c["fp32"] / FP32_LANES, c["mufu"] / MUFU_LANES, c["fp64"] / FP64_LANES)


def roofline(cells_per_launch: float, seconds_per_launch: float, s: int, r_k: int, precision: str = "fp32",
             sm_mhz_measured: float | None = None, traffic=None, comps: int = 15, fma_pipe_pct=None) -> dict:
    """The `roofline` object of bench.py's JSON line.  achieved and peak count thread-level instructions of the
    binding pipe per second (fp32 ALU lanes, or fp64 lanes in fp64 mode); frac = roofline time / measured time."""
    c = census(s, r_k, precision, comps)
    ct = census(s, r_k, precision, comps, "tight")
    pipe = "fp64" if precision == "fp64" else "fp32"
    lanes = FP64_LANES if precision == "fp64" else FP32_LANES
    fmax = sm_max_mhz() * 1e6
    peak = N_SM * lanes * fmax                               # instr/s of the binding pipe
    t_roof = cells_per_launch * clocks_per_cell(s, r_k, precision, comps) / (N_SM * fmax)
    t_tight = cells_per_launch * clocks_per_cell(s, r_k, precision, comps, "tight") / (N_SM * fmax)
    achieved = cells_per_launch * c[pipe] / seconds_per_launch
    # when MUFU binds harder than the ALU pipe, frac is the time ratio (achieved/peak would overstate the headroom)
    frac = t_roof / seconds_per_launch
    out = {"bound": "alu", "pipe": pipe, "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "Tinstr/s",
           "frac": frac, "frac_tight": t_tight / seconds_per_launch, "traffic": traffic,
           "peak_source": f"derived: {N_SM} SMs x {lanes} {pipe} lanes x {sm_max_mhz():.0f} MHz (clocks.max.sm, MEASURED_PEAKS.json)",
           "census": "survey (SURVEY.md 8d, per component mask); frac_tight: exact census of the tabulated method (DESIGN.md sec. 7)",
           "instr_per_cell": c[pipe], "mufu_per_cell": c["mufu"], "instr_per_cell_tight": ct[pipe], "mufu_per_cell_tight": ct["mufu"],
           "clk_per_cell_roof": clocks_per_cell(s, r_k, precision, comps),
           "clk_per_cell_measured": seconds_per_launch * N_SM * fmax / cells_per_launch,
           "cells_per_launch": cells_per_launch}
    if precision == "fp64":
        out["assumption"] = f"each transcendental counted as {FP64_PER_TRANSCENDENTAL:g} fp64 instructions"
    if fma_pipe_pct is not None:
        out["ncu_sm__pipe_fma_cycles_active_pct"] = fma_pipe_pct
    if sm_mhz_measured:
        out["frac_at_measured_clock"] = frac * sm_max_mhz() / sm_mhz_measured
    return out
