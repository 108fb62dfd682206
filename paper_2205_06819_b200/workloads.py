"""Seeded synthetic workloads for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path (tests, bench.py).
It holds none of the method's arithmetic: it only draws parameter vectors, noise, masks and error
scales from a counter-seeded numpy generator and states the grid / PSF / model settings of each
config.  Model maps are always passed IN (by whoever computed them) to make_data().

The inputs stand in for the paper's CALIFA + SDSS maps of NGC 7683, which are not
available: ~1 arcsec spaxels, Gaussian PSF sigma ~ 1 px, errors 5 % on B, 10 km/s on v and sigma,
0.1 on M/L (BASELINE.json configs; recipe in DESIGN.md "Synthetic inputs").
"""
from __future__ import annotations

import math

import numpy as np

BULGE, DISC1, DISC2, HALO = 1, 2, 4, 8
HALO_HERNQUIST, HALO_NFW = 0, 1
NTHETA = 17
SEED0 = 220506819
N_NEAR_TRUTH = 16

# theta layout (include/bang.h): x0 y0 [arcsec], PA i [deg], log10 Mb, Rb, log10 Md1, Rd1, log10 Md2, Rd2,
# log10 Mh|M200, Rh|c, (M/L)b, (M/L)d1, (M/L)d2, k1, k2
THETA_NAMES = ["x0", "y0", "PA", "inc", "log10Mb", "Rb", "log10Md1", "Rd1", "log10Md2", "Rd2",
               "log10Mh", "Rh_or_c", "MLb", "MLd1", "MLd2", "k1", "k2"]

# BASELINE.json config 1 (given explicitly there); disc 2 and halo are absent (entries ignored)
THETA_TRUE_1 = np.array([0.0, 0.0, 30.0, 60.0, 10.0, 0.8, 10.5, 3.0, 10.0, 5.0, 12.0, 20.0,
                         3.0, 2.0, 2.0, 0.9, 0.9])
# configs 2-5: Table 2 medians, centre (0,0), NFW halo log10 M200 = 12.5, c = 8
THETA_TRUE_4C = np.array([0.0, 0.0, 44.12, math.degrees(math.asin(0.829)), 10.67, 10 ** -0.65,
                          10.42, 10 ** -0.015, 10.865, 10 ** 0.603, 12.5, 8.0, 10.5, 2.12, 2.62, 0.299, 0.700])

# prior box of BASELINE.json config 2 (lo, hi) per theta entry
PRIOR_LO = np.array([-2.0, -2.0, 0.0, 20.0, 8.0, 0.1, 9.0, 0.5, 9.0, 0.5, 10.0, 3.0, 0.5, 0.5, 0.5, 0.0, 0.0])
PRIOR_HI = np.array([2.0, 2.0, 180.0, 80.0, 11.0, 3.0, 11.5, 10.0, 11.5, 10.0, 13.0, 20.0, 5.0, 5.0, 5.0, 1.0, 1.0])

_ALL = BULGE | DISC1 | DISC2 | HALO


def _grid(n, s, sigma, nj, comps, halo, precision):
    return dict(nx=n, ny=n, pix_arcsec=1.0, supersample=s, dist_mpc=50.0, sigma_pix=sigma, trunc_nsigma=3.0,
                components=comps, halo_profile=halo, jeans_nodes=nj, precision=precision)


CONFIGS = {
    1: dict(_grid(32, 2, 1.0, 32, BULGE | DISC1, HALO_HERNQUIST, "fp64"), B=1, name="cfg1_tiny_fp64"),
    2: dict(_grid(64, 3, 1.0, 64, _ALL, HALO_NFW, "fp32"), B=1024, name="cfg2_b1024_64px"),
    3: dict(_grid(128, 3, 1.0, 64, _ALL, HALO_NFW, "fp32"), B=16384, name="cfg3_b16384_128px",
            mask_frac=0.30, err_scale=(0.5, 2.0)),
    4: dict(_grid(80, 3, 1.0, 64, _ALL, HALO_NFW, "fp32"), B=4096, name="cfg4_variants_80px",
            variants={"B+D": BULGE | DISC1, "B+2D": BULGE | DISC1 | DISC2,
                      "2D+H": DISC1 | DISC2 | HALO, "B+2D+H": _ALL}),
    5: dict(_grid(200, 4, 1.5, 128, _ALL, HALO_NFW, "fp32"), B=4096, name="cfg5_stress_200px"),
}


def config(idx: int, variant: str | None = None) -> dict:
    cfg = dict(CONFIGS[idx])
    cfg["index"] = idx
    if variant is not None:
        cfg["components"] = cfg["variants"][variant]
        cfg["variant"] = variant
    return cfg


def theta_true(idx: int) -> np.ndarray:
    return (THETA_TRUE_1 if idx == 1 else THETA_TRUE_4C).copy()


def _streams(idx: int):
    """Independent sub-streams (theta, noise, mask, errors, subset) of the config's seed."""
    ss = np.random.SeedSequence(SEED0 + idx)
    return [np.random.Generator(np.random.PCG64(c)) for c in ss.spawn(5)]


def near_truth_slots(idx: int, B: int) -> np.ndarray:
    """Positions inside the batch that hold the near-truth theta (reading Q)."""
    n = min(N_NEAR_TRUTH, B)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED0 + idx, 77])))
    return np.sort(rng.choice(B, size=n, replace=False))


LOG_MASS_SLOTS = [4, 6, 8, 10]          # theta entries that hold log10 of a mass


def theta_batch(idx: int, B: int | None = None) -> np.ndarray:
    """[B][17] parameter vectors: uniform in the prior box, with 16 vectors within +-1 % of theta_true at seeded
    slots (reading Q): +-1 % on every physical quantity (masses, not their logarithms: log10 M +- log10(1.01)),
    additive +-0.01 arcsec on the centre and +-0.1 deg on the angles.  Config 1: theta_true."""
    cfg = CONFIGS[idx]
    B = cfg["B"] if B is None else B
    if idx == 1:
        return np.repeat(theta_true(1)[None, :], B, axis=0)
    rng = _streams(idx)[0]
    th = PRIOR_LO + (PRIOR_HI - PRIOR_LO) * rng.random((B, NTHETA))
    tt = theta_true(idx)
    slots = near_truth_slots(idx, B)
    u = rng.uniform(-1.0, 1.0, size=(len(slots), NTHETA))
    near = tt * (1.0 + 0.01 * u)
    near[:, LOG_MASS_SLOTS] = tt[LOG_MASS_SLOTS] + np.log10(1.0 + 0.01 * u[:, LOG_MASS_SLOTS])
    near[:, 0:2] = tt[0:2] + 0.01 * u[:, 0:2]
    near[:, 2:4] = tt[2:4] + 0.1 * u[:, 2:4]
    near[:, 15:17] = np.clip(near[:, 15:17], -1.0, 1.0)
    th[slots] = near
    return np.ascontiguousarray(th)


def parity_subset(idx: int, B: int, n: int) -> np.ndarray:
    """Seeded subset of batch indices of size <= n that always contains the near-truth slots."""
    if n >= B:
        return np.arange(B)
    slots = near_truth_slots(idx, B)
    rng = _streams(idx)[4]
    rest = np.setdiff1d(np.arange(B), slots)
    pick = rng.choice(rest, size=max(0, n - len(slots)), replace=False)
    return np.sort(np.concatenate([slots, pick]))


def make_data(idx: int, model_true: np.ndarray):
    """data, err, mask ([4][ny][nx] each) from noise-free model maps of theta_true.

    err nominal = 5 % of B, 10 km/s, 10 km/s, 0.1 (BASELINE.json config 1); config 3 multiplies it per
    pixel by a log-uniform factor in [0.5, 2] and masks a Bernoulli 30 % of the spaxels (same mask for
    the four observables).  data = model + err * N(0,1).
    """
    cfg = CONFIGS[idx]
    model_true = np.asarray(model_true, dtype=np.float64)
    assert model_true.shape == (4, cfg["ny"], cfg["nx"])
    _, rng_noise, rng_mask, rng_err, _ = _streams(idx)
    err = np.empty_like(model_true)
    err[0] = 0.05 * np.abs(model_true[0])
    err[1] = 10.0
    err[2] = 10.0
    err[3] = 0.1
    if "err_scale" in cfg:
        lo, hi = cfg["err_scale"]
        err *= np.exp(rng_err.uniform(math.log(lo), math.log(hi), size=err.shape))
    data = model_true + err * rng_noise.standard_normal(model_true.shape)
    mask = np.ones(model_true.shape, dtype=np.uint8)
    if "mask_frac" in cfg:
        keep = rng_mask.random((cfg["ny"], cfg["nx"])) >= cfg["mask_frac"]
        mask[:] = keep[None, :, :].astype(np.uint8)
    return np.ascontiguousarray(data), np.ascontiguousarray(err), np.ascontiguousarray(mask)
