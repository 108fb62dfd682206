"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 CPU oracle, element by
element on the same seeded inputs, for the five BASELINE.json configs, plus properties that hold at full size.

Sample sizes are SURVEY.md sec. 8(d)'s "Parity sample": ALL theta of configs 1 and 2; seeded subsets (always holding
the 16 near-truth theta) of 256 theta for config 3 (both precisions) and for each config-4 variant, 64 for config 5 --
sized so that the oracle's share stays near two minutes on the GPU box's 16 host cores.

Tolerances (BASELINE.json north_star; readings P and Q), written out here:
  maps, fp64 mode: |g-o| <= 1e-9 |o| per pixel;  fp32 mode: <= 1e-4 |o|;
        v_los crosses zero, so its denominator is max(|o|, 1e-3 max_map|o|) (reading P);
        fp32 B: plus an absolute floor of 1e-30 (fp32 cannot hold the oracle's values below ~1e-38);
  logL, fp32 mode: |dlogL| <= 1e-3 sqrt(N_pix) for the near-truth theta (N_pix = used spaxels per map), and for every
        theta the first-order bound implied by the per-pixel tolerance, |dlogL| <= 1e-4 sum_p |z_p| |m_p| / e_p;
  logL, fp64 mode: the same first-order bound with 1e-9.
  Both logL bounds add the floor of an fp64 sum taken in another order, N 2^-53 sum_p |term_p| (reading Q); the
  first-order bound uses reading P's denominator for v_los, as the per-pixel map tolerance does.
"""
N_PARITY = {2: 1024, 3: 256, 4: 256, 5: 64}
import math

import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL = {"fp64": 1e-9, "fp32": 1e-4}


@pytest.fixture(scope="module")
def bang():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_2205_06819_b200 import bang as b
    b.lib()                                    # fails loudly if libbang.so is missing
    return b


def assert_maps(g, o, prec, what=""):
    g = np.asarray(g, dtype=np.float64)
    o = np.asarray(o, dtype=np.float64)
    assert g.shape == o.shape
    rtol = RTOL[prec]
    worst = []
    for q in range(4):
        gq, oq = g[..., q, :, :], o[..., q, :, :]
        den = np.abs(oq)
        if q == 1:
            den = np.maximum(den, 1e-3 * np.abs(oq).max(axis=(-2, -1), keepdims=True))
        atol = 1e-30 if (prec == "fp32" and q == 0) else 0.0
        bad = np.abs(gq - oq) > rtol * den + atol
        worst.append(float(np.max(np.abs(gq - oq) / (den + atol + 1e-300))))
        assert not bad.any(), f"{what} map {q}: {bad.sum()} pixels beyond {rtol:g}, worst {worst[-1]:.3e}"
    return worst


def first_order_bound(maps_o, data, err, mask):
    """sum_p |z_p| den_p / e_p over used pixels (reading Q), per theta: the change of logL when every model pixel moves by
    its full per-pixel tolerance rtol den_p, den_p = |m_p| (v_los: max(|m_p|, 1e-3 max_map |m|), reading P)."""
    den = np.abs(maps_o).copy()
    den[..., 1, :, :] = np.maximum(den[..., 1, :, :], 1e-3 * den[..., 1, :, :].max(axis=(-2, -1), keepdims=True))
    z = np.abs((data - maps_o) / err) * den / err
    return (z * mask).sum(axis=(-3, -2, -1))


def summation_floor(maps_o, data, err, mask):
    """Rounding of the fp64 sum of eq. 18 taken in another order (the kernel: per thread, per warp, per block; the oracle:
    pixel by pixel): <= N 2^-53 sum_p |term_p|, terms 1/2 z_p^2 and 1/2 ln(2 pi e_p^2)  (reading Q)."""
    z = (data - maps_o) / err
    terms = (0.5 * z * z + np.abs(0.5 * np.log(2 * np.pi * err * err))) * mask
    return mask.sum() * 2.0 ** -53 * terms.sum(axis=(-3, -2, -1))


def assert_logl(g, o, maps_o, data, err, mask, prec, near=None, what=""):
    g, o = np.asarray(g), np.asarray(o)
    bound = RTOL[prec] * first_order_bound(maps_o, data, err, mask) + summation_floor(maps_o, data, err, mask)
    d = np.abs(g - o)
    assert (d <= bound).all(), f"{what}: |dlogL| {d.max():.3e} beyond first-order bound (worst ratio {(d / bound).max():.3e})"
    if near is not None and prec == "fp32" and near.any():
        npix = mask[0].sum()
        lim = 1e-3 * math.sqrt(npix)
        assert (d[near] <= lim).all(), f"{what}: near-truth |dlogL| {d[near].max():.3e} > 1e-3 sqrt(N_pix) = {lim:.3e}"
    return float(d.max())


class Case:
    """Seeded inputs + oracle results for one config (or one config-4 variant) on a parity subset of the batch."""

    def __init__(self, oracle, idx, nsub, variant=None):
        self.idx, self.variant = idx, variant
        self.cfg = W.config(idx, variant)
        richest = W.config(idx)                               # data come from the richest model (config 4)
        self.theta = W.theta_batch(idx)
        self.B = self.theta.shape[0]
        self.sub = W.parity_subset(idx, self.B, nsub)
        slots = W.near_truth_slots(idx, self.B)
        self.near = np.isin(self.sub, slots) if (idx != 1 and variant in (None, "B+2D+H")) else np.zeros(len(self.sub), bool)
        mtrue = oracle.model_maps(W.theta_true(idx), richest)[0]
        self.data, self.err, self.mask = W.make_data(idx, mtrue)
        self.logl_o, self.maps_o = oracle.loglike(self.theta[self.sub], self.cfg, self.data, self.err, self.mask,
                                                  return_maps=True)


_cases = {}


def get_case(oracle, idx, nsub, variant=None):
    key = (idx, variant)
    if key not in _cases:
        _cases[key] = Case(oracle, idx, nsub, variant)
    return _cases[key]


def run_case(bang, case, prec, full_batch):
    import torch
    ctx = bang.Context(case.cfg, precision=prec)
    ctx.set_data(case.data, case.err, case.mask)
    th_sub = case.theta[case.sub]
    maps = ctx.model_maps(th_sub).cpu().numpy()
    if full_batch:                                           # bench.py's launch configuration: the whole batch at once
        ll_all = ctx.loglike(torch.as_tensor(case.theta, device="cuda")).cpu().numpy()
        ll = ll_all[case.sub]
    else:
        ll_all = None
        ll = ctx.loglike(th_sub).cpu().numpy()
    ctx.close()
    return maps, ll, ll_all


# ------------------------------------------------------------------------------------------------ config 1
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_config1_tiny(bang, oracle, prec):
    case = get_case(oracle, 1, 1)
    ctx = bang.Context(case.cfg, precision=prec)
    # intermediate of steps a0-a3: the un-convolved fine maps (Alg. 1 line 3)
    fine = ctx.model_fine(case.theta[:1]).cpu().numpy()[0]
    fine_o = oracle.model_fine(case.theta[0], case.cfg)
    assert fine.shape == fine_o.shape == (4, 32 * 2 + 12, 32 * 2 + 12)
    assert_maps(fine, fine_o, prec, "fine")
    ctx.close()
    maps, ll, _ = run_case(bang, case, prec, full_batch=False)
    assert_maps(maps, case.maps_o, prec, "maps")
    assert_logl(ll, case.logl_o, case.maps_o, case.data, case.err, case.mask, prec, near=np.array([True]), what="cfg1")


def test_config1_matches_the_survey_crosscheck_pixels(bang):
    # tests/golden/config1_survey_crosscheck.txt: an independent prototype's values
    import os
    ctx = bang.Context(W.config(1), precision="fp64")
    m = ctx.model_maps(W.theta_true(1)).cpu().numpy()[0]
    ctx.close()
    path = os.path.join(os.path.dirname(__file__), "golden", "config1_survey_crosscheck.txt")
    for line in open(path):
        if line.startswith("#"):
            continue
        i, j, *vals = line.split()
        for q, v in enumerate(vals):
            assert abs(m[q, int(i), int(j)] / float(v) - 1) < 1e-9


# ------------------------------------------------------------------------------------------------ configs 2, 3, 5
@pytest.mark.parametrize("idx,nsub,prec", [(2, N_PARITY[2], "fp32"), (2, N_PARITY[2], "fp64"), (3, N_PARITY[3], "fp32"),
                                           (3, N_PARITY[3], "fp64"), (5, N_PARITY[5], "fp32")])
def test_config_batches_against_oracle(bang, oracle, idx, nsub, prec):
    case = get_case(oracle, idx, nsub)
    full = prec == "fp32" or idx == 2
    maps, ll, ll_all = run_case(bang, case, prec, full_batch=full)
    assert_maps(maps, case.maps_o, prec, f"cfg{idx}")
    assert_logl(ll, case.logl_o, case.maps_o, case.data, case.err, case.mask, prec, near=case.near, what=f"cfg{idx}")
    if ll_all is not None:
        assert ll_all.shape == (case.B,) and np.isfinite(ll_all).all()


# ------------------------------------------------------------------------------------------------ config 4
@pytest.mark.parametrize("variant", ["B+D", "B+2D", "2D+H", "B+2D+H"])
def test_config4_model_variants(bang, oracle, variant):
    case = get_case(oracle, 4, N_PARITY[4], variant)
    maps, ll, ll_all = run_case(bang, case, "fp32", full_batch=True)
    assert_maps(maps, case.maps_o, "fp32", variant)
    assert_logl(ll, case.logl_o, case.maps_o, case.data, case.err, case.mask, "fp32", near=case.near, what=variant)
    assert np.isfinite(ll_all).all()
    if variant == "B+2D+H":           # the model that generated the data explains it best near the truth
        others = [get_case(oracle, 4, N_PARITY[4], v) for v in ("B+D", "2D+H")]
        for o in others:
            assert case.logl_o[case.near].max() > o.logl_o.max()


# ------------------------------------------------------------------------------------------------ properties at full size
@pytest.mark.parametrize("idx", [2, 3, 4, 5])
def test_fp32_and_fp64_modes_agree_on_the_whole_batch(bang, oracle, idx):
    import torch
    case = get_case(oracle, idx, N_PARITY[idx], "B+2D+H" if idx == 4 else None)
    B = case.B if idx != 5 else 1024
    th = torch.as_tensor(case.theta[:B], device="cuda")
    out = {}
    for prec in ("fp32", "fp64"):
        ctx = bang.Context(case.cfg, precision=prec)
        ctx.set_data(case.data, case.err, case.mask)
        out[prec] = ctx.loglike(th).cpu().numpy()
        ctx.close()
    assert np.isfinite(out["fp64"]).all()
    rel = np.abs(out["fp32"] - out["fp64"]) / np.abs(out["fp64"])
    assert rel.max() < 2e-5, rel.max()          # far from the truth logL ~ -1e8: a 1e-4 per-pixel tolerance allows ~2e-4


def test_batch_results_do_not_depend_on_batch_size_or_order(bang, oracle):
    import torch
    case = get_case(oracle, 2, N_PARITY[2])
    ctx = bang.Context(case.cfg, precision="fp32")
    ctx.set_data(case.data, case.err, case.mask)
    th = torch.as_tensor(case.theta, device="cuda")
    a = ctx.loglike(th).cpu().numpy()
    b = ctx.loglike(th).cpu().numpy()
    assert np.array_equal(a, b)                                     # deterministic
    perm = np.random.default_rng(0).permutation(case.B)
    c = ctx.loglike(th[torch.as_tensor(perm, device="cuda")]).cpu().numpy()
    assert np.array_equal(c, a[perm])                               # each theta independent of its neighbours
    d = ctx.loglike(th[:37]).cpu().numpy()
    assert np.array_equal(d, a[:37])
    e = ctx.loglike_host(case.theta[:100])
    assert np.array_equal(e, a[:100])                               # host-buffer entry point, same kernels
    ctx.close()


def test_logl_equals_likelihood_of_the_returned_maps(bang, oracle):
    # eq. 18 on the library's own maps, evaluated by the oracle's step 11: ties bang_loglike to bang_model_maps
    case = get_case(oracle, 3, N_PARITY[3])
    ctx = bang.Context(case.cfg, precision="fp64")
    ctx.set_data(case.data, case.err, case.mask)
    th = case.theta[case.sub][:6]
    maps = ctx.model_maps(th).cpu().numpy()
    ll = ctx.loglike(th).cpu().numpy()
    ctx.close()
    for b in range(len(th)):
        want = oracle.loglike_of_maps(maps[b], case.data, case.err, case.mask)
        assert abs(ll[b] - want) <= 1e-12 * abs(want)


# ------------------------------------------------------------------------------------------------ Jaffe bulge (App. B)
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_jaffe_bulge_config1_grid(bang, oracle, prec):
    # BASELINE.json config 1 with the bulge profile switched to Jaffe: fine maps, maps and logL
    cfg = dict(W.config(1), bulge_profile=1)
    theta = np.stack([W.theta_true(1), W.theta_true(1) * 1.01, W.theta_true(1) * 0.99])
    theta[1, 0:2] = 0.37, -0.21                              # off-centre: the 1/R cusp is sampled asymmetrically
    logl_o, maps_o = None, oracle.model_maps(theta, cfg)
    data, err, mask = W.make_data(1, maps_o[0])
    logl_o, maps_o = oracle.loglike(theta, cfg, data, err, mask, return_maps=True)
    ctx = bang.Context(cfg, precision=prec)
    fine = ctx.model_fine(theta[:1]).cpu().numpy()[0]
    assert_maps(fine, oracle.model_fine(theta[0], cfg), prec, "jaffe fine")
    ctx.set_data(data, err, mask)
    maps = ctx.model_maps(theta).cpu().numpy()
    ll = ctx.loglike(theta).cpu().numpy()
    ctx.close()
    assert_maps(maps, maps_o, prec, "jaffe maps")
    assert_logl(ll, logl_o, maps_o, data, err, mask, prec, near=np.array([True, False, False]), what="jaffe cfg1")
    # and the switch matters: the Hernquist maps of the same theta are different
    ctx = bang.Context(W.config(1), precision=prec)
    other = ctx.model_maps(theta[:1]).cpu().numpy()[0]
    ctx.close()
    assert np.abs(other[0] / maps_o[0, 0] - 1).max() > 1e-2


def test_jaffe_bulge_prior_batch(bang, oracle):
    # a seeded subset of config 2's prior-drawn batch (four components, NFW halo) with a Jaffe bulge, both precisions
    cfg = dict(W.config(2), bulge_profile=1)
    theta = W.theta_batch(2)
    sub = W.parity_subset(2, theta.shape[0], 24)
    mtrue = oracle.model_maps(W.theta_true(2), cfg)[0]
    data, err, mask = W.make_data(2, mtrue)
    logl_o, maps_o = oracle.loglike(theta[sub], cfg, data, err, mask, return_maps=True)
    near = np.isin(sub, W.near_truth_slots(2, theta.shape[0]))
    for prec in ("fp32", "fp64"):
        ctx = bang.Context(cfg, precision=prec)
        ctx.set_data(data, err, mask)
        maps = ctx.model_maps(theta[sub]).cpu().numpy()
        ll = ctx.loglike(theta[sub]).cpu().numpy()
        ctx.close()
        assert_maps(maps, maps_o, prec, f"jaffe cfg2 {prec}")
        assert_logl(ll, logl_o, maps_o, data, err, mask, prec, near=near, what=f"jaffe cfg2 {prec}")


# ------------------------------------------------------------------------------------------------ flux-weighted PSF (reading G')
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_flux_weighted_psf_config1_grid(bang, oracle, prec):
    cfg = dict(W.config(1), psf_weighting=1)
    theta = np.stack([W.theta_true(1), W.theta_true(1) * 1.01, W.theta_true(1) * 0.99])
    theta[1, 0:2] = 0.37, -0.21
    maps_o = oracle.model_maps(theta, cfg)
    data, err, mask = W.make_data(1, maps_o[0])
    logl_o, maps_o = oracle.loglike(theta, cfg, data, err, mask, return_maps=True)
    ctx = bang.Context(cfg, precision=prec)
    fine = ctx.model_fine(theta[:1]).cpu().numpy()[0]               # the four moment fields before the PSF
    assert_maps(fine, oracle.model_fine(theta[0], cfg), prec, "flux fine")
    ctx.set_data(data, err, mask)
    maps = ctx.model_maps(theta).cpu().numpy()
    ll = ctx.loglike(theta).cpu().numpy()
    ctx.close()
    assert_maps(maps, maps_o, prec, "flux maps")
    assert_logl(ll, logl_o, maps_o, data, err, mask, prec, near=np.array([True, False, False]), what="flux cfg1")
    plain = oracle.model_maps(theta[:1], W.config(1))[0]             # the paper's definition gives different kinematics
    assert np.abs(maps_o[0, 1] / plain[1] - 1).max() > 0.05


def test_flux_weighted_psf_prior_batch(bang, oracle):
    # a seeded subset of config 2's prior-drawn batch, P = 2 launch shape; ragged 13 x 7 map with s = 3 in fp64
    cfg = dict(W.config(2), psf_weighting=1)
    theta = W.theta_batch(2)
    sub = W.parity_subset(2, theta.shape[0], 24)
    mtrue = oracle.model_maps(W.theta_true(2), cfg)[0]
    data, err, mask = W.make_data(2, mtrue)
    logl_o, maps_o = oracle.loglike(theta[sub], cfg, data, err, mask, return_maps=True)
    near = np.isin(sub, W.near_truth_slots(2, theta.shape[0]))
    for prec in ("fp32", "fp64"):
        ctx = bang.Context(cfg, precision=prec)
        ctx.set_data(data, err, mask)
        maps = ctx.model_maps(theta[sub]).cpu().numpy()
        ll = ctx.loglike(theta[sub]).cpu().numpy()
        ctx.close()
        assert_maps(maps, maps_o, prec, f"flux cfg2 {prec}")
        assert_logl(ll, logl_o, maps_o, data, err, mask, prec, near=near, what=f"flux cfg2 {prec}")
    small = dict(cfg, nx=13, ny=7)
    ctx = bang.Context(small, precision="fp64")
    got = ctx.model_maps(theta[sub][:4]).cpu().numpy()
    ctx.close()
    assert_maps(got, oracle.model_maps(theta[sub][:4], small), "fp64", "flux ragged")
