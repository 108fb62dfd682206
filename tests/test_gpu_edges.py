"""GPU edge cases of the C-ABI path: empty batches, out-of-domain theta, masks, ragged and non-square grids, the
degenerate PSF / supersampling settings, tap padding, the model's invariants, error codes."""
import ctypes as C

import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W

pytestmark = pytest.mark.gpu

B_, D1, D2, H_ = W.BULGE, W.DISC1, W.DISC2, W.HALO
THETA = np.array([0.3, -0.4, 35.0, 55.0, 10.2, 0.5, 10.1, 1.2, 10.6, 3.5, 12.0, 9.0, 4.0, 1.5, 2.5, 0.4, 0.8])


@pytest.fixture(scope="module")
def bang():
    import torch
    assert torch.cuda.is_available()
    from paper_2205_06819_b200 import bang as b
    b.lib()
    return b


def small_cfg(**kw):
    cfg = dict(nx=12, ny=10, pix_arcsec=1.0, supersample=2, dist_mpc=50.0, sigma_pix=0.8, trunc_nsigma=3.0,
               components=B_ | D1 | D2 | H_, halo_profile=W.HALO_NFW, jeans_nodes=32)
    cfg.update(kw)
    return cfg


def rel(g, o):
    g, o = np.asarray(g, np.float64), np.asarray(o, np.float64)
    den = np.abs(o)
    den[..., 1, :, :] = np.maximum(den[..., 1, :, :], 1e-3 * den[..., 1, :, :].max())
    return float(np.max(np.abs(g - o) / den))


def synth_data(oracle, cfg, theta, seed=3):
    m = oracle.model_maps(theta, cfg)[0]
    rng = np.random.default_rng(seed)
    err = np.stack([0.05 * np.abs(m[0]), np.full_like(m[1], 10.0), np.full_like(m[2], 10.0), np.full_like(m[3], 0.1)])
    data = m + err * rng.standard_normal(m.shape)
    mask = (rng.random(m.shape) > 0.3).astype(np.uint8)          # a different mask per observable (reading M)
    return data, err, mask


# ------------------------------------------------------------------------------------------------ shapes
@pytest.mark.parametrize("prec,tol", [("fp64", 1e-9), ("fp32", 1e-4)])
@pytest.mark.parametrize("kw", [
    dict(),                                                     # 12 x 10, s = 2
    dict(nx=13, ny=7, supersample=3, sigma_pix=1.0),            # ragged: nx not a multiple of the pixel group
    dict(nx=5, ny=1, supersample=1, sigma_pix=0.0),             # a single row, point sampling (reading F limit)
    dict(nx=1, ny=1, supersample=4, sigma_pix=0.5),             # a single pixel
    dict(nx=9, ny=11, supersample=3, sigma_pix=0.7),            # r_k = 7: 2 r_k + s = 17 taps padded to 21
    dict(nx=20, ny=6, supersample=1, sigma_pix=2.0),            # s = 1, 13-tap footprint
    dict(nx=7, ny=9, supersample=4, sigma_pix=1.5, components=B_ | D1, halo_profile=W.HALO_HERNQUIST),
    dict(nx=8, ny=8, supersample=2, sigma_pix=1.0, components=D1 | D2 | H_, halo_profile=W.HALO_HERNQUIST),
    dict(nx=140, ny=3, supersample=2, sigma_pix=1.0),           # wide row: the P = 4 pixel-group path in fp32
    dict(nx=300, ny=2, supersample=2, sigma_pix=1.0),           # wider still: the 512-thread launch class (fp64: 2 x 300 > 512 is refused)
])
def test_shapes_and_variants_match_the_oracle(bang, oracle, kw, prec, tol):
    cfg = small_cfg(**kw)
    th = np.stack([THETA, THETA * np.array([1, 1, 2.5, 0.6, 1, 3, 1, 0.5, 1, 1, 1, 1, 1, 1, 1, -1, 1])])
    if prec == "fp64" and cfg["nx"] > 256:                       # include/bang.h: fp64 mode holds rows of <= 256 pixels
        with pytest.raises(bang.BangError) as e:
            bang.Context(cfg, precision=prec)
        assert e.value.code == bang.EINVAL
        return
    ctx = bang.Context(cfg, precision=prec)
    maps = ctx.model_maps(th).cpu().numpy()
    fine = ctx.model_fine(th).cpu().numpy()
    want = oracle.model_maps(th, cfg)
    assert rel(maps, want) < tol
    # un-convolved fine cells (a test-only intermediate, not a map pixel): theta[1] has k_1 < 0 < k_2, so the two disc
    # terms of eq. 14 cancel and |v| falls to the fp32 noise of the terms (eps x ~150 km/s = reading P's floor of
    # 1e-3 max|v| x 1e-4); a single fine cell may then sit at 1e-4 of that floor.  The map pixels above keep 1e-4.
    assert rel(fine, np.stack([oracle.model_fine(t, cfg) for t in th])) < (tol if prec == "fp64" else 3 * tol)
    data, err, mask = synth_data(oracle, cfg, THETA)
    ctx.set_data(data, err, mask)
    ll = ctx.loglike(th).cpu().numpy()
    want_ll = oracle.loglike(th, cfg, data, err, mask)
    assert np.all(np.abs(ll - want_ll) <= tol * np.abs(want_ll))
    ctx.close()


def test_empty_batch_is_a_noop(bang, oracle):
    import torch
    ctx = bang.Context(small_cfg(), precision="fp32")
    assert ctx.model_maps(np.zeros((0, 17))).shape == (0, 4, 10, 12)
    data, err, mask = synth_data(oracle, small_cfg(), THETA)
    ctx.set_data(data, err, mask)
    assert ctx.loglike(torch.zeros((0, 17), dtype=torch.float64, device="cuda")).shape == (0,)
    assert ctx.loglike_host(np.zeros((0, 17))).shape == (0,)
    n = ctx.launches
    ctx.loglike(THETA)
    assert ctx.launches == n + 2                                  # one fused kernel per batch + the (empty) direct-path
                                                                  # launch for theta outside the tabulated ranges
    ctx.close()


# ------------------------------------------------------------------------------------------------ domain
@pytest.mark.parametrize("prec", ["fp32", "fp64"])
def test_out_of_domain_theta_gives_minus_infinity_and_nan_maps(bang, oracle, prec):
    cfg = small_cfg()
    bad = []
    for slot, val in [(5, 0.0), (5, -1.0), (7, 0.0), (12, 0.0), (13, -2.0), (15, 1.5), (16, -1.01), (3, 90.0), (3, 95.0),
                      (4, np.nan), (0, np.inf), (11, 0.0), (9, np.nan)]:
        t = THETA.copy()
        t[slot] = val
        bad.append(t)
    th = np.stack([THETA] + bad + [THETA])
    data, err, mask = synth_data(oracle, cfg, THETA)
    ctx = bang.Context(cfg, precision=prec)
    ctx.set_data(data, err, mask)
    ll = ctx.loglike(th).cpu().numpy()
    maps = ctx.model_maps(th).cpu().numpy()
    ctx.close()
    want = oracle.loglike(th, cfg, data, err, mask)
    assert np.isfinite(ll[0]) and np.isfinite(ll[-1]) and ll[0] == ll[-1]
    assert np.all(np.isneginf(ll[1:-1])) and np.all(np.isneginf(want[1:-1]))
    assert np.isfinite(maps[0]).all() and np.isnan(maps[1:-1]).all()


def test_entries_of_absent_components_are_ignored(bang):
    cfg = small_cfg(components=B_ | D1)
    ctx = bang.Context(cfg, precision="fp64")
    t2 = THETA.copy()
    t2[[8, 9, 10, 11, 14, 16]] = [np.nan, -1.0, np.inf, 0.0, -3.0, 7.0]       # disc 2 and halo slots: garbage
    a = ctx.model_maps(THETA).cpu().numpy()
    b = ctx.model_maps(t2).cpu().numpy()
    ctx.close()
    assert np.array_equal(a, b) and np.isfinite(a).all()


def test_centre_far_outside_the_grid_and_extreme_inclination(bang, oracle):
    cfg = small_cfg(nx=16, ny=16)
    th = np.stack([THETA.copy() for _ in range(4)])
    th[0, 0:2] = [40.0, -25.0]                  # centre well outside the field
    th[1, 3] = 89.0                             # nearly edge-on: r = y'/cos i reaches ~57 x R
    th[2, 5] = 0.02                             # tiny bulge: s = R/R_b up to ~300
    th[3, 0:2] = [0.25, 0.25]                   # centre exactly on a fine-cell centre (s = 2): R = 0 -> floor (reading V)
    for prec, tol in (("fp64", 1e-9), ("fp32", 1e-4)):
        ctx = bang.Context(cfg, precision=prec)
        maps = ctx.model_maps(th).cpu().numpy()
        ctx.close()
        assert rel(maps, oracle.model_maps(th, cfg)) < tol


def test_disc_only_model_survives_fp32_underflow_far_outside_small_discs(bang, oracle):
    # exp(-r/R_d) underflows fp32 beyond r ~ 87 R_d; v, sigma and M/L are ratios and must stay finite and right
    cfg = small_cfg(nx=40, ny=40, supersample=1, sigma_pix=0.0, components=D1 | D2 | H_)
    t = THETA.copy()
    t[[3, 7, 9]] = [80.0, 0.1, 0.12]
    ctx = bang.Context(cfg, precision="fp32")
    m = ctx.model_maps(t).cpu().numpy().astype(np.float64)[0]
    ctx.close()
    o = oracle.model_maps(t, cfg)[0]
    assert (o[0] < 1e-38).any()                                  # the case really occurs on this grid
    assert np.isfinite(m).all()
    for q in (1, 2, 3):
        den = np.maximum(np.abs(o[q]), 1e-3 * np.abs(o[q]).max())
        assert np.max(np.abs(m[q] - o[q]) / den) < 1e-4
    big = o[0] > 1e-30
    assert np.max(np.abs(m[0][big] / o[0][big] - 1)) < 1e-4


# ------------------------------------------------------------------------------------------------ invariants
def test_invariants_on_the_gpu_path(bang):
    cfg = small_cfg(nx=16, ny=16, supersample=2, sigma_pix=1.0)
    ctx = bang.Context(cfg, precision="fp64")
    t0 = THETA.copy()
    t0[0:2] = 0.0
    face = t0.copy(); face[3] = 0.0
    flip = t0.copy(); flip[2] += 180.0
    kneg = t0.copy(); kneg[15:17] *= -1
    m0, mf, m180, mk = (ctx.model_maps(t).cpu().numpy()[0] for t in (t0, face, flip, kneg))
    ctx.close()
    assert np.max(np.abs(mf[1])) == 0.0                                        # eq. 11: sin i = 0 -> v_los = 0
    for q in (0, 2, 3):
        assert np.allclose(m180[q], m0[q], rtol=1e-12)                         # P.A. + 180 deg
        assert np.allclose(mk[q], m0[q], rtol=1e-12)
    assert np.allclose(m180[1], -m0[1], rtol=1e-10, atol=1e-10)
    assert np.allclose(mk[1], -m0[1], rtol=1e-12)                              # k -> -k flips v only (reading K)
    assert np.allclose(m0[0], m0[0][::-1, ::-1], rtol=1e-12)                   # point symmetry about the centre
    assert np.allclose(m0[1], -m0[1][::-1, ::-1], rtol=1e-10, atol=1e-10)


def test_psf_leaves_a_constant_field_unchanged(bang):
    # a face-on, very large single disc is flat across a small field: B and M/L must come back flat (eq. 21 normalised)
    cfg = small_cfg(nx=8, ny=8, supersample=3, sigma_pix=1.2, components=D1)
    t = THETA.copy()
    t[[3, 7]] = [0.0, 5e6]
    ctx = bang.Context(cfg, precision="fp64")
    m = ctx.model_maps(t).cpu().numpy()[0]
    ctx.close()
    assert np.ptp(m[0]) / m[0].mean() < 1e-6 and np.ptp(m[3]) < 1e-12
    assert abs(m[3].mean() - t[13]) < 1e-12


# ------------------------------------------------------------------------------------------------ data handling
def test_masked_pixels_may_hold_nan_and_do_not_change_logl(bang, oracle):
    cfg = small_cfg()
    data, err, mask = synth_data(oracle, cfg, THETA)
    ctx = bang.Context(cfg, precision="fp32")
    ctx.set_data(data, err, mask)
    a = ctx.loglike(THETA).cpu().numpy()
    d2, e2 = data.copy(), err.copy()
    d2[mask == 0] = np.nan
    e2[mask == 0] = -1.0
    ctx.set_data(d2, e2, mask)
    b = ctx.loglike(THETA).cpu().numpy()
    assert np.array_equal(a, b)
    none = np.zeros_like(mask)
    ctx.set_data(data, err, none)
    assert ctx.loglike(THETA).cpu().numpy()[0] == 0.0               # nothing used: empty sum
    ctx.close()


def test_model_equal_to_data_gives_the_normalisation_term(bang, oracle):
    cfg = small_cfg()
    ctx = bang.Context(cfg, precision="fp64")
    m = ctx.model_maps(THETA).cpu().numpy()[0]
    err = np.full_like(m, 0.37)
    mask = np.ones(m.shape, np.uint8)
    ctx.set_data(m, err, mask)
    ll = ctx.loglike(THETA).cpu().numpy()[0]
    ctx.close()
    assert abs(ll - (-0.5 * np.log(2 * np.pi * 0.37 ** 2) * m.size)) < 1e-9      # reading L


def test_error_codes(bang, oracle):
    import torch
    cfg = small_cfg()
    ctx = bang.Context(cfg, precision="fp32")
    with pytest.raises(bang.BangError) as ei:
        ctx.loglike(THETA)
    assert ei.value.code == bang.ENODATA
    data, err, mask = synth_data(oracle, cfg, THETA)
    ctx.set_data(data, err, mask)
    good = ctx.loglike(THETA).cpu().numpy()
    e_bad = err.copy()
    e_bad[1, 2, 3] = 0.0
    m_bad = mask.copy()
    m_bad[1, 2, 3] = 1
    with pytest.raises(bang.BangError) as ei:
        ctx.set_data(data, e_bad, m_bad)
    assert ei.value.code == bang.EINVAL and b"err" in bang.lib().bang_last_error(ctx._h)
    assert np.array_equal(ctx.loglike(THETA).cpu().numpy(), good)    # the previous data stay loaded
    L = bang.lib()
    assert L.bang_loglike(ctx._h, None, 3, None) == bang.EINVAL
    assert L.bang_model_maps(ctx._h, None, -1, None) == bang.EINVAL
    assert L.bang_set_data(ctx._h, None, None, None) == bang.EINVAL
    # bang_ns_walk: argument checks, and the degenerate calls that do nothing
    d, K = 3, 8
    u = torch.full((K, d), 0.5, dtype=torch.float64, device="cuda")
    ll = torch.zeros(K, dtype=torch.float64, device="cuda")
    ls = torch.full((K,), -np.inf, dtype=torch.float64, device="cuda")
    grp = torch.zeros(K, dtype=torch.int32, device="cuda")
    chol, free = 0.01 * np.eye(d)[None], [2, 3, 4]
    lo, hi = THETA[free] * 0.99, THETA[free] * 1.01
    assert ctx.ns_walk(u, ll, ls, grp, chol, [1.0], free, lo, hi, THETA, steps=0).tolist() == [0]      # no step: no-op
    assert torch.equal(u, torch.full_like(u, 0.5))
    with pytest.raises(bang.BangError) as ei:
        ctx.ns_walk(u, ll, ls, grp, chol, [1.0], [2, 3, 99], lo, hi, THETA, steps=1)                    # free index out of range
    assert ei.value.code == bang.EINVAL
    import ctypes as C
    n_acc = (C.c_int * 1)()
    fi = (C.c_int * 3)(2, 3, 4)
    assert L.bang_ns_walk(ctx._h, K, 18, fi, lo.ctypes.data, hi.ctypes.data, THETA.ctypes.data, u.data_ptr(), ll.data_ptr(),
                          ls.data_ptr(), grp.data_ptr(), 1, chol.ctypes.data, lo.ctypes.data, 1, 0, n_acc) == bang.EINVAL   # d > 17
    fresh = bang.Context(cfg, precision="fp32")
    with pytest.raises(bang.BangError) as ei:
        fresh.ns_walk(u, ll, ls, grp, chol, [1.0], free, lo, hi, THETA, steps=1)                         # before bang_set_data
    assert ei.value.code == bang.ENODATA
    fresh.close()
    ctx.close()
    # a context on a stream of its own
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c2 = bang.Context(cfg, precision="fp32", stream=s)
        c2.set_data(data, err, mask)
        out = c2.loglike(THETA)
    s.synchronize()
    assert np.array_equal(out.cpu().numpy(), good)
    c2.close()
    # too wide for one CTA's shared memory / thread budget
    with pytest.raises(bang.BangError) as ei:
        bang.Context(small_cfg(nx=4000, ny=4), precision="fp64")
    assert ei.value.code == bang.EINVAL


def test_peak_probe_matches_the_derived_unit_counts(bang):
    # 128 fp32 lanes, 16 MUFU results and 64 fp64 lanes per SM per clock at clocks.max.sm
    import torch
    ctx = bang.Context(small_cfg(), precision="fp32")
    pk = ctx.probe_peaks()
    ctx.close()
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    from paper_2205_06819_b200 import roofline as R
    clk = R.sm_max_mhz() * 1e6
    for key, lanes in (("fp32_fma", 128), ("mufu", 16), ("fp64_fma", 64)):
        frac = pk[key] / (n_sm * lanes * clk)
        assert 0.6 < frac < 1.08, (key, frac)
