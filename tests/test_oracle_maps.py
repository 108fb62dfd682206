"""Pins for the map-level path of the oracle: geometry, light-weighting, PSF + rebin, likelihood (CPU only).

Closed forms on simple models, invariants implied by PAPER.md eqs. 11, 14, 15, brute-force PSF sums on tiny
grids, library routines (scipy.stats) and the survey-time cross-check values under tests/golden/.
"""
import math
import os

import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
B_, D1, D2, H_ = W.BULGE, W.DISC1, W.DISC2, W.HALO


def small_cfg(**kw):
    cfg = dict(nx=12, ny=10, pix_arcsec=1.0, supersample=2, dist_mpc=50.0, sigma_pix=0.8, trunc_nsigma=3.0,
               components=B_ | D1 | D2 | H_, halo_profile=W.HALO_NFW, jeans_nodes=32)
    cfg.update(kw)
    return cfg


THETA = np.array([0.3, -0.4, 35.0, 55.0, 10.2, 0.5, 10.1, 1.2, 10.6, 3.5, 12.0, 9.0, 4.0, 1.5, 2.5, 0.4, 0.8])


# ------------------------------------------------------------------ golden: survey cross-check
def test_config1_matches_survey_crosscheck_values(oracle):
    m = oracle.model_maps(W.theta_true(1), W.config(1))[0]
    n = 0
    for line in open(os.path.join(GOLD, "config1_survey_crosscheck.txt")):
        if line.startswith("#"):
            continue
        i, j, *vals = line.split()
        for q, v in enumerate(vals):
            assert abs(m[q, int(i), int(j)] / float(v) - 1) < 2e-12, (i, j, q)
        n += 1
    assert n == 5


# ------------------------------------------------------------------ geometry: closed form for a bare disc
@pytest.mark.parametrize("pa,inc", [(0.0, 0.0), (0.0, 60.0), (90.0, 60.0), (30.0, 40.0)])
def test_disc_only_point_sampled_surface_brightness(oracle, pa, inc):
    # sigma_psf = 0, s = 1: the map is the model at pixel centres (reading F), pixel j centre = (j-(N-1)/2) p.
    # eq. 7-8: B = M_d/(2 pi R_d^2 cos i)/(M/L) exp(-r/R_d), r from the rotation of fn 2
    cfg = small_cfg(nx=9, ny=7, supersample=1, sigma_pix=0.0, components=D1)
    th = THETA.copy()
    th[[0, 1, 2, 3]] = [0.5, -1.0, pa, inc]
    m = oracle.model_maps(th, cfg)[0]
    kappa = 50.0 * 4.84813681109536e-3
    ys, xs = np.meshgrid((np.arange(7) - 3.0), (np.arange(9) - 4.0), indexing="ij")
    X, Y = (xs - 0.5) * kappa, (ys + 1.0) * kappa
    c, s = math.cos(math.radians(pa)), math.sin(math.radians(pa))
    xp, yp = X * c + Y * s, -X * s + Y * c
    ci = math.cos(math.radians(inc))
    r = np.hypot(xp, yp / ci)
    Md, Rd, ML = 10 ** th[6], th[7], th[13]
    want = Md / (2 * np.pi * Rd**2 * ci) / ML * np.exp(-r / Rd) * 1e-6
    assert np.allclose(m[0], want, rtol=1e-13)
    assert np.allclose(m[3], ML, rtol=1e-13)                      # single component: M/L is its own
    # eq. 11 with eq. 9-10: v = -k sin i cos(phi) v_c(r)
    L = oracle.lib()
    vc = np.sqrt(np.vectorize(lambda rr: L.bo_vc2_expdisc(rr, Md, Rd))(r))
    want_v = -th[15] * math.sin(math.radians(inc)) * (xp / r) * vc
    assert np.allclose(m[1], want_v, rtol=1e-12, atol=1e-12)
    assert np.allclose(m[2], np.sqrt((1 - th[15] ** 2) / 3) * vc, rtol=1e-12)     # eq. 12


def test_major_and_minor_axis_scale_lengths(oracle):
    # along the major axis (P.A. from +x, counter-clockwise) B falls as exp(-d/R_d); along the minor as exp(-d/(R_d cos i))
    cfg = small_cfg(nx=21, ny=21, supersample=1, sigma_pix=0.0, components=D1)
    th = THETA.copy()
    th[[0, 1, 2, 3]] = [0.0, 0.0, 90.0, 60.0]            # major axis along +y
    m = oracle.model_maps(th, cfg)[0][0]
    kappa = 50.0 * 4.84813681109536e-3
    assert abs(math.log(m[11, 10] / m[16, 10]) - 5 * kappa / th[7]) < 1e-12          # 5 px up the major axis
    assert abs(math.log(m[10, 11] / m[10, 16]) - 5 * kappa / (th[7] * 0.5)) < 1e-10  # 5 px along the minor axis


def test_exponential_disc_total_luminosity(oracle):
    # sum(B) x pixel area -> M_d/(M/L)  (PSF and rebin conserve flux; grid out to ~14 R_d)
    cfg = small_cfg(nx=120, ny=120, supersample=2, sigma_pix=1.0, components=D1, dist_mpc=20.0)
    th = THETA.copy()
    th[[0, 1, 2, 3, 6, 7, 13]] = [0.2, 0.1, 20.0, 35.0, 10.0, 0.4, 2.0]
    m = oracle.model_maps(th, cfg)[0][0]
    area_pc2 = (cfg["pix_arcsec"] * cfg["dist_mpc"] * 4.84813681109536e-3 * 1e3) ** 2
    assert abs(m.sum() * area_pc2 / (1e10 / 2.0) - 1) < 2e-3


def test_bulge_only_reduces_to_hernquist_closed_forms(oracle):
    # v == 0 (eq. 14 has no bulge term), sigma_los^2 = I_b/Sigma_b = (G M_b/R_b) ITilde/(6 SigmaTilde) (eq. 4, 6), B = Sigma_b/(M/L)
    cfg = small_cfg(nx=8, ny=8, supersample=1, sigma_pix=0.0, components=B_, jeans_nodes=128)
    th = THETA.copy()
    th[[0, 1]] = [0.3, 0.2]
    m = oracle.model_maps(th, cfg)[0]
    L = oracle.lib()
    kappa = 50.0 * 4.84813681109536e-3
    ys, xs = np.meshgrid(np.arange(8) - 3.5, np.arange(8) - 3.5, indexing="ij")
    R = np.hypot((xs - 0.3) * kappa, (ys - 0.2) * kappa)
    Mb, Rb, ML = 10 ** th[4], th[5], th[12]
    sig = np.vectorize(L.bo_sigma_tilde)(R / Rb)
    it = np.vectorize(L.bo_I_tilde_closed)(R / Rb)
    assert np.all(m[1] == 0.0)
    assert np.allclose(m[0], Mb / (2 * np.pi * Rb**2) * sig / ML * 1e-6, rtol=1e-13)
    assert np.allclose(m[2], np.sqrt(L.bo_G() * Mb / Rb * it / (6 * sig)), rtol=1e-12)
    assert np.allclose(m[3], ML, rtol=1e-13)


def test_two_component_light_weighting_by_hand(oracle):
    # eqs. 13-15, 19 assembled by hand at one pixel from the scalar entry points
    cfg = small_cfg(nx=5, ny=5, supersample=1, sigma_pix=0.0, components=B_ | D1 | H_, halo_profile=W.HALO_HERNQUIST,
                    jeans_nodes=64)
    th = THETA.copy()
    th[[0, 1, 2, 3]] = [0.0, 0.0, 0.0, 50.0]
    th[10], th[11] = 12.0, 25.0
    m = oracle.model_maps(th, cfg)[0]
    L = oracle.lib()
    kappa = 50.0 * 4.84813681109536e-3
    iy, ix = 3, 4                                  # pixel centre at (+2, +1) arcsec
    xp, yp = 2 * kappa, 1 * kappa
    ci, si = math.cos(math.radians(50.0)), math.sin(math.radians(50.0))
    R, r = math.hypot(xp, yp), math.hypot(xp, yp / ci)
    Mb, Rb, Md, Rd, Mh, Rh = 10 ** th[4], th[5], 10 ** th[6], th[7], 10 ** th[10], th[11]
    Sb = L.bo_hernquist_Sigma(R, Mb, Rb)
    Sd = Md / (2 * math.pi * Rd**2 * ci) * math.exp(-r / Rd)
    Bb, Bd = Sb / th[12] * 1e-6, Sd / th[13] * 1e-6
    vc2 = L.bo_vc2_hernquist(r, Mb, Rb) + L.bo_vc2_expdisc(r, Md, Rd) + L.bo_vc2_hernquist(r, Mh, Rh)
    vd = -th[15] * si * (xp / r) * math.sqrt(vc2)
    sd2 = (1 - th[15] ** 2) * vc2 / 3
    sb2 = L.bo_Ib_quadrature(R, Mb, Rb, 64) / Sb
    assert abs(m[0, iy, ix] / (Bb + Bd) - 1) < 1e-13
    assert abs(m[1, iy, ix] / (Bd * vd / (Bb + Bd)) - 1) < 1e-13
    assert abs(m[2, iy, ix] / math.sqrt((Bb * sb2 + Bd * sd2) / (Bb + Bd)) - 1) < 1e-13
    assert abs(m[3, iy, ix] / ((Sb + Sd) * 1e-6 / (Bb + Bd)) - 1) < 1e-13


# ------------------------------------------------------------------ invariants
def test_face_on_has_zero_velocity(oracle):
    th = THETA.copy()
    th[3] = 0.0
    m = oracle.model_maps(th, small_cfg())[0]
    assert np.all(m[1] == 0.0)


def test_position_angle_plus_180(oracle):
    cfg = small_cfg()
    a = oracle.model_maps(THETA, cfg)[0]
    th = THETA.copy()
    th[2] += 180.0
    b = oracle.model_maps(th, cfg)[0]
    for q in (0, 2, 3):
        assert np.allclose(a[q], b[q], rtol=1e-12)
    assert np.allclose(a[1], -b[1], rtol=1e-10, atol=1e-10)


def test_point_symmetry_about_the_centre(oracle):
    cfg = small_cfg(nx=12, ny=12)
    th = THETA.copy()
    th[[0, 1]] = 0.0
    m = oracle.model_maps(th, cfg)[0]
    for q, sgn in ((0, 1), (1, -1), (2, 1), (3, 1)):
        assert np.allclose(m[q], sgn * m[q, ::-1, ::-1], rtol=1e-12, atol=1e-10)


def test_k_sign_flips_velocity_only(oracle):
    cfg = small_cfg()
    a = oracle.model_maps(THETA, cfg)[0]
    th = THETA.copy()
    th[15:17] *= -1
    b = oracle.model_maps(th, cfg)[0]
    assert np.allclose(a[1], -b[1], rtol=1e-13) and np.allclose(a[[0, 2, 3]], b[[0, 2, 3]], rtol=1e-14)


def test_cold_disc_has_zero_dispersion(oracle):
    th = THETA.copy()
    th[15] = 1.0
    m = oracle.model_maps(th, small_cfg(components=D1))[0]
    assert np.all(np.abs(m[2]) < 1e-12)


def test_centre_shift_by_one_pixel_shifts_the_map(oracle):
    cfg = small_cfg(nx=14, ny=12)
    th = THETA.copy()
    a = oracle.model_maps(th, cfg)[0]
    th[0] += 1.0
    th[1] += 2.0                                   # +x = +column, +y = +row (reading S)
    b = oracle.model_maps(th, cfg)[0]
    assert np.allclose(a[:, :-2, :-1], b[:, 2:, 1:], rtol=1e-11, atol=1e-10)


def test_absent_components_ignore_their_parameters(oracle):
    cfg = small_cfg(components=B_ | D1)
    a = oracle.model_maps(THETA, cfg)[0]
    th = THETA.copy()
    th[[8, 9, 10, 11, 14, 16]] = [3.0, -1.0, np.nan, -5.0, -2.0, 7.0]
    assert np.array_equal(a, oracle.model_maps(th, cfg)[0])


def test_out_of_domain_theta(oracle):
    cfg = small_cfg()
    data = np.zeros((4, cfg["ny"], cfg["nx"]))
    err = np.ones_like(data)
    mask = np.ones(data.shape, np.uint8)
    for idx, val in ((5, 0.0), (7, -1.0), (12, 0.0), (15, 1.5), (3, 90.0), (3, 120.0), (4, np.nan), (11, 0.0)):
        th = THETA.copy()
        th[idx] = val
        ll, maps = oracle.loglike(th, cfg, data, err, mask, return_maps=True)
        assert ll[0] == -np.inf and np.all(np.isnan(maps))


# ------------------------------------------------------------------ PSF + rebin (eq. 21, reading F)
def test_psf_taps(oracle):
    for sigma, s in ((1.0, 2), (1.0, 3), (1.5, 4), (0.7, 3), (0.0, 1)):
        g = oracle.psf_taps(sigma, s)
        rk = (len(g) - 1) // 2
        assert rk == math.ceil(3 * sigma * s - 1e-9)
        assert abs(g.sum() - 1) < 1e-15 and np.allclose(g, g[::-1], rtol=0, atol=0)
        if sigma > 0:
            m = np.arange(-rk, rk + 1)
            assert np.allclose(g / g[rk], np.exp(-m**2 / (2 * (sigma * s) ** 2)), rtol=1e-14)
    assert oracle.lib().bo_psf_halfwidth(1.0, 2, 3.0) == 6 and oracle.lib().bo_psf_halfwidth(1.5, 4, 3.0) == 18


def test_convolve_rebin_brute_force_2d(oracle):
    # eq. 21 written as the full 2-D double sum (normalised by the sum of the weights), then the s x s mean
    rng = np.random.default_rng(5)
    nx, ny, s, sigma = 5, 4, 3, 0.6
    rk = math.ceil(3 * sigma * s - 1e-9)
    fine = rng.uniform(0.5, 2.0, size=(4, ny * s + 2 * rk, nx * s + 2 * rk))
    got = oracle.convolve_rebin(fine, nx, ny, s, sigma)
    mm = np.arange(-rk, rk + 1)
    w2 = np.exp(-(mm[:, None] ** 2 + mm[None, :] ** 2) / (2 * (sigma * s) ** 2))
    for q in range(4):
        conv = np.zeros((ny * s, nx * s))
        for iy in range(ny * s):
            for ix in range(nx * s):
                patch = fine[q, iy:iy + 2 * rk + 1, ix:ix + 2 * rk + 1]
                conv[iy, ix] = (patch * w2).sum() / w2.sum()
        reb = conv.reshape(ny, s, nx, s).mean(axis=(1, 3))
        want = 1.0 / reb if q == 3 else reb
        assert np.allclose(got[q], want, rtol=1e-13)


def test_psf_leaves_constant_and_linear_fields_unchanged(oracle):
    nx, ny, s, sigma = 6, 5, 2, 1.0
    rk = 6
    fine = np.ones((4, ny * s + 2 * rk, nx * s + 2 * rk)) * np.array([3.0, -2.0, 7.0, 0.25])[:, None, None]
    got = oracle.convolve_rebin(fine, nx, ny, s, sigma)
    assert np.allclose(got[0], 3.0, rtol=1e-14) and np.allclose(got[1], -2.0, rtol=1e-14)
    assert np.allclose(got[2], 7.0, rtol=1e-14) and np.allclose(got[3], 4.0, rtol=1e-14)
    # a symmetric normalised kernel also preserves a linear ramp: rebinned value = ramp at the pixel centre
    jx = np.arange(nx * s + 2 * rk) - rk
    ramp = np.broadcast_to(0.5 * jx[None, :] + 1.0, fine.shape[1:])
    fine2 = np.stack([ramp, ramp, ramp, ramp])
    got2 = oracle.convolve_rebin(fine2, nx, ny, s, sigma)
    centre = 0.5 * (np.arange(nx) * s + (s - 1) / 2.0) + 1.0
    assert np.allclose(got2[0], np.broadcast_to(centre, (ny, nx)), rtol=1e-13)


def test_psf_flux_conservation_of_a_compact_source(oracle):
    nx, ny, s, sigma = 16, 16, 2, 1.0
    rk = 6
    fine = np.zeros((4, ny * s + 2 * rk, nx * s + 2 * rk))
    fine[:, rk + 15, rk + 17] = 1.0
    fine[3] += 1.0
    got = oracle.convolve_rebin(fine, nx, ny, s, sigma)
    assert abs(got[0].sum() * s * s - 1.0) < 1e-14


def test_model_maps_equal_fine_maps_pushed_through_psf(oracle):
    cfg = small_cfg()
    fine = oracle.model_fine(THETA, cfg)
    a = oracle.convolve_rebin(fine, cfg["nx"], cfg["ny"], cfg["supersample"], cfg["sigma_pix"])
    assert np.array_equal(a, oracle.model_maps(THETA, cfg)[0])
    # fine-grid convention (step 1): cell J in [-r_k, N s + r_k); with s = 1, sigma = 0 fine == map
    cfg1 = small_cfg(supersample=1, sigma_pix=0.0)
    f1 = oracle.model_fine(THETA, cfg1)
    m1 = oracle.model_maps(THETA, cfg1)[0]
    assert np.array_equal(f1[:3], m1[:3]) and np.allclose(1.0 / f1[3], m1[3], rtol=1e-15)


def test_supersampled_map_converges_to_the_pixel_integral(oracle):
    # with s -> large and no PSF the rebinned B tends to the pixel average of the analytic disc (midpoint rule, O(1/s^2))
    th = THETA.copy()
    errs = []
    ref = oracle.model_maps(th, small_cfg(nx=6, ny=6, supersample=16, sigma_pix=0.0, components=D1))[0][0]
    for s in (1, 2, 4):
        m = oracle.model_maps(th, small_cfg(nx=6, ny=6, supersample=s, sigma_pix=0.0, components=D1))[0][0]
        errs.append(np.abs(m / ref - 1).max())
    assert errs[0] > 3.5 * errs[1] > 3.5 * 3.5 * errs[2] * 0.9


# ------------------------------------------------------------------ likelihood (eq. 18, readings L, M)
def test_loglike_against_scipy_norm(oracle):
    from scipy.stats import norm
    cfg = small_cfg()
    rng = np.random.default_rng(11)
    maps = oracle.model_maps(THETA, cfg)[0]
    err = rng.uniform(0.5, 2.0, size=maps.shape)
    data = maps + err * rng.standard_normal(maps.shape)
    mask = (rng.random(maps.shape) > 0.3).astype(np.uint8)
    want = norm.logpdf(data, loc=maps, scale=err)[mask == 1].sum()
    got = oracle.loglike(THETA, cfg, data, err, mask)[0]
    assert abs(got - want) < 1e-9 * abs(want)
    # masked pixels may hold anything
    data2 = data.copy()
    data2[mask == 0] = np.nan
    assert oracle.loglike(THETA, cfg, data2, err, mask)[0] == got
    # data == model: only the normalisation remains
    full = np.ones(maps.shape, np.uint8)
    assert abs(oracle.loglike(THETA, cfg, maps, err, full)[0] + 0.5 * np.log(2 * np.pi * err**2).sum()) < 1e-9


def test_loglike_batch_matches_single_calls(oracle):
    cfg = small_cfg(jeans_nodes=16)
    rng = np.random.default_rng(3)
    th = np.stack([THETA, THETA * 1.01, THETA * 0.99])
    maps = oracle.model_maps(THETA, cfg)[0]
    err = np.ones_like(maps)
    mask = np.ones(maps.shape, np.uint8)
    ll = oracle.loglike(th, cfg, maps, err, mask)
    for b in range(3):
        assert ll[b] == oracle.loglike(th[b], cfg, maps, err, mask)[0]
    assert ll[0] > ll[1] and ll[0] > ll[2]


def test_jeans_node_count_barely_matters_on_config1(oracle):
    # N_J = 32/64/128 give the same central sigma to ~1e-15 on config 1 (s >= 0.1 everywhere)
    th, c = W.theta_true(1), W.config(1)
    vals = [oracle.model_maps(th, dict(c, jeans_nodes=nj))[0][2, 16, 16] for nj in (32, 64, 128)]
    assert abs(vals[0] / vals[2] - 1) < 1e-12 and abs(vals[1] / vals[2] - 1) < 1e-13
