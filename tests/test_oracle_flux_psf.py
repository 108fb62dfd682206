"""Pins for the flux-weighted PSF variant of the oracle (reading G').  CPU only.

The paper convolves B, v, sigma and <L/M> separately (eq. 21; reading G).  The variant hands the PSF
the light moments B, B v, B (sigma^2 + v^2) and the mass surface density, and forms v = M1/M0,
sigma^2 = M2/M0 - v^2, M/L = M3/M0 per data pixel.  Checked against brute-force weighted sums, closed forms for simple
fields, and its reduction to the paper's path when the beam is trivial."""
import numpy as np

from paper_2205_06819_b200 import workloads as W


def _kernel2d(oracle, s, sigma_pix):
    """Weights K[dy][dx] with which fine cell (s py + dy - r_k ...) enters data pixel (py, px): taps (*) s-cell box."""
    g = oracle.psf_taps(sigma_pix, s)
    rk = (len(g) - 1) // 2
    w = np.zeros(2 * rk + s)
    for b in range(s):
        w[b:b + 2 * rk + 1] += g / s
    return np.outer(w, w), rk


def test_trivial_beam_reduces_to_the_papers_path(oracle):
    cfg = dict(W.config(1), supersample=1, sigma_pix=0.0)
    th = W.theta_true(1)
    a = oracle.model_maps(th, cfg)
    b = oracle.model_maps(th, dict(cfg, psf_weighting=1))
    assert np.allclose(a, b, rtol=1e-13, atol=1e-13 * np.abs(a[:, 1]).max())
    # with a beam the two definitions differ (the light is concentrated, the velocity field is not flat)
    c = oracle.model_maps(th, W.config(1))[0]
    d = oracle.model_maps(th, dict(W.config(1), psf_weighting=1))[0]
    assert np.array_equal(c[0], d[0]) and np.abs(d[1] / c[1] - 1).max() > 0.05


def test_brute_force_weighted_sums(oracle):
    rng = np.random.default_rng(5)
    nx, ny, s, sig = 4, 3, 2, 0.7
    K, rk = _kernel2d(oracle, s, sig)
    nfx, nfy = nx * s + 2 * rk, ny * s + 2 * rk
    B = rng.uniform(0.5, 3.0, (nfy, nfx))
    v = rng.uniform(-200, 200, (nfy, nfx))
    sg = rng.uniform(20, 120, (nfy, nfx))
    ml = rng.uniform(0.5, 4.0, (nfy, nfx))
    fine = np.stack([B, B * v, B * (sg**2 + v**2), B * ml])              # the moments the variant's fine cells hold
    got = oracle.convolve_rebin(fine, nx, ny, s, sig, psf_weighting=1)
    n = K.shape[0]
    for py in range(ny):
        for px in range(nx):
            sl = (slice(py * s, py * s + n), slice(px * s, px * s + n))
            M0 = (K * B[sl]).sum()
            vv = (K * B[sl] * v[sl]).sum() / M0
            s2 = (K * B[sl] * (sg[sl] ** 2 + v[sl] ** 2)).sum() / M0 - vv**2
            assert abs(got[0, py, px] / M0 - 1) < 1e-13
            assert abs(got[1, py, px] - vv) < 1e-10
            assert abs(got[2, py, px] / np.sqrt(s2) - 1) < 1e-11
            assert abs(got[3, py, px] / ((K * B[sl] * ml[sl]).sum() / M0) - 1) < 1e-13


def test_uniform_light_linear_velocity_beam_smearing(oracle):
    # B constant, v = g x, sigma constant: v is unchanged (symmetric beam) and sigma^2 gains g^2 Var_K(x), the
    # classical beam-smearing term, Var_K being the variance of the composite kernel along x (in fine cells)
    nx, ny, s, sig = 6, 5, 3, 1.0
    K, rk = _kernel2d(oracle, s, sig)
    nfx, nfy = nx * s + 2 * rk, ny * s + 2 * rk
    x = np.arange(nfx)[None, :] * np.ones((nfy, 1))
    g, s0, B0 = 7.5, 40.0, 2.0
    v = g * (x - nfx / 2)
    fine = np.stack([np.full_like(x, B0), B0 * v, B0 * (s0**2 + v**2), np.full_like(x, 3.0 * B0)])
    got = oracle.convolve_rebin(fine, nx, ny, s, sig, psf_weighting=1)
    w = K.sum(axis=0)
    pos = np.arange(len(w))
    var = (w * pos**2).sum() - (w * pos).sum() ** 2
    centre = (w * pos).sum()
    for px in range(nx):
        assert np.allclose(got[1, :, px], g * (px * s + centre - nfx / 2), atol=1e-10)
    assert np.allclose(got[2], np.sqrt(s0**2 + g**2 * var), rtol=1e-12)
    assert np.allclose(got[3], 3.0, rtol=1e-13) and np.allclose(got[0], B0, rtol=1e-13)


def test_invariants_survive(oracle):
    cfg = dict(W.config(1), psf_weighting=1)
    th = W.theta_true(1)
    m = oracle.model_maps(th, cfg)[0]
    th2 = th.copy()
    th2[2] += 180.0
    m2 = oracle.model_maps(th2, cfg)[0]
    assert np.allclose(m2[1], -m[1], atol=1e-9 * np.abs(m[1]).max())
    for q in (0, 2, 3):
        assert np.allclose(m2[q], m[q], rtol=1e-11)
    th3 = th.copy()
    th3[3] = 0.0
    assert np.abs(oracle.model_maps(th3, cfg)[0][1]).max() == 0.0
