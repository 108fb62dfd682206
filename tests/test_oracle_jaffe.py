"""Pins for the Jaffe bulge of the oracle (Appendix B; reading J).  CPU only.

Each function is checked against something other than itself: the printed closed forms B4/B5 evaluated by mpmath,
the integrals that DEFINE the quantities (Abel projection of eq. B1, the isotropic Jeans integral, the line-of-sight
integral of rho v_r^2), textbook facts (total mass, enclosed mass, central dispersion) and the map-level reductions.
"""
import mpmath as mp
import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W

mp.mp.dps = 50


def _X(s):
    s = mp.mpf(s)
    if s < 1:
        return mp.asech(s) / mp.sqrt(1 - s * s)          # PAPER.md:100 eq. 5
    return mp.asec(s) / mp.sqrt(s * s - 1)


def _B4(s):                                              # PAPER.md:582 eq. B4, in units of M_b/R_b^2
    s = mp.mpf(s)
    return 1 / (4 * s) + (1 - (2 - s * s) * _X(s)) / (2 * mp.pi * (1 - s * s))


def _B5(s):                                              # PAPER.md:586 eq. B5 x Sigma_b, in units of G M_b^2/(4 pi R_b^3)
    s = mp.mpf(s)
    return (mp.pi / (2 * s) + 11 - mp.mpf(13) / 2 * mp.pi * s - 12 * s**2 + 6 * mp.pi * s**3
            - _X(s) * (6 - 19 * s**2 + 12 * s**4)) / (1 - s * s)


def _rho(r):                                             # PAPER.md:566 eq. B1, M_b = R_b = 1
    r = mp.mpf(r)
    return 1 / (4 * mp.pi * r**2 * (1 + r) ** 2)


def _jeans(r):                                           # int_r^inf rho G M(<x)/x^2 dx with M(<x) = x/(1+x), G = 1
    return mp.quad(lambda x: _rho(x) * (x / (1 + x)) / x**2, [r, 2 * r + 1, 10 * r + 10, mp.inf])


S_GRID = [1e-4, 1e-2, 0.1, 0.5, 0.9, 0.99, 1 - 1e-6, 1 - 1e-9, 1.0, 1 + 1e-9, 1 + 1e-6, 1.01, 1.5, 1.9999, 2.0001, 10.0, 300.0]


@pytest.mark.parametrize("s", S_GRID)
def test_jaffe_sigma_tilde_vs_mpmath_closed_form(oracle, s):
    want = mp.mpf(1) / 4 - 2 / (3 * mp.pi) if s == 1.0 else _B4(s)
    assert abs(oracle.lib().bo_jaffe_sigma_tilde(s) / float(want) - 1) < 5e-15


@pytest.mark.parametrize("s", [0.05, 0.7, 1.3, 6.0])
def test_jaffe_sigma_tilde_is_the_abel_projection_of_eq_B1(oracle, s):
    s = mp.mpf(s)
    proj = 2 * mp.quad(lambda z: _rho(mp.sqrt(s * s + z * z)), [0, s, 1 + s, 10 + 10 * s, mp.inf])
    assert abs(oracle.lib().bo_jaffe_sigma_tilde(float(s)) / float(proj) - 1) < 1e-13


def test_jaffe_total_and_enclosed_mass(oracle):
    # 4 pi int rho r^2 dr = r/(1+r) (M_b = R_b = 1) -> v_c^2 = G M(<r)/r = G M_b/(r + R_b), eq. B2
    L = oracle.lib()
    for r in (0.01, 0.3, 2.0, 50.0):
        m = 4 * mp.pi * mp.quad(lambda x: _rho(x) * x * x, [0, r])
        assert abs(float(m) - r / (1 + r)) < 1e-14
        assert abs(L.bo_vc2_jaffe(r * 0.7, 3e10, 0.7) / (L.bo_G() * 3e10 * float(m) / (r * 0.7)) - 1) < 1e-13
    # projected density integrates to the total mass: 2 pi int_0^S SigmaTildeJ s ds + pi/(4 S) = 1, the second term being
    # the mass projected beyond S >> 1, where Sigma -> M_b R_b/(8 R^3) (from rho -> M_b R_b/(4 pi r^4))
    f = lambda x: mp.mpf(L.bo_jaffe_sigma_tilde(float(x))) * x
    S = mp.mpf(10000)
    inner = mp.quad(f, [0, 0.25, 0.5, 0.75, 0.9, 0.99, 1, 1.01, 1.1, 1.5, 2, 5, 10, 100, 1000, S])
    assert abs(2 * mp.pi * inner + mp.pi / (4 * S) - 1) < 1e-7


@pytest.mark.parametrize("x", [1e-3, 0.03, 0.5, 1.0, 1.01, 3.0, 30.0, 1e3])
def test_jaffe_rho_vr2_is_the_isotropic_jeans_integral(oracle, x):
    L = oracle.lib()
    G, M, a = L.bo_G(), 2.5e10, 0.8
    got = L.bo_rho_vr2_jaffe(x * a, M, a)
    want = mp.mpf(G) * M * M / a**4 * _jeans(mp.mpf(x))
    assert abs(got / float(want) - 1) < 1e-12


@pytest.mark.parametrize("x", [0.01, 0.1, 0.7, 1.0, 4.0, 10.0])
def test_eq_B3_with_reading_J_equals_the_jeans_form(oracle, x):
    # eq. B3 with a = R_b and the braces' sign reversed (reading J): v_r^2 = rho v_r^2 / rho
    L = oracle.lib()
    G, M, a = L.bo_G(), 2.5e10, 0.8
    rho = M / a**3 * float(_rho(x))
    assert abs(L.bo_rho_vr2_jaffe(x * a, M, a) / rho / L.bo_vr2_jaffe_corrected(x * a, M, a) - 1) < 1e-12
    # ... and the printed sign gives a NEGATIVE square: the reading is forced
    xx = mp.mpf(x)
    printed = xx**2 * (1 + xx) ** 2 * (3 / xx + (6 * xx + 7) / (2 * (1 + xx) ** 2) - 1 / (2 * xx**2) - 6 * mp.log(1 + 1 / xx))
    assert printed < 0


def test_jaffe_dispersion_limits(oracle):
    # centre: v_r^2 -> G M_b/(2 R_b) (Jaffe 1983); far out: v_r^2 -> G M_b/(5 r), like any finite-mass r^-4 halo
    L = oracle.lib()
    G, M, a = L.bo_G(), 1e11, 1.3
    r = 1e-6 * a
    rho = M / a**3 * float(_rho(r / a))
    assert abs(L.bo_rho_vr2_jaffe(r, M, a) / rho / (G * M / (2 * a)) - 1) < 1e-4
    r = 1e5 * a
    rho = M / a**3 * float(_rho(r / a))
    assert abs(L.bo_rho_vr2_jaffe(r, M, a) / rho / (G * M / (5 * r)) - 1) < 1e-4


def test_J3_branches_agree(oracle):
    L = oracle.lib()
    for t in (0.999999, 1.0, 1.000001, 1e-9, 1e3):     # closed form (cancels ~100x at t = 1) / series
        tt = mp.mpf(t)
        want = mp.quad(lambda x: 1 / (x**3 * (1 + x) ** 3), [tt, 2 * tt + 1, 10 * tt + 10, mp.inf])
        assert abs(L.bo_J3(t) / float(want) - 1) < 1e-12


@pytest.mark.parametrize("s", S_GRID)
def test_jaffe_I_tilde_closed_vs_mpmath(oracle, s):
    want = mp.limit(_B5, 1) if s == 1.0 else _B5(s)
    assert abs(oracle.lib().bo_jaffe_I_tilde_closed(s) / float(want) - 1) < 1e-12


@pytest.mark.parametrize("s", [0.02, 0.4, 1.7, 25.0])
def test_jaffe_I_tilde_is_the_los_integral_of_rho_vr2(oracle, s):
    # eq. B5 x B4 = 2 int_0^inf dz int_{sqrt(s^2+z^2)}^inf rho G M(<x)/x^2 dx (the DEFINING integrals, not the oracle's
    # J3); exchanging the order of integration, = 2 int_s^inf rho G M(<x)/x^2 sqrt(x^2 - s^2) dx, a single quadrature
    s = mp.mpf(s)
    los = 2 * mp.quad(lambda x: 4 * mp.pi * _rho(x) * (x / (1 + x)) / x**2 * mp.sqrt(x * x - s * s),
                      [s, 2 * s, 1 + 2 * s, 10 + 10 * s, mp.inf])
    assert abs(oracle.lib().bo_jaffe_I_tilde_closed(float(s)) / float(los) - 1) < 1e-10


@pytest.mark.parametrize("NJ,bound,bound_inner", [(32, 1e-9, 5e-4), (64, 1e-12, 2e-7), (128, 1e-12, 1e-12)])
def test_jaffe_jeans_quadrature_vs_closed_form(oracle, NJ, bound, bound_inner):
    # the N_J-node rule of reading B applied to the Jaffe integrand, against eq. B5 x B4 (bounds measured with mpmath)
    L = oracle.lib()
    G, M, a = L.bo_G(), 4e10, 0.6
    for s in (1e-3, 1e-2, 0.1, 0.5, 0.999, 1.0, 3.0, 30.0, 300.0):
        want = G * M * M / (4 * np.pi * a**3) * L.bo_jaffe_I_tilde_closed(s)
        got = L.bo_Ib_quadrature_jaffe(s * a, M, a, NJ)
        assert abs(got / want - 1) < (bound if s >= 0.1 else bound_inner), (NJ, s)


# ---------------------------------------------------------------------------------------------- maps
def _cfg(**kw):
    cfg = W.config(1)
    cfg.update(bulge_profile=1, **kw)
    return cfg


def test_jaffe_bulge_only_map_reduces_to_closed_forms(oracle):
    # point-sampled (s = 1, no PSF), bulge only: B = Sigma_b/(M/L), sigma_los^2 = (B5 x B4)/B4, v = 0, M/L = (M/L)_b
    cfg = _cfg(components=W.BULGE, supersample=1, sigma_pix=0.0, nx=16, ny=16, jeans_nodes=128)
    th = W.theta_true(1)
    th[0], th[1] = 0.31, -0.17
    m = oracle.model_maps(th, cfg)[0]
    L = oracle.lib()
    Mb, Rb, MLb = 10 ** th[4], th[5], th[12]
    kap = L.bo_kappa(cfg["dist_mpc"])
    for (i, j) in [(0, 0), (7, 8), (8, 8), (15, 3)]:
        x = (j - 7.5) * cfg["pix_arcsec"] - th[0]
        y = (i - 7.5) * cfg["pix_arcsec"] - th[1]
        s = float(np.hypot(x, y)) * kap / Rb
        Sig = Mb / Rb**2 * float(_B4(s))
        assert abs(m[0, i, j] / (Sig / MLb * 1e-6) - 1) < 1e-12
        sig2 = L.bo_G() * Mb**2 / (4 * np.pi * Rb**3) * float(_B5(s)) / Sig
        assert abs(m[2, i, j] / np.sqrt(sig2) - 1) < 1e-10
        assert m[1, i, j] == 0.0
        assert abs(m[3, i, j] / MLb - 1) < 1e-13


def test_jaffe_and_hernquist_share_everything_but_the_bulge(oracle):
    # discs only: the bulge profile switch must not matter
    cfg_h = W.config(1)
    cfg_h["components"] = W.DISC1
    cfg_j = dict(cfg_h, bulge_profile=1)
    th = W.theta_true(1)
    assert np.array_equal(oracle.model_maps(th, cfg_h), oracle.model_maps(th, cfg_j))
    # with the bulge on, the maps differ, and the Jaffe centre is brighter (Sigma ~ 1/R against ~ ln 1/R)
    a = oracle.model_maps(th, W.config(1))[0]
    b = oracle.model_maps(th, _cfg())[0]
    assert b[0, 16, 16] > a[0, 16, 16] and not np.allclose(a[2], b[2])


def test_jaffe_invariants(oracle):
    cfg = _cfg()
    th = W.theta_true(1)
    m = oracle.model_maps(th, cfg)[0]
    th2 = th.copy()
    th2[2] += 180.0                                       # P.A. + 180 deg: v flips, the rest is unchanged
    m2 = oracle.model_maps(th2, cfg)[0]
    assert np.allclose(m2[1], -m[1], rtol=0, atol=1e-9 * np.abs(m[1]).max())
    for q in (0, 2, 3):
        assert np.allclose(m2[q], m[q], rtol=1e-11)
    for q, sgn in ((0, 1), (1, -1), (2, 1), (3, 1)):      # point symmetry about the centre (x0 = y0 = 0)
        assert np.allclose(m[q][::-1, ::-1], sgn * m[q], rtol=1e-10, atol=1e-9)
    th3 = th.copy()
    th3[3] = 0.0                                          # face-on: no line-of-sight rotation
    assert np.abs(oracle.model_maps(th3, cfg)[0][1]).max() == 0.0
