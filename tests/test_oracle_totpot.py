"""Pins for the oracle's total-potential bulge dispersion (reading U'; the limitation
the paper names at PAPER.md:107 and :417-419).

    rho_b v_r^2 (r) = int_r^inf rho_b(x) v_c,tot^2(x)/x dx          (isotropic spherical Jeans, G M(<x) = x v_c,tot^2)
    I_b(R) = 2 int_0^inf rho_b v_r^2 (sqrt(R^2+z^2)) dz            (eq. 6, first form)
           = I_b,self(R) [the paper's path] + I_ext(R),   I_ext = 2 int_R^inf rho_b v_ext^2 sqrt(x^2-R^2)/x dx.

The oracle's N_J-node rule for I_ext is pinned to things other than itself:
  * the paper's own closed form of eq. 6 (reading A): a Hernquist "halo" with the bulge's mass and scale radius pulls on
    the bulge exactly as the bulge pulls on itself, so I_ext must equal G M_b^2/(12 pi R_b^3) ITilde(s);
  * brute force: the DOUBLE integral as defined (Jeans integral inside, l.o.s. integral outside) by adaptive quadrature
    with scipy's Bessel functions, for an exponential disc + NFW halo and for the Jaffe bulge, at three radii;
  * the reduction to the paper's path when nothing but the bulge is there, linearity in the external mass, and what the
    variant may and may not change in the maps.
"""
import math

import numpy as np
import pytest
from scipy import integrate, special

from paper_2205_06819_b200 import workloads as W

G = 4.30091727004e-6
B_, D1, D2, H = 1, 2, 4, 8


@pytest.fixture(scope="module")
def L(oracle):
    return oracle.lib()


def iext(L, R, Mb=1e10, Rb=0.8, bulge=0, Md1=0.0, Rd1=1.0, Md2=0.0, Rd2=1.0, Mh=0.0, Rh=1.0, halo=0, comps=B_, NJ=64):
    return L.bo_Ib_ext_quadrature(R, Mb, Rb, bulge, Md1, Rd1, Md2, Rd2, Mh, Rh, halo, comps, NJ)


# ------------------------------------------------------------------------------------------------ the paper's eq. 6
@pytest.mark.parametrize("NJ,tol", [(32, 2e-6), (64, 1e-9), (128, 1e-12)])
def test_a_hernquist_halo_equal_to_the_bulge_reproduces_eq6(L, NJ, tol):
    Mb, Rb = 3e10, 0.7
    for s in (0.01, 0.1, 0.5, 0.9, 1.3, 2.0, 10.0, 100.0):
        got = iext(L, s * Rb, Mb, Rb, Mh=Mb, Rh=Rb, halo=0, comps=B_ | H, NJ=NJ)
        want = G * Mb * Mb / (12 * math.pi * Rb ** 3) * L.bo_I_tilde_closed(s)      # reading A, binary128
        assert abs(got / want - 1) < tol, (s, got / want - 1)


# ------------------------------------------------------------------------------------------------ brute force
def freeman_vc2(x, Md, Rd):
    y = x / (2 * Rd)
    return 2 * G * Md / Rd * y * y * (special.i0e(y) * special.k0e(y) - special.i1e(y) * special.k1e(y))


def nfw_vc2(x, M200, c):
    rho_c = 3 * 0.07 ** 2 / (8 * math.pi * G)
    r200 = (3 * M200 / (4 * math.pi * 200 * rho_c)) ** (1 / 3)
    mu = lambda u: math.log1p(u) - u / (1 + u)
    return G * M200 * mu(x * c / r200) / (x * mu(c))


def brute(R, rho, vext2):
    """2 int_0^inf dz int_{sqrt(R^2+z^2)}^inf rho(x) vext2(x)/x dx, as defined (nested adaptive quadrature in ln x, ln z)."""
    def P(r):
        f = lambda w: rho(math.exp(w)) * vext2(math.exp(w))                  # dx/x = dw
        return integrate.quad(f, math.log(r), math.log(r) + 40, epsrel=1e-12, epsabs=0, limit=400)[0]
    g = lambda z: P(math.hypot(R, z))
    a = integrate.quad(g, 0, R, epsrel=1e-10, epsabs=0, limit=200)[0]
    b = integrate.quad(lambda w: g(math.exp(w)) * math.exp(w), math.log(R), math.log(R) + 30, epsrel=1e-10, epsabs=0, limit=400)[0]
    return 2 * (a + b)


@pytest.mark.parametrize("bulge", [0, 1])
@pytest.mark.parametrize("R", [0.05, 0.8, 6.0])
def test_rule_against_the_double_integral_as_defined(L, bulge, R):
    Mb, Rb, Md, Rd, M200, c = 10 ** 10.3, 0.6, 10 ** 10.8, 2.5, 10 ** 12.2, 9.0
    rho = lambda x: L.bo_rho_bulge(x, Mb, Rb, bulge)
    want = brute(R, rho, lambda x: freeman_vc2(x, Md, Rd) + nfw_vc2(x, M200, c))
    for NJ, tol in ((32, 3e-5), (64, 2e-8), (128, 2e-9)):
        got = iext(L, R, Mb, Rb, bulge, Md1=Md, Rd1=Rd, Mh=M200, Rh=c, halo=1, comps=B_ | D1 | H, NJ=NJ)
        assert abs(got / want - 1) < tol, (NJ, got / want - 1)


def test_rho_bulge_is_eq1_and_eqB1_and_integrates_to_the_mass(L):
    Mb, Rb = 2e10, 0.9
    for prof in (0, 1):
        m = integrate.quad(lambda w: 4 * math.pi * math.exp(3 * w) * L.bo_rho_bulge(math.exp(w), Mb, Rb, prof), -40, 40,
                           epsrel=1e-12, limit=400)[0]
        assert abs(m / Mb - 1) < 1e-9
    x = 1.7
    assert abs(L.bo_rho_bulge(x, Mb, Rb, 0) / (Mb / (2 * math.pi) * Rb / x / (x + Rb) ** 3) - 1) < 1e-14      # eq. 1
    assert abs(L.bo_rho_bulge(x, Mb, Rb, 1) / (Mb / (4 * math.pi) * Rb / x ** 2 / (x + Rb) ** 2) - 1) < 1e-14  # eq. B1


def test_linear_in_the_external_mass_and_additive_over_components(L):
    a = iext(L, 1.1, Md1=1e10, Rd1=2.0, comps=B_ | D1)
    b = iext(L, 1.1, Md1=3e10, Rd1=2.0, comps=B_ | D1)
    h = iext(L, 1.1, Mh=1e12, Rh=8.0, halo=1, comps=B_ | H)
    both = iext(L, 1.1, Md1=1e10, Rd1=2.0, Mh=1e12, Rh=8.0, halo=1, comps=B_ | D1 | H)
    assert abs(b / a - 3) < 1e-13 and abs(both / (a + h) - 1) < 1e-13
    assert iext(L, 1.1, Md1=1e10, Rd1=2.0, comps=B_) == 0.0                    # an absent component does not pull


# ------------------------------------------------------------------------------------------------ maps
def small(**kw):
    cfg = dict(W.config(1), nx=12, ny=10, jeans_nodes=32)
    cfg.update(kw)
    return cfg


def test_reduces_to_the_papers_path_without_external_components(oracle):
    th = W.theta_true(1)
    a = oracle.model_maps(th, small(components=B_))
    b = oracle.model_maps(th, small(components=B_, bulge_potential=1))
    assert np.array_equal(a, b)
    th2 = th.copy()
    th2[6] = 0.0                                           # a disc of one solar mass: nothing changes beyond 1e-9
    a = oracle.model_maps(th2, small())
    b = oracle.model_maps(th2, small(bulge_potential=1))
    assert np.allclose(a, b, rtol=1e-9, atol=0)


def test_only_the_dispersion_changes_and_it_grows(oracle):
    for idx, cfg in ((1, small()), (2, dict(W.config(2), nx=12, ny=10, jeans_nodes=32))):
        th = W.theta_true(idx)
        a = oracle.model_fine(th, cfg)
        b = oracle.model_fine(th, dict(cfg, bulge_potential=1))
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[3], b[3])
        assert (b[2] > a[2]).all()
        # by hand at one cell: sigma^2 B_tot gains I_ext / (M/L)_b 1e-6
        Lb = oracle.lib()
        rk = oracle.psf_halfwidth(cfg)
        jy, jx = rk + 7, rk + 9
        s = cfg["supersample"]
        kappa = 50.0 * 4.84813681109536e-3
        X = (((jx - rk) + 0.5) / s - 0.5 * cfg["nx"]) * kappa - th[0] * kappa
        Y = (((jy - rk) + 0.5) / s - 0.5 * cfg["ny"]) * kappa - th[1] * kappa
        R = math.hypot(X, Y)
        comps = cfg["components"]
        ie = Lb.bo_Ib_ext_quadrature(R, 10 ** th[4], th[5], 0, 10 ** th[6], th[7], 10 ** th[8], th[9], 10 ** th[10], th[11],
                                     cfg["halo_profile"], comps, cfg["jeans_nodes"])
        gain = (b[2, jy, jx] ** 2 - a[2, jy, jx] ** 2) * a[0, jy, jx]
        assert abs(gain / (ie / th[12] * 1e-6) - 1) < 1e-10
