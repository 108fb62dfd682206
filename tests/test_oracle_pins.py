"""Pins for the scalar building blocks of oracle/bang_oracle.cpp (CPU only).

Each block is checked against something other than itself: high-precision mpmath evaluation of the
paper's printed closed forms, direct numerical integration of the defining integrals, textbook limits
and library routines.  Citations are PAPER.md:<line> (section / equation).
"""
import os

import mpmath as mp
import numpy as np
import pytest

mp.mp.dps = 50
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _X(s):
    s = mp.mpf(s)
    if s < 1:
        return mp.asech(s) / mp.sqrt(1 - s * s)          # PAPER.md:100 eq. 5, first branch
    return mp.asec(s) / mp.sqrt(s * s - 1)               # second branch


def _sigma_tilde_mp(s):
    s = mp.mpf(s)
    return ((2 + s * s) * _X(s) - 3) / (1 - s * s) ** 2   # PAPER.md:96 eq. 4


def _I_tilde_mp(s):
    s = mp.mpf(s)                                        # PAPER.md:105 eq. 6 second form (reading A)
    br = (-3 * s**2 * _X(s) * (8 * s**6 - 28 * s**4 + 35 * s**2 - 20) - 24 * s**6 + 68 * s**4 - 65 * s**2 + 6)
    return br / (2 * (1 - s * s) ** 3) - 6 * mp.pi * s


def _rho(r, M, a):
    r, M, a = mp.mpf(r), mp.mpf(M), mp.mpf(a)
    return M / (2 * mp.pi) * a / (r * (r + a) ** 3)      # PAPER.md:78 eq. 1


def _vr2(r, M, a, G):
    r, M, a, G = mp.mpf(r), mp.mpf(M), mp.mpf(a), mp.mpf(G)
    x = r / a                                            # PAPER.md:89 eq. 3
    return G * M / (12 * a) * (12 * r * (r + a) ** 3 / a**4 * mp.log((r + a) / r)
                               - r / (r + a) * (25 + 52 * x + 42 * x**2 + 12 * x**3))


# ---------------------------------------------------------------- eq. 5 / eq. 4
@pytest.mark.parametrize("s", [1e-6, 1e-3, 0.1, 0.5, 0.9, 0.95, 0.99, 0.999, 1 - 1e-5, 1 - 1e-6, 1 - 3e-8, 1 - 1e-9,
                               1.0, 1 + 1e-9, 1 + 3e-8, 1 + 1e-6, 1 + 1e-5, 1.001, 1.01, 1.05, 1.0999, 1.1001, 0.4999, 0.5001, 1.9999, 2.0001,
                               2.0, 10.0, 300.0, 1e4])
def test_sigma_tilde_vs_mpmath_closed_form(oracle, s):
    L = oracle.lib()
    want = mp.mpf(4) / 15 if s == 1.0 else _sigma_tilde_mp(s)
    assert abs(L.bo_sigma_tilde(s) / float(want) - 1) < 5e-15


@pytest.mark.parametrize("s", [0.05, 0.7, 1.3, 6.0])
def test_sigma_tilde_is_abel_projection_of_eq1(oracle, s):
    # PAPER.md:96 eq. 4, first equality: Sigma_b(R) = 2 int_R^inf rho r / sqrt(r^2 - R^2) dr, in units M=a=1
    L = oracle.lib()
    R = mp.mpf(s)
    f = lambda t: 2 * _rho(mp.sqrt(R * R + t * t), 1, 1)      # z-integral form, same thing
    val = mp.quad(f, [0, 1, 10, mp.inf])
    assert abs(float(val * 2 * mp.pi) / L.bo_sigma_tilde(s) - 1) < 1e-13


def test_hernquist_total_mass_from_projected_density(oracle):
    # 2 pi int Sigma_b R dR = M_b  (1-D; SURVEY.md §8(c) pins)
    L = oracle.lib()
    from scipy.integrate import quad
    f = lambda lnR: 2 * np.pi * L.bo_hernquist_Sigma(np.exp(lnR), 3.0e10, 0.7) * np.exp(2 * lnR)
    tot = quad(f, np.log(1e-8), np.log(1e7), limit=400, epsabs=0, epsrel=1e-11)[0]
    assert abs(tot / 3.0e10 - 1) < 1e-6      # the 1/R^3 tail beyond 1e7 a holds < 1e-7 of the mass


def test_sigma_tilde_series_coefficients(oracle):
    # reading I: 4/15 - (16/35) e + (8/15) e^2 from the printed form in 60 digits
    mp.mp.dps = 80
    try:
        h = mp.mpf("1e-12")
        f0 = mp.mpf(4) / 15
        fp, fm = _sigma_tilde_mp(1 + h), _sigma_tilde_mp(1 - h)
        assert abs((fp - fm) / (2 * h) + mp.mpf(16) / 35) < 1e-20
        assert abs((fp - 2 * f0 + fm) / (h * h) / 2 - mp.mpf(8) / 15) < 1e-10
    finally:
        mp.mp.dps = 50


# ---------------------------------------------------------------- eq. 1, 2, 3 and the Jeans integral
@pytest.mark.parametrize("x", [1e-3, 0.03, 0.5, 1.0, 7.0, 30.0, 300.0, 1e3])
def test_rho_vr2_equals_eq1_times_eq3(oracle, x):
    L = oracle.lib()
    M, a = 2.0e10, 0.6
    G = mp.mpf(L.bo_G())
    want = _rho(mp.mpf(x) * a, M, a) * _vr2(mp.mpf(x) * a, M, a, G)
    assert abs(L.bo_rho_vr2(x * a, M, a) / float(want) - 1) < 2e-14
    assert abs(L.bo_vr2_printed(x * a, M, a) / float(_vr2(mp.mpf(x) * a, M, a, G)) - 1) < 1e-14


def test_rho_vr2_is_the_isotropic_jeans_integral(oracle):
    # rho v_r^2 = int_r^inf rho G M(<x)/x^2 dx with M(<x) = M x^2/(x+a)^2 (Hernquist 1990)
    L = oracle.lib()
    M, a, G = mp.mpf(1e10), mp.mpf(1.3), mp.mpf(L.bo_G())
    for r in (0.01, 0.4, 2.0, 25.0):
        val = mp.quad(lambda x: _rho(x, M, a) * G * M * x * x / (x + a) ** 2 / (x * x), [r, 10 * r + 10, mp.inf])
        assert abs(L.bo_rho_vr2(r, float(M), float(a)) / float(val) - 1) < 1e-13


def test_vr2_large_radius_limit(oracle):
    # v_r^2 -> G M/(5 r) for r >> R_b
    L = oracle.lib()
    M, a, r = 1e10, 0.5, 5e4
    vr2 = L.bo_rho_vr2(r, M, a) / float(_rho(mp.mpf(r), M, a))
    assert abs(vr2 / (L.bo_G() * M / (5 * r)) - 1) < 1e-4


def test_T5_branches_agree(oracle):
    L = oracle.lib()
    for u in (1e-6, 0.1, 0.4999999, 0.5, 0.5000001, 0.9, 0.999999):
        want = -mp.log(1 - mp.mpf(u)) - sum(mp.mpf(u) ** n / n for n in range(1, 5))
        assert abs(L.bo_T5(u) / float(want) - 1) < 1e-14 or u > 0.49 and abs(L.bo_T5(u) / float(want) - 1) < 2e-13


def test_hernquist_vcirc_from_enclosed_mass(oracle):
    # PAPER.md:84 eq. 2 against G M(<r)/r with M(<r) = int 4 pi x^2 rho dx (eq. 1)
    L = oracle.lib()
    M, a = 4e10, 0.9
    for r in (0.05, 0.9, 12.0):
        Menc = mp.quad(lambda x: 4 * mp.pi * x * x * _rho(x, M, a), [0, r])
        assert abs(L.bo_vc2_hernquist(r, M, a) / (L.bo_G() * float(Menc) / r) - 1) < 1e-13


# ---------------------------------------------------------------- eq. 6
@pytest.mark.parametrize("s", [0.01, 0.1, 0.5, 0.97, 1.0, 1.04, 2.0, 10.0, 100.0, 1000.0])
def test_I_tilde_closed_vs_mpmath(oracle, s):
    L = oracle.lib()
    want = 664 / mp.mpf(35) - 6 * mp.pi if s == 1.0 else _I_tilde_mp(s)
    assert abs(L.bo_I_tilde_closed(s) / float(want) - 1) < 1e-14


@pytest.mark.parametrize("s", [0.2, 1.7])
def test_I_tilde_is_the_los_integral_of_eq1_eq3(oracle, s):
    # PAPER.md:105 eq. 6 first line, with eq. 1 and eq. 3 as printed, units G = M = R_b = 1:
    # Sigma_b sigma_b^2 = 2 int_0^inf rho v_r^2 dz = ITilde/(12 pi)
    # (eq. 3 cancels like x^5, so the integral is cut at z = 1e5 R_b where the z^-5 tail holds < 1e-20 of it)
    mp.mp.dps = 70
    try:
        val = mp.quad(lambda z: 2 * _rho(mp.sqrt(s * s + z * z), 1, 1) * _vr2(mp.sqrt(s * s + z * z), 1, 1, 1),
                      [0, 1, 10, 100, 1e3, 1e4, 1e5])
    finally:
        mp.mp.dps = 50
    assert abs(float(val * 12 * mp.pi) / oracle.lib().bo_I_tilde_closed(s) - 1) < 1e-12


def test_I_tilde_limits_and_series(oracle):
    L = oracle.lib()
    assert abs(L.bo_I_tilde_closed(1e-9) - 3.0) < 1e-7                       # ITilde(0) = 3
    mp.mp.dps = 80
    try:
        h = mp.mpf("1e-10")
        d1 = (_I_tilde_mp(1 + h) - _I_tilde_mp(1 - h)) / (2 * h)
        d2 = (_I_tilde_mp(1 + h) - 2 * (664 / mp.mpf(35) - 6 * mp.pi) + _I_tilde_mp(1 - h)) / (h * h) / 2
        assert abs(d1 + mp.mpf("0.259079731063")) < 1e-11
        assert abs(d2 - mp.mpf(80) / 231) < 1e-8
    finally:
        mp.mp.dps = 50
    # continuity across the series / binary128 switch
    a, b = L.bo_I_tilde_closed(1 + 0.99e-5), L.bo_I_tilde_closed(1 + 1.01e-5)
    assert abs(a - b) < 1e-7


@pytest.mark.parametrize("NJ,bound,bound_inner", [(32, 1e-6, 1e-11), (64, 1e-10, 5e-14), (128, 5e-14, 5e-14)])
def test_jeans_quadrature_vs_closed_form(oracle, NJ, bound, bound_inner):
    # reading B: N_J-node Gauss-Legendre rule against eq. 6's closed form; bounds of SURVEY.md §8(c) item B
    L = oracle.lib()
    M, a = 3e10, 0.8
    pref = L.bo_G() * M * M / (12 * np.pi * a**3)
    for s in np.logspace(-3, np.log10(300), 40):
        q = L.bo_Ib_quadrature(s * a, M, a, NJ) / pref
        rel = abs(q / L.bo_I_tilde_closed(s) - 1)
        assert rel < (bound if s < 0.1 else bound_inner), (s, rel)


def test_gauss_legendre_nodes(oracle):
    for n in (1, 2, 5, 32, 64, 128):
        x, w = oracle.gauss_legendre(n)
        xr, wr = np.polynomial.legendre.leggauss(n)
        assert np.allclose(x, xr, atol=2e-15, rtol=0) and np.allclose(w, wr, atol=1e-14, rtol=0)
        assert abs(w.sum() - 2) < 2e-15
        # exactness: integrates x^(2n-2) exactly
        assert abs(np.sum(w * x ** (2 * n - 2)) / (2.0 / (2 * n - 1)) - 1) < 1e-13
    # weights against 40-digit Newton-refined nodes (numpy's own weights are only good to ~1e-11 at n = 128)
    n = 64
    x, w = oracle.gauss_legendre(n)
    for xi, wi in zip(x[:8], w[:8]):
        z = mp.mpf(float(xi))
        for _ in range(3):
            dp = n * (z * mp.legendre(n, z) - mp.legendre(n - 1, z)) / (z * z - 1)
            z -= mp.legendre(n, z) / dp
        dp = n * (z * mp.legendre(n, z) - mp.legendre(n - 1, z)) / (z * z - 1)
        assert abs(wi / float(2 / ((1 - z * z) * dp * dp)) - 1) < 1e-12


# ---------------------------------------------------------------- eq. 9 (reading D)
@pytest.mark.parametrize("y", [1e-4, 0.05, 0.25, 1.075, 2.5, 10.0, 19.9, 29.9, 30.0, 30.1, 40.0, 200.0, 650.0, 5000.0])
def test_freeman_F_vs_mpmath_bessel(oracle, y):
    ym = mp.mpf(y)
    want = ym * ym * (mp.besseli(0, ym) * mp.besselk(0, ym) - mp.besseli(1, ym) * mp.besselk(1, ym))
    assert abs(oracle.lib().bo_freeman_F(y) / float(want) - 1) < 5e-15


@pytest.mark.parametrize("x", [0.3, 2.15, 6.0])
def test_freeman_disc_vs_direct_integration_of_the_potential(oracle, x):
    # razor-thin exponential disc, Sigma0 exp(-r/Rd): Phi(r,0) = -2 pi G int_0^inf J0(k r) S(k) dk with
    # S(k) = Sigma0 Rd^2 (1 + k^2 Rd^2)^(-3/2) (Hankel transform; Binney & Tremaine), so
    # v_c^2 = r dPhi/dr = 2 pi G Sigma0 Rd^2 r int_0^inf k J1(k r) (1 + k^2 Rd^2)^(-3/2) dk.
    L = oracle.lib()
    Md, Rd = 5e10, 2.0
    r = x * Rd
    Sigma0 = Md / (2 * mp.pi * Rd**2)
    integ = mp.quadosc(lambda k: k * mp.besselj(1, k * r) * (1 + k * k * Rd * Rd) ** mp.mpf(-1.5), [0, mp.inf],
                       omega=r)
    want = 2 * mp.pi * L.bo_G() * Sigma0 * Rd**2 * r * integ
    assert abs(L.bo_vc2_expdisc(r, Md, Rd) / float(want) - 1) < 1e-9


def test_freeman_disc_kepler_limit_and_peak(oracle):
    L = oracle.lib()
    Md, Rd = 1e10, 1.0
    assert abs(L.bo_vc2_expdisc(400.0, Md, Rd) / (L.bo_G() * Md / 400.0) - 1) < 1e-4     # 4 y F(y) -> 1
    rr = np.linspace(1.5, 3.0, 301)
    v = np.array([L.bo_vc2_expdisc(r, Md, Rd) for r in rr])
    assert abs(rr[np.argmax(v)] - 2.15) < 0.02 and abs(v.max() / (L.bo_G() * Md / Rd) - 0.38705) < 1e-4


# ---------------------------------------------------------------- reading H (NFW)
def test_nfw_worked_values(oracle):
    L = oracle.lib()
    G = L.bo_G()
    rho_c = 3 * 0.07**2 / (8 * np.pi * G)
    assert abs(rho_c - 135.9929474) < 1e-6
    for logM, c in ((12.5, 8.0), (10.0, 3.0), (13.0, 20.0)):
        M = 10**logM
        r200 = L.bo_nfw_r200(M)
        assert abs(M / (4 / 3 * np.pi * r200**3) / (200 * rho_c) - 1) < 1e-13            # mean density = 200 rho_c
        assert abs(L.bo_vc2_nfw(r200, M, c) / (G * M / r200) - 1) < 1e-13               # v_c^2(r200) = G M200/r200
        # enclosed mass of rho = rho_s / (x (1+x)^2) by direct integration
        rs = r200 / c
        for r in (0.3 * rs, 2.5 * rs):
            m_enc = mp.quad(lambda x: x * x / (x * (1 + x) ** 2), [0, r / rs])
            m_200 = mp.quad(lambda x: x * x / (x * (1 + x) ** 2), [0, c])
            assert abs(L.bo_vc2_nfw(r, M, c) / (G * M * float(m_enc / m_200) / r) - 1) < 1e-12
    assert abs(np.sqrt(G * 10**12.5 / L.bo_nfw_r200(10**12.5)) - 211.94331) < 1e-4
    assert abs(np.sqrt(G * 1e13 / L.bo_nfw_r200(1e13)) - 311.09023) < 1e-4


def test_nfw_mu_series_switch(oracle):
    L = oracle.lib()
    for x in (1e-8, 1e-4, 0.99e-2, 1.01e-2, 0.5):
        xm = mp.mpf(x)
        assert abs(L.bo_nfw_mu(x) / float(mp.log(1 + xm) - xm / (1 + xm)) - 1) < 1e-13


# ---------------------------------------------------------------- golden text fixtures
def test_golden_scalar_values(oracle):
    L = oracle.lib()
    fn = {"sigma_tilde": L.bo_sigma_tilde, "I_tilde": L.bo_I_tilde_closed, "freeman_F": L.bo_freeman_F,
          "nfw_r200": lambda lm: L.bo_nfw_r200(10.0**lm)}
    n = 0
    for line in open(os.path.join(GOLD, "hernquist_freeman_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, arg, val = line.split()
        digits = len(val.replace("-", "").replace(".", "").split("e")[0].lstrip("0"))
        assert abs(fn[kind](float(arg)) / float(val) - 1) < 2 * 10.0 ** (1 - digits), line
        n += 1
    assert n == 19
