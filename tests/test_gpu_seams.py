"""GPU parity on parameter vectors BUILT to hit the seams of the CUDA path's tables and branches, instead of hoping that a
prior draw finds them ("parity is thin where it matters"):

  * the SigmaTilde series / closed-form switch at |1 - s^2| = 1/4 (s^2 = 0.75, 1.25) with many cells on both sides;
  * the first and the last octave of the per-theta radial tables: centre exactly on a fine-cell centre (R = 0 -> the
    floor of reading V), centre far outside the field, corners at i = 80 deg and 85 deg;
  * R_b = 0.1 kpc (prior edge) and 0.02 kpc: s = R/R_b up to ~600 at the map corner;
  * Freeman-disc argument y = r/2R_d across y = 2 and y = 32 (series / quadrature / asymptotic switches of the table
    build) and NFW r/r_s across the series switch;
  * P.A. = 0, 90, 180 deg (x' or y' exactly zero along a row or a column), k = 0, +-1, extreme M/L.

Everything is compared element by element with the oracle: the un-convolved fine maps (steps a0-a3) and the final maps
(a4-a5), in both precisions, plus logL (a6).  Tolerances: BASELINE.json's 1e-9 / 1e-4 per pixel with reading P's
denominator for v_los; logL as in tests/test_gpu_parity.py (reading Q).
"""
import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W
from test_gpu_parity import assert_logl, assert_maps

pytestmark = pytest.mark.gpu

# the config-2 grid (64 x 64, s = 3, sigma = 1 px, N_J = 64, four components, NFW halo)
CFG = W.config(2)
ON_CELL = 1.0 / 6.0           # s = 3, even N: fine-cell centres sit at ((J + 1/2)/3 - N/2) arcsec -> 1/6 arcsec for J = 3N/2


def seam_thetas():
    t0 = W.theta_true(2)
    t0[12] = 4.0                                   # (M/L)_b inside the prior box
    out = {}

    def add(name, **kw):
        t = t0.copy()
        for k, v in kw.items():
            t[W.THETA_NAMES.index(k)] = v
        out[name] = t

    add("truth")
    add("Rb3_many_cells_at_s_eq_1", Rb=3.0, log10Mb=11.0)
    add("Rb_prior_min", Rb=0.1)
    add("Rb_tiny", Rb=0.02, log10Mb=9.0)
    add("centre_on_cell", x0=ON_CELL, y0=ON_CELL)
    add("centre_on_cell_i80", x0=ON_CELL, y0=ON_CELL, inc=80.0)
    add("centre_on_corner_cell", x0=ON_CELL - 32.0, y0=ON_CELL - 32.0)
    add("centre_outside_field", x0=45.0, y0=-38.0)
    add("i80_Rd_min", inc=80.0, Rd1=0.5, Rd2=0.5)                       # y = r/2R_d up to ~70: all three Freeman branches
    add("i85", inc=85.0)
    add("i20_Rd_max", inc=20.0, Rd1=10.0, Rd2=10.0)
    add("nfw_c20_M10", log10Mh=10.0, Rh_or_c=20.0)                      # r_s = 2.2 kpc: r/r_s from 0.01 to 30
    add("nfw_c3_M13", log10Mh=13.0, Rh_or_c=3.0)                        # r_s = 148 kpc: the series branch everywhere
    add("PA0", PA=0.0)
    add("PA90", PA=90.0, x0=0.0, y0=ON_CELL)
    add("PA180_k1", PA=180.0, k1=1.0, k2=1.0)
    add("k0", k1=0.0, k2=0.0)
    add("k_minus1", k1=-1.0, k2=-1.0)
    add("ML_extremes", MLb=0.5, MLd1=5.0, MLd2=0.5)
    add("light_bulge_heavy_discs", log10Mb=8.0, log10Md1=11.5, log10Md2=11.5)
    add("heavy_bulge_light_discs", log10Mb=11.0, log10Md1=9.0, log10Md2=9.0, Rb=0.1)
    return out


@pytest.fixture(scope="module")
def bang():
    import torch
    assert torch.cuda.is_available()
    from paper_2205_06819_b200 import bang as b
    b.lib()
    return b


@pytest.fixture(scope="module")
def seam_case(oracle):
    th = seam_thetas()
    names = list(th)
    theta = np.stack([th[n] for n in names])
    mtrue = oracle.model_maps(W.theta_true(2), CFG)[0]
    data, err, mask = W.make_data(2, mtrue)
    logl_o, maps_o = oracle.loglike(theta, CFG, data, err, mask, return_maps=True)
    fine_o = np.stack([oracle.model_fine(t, CFG) for t in theta])
    return names, theta, data, err, mask, logl_o, maps_o, fine_o


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_seam_thetas_match_the_oracle(bang, seam_case, prec):
    names, theta, data, err, mask, logl_o, maps_o, fine_o = seam_case
    ctx = bang.Context(CFG, precision=prec)
    ctx.set_data(data, err, mask)
    fine = ctx.model_fine(theta).cpu().numpy()
    maps = ctx.model_maps(theta).cpu().numpy()
    ll = ctx.loglike(theta).cpu().numpy()
    ctx.close()
    assert np.isfinite(maps).all() and np.isfinite(ll).all()
    for b, name in enumerate(names):
        assert_maps(fine[b], fine_o[b], prec, f"{name} fine")
        assert_maps(maps[b], maps_o[b], prec, f"{name} maps")
    assert_logl(ll, logl_o, maps_o, data, err, mask, prec, near=np.array([n == "truth" for n in names]), what="seams")


# ------------------------------------------------------------------------------------------------ the edge of the tables
def extreme_thetas():
    """Valid parameter vectors (in the sense of include/bang.h) whose radii leave the tabulated ranges of the fast path:
    more octaves of r^2 on the grid than the per-theta table holds, or R/R_b outside the scale-free bulge tables."""
    t0 = W.theta_true(2)
    t0[12] = 4.0
    out = []
    a = t0.copy(); a[[0, 1, 3]] = [ON_CELL_SMALL, ON_CELL_SMALL, 89.999]     # R = 0 at one cell, r up to ~1e6 kpc
    out.append(a)
    b = t0.copy(); b[5] = 1e-6                                               # R/R_b up to ~1e7 > 2^18
    out.append(b)
    c = t0.copy(); c[[0, 1, 5]] = [ON_CELL_SMALL, ON_CELL_SMALL, 200.0]      # floor/R_b = 2^-16/200 < 2^-22
    out.append(c)
    d = t0.copy(); d[3] = 89.9                                               # r/2R_d ~ 1e4
    out.append(d)
    return np.stack(out)


SMALL_BASE = dict(W.config(2), nx=16, ny=12, supersample=2, jeans_nodes=32)
ON_CELL_SMALL = 0.25          # s = 2, even N: fine-cell centres at ((J + 1/2)/2 - N/2) arcsec


@pytest.mark.parametrize("variant", [{}, {"psf_weighting": 1}, {"bulge_potential": 1}, {"bulge_profile": 1}],
                         ids=["paper", "flux_psf", "total_potential", "jaffe"])
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_radii_outside_the_tabulated_ranges_take_the_direct_path(bang, oracle, prec, variant):
    """include/bang.h: the library's domain is the model's (R_b, R_d > 0, |i| < 90 deg, ...), not the tables': a theta
    whose grid leaves the tabulated ranges is evaluated directly (slow path), cell by cell, and must match the oracle
    like any other -- in the paper's model and in the widened variants (readings G', U', App. B)."""
    SMALL = dict(SMALL_BASE, **variant)
    theta = extreme_thetas()
    t0 = W.theta_true(2)
    t0[12] = 4.0
    both = np.concatenate([t0[None], theta, t0[None]])               # fast-path theta around the slow ones, one batch
    mtrue = oracle.model_maps(t0, SMALL)[0]
    rng = np.random.default_rng(7)
    err = np.stack([0.05 * np.abs(mtrue[0]), np.full_like(mtrue[1], 10.0), np.full_like(mtrue[2], 10.0),
                    np.full_like(mtrue[3], 0.1)])
    data = mtrue + err * rng.standard_normal(mtrue.shape)
    mask = rng.random(mtrue.shape) > 0.2
    logl_o, want = oracle.loglike(both, SMALL, data, err, mask, return_maps=True)
    assert np.isfinite(want).all()
    ctx = bang.Context(SMALL, precision=prec)
    ctx.set_data(data, err, mask)
    got = ctx.model_maps(both).cpu().numpy()
    fine = ctx.model_fine(both).cpu().numpy()
    ll = ctx.loglike(both).cpu().numpy()
    ll_again = ctx.loglike(both).cpu().numpy()                        # the list of slow theta is emptied between calls
    ctx.close()
    for b in range(len(both)):
        assert_maps(got[b], want[b], prec, f"extreme theta {b}")
        assert_maps(fine[b], oracle.model_fine(both[b], SMALL), prec, f"extreme theta {b} fine")
    assert_logl(ll, logl_o, want, data, err, mask, prec, what="direct path")
    assert np.array_equal(ll, ll_again) and ll[0] == ll[-1]
