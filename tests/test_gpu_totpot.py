"""GPU parity for the bulge dispersion in the TOTAL potential (bang_model.bulge_potential = BANG_POTENTIAL_TOTAL; reading
U'; the limitation the paper names at PAPER.md:107 and :417-419).

The CUDA path tabulates Itilde_ext per theta inside the fused kernel (build_bulge_tables: north_star's per-theta kernel
(1)); the oracle evaluates the same N_J-node rule directly at every fine cell (oracle/bang_oracle.cpp,
Ib_ext_quadrature, pinned in tests/test_oracle_totpot.py).  Compared element by element on fine maps, maps and logL in
both precisions at the tolerances of tests/test_gpu_parity.py (1e-9 / 1e-4 per pixel; readings P and Q).
"""
import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W
from test_gpu_parity import assert_logl, assert_maps, bang  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


def _three_theta():
    theta = np.stack([W.theta_true(1), W.theta_true(1) * 1.01, W.theta_true(1) * 0.99])
    theta[1, 0:2] = 0.37, -0.21                              # off-centre
    theta[2, 0:2] = 0.0, 0.0                                 # the centre exactly between cells: R_min = h/sqrt(2)
    return theta


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
@pytest.mark.parametrize("bulge_profile", [0, 1])
def test_total_potential_config1_grid(bang, oracle, prec, bulge_profile):
    # BASELINE.json config 1 (bulge + one disc, no halo) plus the same grid with a second disc and a Hernquist halo
    for comps, halo in ((W.config(1)["components"], 0), (15, 0), (15, 1)):
        cfg = dict(W.config(1), bulge_potential=1, bulge_profile=bulge_profile, components=comps, halo_profile=halo)
        theta = _three_theta()
        if comps == 15:
            theta[:, 8:10] = 10.2, 6.0                       # outer disc
            theta[:, 10:12] = (12.0, 8.0) if halo == 1 else (11.5, 15.0)
            theta[:, 14], theta[:, 16] = 1.5, 0.7
        maps_o = oracle.model_maps(theta, cfg)
        data, err, mask = W.make_data(1, maps_o[0])
        logl_o, maps_o = oracle.loglike(theta, cfg, data, err, mask, return_maps=True)
        ctx = bang.Context(cfg, precision=prec)
        fine = ctx.model_fine(theta[:2]).cpu().numpy()
        for b in range(2):
            assert_maps(fine[b], oracle.model_fine(theta[b], cfg), prec, f"totpot fine {comps}/{halo}")
        ctx.set_data(data, err, mask)
        maps = ctx.model_maps(theta).cpu().numpy()
        ll = ctx.loglike(theta).cpu().numpy()
        ctx.close()
        assert_maps(maps, maps_o, prec, f"totpot maps {comps}/{halo}")
        assert_logl(ll, logl_o, maps_o, data, err, mask, prec, near=np.array([True, False, False]), what="totpot cfg1")
        # the switch matters (sigma_los rises where the bulge shines) and touches nothing but sigma_los
        plain = oracle.model_maps(theta[:1], dict(cfg, bulge_potential=0))[0]
        assert (maps_o[0, 2] >= plain[2] * (1 - 1e-12)).all() and (maps_o[0, 2] / plain[2]).max() > 1.02
        for q in (0, 1, 3):
            assert np.array_equal(maps_o[0, q], plain[q])


def test_total_potential_prior_batch(bang, oracle):
    # a seeded subset of config 2's prior-drawn batch (four components, NFW halo), both precisions, fused launch shape
    cfg = dict(W.config(2), bulge_potential=1)
    theta = W.theta_batch(2)
    sub = W.parity_subset(2, theta.shape[0], 32)
    mtrue = oracle.model_maps(W.theta_true(2), cfg)[0]
    data, err, mask = W.make_data(2, mtrue)
    logl_o, maps_o = oracle.loglike(theta[sub], cfg, data, err, mask, return_maps=True)
    near = np.isin(sub, W.near_truth_slots(2, theta.shape[0]))
    for prec in ("fp32", "fp64"):
        ctx = bang.Context(cfg, precision=prec)
        ctx.set_data(data, err, mask)
        maps = ctx.model_maps(theta[sub]).cpu().numpy()
        ll_all = ctx.loglike(theta).cpu().numpy()               # the whole batch in bench.py's launch configuration
        ctx.close()
        assert np.isfinite(ll_all).all()
        assert_maps(maps, maps_o, prec, f"totpot cfg2 {prec}")
        assert_logl(ll_all[sub], logl_o, maps_o, data, err, mask, prec, near=near, what=f"totpot cfg2 {prec}")


def test_total_potential_reduces_to_the_paper_for_a_lone_bulge(bang):
    # nothing but the bulge: v_ext = 0, the variant is the paper's path bit for bit
    cfg = dict(W.config(1), components=1)
    theta = _three_theta()
    out = []
    for pot in (0, 1):
        ctx = bang.Context(dict(cfg, bulge_potential=pot), precision="fp64")
        out.append(ctx.model_maps(theta).cpu().numpy())
        ctx.close()
    assert np.array_equal(out[0], out[1])
