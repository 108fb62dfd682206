"""The nested-sampling driver (paper_2205_06819_b200/nested.py; eq. 16-17) against analytic evidences.

CPU only: the driver takes any batched likelihood, so it is pinned on toy likelihoods whose evidence is known in closed
form (uniform prior on the unit cube): a Gaussian, a sum of two Gaussians, and a plateau with a sharp edge.
"""
import math

import numpy as np

from paper_2205_06819_b200.nested import NestedSampler, box_transform


def gauss_loglike(mu, sigma):
    mu = np.asarray(mu)

    def f(u):
        return -0.5 * (((u - mu) / sigma) ** 2).sum(axis=1) - u.shape[1] * math.log(sigma * math.sqrt(2 * math.pi))
    return f


def test_gaussian_evidence_is_one():
    # a NORMALISED Gaussian well inside the unit cube integrates to 1 under the uniform prior: ln Z = 0
    for d, sigma, seed in ((2, 0.03, 1), (4, 0.05, 2), (6, 0.07, 3)):
        ns = NestedSampler(gauss_loglike([0.5] * d, sigma), d, nlive=400, batch=50, mcmc_steps=25, seed=seed)
        r = ns.run()
        assert abs(r.logZ) < 3 * r.logZ_err + 0.05, (d, r.logZ, r.logZ_err)
        # information of a Gaussian posterior against a unit-volume prior: H = -d/2 ln(2 pi e sigma^2)
        H = -0.5 * d * math.log(2 * math.pi * math.e * sigma**2)
        assert abs(r.information - H) < 0.15 * H
        mean, std = r.posterior_mean_std()
        assert np.all(np.abs(mean - 0.5) < 4 * sigma / math.sqrt(50)) and np.all(np.abs(std / sigma - 1) < 0.15)
        assert abs(np.exp(r.logw).sum() - 1) < 1e-9


def test_two_modes_and_bayes_factor():
    # Z of a mixture is the sum of the parts; ln B_12 between a broad and a narrow UNNORMALISED Gaussian of equal peak
    # height is d ln(sigma_1/sigma_2) (eq. 17)
    d = 3
    g1, g2 = gauss_loglike([0.3] * d, 0.04), gauss_loglike([0.7] * d, 0.04)
    mix = lambda u: np.logaddexp(g1(u), g2(u)) + math.log(0.5) + 7.0
    r = NestedSampler(mix, d, nlive=600, batch=60, mcmc_steps=30, seed=5).run()
    assert abs(r.logZ - 7.0) < 3 * r.logZ_err + 0.05
    mean, _ = r.posterior_mean_std()
    assert np.all(np.abs(mean - 0.5) < 0.05)                         # both modes found, equally weighted
    peak = lambda s: (lambda u: -0.5 * (((u - 0.5) / s) ** 2).sum(axis=1))
    za = NestedSampler(peak(0.08), d, nlive=400, batch=40, mcmc_steps=25, seed=6).run()
    zb = NestedSampler(peak(0.04), d, nlive=400, batch=40, mcmc_steps=25, seed=7).run()
    assert abs((za.logZ - zb.logZ) - d * math.log(2.0)) < 3 * math.hypot(za.logZ_err, zb.logZ_err) + 0.05


def test_shrinkage_modes_determinism_and_batch_size():
    f = gauss_loglike([0.4, 0.6, 0.5], 0.05)
    a = NestedSampler(f, 3, nlive=300, batch=30, seed=11).run()
    b = NestedSampler(f, 3, nlive=300, batch=30, seed=11).run()
    assert a.logZ == b.logZ and a.n_evals == b.n_evals                # same seed, same run
    c = NestedSampler(f, 3, nlive=300, batch=30, seed=12, shrink="sampled").run()   # X_tau = t_tau X_(tau-1), t drawn
    d1 = NestedSampler(f, 3, nlive=300, batch=1, mcmc_steps=15, seed=13).run()       # the paper's one-at-a-time loop
    for r in (a, c, d1):
        assert abs(r.logZ) < 3 * r.logZ_err + 0.06, r.logZ
    # the batched run needs far fewer likelihood CALLS for the same number of evaluations per replacement
    assert a.n_iter * 30 < 2 * d1.n_iter


def test_box_transform_and_out_of_domain_points():
    th0 = np.arange(17.0)
    tr = box_transform(th0, [2, 5], np.array([10.0, -1.0]), np.array([20.0, 1.0]))
    th = tr(np.array([[0.0, 0.5], [1.0, 1.0]]))
    assert th.shape == (2, 17) and th[0, 2] == 10.0 and th[0, 5] == 0.0 and th[1, 2] == 20.0 and th[1, 5] == 1.0
    assert np.array_equal(np.delete(th[1], [2, 5]), np.delete(th0, [2, 5]))
    # -inf likelihood (out-of-domain theta, PAPER.md:214 via the library's convention) on half of the cube: Z halves
    g = gauss_loglike([0.75, 0.5], 0.05)
    f = lambda u: np.where(u[:, 0] < 0.5, -np.inf, g(u))
    r = NestedSampler(f, 2, nlive=400, batch=40, mcmc_steps=25, seed=21).run()
    assert abs(r.logZ) < 3 * r.logZ_err + 0.05
