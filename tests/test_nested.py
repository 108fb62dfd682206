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


def test_philox_restatement_against_the_published_known_answers():
    # the numpy restatement of Philox4x32-10 that tests/test_gpu_nested.py uses to check bang_ns_walk's proposals,
    # against Random123's known-answer vectors for philox4x32-10 (Salmon et al. 2011)
    from test_gpu_nested import _philox4x32_10
    out = _philox4x32_10([0], [0], [0], [0], 0, 0)
    assert [int(x[0]) for x in out] == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]
    out = _philox4x32_10([0xFFFFFFFF], [0xFFFFFFFF], [0xFFFFFFFF], [0xFFFFFFFF], 0xFFFFFFFF, 0xFFFFFFFF)
    assert [int(x[0]) for x in out] == [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]
    out = _philox4x32_10([0x243F6A88], [0x85A308D3], [0x13198A2E], [0x03707344], 0xA4093822, 0x299F31D0)
    assert [int(x[0]) for x in out] == [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]


def test_combine_runs():
    from paper_2205_06819_b200.nested import NestedResult, combine_runs
    mk = lambda z, e: NestedResult(z, e, 1.0, np.zeros((1, 1)), np.zeros(1), np.zeros(1), 1, 1, 0.3)
    assert combine_runs([mk(-5.0, 0.2)]) == (-5.0, 0.2)
    lz, err = combine_runs([mk(math.log(1.0), 0.1), mk(math.log(3.0), 0.1)])
    assert abs(lz - math.log(2.0)) < 1e-12 and abs(err - math.sqrt(2.0) / math.sqrt(2) / 2.0) < 1e-12
    lz, _ = combine_runs([mk(-1e6 + 1.0, 0.1), mk(-1e6, 0.1)])          # no overflow far from zero
    assert abs(lz - (-1e6 + math.log((math.e + 1) / 2))) < 1e-9


class _StubContext:
    """A stand-in for bang.Context on the CPU: a Gaussian likelihood in the unit cube and a numpy restatement of what
    bang_ns_walk does (lock-step constrained Metropolis walks, per-group Cholesky factor and scale, per-walker bound),
    so that run_device's host side -- several runs in lock-step, retire / replace bookkeeping, evidence -- is tested
    without a GPU."""
    device = "cpu"

    def __init__(self, mu, sigma, free, lo, hi):
        self.mu, self.sigma, self.free, self.lo, self.hi = np.asarray(mu), sigma, list(free), np.asarray(lo), np.asarray(hi)
        self.calls, self.max_walkers = 0, 0

    def _ll(self, u):
        d = u.shape[1]
        return -0.5 * (((u - self.mu) / self.sigma) ** 2).sum(axis=1) - d * math.log(self.sigma * math.sqrt(2 * math.pi))

    def loglike(self, theta):
        import torch
        theta = np.asarray(theta)
        return torch.as_tensor(self._ll((theta[:, self.free] - self.lo) / (self.hi - self.lo)))

    def ns_walk(self, u, logL, Lstar, group, chol, scale, free, lo, hi, theta0, steps, seed=0):
        rng = np.random.default_rng(seed)
        un, ln, ls, g = u.numpy(), logL.numpy(), Lstar.numpy(), group.numpy()      # views: updated in place
        K, d = un.shape
        self.calls += 1
        self.max_walkers = max(self.max_walkers, K)
        n_acc = np.zeros(chol.shape[0], dtype=np.int32)
        for _ in range(steps):
            z = rng.standard_normal((K, d))
            prop = un + (np.asarray(scale)[g] * 2.38 / math.sqrt(d))[:, None] * np.einsum("kij,kj->ki", np.asarray(chol)[g], z)
            inside = np.all((prop >= 0) & (prop <= 1), axis=1)
            pl = np.where(inside, self._ll(np.clip(prop, 0, 1)), -np.inf)
            ok = pl > ls
            un[ok], ln[ok] = prop[ok], pl[ok]
            np.add.at(n_acc, g[ok], 1)
        return n_acc


def test_run_device_host_side_with_a_stub_context():
    from paper_2205_06819_b200.nested import combine_runs, run_device
    d, sigma = 3, 0.05
    free = [2, 5, 7]
    theta0 = np.arange(17.0)
    lo, hi = np.array([10.0, -1.0, 0.5]), np.array([20.0, 1.0, 2.5])
    ctx = _StubContext([0.4, 0.6, 0.5], sigma, free, lo, hi)
    runs = run_device(ctx, free, lo, hi, theta0, nlive=300, batch=100, mcmc_steps=25, n_runs=4, seed=7)
    assert len(runs) == 4 and ctx.max_walkers == 400                # 4 runs x 100 walkers share every call
    assert ctx.calls == max(r.n_iter for r in runs)                 # one device call per lock-step iteration
    for r in runs:                                                  # a normalised Gaussian inside the cube: ln Z = 0
        assert abs(r.logZ) < 3 * r.logZ_err + 0.06, r.logZ
        assert abs(np.exp(r.logw).sum() - 1) < 1e-9
    lz, err = combine_runs(runs)
    assert abs(lz) < 4 * err + 0.05
    mean, std = runs[0].posterior_mean_std(lambda u: lo + (hi - lo) * u)
    want = lo + (hi - lo) * np.array([0.4, 0.6, 0.5])
    assert np.all(np.abs(mean - want) < 5 * sigma * (hi - lo) / math.sqrt(30))
    again = run_device(_StubContext([0.4, 0.6, 0.5], sigma, free, lo, hi), free, lo, hi, theta0, nlive=300, batch=100,
                       mcmc_steps=25, n_runs=4, seed=7)
    assert [r.logZ for r in again] == [r.logZ for r in runs]        # same seed, same runs
