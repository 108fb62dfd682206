"""Nested sampling around the batched likelihood (SURVEY.md sec. 8f item 2, eq. 16-17 at :209, :218-221).

The paper drives its likelihood with CPNest: N live points drawn from the prior, the worst one replaced at every
iteration by a point of higher likelihood found by MCMC, the prior mass shrinking as X_tau = t_tau X_(tau-1) with t_tau
the largest of N uniform numbers, the evidence growing by L_tau (X_(tau-1) - X_tau), until further growth cannot change
Z by more than a fraction f.  One likelihood per call leaves a GPU idle, so this driver is BATCHED: every iteration
retires the K worst live points one after the other (the live set shrinking N, N-1, ..., N-K+1, so that the
shrinkage statistics are exactly those of K ordinary iterations), then draws K replacements above the K-th retired
likelihood with K constrained random walks that advance in lock-step -- one batched likelihood call (K evaluations) per
MCMC step.  The likelihood is any callable theta[K][d_full] -> logL[K]; with `bang.Context.loglike_host` every
evaluation runs in the fused CUDA kernel.  This module holds no model arithmetic.

Parameters live in the unit cube u in [0,1]^d with a uniform prior; `transform(u) -> theta` maps them to the physical
vector (affine for uniform priors, a power of ten for log-uniform ones, ...).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np


def box_transform(theta0: np.ndarray, free: list[int], lo: np.ndarray, hi: np.ndarray):
    """transform for uniform priors on the entries `free` of a template theta0: theta[free] = lo + (hi - lo) u."""
    theta0 = np.asarray(theta0, dtype=np.float64)
    free = np.asarray(free, dtype=np.int64)
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)

    def transform(u: np.ndarray) -> np.ndarray:
        th = np.repeat(theta0[None, :], u.shape[0], axis=0)
        th[:, free] = lo + (hi - lo) * u
        return th

    return transform


def logaddexp(a: float, b: float) -> float:
    if a == -math.inf:
        return b
    if b == -math.inf:
        return a
    m = max(a, b)
    return m + math.log(math.exp(a - m) + math.exp(b - m))


@dataclass
class NestedResult:
    logZ: float
    logZ_err: float                 # sqrt(H / N) (Skilling 2004)
    information: float              # H [nats]
    samples_u: np.ndarray           # dead + final live points, unit cube [n][d]
    logL: np.ndarray                # their likelihoods
    logw: np.ndarray                # log posterior weights (normalised: logsumexp = 0)
    n_iter: int
    n_evals: int
    acceptance: float
    history: list = field(default_factory=list)

    def posterior_mean_std(self, transform=None):
        w = np.exp(self.logw)
        x = self.samples_u if transform is None else transform(self.samples_u)
        mean = (w[:, None] * x).sum(0)
        var = (w[:, None] * (x - mean) ** 2).sum(0)
        return mean, np.sqrt(var)


class NestedSampler:
    """Batched nested sampling with constrained random-walk replacement (see the module docstring)."""

    def __init__(self, loglike, ndim: int, transform=None, nlive: int = 400, batch: int = 64, mcmc_steps: int = 20,
                 f: float = 1e-3, seed: int = 0, shrink: str = "expected", max_iter: int = 100000):
        assert 1 <= batch < nlive and shrink in ("expected", "sampled")
        self.loglike, self.ndim = loglike, ndim
        self.transform = transform if transform is not None else (lambda u: u)
        self.N, self.K, self.steps, self.f = nlive, batch, mcmc_steps, f
        self.rng = np.random.Generator(np.random.PCG64(seed))
        self.shrink, self.max_iter = shrink, max_iter
        self.n_evals = 0

    def _L(self, u: np.ndarray) -> np.ndarray:
        self.n_evals += u.shape[0]
        out = np.asarray(self.loglike(self.transform(u)), dtype=np.float64)
        return np.where(np.isnan(out), -np.inf, out)

    def run(self) -> NestedResult:
        N, K, d, rng = self.N, self.K, self.ndim, self.rng
        u = rng.random((N, d))
        L = self._L(u)
        logX, logZ, H = 0.0, -math.inf, 0.0
        dead_u, dead_L, dead_logw = [], [], []
        scale, acc_hist, history = 1.0, [], []
        it = 0
        while it < self.max_iter:
            order = np.argsort(L, kind="stable")
            worst = order[:K]
            for i, j in enumerate(worst):                       # retire the K worst, the live set shrinking N-i
                n = N - i
                dlog = 1.0 / n if self.shrink == "expected" else -math.log(rng.random()) / n   # -ln t, t = max of n uniforms
                logX_new = logX - dlog
                logw = logX + math.log1p(-math.exp(logX_new - logX))                            # ln(X_prev - X_new)
                if L[j] > -math.inf:
                    logZ_new = logaddexp(logZ, L[j] + logw)
                    # information (Skilling 2004 eq. 13), updated incrementally
                    H = (math.exp(L[j] + logw - logZ_new) * L[j]
                         + (math.exp(logZ - logZ_new) * (H + logZ) if logZ > -math.inf else 0.0) - logZ_new)
                    logZ = logZ_new
                dead_u.append(u[j].copy()); dead_L.append(L[j]); dead_logw.append(L[j] + logw)
                logX = logX_new
            Lstar = L[worst[-1]]
            keep = order[K:]
            # K constrained random walks from random survivors, in lock-step: proposals from the survivors' covariance
            cov = np.cov(u[keep].T).reshape(d, d) + 1e-12 * np.eye(d)
            chol = np.linalg.cholesky(cov)
            cur = u[rng.choice(keep, size=K, replace=True)].copy()
            curL = np.full(K, np.nan)
            n_acc = 0
            for _ in range(self.steps):
                prop = cur + scale * (2.38 / math.sqrt(d)) * rng.standard_normal((K, d)) @ chol.T
                inside = np.all((prop >= 0.0) & (prop <= 1.0), axis=1)
                pl = np.full(K, -np.inf)
                if inside.any():
                    pl[inside] = self._L(prop[inside])
                ok = inside & (pl > Lstar)
                cur[ok], curL[ok] = prop[ok], pl[ok]
                n_acc += int(ok.sum())
            never = np.isnan(curL)                               # walkers that never moved keep their start point:
            if never.any():                                      # re-evaluate nothing, copy the survivor's likelihood
                for k in np.flatnonzero(never):
                    match = np.flatnonzero((u[keep] == cur[k]).all(axis=1))
                    curL[k] = L[keep[match[0]]]
            acc = n_acc / (self.steps * K)
            acc_hist.append(acc)
            scale *= math.exp((acc - 0.3) * 0.5)                 # steer the acceptance towards ~30 %
            scale = min(max(scale, 1e-4), 4.0)
            u[worst], L[worst] = cur, curL
            it += 1
            history.append((it, logZ, logX, float(L.max()), acc, scale))
            if L.max() + logX < math.log(self.f) + logZ:         # the live points cannot add more than f Z
                break
        # the remaining live points share the remaining prior mass
        logw_live = logX - math.log(N)
        for j in np.argsort(L, kind="stable"):
            if L[j] > -math.inf:
                logZ_new = logaddexp(logZ, L[j] + logw_live)
                H = (math.exp(L[j] + logw_live - logZ_new) * L[j]
                     + (math.exp(logZ - logZ_new) * (H + logZ) if logZ > -math.inf else 0.0) - logZ_new)
                logZ = logZ_new
            dead_u.append(u[j].copy()); dead_L.append(L[j]); dead_logw.append(L[j] + logw_live)
        logw = np.asarray(dead_logw) - logZ
        return NestedResult(logZ=logZ, logZ_err=math.sqrt(max(H, 0.0) / N), information=H,
                            samples_u=np.asarray(dead_u), logL=np.asarray(dead_L), logw=logw, n_iter=it,
                            n_evals=self.n_evals, acceptance=float(np.mean(acc_hist)) if acc_hist else 0.0, history=history)
