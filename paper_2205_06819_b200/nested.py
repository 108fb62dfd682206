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

`run_device` is the form that feeds a GPU: R independent runs (different seeds) advance in lock-step and share every
call, so that R x K walkers (>= 1024 for the defaults) are in flight; the walks themselves -- proposal, likelihood,
accept/reject for all MCMC steps -- run on the device through `bang.Context.ns_walk` (C ABI: bang_ns_walk) with the
walkers resident in device memory; the host keeps the live sets and the evidence sums.  The scatter of log Z over the R
runs is an empirical check of the sqrt(H/N) error estimate.

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


class _Evidence:
    """The bookkeeping of one run: prior-mass shrinkage, evidence and information sums, dead points (eq. 16)."""

    def __init__(self, N: int, shrink: str, rng):
        self.N, self.shrink, self.rng = N, shrink, rng
        self.logX, self.logZ, self.H = 0.0, -math.inf, 0.0
        self.dead_u, self.dead_L, self.dead_logw = [], [], []

    def _add(self, Lj: float, logw: float):
        if Lj > -math.inf:
            logZ_new = logaddexp(self.logZ, Lj + logw)
            # information (Skilling 2004 eq. 13), updated incrementally
            self.H = (math.exp(Lj + logw - logZ_new) * Lj
                      + (math.exp(self.logZ - logZ_new) * (self.H + self.logZ) if self.logZ > -math.inf else 0.0) - logZ_new)
            self.logZ = logZ_new

    def retire(self, u: np.ndarray, L: np.ndarray, K: int):
        """Retire the K worst live points one after the other, the live set shrinking N, N-1, ..., N-K+1.
        Returns (indices retired, indices kept, L* = the K-th retired likelihood)."""
        order = np.argsort(L, kind="stable")
        worst = order[:K]
        for i, j in enumerate(worst):
            n = self.N - i
            dlog = 1.0 / n if self.shrink == "expected" else -math.log(self.rng.random()) / n   # -ln t, t = max of n uniforms
            logX_new = self.logX - dlog
            logw = self.logX + math.log1p(-math.exp(logX_new - self.logX))                      # ln(X_prev - X_new)
            self._add(L[j], logw)
            self.dead_u.append(u[j].copy()); self.dead_L.append(L[j]); self.dead_logw.append(L[j] + logw)
            self.logX = logX_new
        return worst, order[K:], L[worst[-1]]

    def converged(self, L: np.ndarray, f: float) -> bool:
        return L.max() + self.logX < math.log(f) + self.logZ         # the live points cannot add more than f Z

    def finish(self, u, L, n_iter, n_evals, acc_hist, history) -> NestedResult:
        logw_live = self.logX - math.log(self.N)                      # the remaining live points share the remaining mass
        for j in np.argsort(L, kind="stable"):
            self._add(L[j], logw_live)
            self.dead_u.append(u[j].copy()); self.dead_L.append(L[j]); self.dead_logw.append(L[j] + logw_live)
        logw = np.asarray(self.dead_logw) - self.logZ
        return NestedResult(logZ=self.logZ, logZ_err=math.sqrt(max(self.H, 0.0) / self.N), information=self.H,
                            samples_u=np.asarray(self.dead_u), logL=np.asarray(self.dead_L), logw=logw, n_iter=n_iter,
                            n_evals=n_evals, acceptance=float(np.mean(acc_hist)) if acc_hist else 0.0, history=history)


def _next_scale(scale: float, acc: float) -> float:
    return min(max(scale * math.exp((acc - 0.3) * 0.5), 1e-4), 4.0)   # steer the acceptance towards ~30 %


def _proposal_cholesky(u_keep: np.ndarray) -> np.ndarray:
    d = u_keep.shape[1]
    cov = np.cov(u_keep.T).reshape(d, d) + 1e-12 * np.eye(d)
    return np.linalg.cholesky(cov)


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
        ev = _Evidence(N, self.shrink, rng)
        scale, acc_hist, history = 1.0, [], []
        it = 0
        while it < self.max_iter:
            worst, keep, Lstar = ev.retire(u, L, K)
            # K constrained random walks from random survivors, in lock-step: proposals from the survivors' covariance
            chol = _proposal_cholesky(u[keep])
            start = rng.choice(keep, size=K, replace=True)       # a walker that never moves keeps its survivor's point
            cur, curL = u[start].copy(), L[start].copy()         # and likelihood (carried by index)
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
            acc = n_acc / (self.steps * K)
            acc_hist.append(acc)
            scale = _next_scale(scale, acc)
            u[worst], L[worst] = cur, curL
            it += 1
            history.append((it, ev.logZ, ev.logX, float(L.max()), acc, scale))
            if ev.converged(L, self.f):
                break
        return ev.finish(u, L, it, self.n_evals, acc_hist, history)


def run_device(ctx, free: list[int], lo, hi, theta0, nlive: int = 400, batch: int = 256, mcmc_steps: int = 20,
               n_runs: int = 4, f: float = 1e-3, seed: int = 0, shrink: str = "expected",
               max_iter: int = 100000) -> list[NestedResult]:
    """n_runs independent nested-sampling runs in lock-step on one `bang.Context` (data loaded): every device call advances
    n_runs x batch walkers for mcmc_steps steps (Context.ns_walk: proposals, likelihoods and accept/reject on the device,
    theta resident).  Box prior: theta[free[j]] uniform in [lo[j], hi[j]], the other entries from theta0.
    Returns one NestedResult per run (combine with `combine_runs`)."""
    import torch
    free = [int(i) for i in free]
    d, N, K, R = len(free), nlive, batch, n_runs
    assert 1 <= K < N and R >= 1
    lo, hi, theta0 = (np.asarray(a, dtype=np.float64) for a in (lo, hi, theta0))
    tr = box_transform(theta0, free, lo, hi)
    rngs = [np.random.Generator(np.random.PCG64([seed, r])) for r in range(R)]
    u = [rng.random((N, d)) for rng in rngs]
    L0 = ctx.loglike(np.concatenate([tr(x) for x in u])).cpu().numpy()
    L = [np.where(np.isnan(x), -np.inf, x) for x in np.split(L0, R)]
    ev = [_Evidence(N, shrink, rng) for rng in rngs]
    scale, acc_hist, history = [1.0] * R, [[] for _ in range(R)], [[] for _ in range(R)]
    n_evals, n_iter, active = [N] * R, [0] * R, list(range(R))
    dev = ctx.device
    call = 0
    while active and max(n_iter) < max_iter:
        G = len(active)
        worst, chol, cur, curL, Lstar = [], [], [], [], []
        for r in active:
            w, keep, ls = ev[r].retire(u[r], L[r], K)
            start = rngs[r].choice(keep, size=K, replace=True)
            worst.append(w); chol.append(_proposal_cholesky(u[r][keep]))
            cur.append(u[r][start]); curL.append(L[r][start]); Lstar.append(np.full(K, ls))
        u_dev = torch.as_tensor(np.concatenate(cur), device=dev)
        l_dev = torch.as_tensor(np.concatenate(curL), device=dev)
        ls_dev = torch.as_tensor(np.concatenate(Lstar), device=dev)
        g_dev = torch.as_tensor(np.repeat(np.arange(G, dtype=np.int32), K), device=dev)
        n_acc = ctx.ns_walk(u_dev, l_dev, ls_dev, g_dev, np.stack(chol), np.asarray([scale[r] for r in active]),
                            free, lo, hi, theta0, mcmc_steps, seed=(seed << 20) + call)
        call += 1
        new_u, new_L = u_dev.cpu().numpy().reshape(G, K, d), l_dev.cpu().numpy().reshape(G, K)
        still = []
        for gi, r in enumerate(active):
            u[r][worst[gi]], L[r][worst[gi]] = new_u[gi], new_L[gi]
            acc = n_acc[gi] / (mcmc_steps * K)
            acc_hist[r].append(acc)
            scale[r] = _next_scale(scale[r], acc)
            n_iter[r] += 1
            n_evals[r] += mcmc_steps * K
            history[r].append((n_iter[r], ev[r].logZ, ev[r].logX, float(L[r].max()), acc, scale[r]))
            if not ev[r].converged(L[r], f):
                still.append(r)
        active = still
    return [ev[r].finish(u[r], L[r], n_iter[r], n_evals[r], acc_hist[r], history[r]) for r in range(R)]


def combine_runs(results: list[NestedResult]) -> tuple[float, float]:
    """ln of the mean evidence of independent runs and its standard error (from the scatter when there are several runs,
    else the single run's sqrt(H/N))."""
    lz = np.asarray([r.logZ for r in results])
    if len(lz) == 1:
        return float(lz[0]), float(results[0].logZ_err)
    m = lz.max()
    z = np.exp(lz - m)
    mean = z.mean()
    return float(m + math.log(mean)), float(z.std(ddof=1) / math.sqrt(len(z)) / mean)
