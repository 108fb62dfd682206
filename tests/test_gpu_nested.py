"""Nested sampling with the CUDA likelihood: parameter recovery and the shape of the paper's
model comparison (Table 3: the model that generated the data has the larger evidence) on synthetic
data of BASELINE.json config 1's grid.  Every likelihood evaluation runs in the fused kernel through bang_loglike_host."""
import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W
from paper_2205_06819_b200.nested import NestedSampler, box_transform

pytestmark = pytest.mark.gpu

FREE = [2, 3, 4, 5, 6, 7, 12, 13, 15]        # PA, inc, log10 Mb, Rb, log10 Md1, Rd1, (M/L)b, (M/L)d1, k1
HALF = np.array([5.0, 5.0, 0.15, 0.15, 0.15, 0.4, 0.5, 0.4, 0.1])   # half-widths of the uniform prior box about theta_true


def test_nested_sampling_recovers_theta_and_prefers_the_true_model(oracle):
    import torch
    assert torch.cuda.is_available()
    from paper_2205_06819_b200 import bang
    cfg = W.config(1)
    tt = W.theta_true(1)
    mtrue = oracle.model_maps(tt, cfg)[0]
    data, err, mask = W.make_data(1, mtrue)
    lo, hi = tt[FREE] - HALF, tt[FREE] + HALF
    hi[-1] = min(hi[-1], 1.0)
    tr = box_transform(tt, FREE, lo, hi)

    ctx = bang.Context(cfg, precision="fp32")
    ctx.set_data(data, err, mask)
    n0 = ctx.launches
    ns = NestedSampler(ctx.loglike_host, len(FREE), transform=tr, nlive=300, batch=64, mcmc_steps=20, seed=1)
    r = ns.run()
    assert ctx.launches - n0 >= r.n_iter * 20                      # the evaluations were kernel launches
    mean, std = r.posterior_mean_std(tr)
    z = (mean[FREE] - tt[FREE]) / std[FREE]
    assert np.all(np.abs(z) < 5), z                                # truth within the posterior (one noise realisation)
    assert np.all(std[FREE] < 0.5 * HALF)                          # and the data, not the prior, set the widths
    # the kernel's logL at posterior samples is the oracle's (reading Q bound for fp32 near the truth)
    top = np.argsort(r.logw)[-3:]
    th = tr(r.samples_u[top])
    lo_ = oracle.loglike(th, cfg, data, err, mask)
    assert np.all(np.abs(ctx.loglike_host(th) - lo_) <= 1e-3 * np.sqrt(mask[0].sum()) + 1e-9 * np.abs(lo_))
    ctx.close()

    # a model without the bulge cannot explain data that contain one: ln B >> 0 (eq. 17)
    cfg_d = dict(cfg, components=W.DISC1)
    free_d = [2, 3, 6, 7, 13, 15]
    sel = [FREE.index(i) for i in free_d]
    tr_d = box_transform(tt, free_d, lo[sel], hi[sel])
    ctx = bang.Context(cfg_d, precision="fp32")
    ctx.set_data(data, err, mask)
    rd = NestedSampler(ctx.loglike_host, len(free_d), transform=tr_d, nlive=300, batch=64, mcmc_steps=20, seed=2).run()
    ctx.close()
    assert r.logZ - rd.logZ > 100.0, (r.logZ, rd.logZ)
    assert r.logZ_err < 1.0 and rd.logZ_err < 1.0
