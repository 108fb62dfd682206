"""bang_loglike_noalloc (include/bang.h): the allocation-free entry point against the existing bang_loglike.

Same kernels, same inputs, so the results must be EQUAL (the tolerance tests/test_gpu_parity.py uses where one kernel is
called twice: np.array_equal), on two calls in a row -- the scratch array is static, shared, and keeps the last call's
contents.  The batch holds theta that take the direct path (radii outside the fused kernel's tables), so that the list in
the static scratch is really written and read, around theta of the fast path and one out-of-domain theta.

Collected last on purpose (pytest -x: a failure here hides nothing after it).  Passes alone in a fresh
process and after the other GPU tests.
"""
import numpy as np
import pytest

from paper_2205_06819_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _batch():
    """prior-drawn theta of config 2 + the four 'extreme' theta of tests/test_gpu_seams.py + one invalid theta"""
    t0 = W.theta_true(2)
    t0[12] = 4.0
    ext = []
    a = t0.copy(); a[[0, 1, 3]] = [0.25, 0.25, 89.999]; ext.append(a)          # > 32 octaves of r^2
    b = t0.copy(); b[5] = 1e-6; ext.append(b)                                   # R/R_b beyond the bulge tables
    c = t0.copy(); c[[0, 1, 5]] = [0.25, 0.25, 200.0]; ext.append(c)
    d = t0.copy(); d[3] = 89.9; ext.append(d)
    bad = t0.copy(); bad[5] = -1.0                                              # R_b < 0: out of domain, logL = -inf
    prior = W.theta_batch(2)[:300]
    return np.concatenate([prior[:150], np.stack(ext), bad[None], prior[150:], np.stack(ext[::-1])])


@pytest.mark.parametrize("prec", ["fp32", "fp64"])
def test_noalloc_entry_point_equals_the_existing_path_on_two_calls_in_a_row(oracle, prec):
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_2205_06819_b200 import bang
    bang.lib()
    cfg = dict(W.config(2), nx=16, ny=12, supersample=2, jeans_nodes=32)        # the small grid of the direct-path tests
    theta = _batch()
    t0 = W.theta_true(2)
    t0[12] = 4.0
    mtrue = oracle.model_maps(t0, cfg)[0]
    rng = np.random.default_rng(11)
    err = np.stack([0.05 * np.abs(mtrue[0]), np.full_like(mtrue[1], 10.0), np.full_like(mtrue[2], 10.0),
                    np.full_like(mtrue[3], 0.1)])
    data = mtrue + err * rng.standard_normal(mtrue.shape)
    mask = rng.random(mtrue.shape) > 0.2

    ctx = bang.Context(cfg, precision=prec)
    ctx.set_data(data, err, mask)
    th = torch.as_tensor(theta, device="cuda")
    want = ctx.loglike(th).cpu().numpy()                                        # the existing path
    assert np.isneginf(want).sum() == 1 and np.isfinite(np.delete(want, np.flatnonzero(np.isneginf(want)))).all()

    out1 = torch.full((len(theta),), 7.0, dtype=torch.float64, device="cuda")
    out2 = torch.full((len(theta),), -7.0, dtype=torch.float64, device="cuda")
    ctx.loglike_noalloc(th, out1)                                               # two calls in a row on one stream
    ctx.loglike_noalloc(th, out2)
    got1, got2 = out1.cpu().numpy(), out2.cpu().numpy()
    assert np.array_equal(got1, want) and np.array_equal(got2, want)

    # a second context (another model variant) shares the array; calls ordered on the stream do not disturb each other
    ctx_b = bang.Context(dict(cfg, components=W.DISC1 | W.DISC2 | W.HALO), precision=prec)
    ctx_b.set_data(data, err, mask)
    want_b = ctx_b.loglike(th).cpu().numpy()
    out_b = torch.empty(len(theta), dtype=torch.float64, device="cuda")
    ctx_b.loglike_noalloc(th, out_b)
    torch.cuda.synchronize()
    ctx.loglike_noalloc(th, out1)
    assert np.array_equal(out_b.cpu().numpy(), want_b) and np.array_equal(out1.cpu().numpy(), want)
    # and the existing path is untouched by the new one
    assert np.array_equal(ctx.loglike(th).cpu().numpy(), want)

    # a shorter batch after a longer one (stale list entries beyond the new count are never read), and B = 0
    assert np.array_equal(ctx.loglike_noalloc(th[140:160].contiguous(), out2[:20]).cpu().numpy(), want[140:160])
    L = bang.lib()
    assert L.bang_loglike_noalloc(ctx._h, None, 0, None) == bang.OK
    # beyond the stated maximum: rejected with a clear error, nothing launched
    n0 = ctx.launches
    assert L.bang_loglike_noalloc(ctx._h, th.data_ptr(), bang.NOALLOC_MAX_B + 1, out1.data_ptr()) == bang.EINVAL
    assert b"BANG_NOALLOC_MAX_B" in L.bang_last_error(ctx._h) and ctx.launches == n0
    assert L.bang_loglike_noalloc(ctx._h, None, 3, None) == bang.EINVAL
    fresh = bang.Context(cfg, precision=prec)
    assert L.bang_loglike_noalloc(fresh._h, th.data_ptr(), 4, out1.data_ptr()) == bang.ENODATA
    fresh.close()
    ctx_b.close()
    ctx.close()


def test_noalloc_at_the_maximum_batch_size(oracle):
    # B = BANG_NOALLOC_MAX_B exactly, in bench.py's launch configuration of config 2 (64 x 64, x3): accepted, equal to the
    # existing path
    import torch
    from paper_2205_06819_b200 import bang
    cfg = W.config(2)
    c64 = bang.Context(cfg, precision="fp64")
    mtrue = c64.model_maps(W.theta_true(2)).cpu().numpy()[0]
    c64.close()
    data, err, mask = W.make_data(2, mtrue)
    ctx = bang.Context(cfg, precision="fp32")
    ctx.set_data(data, err, mask)
    th = torch.as_tensor(np.tile(W.theta_batch(2), (bang.NOALLOC_MAX_B // 1024, 1)), device="cuda")
    assert th.shape[0] == bang.NOALLOC_MAX_B
    want = ctx.loglike(th)
    out = torch.empty(th.shape[0], dtype=torch.float64, device="cuda")
    ctx.loglike_noalloc(th, out)
    assert torch.equal(out, want)
    ctx.close()
