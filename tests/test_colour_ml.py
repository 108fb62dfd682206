"""Colour-M/L pre-step, eq. 20 with App. C's error model."""
import math

import numpy as np
import pytest


def test_oracle_colour_ml_hand_values_and_error_propagation(oracle):
    # the paper's constants a = -0.70, b = 0.89, sigma = 0.07: g - i = 1.2 -> log10 M/L = 0.368
    ml, err = oracle.ml_from_colour([1.2], [0.0], [0.0], [0.0])
    assert abs(ml[0] - 10 ** 0.368) < 1e-13
    assert abs(err[0] - math.log(10) * 10 ** 0.368 * 0.07) < 1e-13           # only the scatter of the relation
    # a zero colour gives 10^a; b = 0 makes the colour irrelevant
    assert abs(oracle.ml_from_colour([17.3], [17.3], [0.1], [0.1])[0][0] - 10 ** -0.70) < 1e-15
    assert abs(oracle.ml_from_colour([3.0], [1.0], [0.0], [0.0], a=0.3, b=0.0)[0][0] - 10 ** 0.3) < 1e-15
    # first-order propagation: the reported error is the quadrature sum of |d(M/L)/dm| dm and the scatter term,
    # with the derivatives taken by central finite differences of the oracle's own M/L
    rng = np.random.default_rng(0)
    mb, mg = rng.uniform(14, 22, 50), rng.uniform(14, 22, 50)
    dmb, dmg = rng.uniform(0.01, 0.2, 50), rng.uniform(0.01, 0.2, 50)
    a, b, sig = -0.52, 1.1, 0.05
    ml, err = oracle.ml_from_colour(mb, mg, dmb, dmg, a, b, sig)
    h = 1e-6
    z = np.zeros(50)
    dfb = (oracle.ml_from_colour(mb + h, mg, z, z, a, b, sig)[0] - oracle.ml_from_colour(mb - h, mg, z, z, a, b, sig)[0]) / (2 * h)
    dfg = (oracle.ml_from_colour(mb, mg + h, z, z, a, b, sig)[0] - oracle.ml_from_colour(mb, mg - h, z, z, a, b, sig)[0]) / (2 * h)
    want = np.sqrt((dfb * dmb) ** 2 + (dfg * dmg) ** 2 + (math.log(10) * ml * sig) ** 2)
    assert np.allclose(err, want, rtol=1e-8)
    assert np.allclose(dfb, -dfg, rtol=1e-8)                                    # only the COLOUR matters


@pytest.mark.gpu
def test_gpu_colour_ml_matches_the_oracle(oracle):
    import torch
    assert torch.cuda.is_available()
    from paper_2205_06819_b200 import bang
    rng = np.random.default_rng(7)
    shape = (200, 203)                                                          # a ragged map, several grid strides
    mb, mg = rng.uniform(14, 24, shape), rng.uniform(14, 24, shape)
    dmb, dmg = rng.uniform(0.0, 0.3, shape), rng.uniform(0.0, 0.3, shape)
    mb[3, 5] = np.nan                                                           # a bad pixel stays bad, and only it
    ml, err = bang.ml_from_colour(mb, mg, dmb, dmg)
    ml_o, err_o = oracle.ml_from_colour(mb, mg, dmb, dmg)
    ml, err = ml.cpu().numpy(), err.cpu().numpy()
    good = np.isfinite(ml_o)
    assert not good[3, 5] and good.sum() == good.size - 1 and np.array_equal(np.isfinite(ml), good)
    assert np.max(np.abs(ml[good] / ml_o[good] - 1)) < 1e-13 and np.max(np.abs(err[good] / err_o[good] - 1)) < 1e-13
    assert bang.ml_from_colour(np.zeros((0,)), np.zeros((0,)), np.zeros((0,)), np.zeros((0,)))[0].numel() == 0
