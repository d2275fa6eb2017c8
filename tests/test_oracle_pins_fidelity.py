"""Pins for `oracle/fidelity.py` (the tokeniser oracle, NEXT-4) -- CPU only.

Pinned to things other than itself: a hand fixture (tests/golden/fidelity_k3.json), closed forms
(constant field, k = 1, k = 2 box filter, affine field, unit impulse), brute-force Python loops and a
library second opinion (torch conv3d in fp64 with stride k).
"""
import json
import math
import os

import numpy as np
import pytest
import torch

from oracle import fidelity as fid

RNG = np.random.default_rng(20250722)


def test_golden_k3(golden_dir):
    with open(os.path.join(golden_dir, "fidelity_k3.json")) as f:
        g = json.load(f)
    k = g["k"]
    sigma = math.sqrt(g["sigma_squared_times_2ln2"] / (2.0 * math.log(2.0)))
    np.testing.assert_allclose(fid.gaussian_weights_1d(k, sigma), g["weights_1d"], atol=1e-15)
    y = np.zeros(g["shape_MDHWC"])
    for z, yy, x, c, val in g["nonzero_zyxc_value"]:
        y[0, z, yy, x, c] = val
    t = fid.fidelity_tokens(y, (0, 0, 0), (3, 3, 6), k, sigma)
    assert t.shape == (1, 1, 1, 2, 2)
    np.testing.assert_allclose(t[0, 0, 0, 0], g["tokens_x0"], atol=1e-14)
    np.testing.assert_allclose(t[0, 0, 0, 1], g["tokens_x1"], atol=1e-14)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 8])
def test_constant_field_and_weight_sum(k):
    G = fid.gaussian_kernel_3d(k, fid.default_sigma(k))
    assert abs(G.sum() - 1.0) < 1e-14 and G.min() > 0
    np.testing.assert_allclose(G, G.transpose(2, 1, 0), atol=0)          # symmetric in the axes
    np.testing.assert_allclose(G, G[::-1, ::-1, ::-1], atol=1e-17)       # and under reflection
    y = np.full((2, 2 * k, 3 * k, 4 * k, 4), 2.5)
    t = fid.fidelity_tokens(y, (0, 0, 0), (2 * k, 3 * k, 4 * k), k)
    assert t.shape == (2, 2, 3, 4, 4)
    np.testing.assert_allclose(t, 2.5, atol=1e-14)


def test_k1_is_the_crop():
    y = RNG.standard_normal((2, 5, 6, 7, 4))
    t = fid.fidelity_tokens(y, (1, 2, 3), (3, 4, 2), 1)
    np.testing.assert_array_equal(t, y[:, 1:4, 2:6, 3:5, :])


def test_k2_is_the_box_filter():
    y = RNG.standard_normal((1, 4, 6, 8, 4))
    t = fid.fidelity_tokens(y, (0, 0, 0), (4, 6, 8), 2, sigma=0.7)       # any sigma: 8 equal weights
    ref = y.reshape(1, 2, 2, 3, 2, 4, 2, 4).mean(axis=(2, 4, 6))
    np.testing.assert_allclose(t, ref, atol=1e-15)


def test_sigma_default_is_the_les_filter_width():
    # G(r) ~ exp(-6 r^2 / Delta^2) with Delta = k  <=>  sigma^2 = k^2 / 12
    k = 4
    w = fid.gaussian_weights_1d(k, fid.default_sigma(k))
    assert abs(w[0] / w[1] - math.exp(-6.0 * (1.5 ** 2 - 0.5 ** 2) / k ** 2)) < 1e-15


def test_impulse_reads_the_kernel():
    k, sigma = 4, 1.3
    G = fid.gaussian_kernel_3d(k, sigma)
    w = np.exp(-((np.arange(k) - 1.5) ** 2) / (2 * sigma ** 2))
    for (a, b, e) in [(0, 0, 0), (1, 2, 3), (3, 0, 2), (2, 2, 1)]:
        y = np.zeros((1, 2 * k, 2 * k, 2 * k, 1))
        y[0, k + a, b, k + e, 0] = 1.0                                     # window (z'=1, y'=0, x'=1)
        t = fid.fidelity_tokens(y, (0, 0, 0), (2 * k,) * 3, k, sigma)
        assert abs(t[0, 1, 0, 1, 0] - w[a] * w[b] * w[e] / w.sum() ** 3) < 1e-16
        assert abs(t[0, 1, 0, 1, 0] - G[a, b, e]) < 1e-18
        assert np.count_nonzero(t) == 1


@pytest.mark.parametrize("k", [2, 3, 4])
def test_affine_field_gives_window_centre(k):
    D, H, W = 2 * k, 3 * k, 2 * k
    z, yy, x = np.meshgrid(np.arange(D + 2), np.arange(H + 1), np.arange(W + 3), indexing="ij")
    coef = np.array([[0.5, -1.25, 2.0, 0.75], [1.0, 0.0, -3.0, 0.1], [0.0, 2.0, 0.5, -0.2]])   # per channel
    field = (z[..., None] * coef[0] + yy[..., None] * coef[1] + x[..., None] * coef[2] + np.array([1.0, 2.0, 3.0, 4.0]))[None]
    org = (2, 1, 3)
    t = fid.fidelity_tokens(field, org, (D, H, W), k)
    zc = org[0] + k * np.arange(D // k) + 0.5 * (k - 1)
    yc = org[1] + k * np.arange(H // k) + 0.5 * (k - 1)
    xc = org[2] + k * np.arange(W // k) + 0.5 * (k - 1)
    ref = (zc[:, None, None, None] * coef[0] + yc[None, :, None, None] * coef[1] + xc[None, None, :, None] * coef[2]
           + np.array([1.0, 2.0, 3.0, 4.0]))[None]
    np.testing.assert_allclose(t, ref, atol=1e-12)


def test_brute_force_loops():
    k, sigma = 3, 0.9
    y = RNG.standard_normal((2, 7, 8, 10, 3))
    org, size = (1, 2, 1), (6, 3, 9)
    t = fid.fidelity_tokens(y, org, size, k, sigma)
    g = [math.exp(-((a - 1.0) ** 2) / (2 * sigma ** 2)) for a in range(k)]
    s = sum(g)
    for m in range(2):
        for zo in range(size[0] // k):
            for yo in range(size[1] // k):
                for xo in range(size[2] // k):
                    for c in range(3):
                        acc = 0.0
                        for a in range(k):
                            for b in range(k):
                                for e in range(k):
                                    acc += (g[a] / s) * (g[b] / s) * (g[e] / s) * y[m, org[0] + k * zo + a, org[1] + k * yo + b, org[2] + k * xo + e, c]
                        assert abs(t[m, zo, yo, xo, c] - acc) < 1e-13


@pytest.mark.parametrize("k", [2, 4])
def test_library_second_opinion_conv3d(k):
    y = RNG.standard_normal((2, 8, 12, 16, 4))
    org, size = (0, 4, 8), (8, 8, 8)
    t = fid.fidelity_tokens(y, org, size, k)
    G = torch.from_numpy(fid.gaussian_kernel_3d(k, fid.default_sigma(k)))[None, None]
    c = torch.from_numpy(y[:, org[0]:org[0] + 8, org[1]:org[1] + 8, org[2]:org[2] + 8]).permute(0, 4, 1, 2, 3).reshape(8, 1, 8, 8, 8)
    ref = torch.nn.functional.conv3d(c, G, stride=k).reshape(2, 4, 8 // k, 8 // k, 8 // k).permute(0, 2, 3, 4, 1).numpy()
    np.testing.assert_allclose(t, ref, atol=1e-14)


def test_crop_origin_and_rejections():
    assert fid.crop_origin((8, 8, 9), (4, 6, 8)) == (6, 5, 5)
    y = np.zeros((1, 4, 4, 4, 1))
    with pytest.raises(ValueError):
        fid.fidelity_tokens(y, (1, 0, 0), (4, 4, 4), 2)
    with pytest.raises(ValueError):
        fid.fidelity_tokens(y, (0, 0, 0), (3, 4, 4), 2)
