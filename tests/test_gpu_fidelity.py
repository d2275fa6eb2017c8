"""GPU parity of `ringx_fidelity_tokens` (the Turbulence-Transformer tokeniser; SURVEY.md §8(f)
NEXT-4) against the fp64 oracle `oracle/fidelity.py`, element by element on the same seeded field.

Tolerance (fp32 output), derived from the arithmetic: the kernel forms k*k fused multiply-adds with weights
w[a]*w[b] (each weight rounded to fp32, the product rounded once), one multiply by w[e], and a sum of k terms; the
weights sum to 1, so the worst-case error is (k*k + k + 8) * 2^-24 * max|Y| (sequential-sum bound gamma_n * sum|terms|).
bf16 output adds one RN-even rounding: unit roundoff 2^-8 * |T|."""
import math

import numpy as np
import pytest
import torch

from oracle import fidelity as fid
from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rx():
    from paper_2507_16697_b200 import ringx
    from paper_2507_16697_b200.build import build_library
    build_library()
    assert torch.cuda.is_available(), "GPU tests need a B200"
    ringx.lib()
    return ringx


def tol_f32(k, ymax):
    return (k * k + k + 8) * 2.0 ** -24 * ymax


CASES = [
    # M, D, H, W, origin, size, k
    (1, 8, 8, 16, (0, 0, 0), (8, 8, 16), 1),
    (2, 8, 12, 40, (0, 0, 0), (8, 12, 40), 2),
    (1, 9, 9, 300, (0, 0, 0), (9, 9, 300), 3),            # span 255, ragged tail of 45
    (2, 16, 20, 1100, (4, 4, 64), (8, 12, 1024), 4),      # several CTAs along x, crop with offsets
    (1, 10, 15, 525, (0, 5, 20), (10, 10, 505), 5),       # span 255: two CTAs, second ragged
    (1, 16, 24, 530, (8, 0, 2), (8, 24, 528), 8),
    (1, 32, 64, 64, (0, 32, 32), (32, 32, 32), 32),       # the largest k; narrow crop (8 rows per CTA)
    (3, 12, 36, 48, (2, 3, 5), (8, 28, 36), 4),           # narrow crop, 7 rows per CTA, ragged row group
    (1, 6, 7, 9, (1, 2, 3), (4, 3, 5), 1),                # pure crop, odd sizes
]


@pytest.mark.parametrize("M,D,H,W,origin,size,k", CASES)
@pytest.mark.parametrize("sigma", [0.0, 1.7])
def test_tokens_match_the_oracle(rx, M, D, H, W, origin, size, k, sigma):
    y = wl.make_field(M, D, H, W, seed=100 + k)
    ref = fid.fidelity_tokens(wl.to_f64_numpy(y), origin, size, k, None if sigma == 0.0 else sigma)
    t = rx.ringx_fidelity_tokens(y.cuda(), origin, size, k, sigma)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == 1
    got = t.cpu().numpy().astype(np.float64)
    assert got.shape == ref.shape
    err = np.abs(got - ref).max()
    assert err <= tol_f32(k, float(y.abs().max())), (err, tol_f32(k, float(y.abs().max())))
    if k == 1:
        np.testing.assert_array_equal(got, ref)                # a crop copies bits
    tb = rx.ringx_fidelity_tokens(y.cuda(), origin, size, k, sigma, out_dtype=torch.bfloat16)
    gb = tb.float().cpu().numpy().astype(np.float64)
    assert np.all(np.abs(gb - ref) <= 2.0 ** -8 * np.abs(ref) + tol_f32(k, float(y.abs().max())) + 1e-30)


def test_constant_and_impulse(rx):
    k = 4
    y = torch.full((1, 8, 8, 512, 4), 1.5)
    t = rx.ringx_fidelity_tokens(y.cuda(), (0, 0, 0), (8, 8, 512), k)
    assert float((t - 1.5).abs().max()) <= 4 * 2.0 ** -24 * 1.5
    y.zero_()
    y[0, 4 + 1, 2, 256 + 3, 2] = 1.0                           # window (1, 0, 64), offsets (1, 2, 3), channel 2
    t = rx.ringx_fidelity_tokens(y.cuda(), (0, 0, 0), (8, 8, 512), k).cpu()
    G = fid.gaussian_kernel_3d(k, fid.default_sigma(k))
    assert abs(float(t[0, 1, 0, 64, 2]) - G[1, 2, 3]) <= 4 * 2.0 ** -24 * G[1, 2, 3]
    assert int((t != 0).sum()) == 1


def test_three_fidelity_modes_of_one_state(rx):
    """Low (whole domain, k1), mid (crop, k2), high (crop, k = 1): PAPER.md:195-199, all against the oracle."""
    D = 64
    y = wl.make_field(1, D, D, D, seed=7)
    y64 = wl.to_f64_numpy(y)
    yd = y.cuda()
    modes = [((0, 0, 0), (D, D, D), 8), (fid.crop_origin((30, 34, 28), (32, 32, 32)), (32, 32, 32), 4),
             (fid.crop_origin((40, 20, 33), (8, 8, 8)), (8, 8, 8), 1)]
    L = 0
    for org, size, k in modes:
        t = rx.ringx_fidelity_tokens(yd, org, size, k).cpu().numpy().astype(np.float64)
        ref = fid.fidelity_tokens(y64, org, size, k)
        assert np.abs(t - ref).max() <= tol_f32(k, float(y.abs().max()))
        L += t.shape[1] * t.shape[2] * t.shape[3]
    assert L == 3 * 512


def test_full_size_sampled_blocks(rx):
    """bench.py's tokeniser workload (512^3 x 4 fp32 = 2.1 GB, k = 4): the field is generated on the GPU, the same
    bits are copied to the host for sampled sub-blocks (windows are independent, so a block of tokens is exactly the
    oracle applied to the matching block of the field), incl. the first/last window and CTA-span boundaries."""
    G, k = 512, 4
    y = wl.make_field(1, G, G, G, seed=20250722, device="cuda")
    t = rx.ringx_fidelity_tokens(y, (0, 0, 0), (G, G, G), k)
    torch.cuda.synchronize()
    ymax = float(y.abs().max())
    assert bool(torch.isfinite(t).all())
    blocks = [(0, 0, 0), (G - 8, G - 8, G - 64), (128, 252, 224), (300, 8, 448), (508 - 4, 0, 248)]
    for (z, yy, x) in blocks:
        sub = y[:, z:z + 8, yy:yy + 8, x:x + 64].cpu()
        ref = fid.fidelity_tokens(wl.to_f64_numpy(sub), (0, 0, 0), (8, 8, 64), k)
        got = t[:, z // k:z // k + 2, yy // k:yy // k + 2, x // k:x // k + 16].cpu().numpy().astype(np.float64)
        assert np.abs(got - ref).max() <= tol_f32(k, ymax)
    # a property of the whole output: with non-negative weights summing to 1, tokens lie in the field's range
    assert float(t.max()) <= float(y.max()) + 1e-5 and float(t.min()) >= float(y.min()) - 1e-5
    # and (k = 2: box filter) the global mean is preserved
    t2 = rx.ringx_fidelity_tokens(y, (0, 0, 0), (G, G, G), 2)
    assert abs(float(t2.double().mean()) - float(y.double().mean())) <= 1e-6


def test_error_codes(rx):
    y = torch.zeros((1, 8, 8, 8, 4), device="cuda")
    bad = [((0, 0, 0), (8, 8, 8), 0), ((0, 0, 0), (8, 8, 8), 33), ((0, 0, 0), (6, 8, 8), 4), ((1, 0, 0), (8, 8, 8), 2),
           ((0, 0, -1), (8, 8, 8), 2), ((0, 0, 0), (8, 8, 0), 2)]
    for org, size, k in bad:
        with pytest.raises(rx.RingxError) as e:
            rx.ringx_fidelity_tokens(y, org, size, k, tokens=torch.zeros(8, device="cuda"))
        assert e.value.status == 2, (org, size, k)
    y3 = torch.zeros((1, 8, 8, 8, 3), device="cuda")
    with pytest.raises(rx.RingxError):
        rx.ringx_fidelity_tokens(y3, (0, 0, 0), (8, 8, 8), 2)
    with pytest.raises(ValueError):
        rx.ringx_fidelity_tokens(torch.zeros((1, 8, 8, 8, 4)), (0, 0, 0), (8, 8, 8), 2)
