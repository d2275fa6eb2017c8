"""Multi-head latent attention shapes (PAPER.md:376 names MLA among the layer designs RingX is
compatible with): d_qk = 192, d_v = 128, forward.  The oracle is the same definition (oracle.attention takes d != dv;
pinned by tests/test_oracle_pins.py::test_brute_force_forward_nonsquare); tolerances are the bf16 forward's."""
import math

import numpy as np
import pytest
import torch

from oracle import attention as orc
from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu
DQK, DV = 192, 128


@pytest.fixture(scope="module")
def rx():
    from paper_2507_16697_b200 import ringx
    from paper_2507_16697_b200.build import build_library
    build_library()
    assert torch.cuda.is_available(), "GPU tests need a B200"
    ringx.lib()
    return ringx


def make(B, H, N, seed, gain=1.0, device="cpu"):
    q = wl.make_tensor((B, H, N, DQK), "q", seed=seed, dtype="bf16", gain=gain, device=device)
    k = wl.make_tensor((B, H, N, DQK), "k", seed=seed, dtype="bf16", gain=gain, device=device)
    v = wl.make_tensor((B, H, N, DV), "v", seed=seed, dtype="bf16", device=device)
    return q, k, v


def f64(t):
    return wl.to_f64_numpy(t)


@pytest.mark.parametrize("B,H,N,chunk,gain", [(1, 1, 256, 256, 1.0), (1, 2, 512, 128, 1.0), (2, 3, 1280, 256, 1.0),
                                              (1, 2, 2304, 768, 1.0), (1, 2, 2048, 2048, 3.0), (1, 1, 4096, 512, 3.0),
                                              (1, 4, 1024, 512, 0.05)])
def test_mla_forward_matches_oracle(rx, B, H, N, chunk, gain):
    q, k, v = make(B, H, N, seed=101, gain=gain)
    scale = 1.0 / math.sqrt(DQK)
    o, lse = rx.ringx_attn_fwd_mla(q.cuda(), k.cuda(), v.cuda(), chunk, scale)
    assert rx.ringx_last_launch_count() == N // chunk and o.shape == (B, H, N, DV)
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    og, lg = f64(o), f64(lse)
    assert np.isfinite(og).all()
    assert np.abs(og - o_ref).max() <= 1e-2 * np.abs(f64(v)).max()
    assert np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref) <= 1e-2
    assert np.abs(lg - lse_ref).max() <= 5e-5


def test_mla_one_hot_v_reads_P(rx):
    """V = unit rows at chosen keys => O[:, c] = P[:, key(c)] (two bf16 roundings): every 64-key half of every key tile,
    both 64-column panels of V, all three 64-column panels of Q and K are probed element by element."""
    B, H, N = 1, 1, 512
    q, k, _ = make(B, H, N, seed=103)
    keys = np.unique((np.arange(DV) * 37 + 5) % N)[:DV]
    v = torch.zeros(B, H, N, DV, dtype=torch.bfloat16)
    for c, j in enumerate(keys):
        v[0, 0, j, c] = 1.0
    scale = 0.25
    # make each 64-column panel of q matter on its own: compare with the oracle on the full 192 columns
    o, _ = rx.ringx_attn_fwd_mla(q.cuda(), k.cuda(), v.cuda(), 128, scale)
    P = orc.softmax_probs(f64(q[0, 0]), f64(k[0, 0]), scale)
    og = f64(o[0, 0])
    for c, j in enumerate(keys):
        assert np.abs(og[:, c] - P[:, j]).max() <= 2 ** -7 * max(P[:, j].max(), 1e-3) + 1e-6, (c, j)
    # dropping any one panel of q from the oracle must break the agreement (the kernel really contracts over all 192)
    for p in range(3):
        qz = f64(q[0, 0]).copy()
        qz[:, 64 * p:64 * p + 64] = 0.0
        Pz = orc.softmax_probs(qz, f64(k[0, 0]), scale)
        assert np.abs(og[:, 0] - Pz[:, keys[0]]).max() > 10 * (2 ** -7 * P[:, keys[0]].max())


def test_mla_long_sequence_sampled_rows(rx):
    """N = 65536, four passes of 16384 keys: oracle on sampled query rows of two heads against all keys."""
    B, H, N, chunk = 1, 2, 65536, 16384
    q, k, v = make(B, H, N, seed=107, device="cuda")
    scale = 1.0 / math.sqrt(DQK)
    o, lse = rx.ringx_attn_fwd_mla(q, k, v, chunk, scale)
    assert torch.isfinite(o.float()).all() and torch.isfinite(lse).all()
    rows = np.array(sorted(set([0, 1, 127, 128, 255, 256, 257, N // 2, N - 257, N - 256, N - 129, N - 128, N - 1])
                           | set(np.random.default_rng(3).integers(0, N, 50).tolist())))
    for h in range(H):
        k64, v64 = f64(k[0, h]), f64(v[0, h])
        o_ref, lse_ref = orc.attention_fwd(f64(q[0, h][rows]), k64, v64, scale)
        og = f64(o[0, h][rows])
        assert np.abs(og - o_ref).max() <= 1e-2 * np.abs(v64).max()
        assert np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref) <= 1e-2
        assert np.abs(f64(lse[0, h][rows]) - lse_ref).max() <= 1e-3
    o1, lse1 = rx.ringx_attn_fwd_mla(q, k, v, N, scale)                       # chunk independence at this size
    assert (lse1 - lse).abs().max().item() <= 5e-5
    assert ((o1.float() - o.float()).norm() / o.float().norm()).item() <= 4e-3


def test_mla_errors(rx):
    L = rx.lib()
    t = torch.zeros(1, 1, 256, 192, dtype=torch.bfloat16, device="cuda")
    v = torch.zeros(1, 1, 256, 128, dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros(1, 1, 256, device="cuda")
    call = lambda dqk, dv, N, chunk, dt: L.ringx_attn_fwd_mla(t.data_ptr(), t.data_ptr(), v.data_ptr(), v.data_ptr(),
                                                              lse.data_ptr(), 1, 1, N, dqk, dv, chunk, 0.1, dt, None, 0, None)
    assert call(192, 128, 256, 256, 1) == 0
    assert call(128, 128, 256, 256, 1) == 2       # only the 192 / 128 pair: BAD_SHAPE
    assert call(192, 64, 256, 256, 1) == 2
    assert call(192, 128, 256, 256, 0) == 3       # bf16 only
    assert call(192, 128, 256, 128, 1) == 1       # two passes need a workspace: NULL_PTR
    assert call(192, 128, 384, 384, 1) == 2       # N % 256
    torch.cuda.synchronize()
