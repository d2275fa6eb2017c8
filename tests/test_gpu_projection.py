"""GPU parity of Table II's projection GEMMs and the attention block (`ringx_qkv_proj`, `ringx_out_proj`,
`ringx_attn_block_fwd`) against the fp64 oracle `oracle/projection.py`.

Tolerance, from the arithmetic: bf16 products are exact in fp32, the fp32 accumulation of K terms is bounded by
K * 2^-24 * sum|x||w| in any order, and the result is rounded once to bf16 (unit roundoff 2^-8):
    |y - y_ref| <= 2^-8 |y_ref| + K 2^-24 (|x| |W|^T)   element by element.
The block feeds bf16-rounded q, k, v and o through two more stages, so it is held to a relative Frobenius error of
2e-2 (measured ~5e-3) like the gradients of BASELINE.json."""
import math

import numpy as np
import pytest
import torch

from oracle import projection as proj
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


def f64(t):
    return wl.to_f64_numpy(t)


def check(got, ref, bound_abs):
    got = got.float().cpu().numpy().astype(np.float64)
    assert got.shape == ref.shape
    excess = np.abs(got - ref) - (2.0 ** -8 * np.abs(ref) + bound_abs)
    assert excess.max() <= 0, excess.max()
    return np.linalg.norm(got - ref) / np.linalg.norm(ref)


SHAPES = [(1, 128, 2, 64), (2, 256, 4, 64), (1, 384, 2, 128), (1, 256, 15, 64), (3, 128, 3, 128), (1, 4096, 8, 128),
          (2, 19 * 128, 5, 64)]


@pytest.mark.parametrize("B,S,H,d", SHAPES)
def test_qkv_and_out_projection_match_the_oracle(rx, B, S, H, d):
    h = H * d
    x, w_qkv, w_o = wl.make_block_inputs(B, S, H, d, seed=B * 1000 + S + H)
    refs = proj.qkv_projection(f64(x), f64(w_qkv), H)
    q, k, v = rx.ringx_qkv_proj(x.cuda(), w_qkv.cuda(), H)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == 1
    ax = np.abs(f64(x))
    for i, (got, ref) in enumerate(zip((q, k, v), refs)):
        bound = proj.split_heads(ax @ np.abs(f64(w_qkv[i * h:(i + 1) * h])).T, H) * (h * 2.0 ** -24)
        rel = check(got, ref, bound)
        assert rel <= 4e-3, rel
    # out-projection of a seeded o (not the GEMM's own output: the two entry points are checked independently)
    o = wl.make_tensor((B, H, S, d), "q", seed=99)
    ref = proj.out_projection(f64(o), f64(w_o))
    y = rx.ringx_out_proj(o.cuda(), w_o.cuda())
    torch.cuda.synchronize()
    bound = (proj.merge_heads(np.abs(f64(o))) @ np.abs(f64(w_o)).T) * (h * 2.0 ** -24)
    assert check(y, ref, bound) <= 4e-3


def test_identity_weights_copy_bits(rx):
    """W = I makes both GEMMs pure layout permutations; bf16 values must come through bit-exactly."""
    B, S, H, d = 2, 256, 4, 64
    h = H * d
    x = wl.make_tensor((B, S, h), "x", seed=5)
    eye = torch.eye(h, dtype=torch.bfloat16)
    w = torch.cat([eye, 2 * eye, -eye], dim=0).contiguous()
    q, k, v = rx.ringx_qkv_proj(x.cuda(), w.cuda(), H)
    xs = x.view(B, S, H, d).permute(0, 2, 1, 3)
    assert torch.equal(q.cpu(), xs) and torch.equal(k.cpu(), 2 * xs) and torch.equal(v.cpu(), -xs)
    y = rx.ringx_out_proj(q, eye.cuda())
    assert torch.equal(y.cpu(), x)


@pytest.mark.parametrize("B,S,H,d,chunk", [(1, 1024, 4, 64, 256), (2, 512, 2, 128, 512)])
def test_attention_block_matches_the_oracle(rx, B, S, H, d, chunk):
    x, w_qkv, w_o = wl.make_block_inputs(B, S, H, d, seed=31)
    scale = 1.0 / math.sqrt(d)
    ref = proj.attention_block_fwd(f64(x), f64(w_qkv), f64(w_o), H, scale)
    y = rx.ringx_attn_block_fwd(x.cuda(), w_qkv.cuda(), w_o.cuda(), H, chunk, scale)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == 2 + S // chunk
    got = y.float().cpu().numpy().astype(np.float64)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert rel <= 2e-2, rel
    assert np.abs(got - ref).max() <= 1e-2 * np.abs(f64(x)).max()


def test_full_size_sampled(rx):
    """bench.py's projection workload (C3's block: B=1, S=262144, h=1024): sampled 128-row blocks of tokens against
    the oracle (rows are independent in a GEMM), incl. the first and last tile."""
    B, S, H, d = 1, 262144, 8, 128
    h = H * d
    x, w_qkv, w_o = wl.make_block_inputs(B, S, H, d, device="cuda")
    q, k, v = rx.ringx_qkv_proj(x, w_qkv, H)
    y = rx.ringx_out_proj(q, w_o)
    torch.cuda.synchronize()
    wq64, wo64 = f64(w_qkv), f64(w_o)
    for s0 in (0, S - 128, 128 * 1000 + 64, 128 * 1481):
        xs = f64(x[:, s0:s0 + 128])
        refs = proj.qkv_projection(xs, wq64, H)
        for i, (got, ref) in enumerate(zip((q, k, v), refs)):
            bound = proj.split_heads(np.abs(xs) @ np.abs(wq64[i * h:(i + 1) * h]).T, H) * (h * 2.0 ** -24)
            check(got[:, :, s0:s0 + 128], ref, bound)
        qs = f64(q[:, :, s0:s0 + 128])
        bound = (proj.merge_heads(np.abs(qs)) @ np.abs(wo64).T) * (h * 2.0 ** -24)
        check(y[:, s0:s0 + 128], proj.out_projection(qs, wo64), bound)


def test_error_codes(rx):
    x = torch.zeros((1, 128, 128), dtype=torch.bfloat16, device="cuda")
    w = torch.zeros((384, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_qkv_proj(x[:, :100].contiguous(), w, 2)           # S % 128 != 0
    assert e.value.status == 2
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_qkv_proj(x, w, 4)                                  # d = 32
    assert e.value.status == 2
    with pytest.raises(ValueError):
        rx.ringx_qkv_proj(x.float(), w, 2)
    with pytest.raises(ValueError):
        rx.ringx_qkv_proj(x.cpu(), w.cpu(), 2)


# ------------------------------------------------------------------------------------------------ backward
BWD_SHAPES = [(1, 128, 4, 64), (2, 256, 2, 128), (1, 384, 8, 64), (3, 128, 4, 128), (1, 2048, 8, 128)]


@pytest.mark.parametrize("B,S,H,d", BWD_SHAPES)
def test_projection_backward_matches_the_oracle(rx, B, S, H, d):
    """Data gradients (bf16) within 2^-8 |ref| + K 2^-24 (|A||B|); weight gradients (fp32, split-K reduce-adds in any order)
    within T 2^-24 (|A|^T |B|) with T = B*S the reduction length."""
    h = H * d
    x, w_qkv, w_o = wl.make_block_inputs(B, S, H, d, seed=7 + S)
    dy = wl.make_tensor((B, S, h), "do", seed=8)
    o = wl.make_tensor((B, H, S, d), "v", seed=9)
    dq, dk, dv = (wl.make_tensor((B, H, S, d), w, seed=10) for w in ("q", "k", "do"))
    T = B * S
    # ---- output projection
    do_ref, dwo_ref = proj.out_projection_bwd(f64(dy), f64(o), f64(w_o))
    d_o, dwo = rx.ringx_out_proj_bwd(dy.cuda(), o.cuda(), w_o.cuda())
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == 2
    bound = proj.split_heads(np.abs(f64(dy)) @ np.abs(f64(w_o)), H) * (h * 2.0 ** -24)
    assert check(d_o, do_ref, bound) <= 4e-3
    wb = np.einsum("bsn,bsi->ni", np.abs(f64(dy)), proj.merge_heads(np.abs(f64(o)))) * (T * 2.0 ** -24)
    assert (np.abs(dwo.cpu().numpy().astype(np.float64) - dwo_ref) - wb).max() <= 0
    assert np.linalg.norm(dwo.cpu().numpy() - dwo_ref) / np.linalg.norm(dwo_ref) <= 1e-5
    # ---- input projections
    dx_ref, dwq_ref = proj.qkv_projection_bwd(f64(dq), f64(dk), f64(dv), f64(x), f64(w_qkv))
    dx, dwq = rx.ringx_qkv_proj_bwd(dq.cuda(), dk.cuda(), dv.cuda(), x.cuda(), w_qkv.cuda())
    torch.cuda.synchronize()
    g = np.concatenate([proj.merge_heads(np.abs(f64(t))) for t in (dq, dk, dv)], axis=-1)
    assert check(dx, dx_ref, (g @ np.abs(f64(w_qkv))) * (3 * h * 2.0 ** -24)) <= 4e-3
    wb = np.einsum("bsn,bsi->ni", g, np.abs(f64(x))) * (T * 2.0 ** -24)
    assert (np.abs(dwq.cpu().numpy().astype(np.float64) - dwq_ref) - wb).max() <= 0
    assert np.linalg.norm(dwq.cpu().numpy() - dwq_ref) / np.linalg.norm(dwq_ref) <= 1e-5


def test_projection_backward_identity_weights_copy_bits(rx):
    B, S, H, d = 1, 256, 4, 64
    h = H * d
    eye = torch.eye(h, dtype=torch.bfloat16)
    dy = wl.make_tensor((B, S, h), "do", seed=3)
    o = wl.make_tensor((B, H, S, d), "v", seed=3)
    d_o, _ = rx.ringx_out_proj_bwd(dy.cuda(), o.cuda(), eye.cuda())
    assert torch.equal(d_o.cpu(), dy.view(B, S, H, d).permute(0, 2, 1, 3))          # dO = split_heads(dY)


@pytest.mark.parametrize("B,S,H,d,chunk", [(1, 1024, 4, 64, 256), (2, 512, 2, 128, 512)])
def test_attention_block_backward_matches_the_oracle(rx, B, S, H, d, chunk):
    x, w_qkv, w_o = wl.make_block_inputs(B, S, H, d, seed=31)
    dy = wl.make_tensor((B, S, H * d), "do", seed=32)
    scale = 1.0 / math.sqrt(d)
    ref = proj.attention_block_bwd(f64(x), f64(w_qkv), f64(w_o), f64(dy), H, scale)
    ws = torch.empty(rx.ringx_attn_block_fwd_workspace_bytes(B, S, H, d, chunk), dtype=torch.uint8, device="cuda")
    xd, wq, wo, dyd = x.cuda(), w_qkv.cuda(), w_o.cuda(), dy.cuda()
    rx.ringx_attn_block_fwd(xd, wq, wo, H, chunk, scale, workspace=ws)
    got = rx.ringx_attn_block_bwd(xd, wq, wo, dyd, ws, H, chunk, scale)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == 2 + (S // chunk + 2) + 2
    for name, g, r in zip(("dx", "dw_qkv", "dw_o"), got, ref):
        rel = np.linalg.norm(g.float().cpu().numpy() - r) / np.linalg.norm(r)
        assert rel <= 2e-2, (name, rel)


def test_projection_backward_rejects_h_not_multiple_of_256(rx):
    o = torch.zeros((1, 2, 128, 64), dtype=torch.bfloat16, device="cuda")       # h = 128
    dy = torch.zeros((1, 128, 128), dtype=torch.bfloat16, device="cuda")
    w = torch.zeros((128, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_out_proj_bwd(dy, o, w)
    assert e.value.status == 2
