"""GPU checks of `ringx_sdpa`, the autograd drop-in for torch's scaled_dot_product_attention: forward and
gradients against the fp64 oracle (the authority) and, as a library second opinion, against torch's own SDPA."""
import math

import numpy as np
import pytest
import torch

from oracle import attention as orc
from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sdpa():
    from paper_2507_16697_b200.build import build_library
    from paper_2507_16697_b200 import ringx, sdpa as mod
    build_library()
    assert torch.cuda.is_available(), "GPU tests need a B200"
    ringx.lib()
    return mod.ringx_sdpa


def relf(a, ref):
    return np.linalg.norm(a - ref) / np.linalg.norm(ref)


@pytest.mark.parametrize("B,Hq,Hkv,N,d,chunk", [(1, 2, 2, 1024, 64, 256), (2, 4, 2, 512, 128, None), (1, 6, 2, 768, 64, 768),
                                                (2, 2, 2, 777, 128, None), (1, 4, 2, 1500, 64, 512)])   # ragged lengths
def test_sdpa_forward_and_gradients(sdpa, B, Hq, Hkv, N, d, chunk):
    q = wl.make_tensor((B, Hq, N, d), "q", seed=41).cuda().requires_grad_()
    k = wl.make_tensor((B, Hkv, N, d), "k", seed=41).cuda().requires_grad_()
    v = wl.make_tensor((B, Hkv, N, d), "v", seed=41).cuda().requires_grad_()
    do = wl.make_tensor((B, Hq, N, d), "do", seed=41).cuda()
    o = sdpa(q, k, v, kv_chunk=chunk, enable_gqa=Hq != Hkv)
    o.backward(do)
    # oracle: query head h uses kv head h // G (the heads of a group are adjacent)
    G = Hq // Hkv
    q64, k64, v64, do64 = (wl.to_f64_numpy(t.detach()) for t in (q, k, v, do))
    scale = 1.0 / math.sqrt(d)
    o_ref = np.empty_like(q64)
    dq_ref, dk_ref, dv_ref = np.zeros_like(q64), np.zeros_like(k64), np.zeros_like(v64)
    for b in range(B):
        for h in range(Hq):
            o_ref[b, h], _ = orc.attention_fwd(q64[b, h], k64[b, h // G], v64[b, h // G], scale)
            a, bk, bv = orc.attention_bwd(q64[b, h], k64[b, h // G], v64[b, h // G], do64[b, h], scale)
            dq_ref[b, h] = a
            dk_ref[b, h // G] += bk
            dv_ref[b, h // G] += bv
    assert relf(o.detach().float().cpu().numpy(), o_ref) <= 1e-2
    for g, r in ((q.grad, dq_ref), (k.grad, dk_ref), (v.grad, dv_ref)):
        assert relf(g.float().cpu().numpy(), r) <= 2e-2
    # second opinion: torch's SDPA on the same bits (fp32 math)
    qt, kt, vt = (t.detach().float().requires_grad_() for t in (q, k, v))
    ot = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, enable_gqa=Hq != Hkv)
    ot.backward(do.float())
    assert relf(o.detach().float().cpu().numpy(), ot.detach().cpu().numpy()) <= 1e-2
    assert relf(q.grad.float().cpu().numpy(), qt.grad.cpu().numpy()) <= 2e-2
    assert relf(k.grad.float().cpu().numpy(), kt.grad.cpu().numpy()) <= 2e-2


def test_sdpa_mla_shapes(sdpa):
    """query/key of width 192, value of width 128 (multi-head latent attention) through the same drop-in:
    forward and gradients against the oracle and against torch's SDPA (which takes E != Ev as well)."""
    B, H, N = 1, 2, 512
    q = wl.make_tensor((B, H, N, 192), "q", seed=43).cuda().requires_grad_()
    k = wl.make_tensor((B, H, N, 192), "k", seed=43).cuda().requires_grad_()
    v = wl.make_tensor((B, H, N, 128), "v", seed=43).cuda().requires_grad_()
    do = wl.make_tensor((B, H, N, 128), "do", seed=43).cuda()
    o = sdpa(q, k, v, kv_chunk=256)
    o.backward(do)
    scale = 1.0 / math.sqrt(192)
    q64, k64, v64, do64 = (wl.to_f64_numpy(t.detach()) for t in (q, k, v, do))
    for h in range(H):
        o_ref, _ = orc.attention_fwd(q64[0, h], k64[0, h], v64[0, h], scale)
        refs = orc.attention_bwd(q64[0, h], k64[0, h], v64[0, h], do64[0, h], scale)
        assert relf(o[0, h].detach().float().cpu().numpy(), o_ref) <= 1e-2
        for g, r in zip((q.grad, k.grad, v.grad), refs):
            assert relf(g[0, h].float().cpu().numpy(), r) <= 2e-2
    qt, kt, vt = (t.detach().float().requires_grad_() for t in (q, k, v))
    ot = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt)
    ot.backward(do.float())
    assert relf(o.detach().float().cpu().numpy(), ot.detach().cpu().numpy()) <= 1e-2
    assert relf(k.grad.float().cpu().numpy(), kt.grad.cpu().numpy()) <= 2e-2


def test_sdpa_fp32_forward_only_path(sdpa):
    """fp32 tensors take the tensor-core split path (config C1); it has no backward, which must fail loudly, not fall back."""
    q, k, v = (wl.make_tensor((1, 1, 512, 64), w, seed=2, dtype="f32").cuda() for w in "qkv")
    o = sdpa(q, k, v, kv_chunk=128)
    o_ref, _ = orc.attention_fwd(*(wl.to_f64_numpy(t[0, 0]) for t in (q, k, v)), 0.125)
    assert np.abs(o[0, 0].cpu().numpy() - o_ref).max() <= 1e-5
    q.requires_grad_()
    with pytest.raises(Exception):
        sdpa(q, k, v, kv_chunk=128).sum().backward()


def test_attention_block_autograd(sdpa):
    """The block as one autograd node (projections + attention, forward and backward in libringx) against the oracle."""
    from oracle import projection as proj
    from paper_2507_16697_b200.sdpa import ringx_attention_block
    B, S, H, d = 1, 512, 4, 64
    x, w_qkv, w_o = (t.cuda().requires_grad_() for t in wl.make_block_inputs(B, S, H, d, seed=51))
    dy = wl.make_tensor((B, S, H * d), "do", seed=52).cuda()
    y = ringx_attention_block(x, w_qkv, w_o, H, kv_chunk=256)
    y.backward(dy)
    f = lambda t: wl.to_f64_numpy(t.detach())
    y_ref = proj.attention_block_fwd(f(x), f(w_qkv), f(w_o), H, d ** -0.5)
    refs = proj.attention_block_bwd(f(x), f(w_qkv), f(w_o), f(dy), H, d ** -0.5)
    assert relf(y.detach().float().cpu().numpy(), y_ref) <= 2e-2
    for g, r in zip((x.grad, w_qkv.grad, w_o.grad), refs):
        assert relf(g.float().cpu().numpy(), r) <= 2e-2
