"""Out-of-bounds canaries (compute-sanitizer is not available on the GPU pool): every output and workspace of an entry
point is carved from the middle of a larger sentinel-filled buffer; after the call the guard bands on both sides must be
untouched.  Shapes are the awkward ones: ragged tiles, smallest sizes, split-KV, ragged GEMM N."""
import math

import pytest
import torch

from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu
GUARD = 4096            # bytes on each side (a multiple of 256: carved buffers keep the 256-byte workspace alignment)


@pytest.fixture(scope="module")
def rx():
    from paper_2507_16697_b200 import ringx
    from paper_2507_16697_b200.build import build_library
    build_library()
    assert torch.cuda.is_available(), "GPU tests need a B200"
    ringx.lib()
    return ringx


class Guarded:
    def __init__(self):
        self.bufs = []

    def make(self, shape, dtype):
        n = math.prod(shape) * torch.empty((), dtype=dtype).element_size()
        raw = torch.full((n + 2 * GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
        self.bufs.append((raw, n))
        return raw[GUARD:GUARD + n].view(dtype).view(shape)

    def check(self):
        torch.cuda.synchronize()
        for raw, n in self.bufs:
            assert bool((raw[:GUARD] == 0xA5).all()) and bool((raw[GUARD + n:] == 0xA5).all()), "guard band overwritten"


def test_attention_forward_backward_guards(rx):
    for (B, H, N, d, chunk) in ((1, 1, 256, 64, 128), (2, 3, 768, 128, 256), (1, 2, 4096, 128, 2048),
                                (2, 3, 1000, 128, 384), (1, 2, 77, 64, 128), (1, 2, 1337, 64, 512)):     # the last three: ragged lengths
        g = Guarded()
        q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=3))
        scale = d ** -0.5
        o, lse = g.make((B, H, N, d), torch.bfloat16), g.make((B, H, N), torch.float32)
        ws = g.make((max(256, rx.ringx_attn_fwd_workspace_bytes(B, H, N, d, chunk, torch.bfloat16)),), torch.uint8)
        rx.ringx_attn_fwd(q, k, v, chunk, scale, o=o, lse=lse, workspace=ws)
        dq, dk, dv = (g.make((B, H, N, d), torch.bfloat16) for _ in range(3))
        wsb = g.make((rx.ringx_attn_bwd_workspace_bytes(B, H, N, d, chunk, torch.bfloat16),), torch.uint8)
        rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale, dq=dq, dk=dk, dv=dv, workspace=wsb)
        g.check()
        assert bool(torch.isfinite(dq.float()).all())


def test_mla_forward_backward_guards(rx):
    for (B, H, N, chunk) in ((1, 1, 256, 128), (2, 3, 768, 256), (2, 2, 1000, 384), (1, 1, 77, 128)):   # the last two: ragged
        g = Guarded()
        q, k = (wl.make_tensor((B, H, N, 192), w, seed=5).cuda() for w in "qk")
        v, do = (wl.make_tensor((B, H, N, 128), w, seed=5).cuda() for w in ("v", "do"))
        scale = 192 ** -0.5
        o, lse = g.make((B, H, N, 128), torch.bfloat16), g.make((B, H, N), torch.float32)
        ws = g.make((max(256, rx.ringx_attn_fwd_mla_workspace_bytes(B, H, N, 192, 128, chunk)),), torch.uint8)
        rx.ringx_attn_fwd_mla(q, k, v, chunk, scale, o=o, lse=lse, workspace=ws)
        dq, dk = (g.make((B, H, N, 192), torch.bfloat16) for _ in range(2))
        dv = g.make((B, H, N, 128), torch.bfloat16)
        wsb = g.make((rx.ringx_attn_bwd_mla_workspace_bytes(B, H, N, 192, 128, chunk),), torch.uint8)
        rx.ringx_attn_bwd_mla(q, k, v, o, lse, do, chunk, scale, dq=dq, dk=dk, dv=dv, workspace=wsb)
        g.check()
        assert bool(torch.isfinite(dq.float()).all())


def test_split_kv_guards(rx):
    B, H, Nq, Nk, d = 1, 3, 256, 3072, 128
    g = Guarded()
    q = wl.make_tensor((B, H, Nq, d), "q", seed=1).cuda()
    k, v = (wl.make_tensor((B, H, Nk, d), w, seed=1).cuda() for w in "kv")
    need = rx.ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, Nk, d, torch.bfloat16)
    assert need > 0
    ws = g.make((need,), torch.uint8)
    acc_o, acc_l = g.make((B, H, Nq, d), torch.float32), g.make((B, H, Nq), torch.float32)
    acc_o.zero_()
    acc_l.fill_(float("-inf"))
    rx.ringx_attn_chunk_fwd_ex(q, k, v, d ** -0.5, o_acc=acc_o, lse_acc=acc_l, workspace=ws)
    g.check()
    ref_o, ref_l = rx.ringx_attn_chunk_fwd(q, k, v, d ** -0.5)          # folding into an empty accumulator = the partial
    assert (acc_l - ref_l).abs().max().item() <= 1e-5 and (acc_o - ref_o).abs().max().item() <= 1e-2 * ref_o.abs().max().item()


def test_tokeniser_and_projection_guards(rx):
    g = Guarded()
    y = wl.make_field(2, 10, 9, 35, seed=4).cuda()
    for (org, size, k, dt) in (((1, 0, 2), (9, 9, 33), 3, torch.float32), ((0, 1, 0), (10, 8, 30), 2, torch.bfloat16),
                               ((3, 3, 3), (5, 5, 31), 1, torch.float32)):
        t = g.make((2, size[0] // k, size[1] // k, size[2] // k, 4), dt)
        rx.ringx_fidelity_tokens(y, org, size, k, tokens=t)
    B, S, H, d = 1, 384, 15, 64                                            # h = 960: ragged last GEMM tile
    x, w_qkv, w_o = (t.cuda() for t in wl.make_block_inputs(B, S, H, d, seed=2))
    q, k, v = (g.make((B, H, S, d), torch.bfloat16) for _ in range(3))
    rx.ringx_qkv_proj(x, w_qkv, H, q=q, k=k, v=v)
    yb = g.make((B, S, H * d), torch.bfloat16)
    rx.ringx_out_proj(q, w_o, y=yb)
    g.check()
    assert bool(torch.isfinite(yb.float()).all())
