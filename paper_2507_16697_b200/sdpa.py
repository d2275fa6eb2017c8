"""RingX attention as a drop-in for `torch.nn.functional.scaled_dot_product_attention` ("RingX is a
standalone attention module that can be used as a drop-in replacement for the scaled_dot_product_attention in PyTorch").

`ringx_sdpa(q, k, v, scale=None, kv_chunk=None, ...)` is a `torch.autograd.Function` whose forward and backward are the
libringx entry points (`ringx_attn_fwd[_gqa]`, `ringx_attn_bwd[_gqa]`); with a `torch.distributed` group it runs the
paper's RingX_b or RingX_a schedule (`ringx_dist`) on the local sequence chunks instead.  Argument marshalling only: no
arithmetic of the method lives here, and there is no fallback -- non-CUDA tensors, masks, dropout and causal attention
(none of which the paper's attention has) raise.
"""
from __future__ import annotations

import math

import torch

from . import ringx, ringx_dist


def _default_chunk(n: int) -> int:
    """KV-chunk length when the caller names none: the largest of 32768..128 that divides N (kv_chunk doubles as the
    L2-blocking parameter; one head's K,V chunk of 32768 x 128 bf16 is 16.8 MB of the 126 MB L2)."""
    c = 32768
    while c > 128 and n % c:
        c //= 2
    if n % c == 0:
        return c
    # a ragged length (bf16 entries take any N): passes of 32768 keys, the last one shorter
    return min(32768, (n + 127) // 128 * 128)


class _RingXAttention(torch.autograd.Function):
    @staticmethod
    def forward(ctx, q, k, v, scale, kv_chunk):
        q, k, v = q.contiguous(), k.contiguous(), v.contiguous()
        if q.shape[-1] != v.shape[-1]:        # multi-head latent attention shapes (d_qk = 192, d_v = 128)
            o, lse = ringx.ringx_attn_fwd_mla(q, k, v, kv_chunk, scale)
        elif q.shape[1] == k.shape[1]:
            o, lse = ringx.ringx_attn_fwd(q, k, v, kv_chunk, scale)
        else:
            o, lse = ringx.ringx_attn_fwd_gqa(q, k, v, kv_chunk, scale)
        ctx.save_for_backward(q, k, v, o, lse)
        ctx.scale, ctx.kv_chunk = scale, kv_chunk
        return o

    @staticmethod
    def backward(ctx, dO):
        q, k, v, o, lse = ctx.saved_tensors
        dO = dO.contiguous()
        if q.shape[-1] != v.shape[-1]:
            dq, dk, dv = ringx.ringx_attn_bwd_mla(q, k, v, o, lse, dO, ctx.kv_chunk, ctx.scale)
        elif q.shape[1] == k.shape[1]:
            dq, dk, dv = ringx.ringx_attn_bwd(q, k, v, o, lse, dO, ctx.kv_chunk, ctx.scale)
        else:
            dq, dk, dv = ringx.ringx_attn_bwd_gqa(q, k, v, o, lse, dO, ctx.kv_chunk, ctx.scale)
        return dq, dk, dv, None, None


class _RingXDistAttention(torch.autograd.Function):
    """q, k, v are this rank's sequence chunks [B,H,N/W,d]; the schedule is RingX_b (default) or RingX_a."""

    @staticmethod
    def forward(ctx, q, k, v, scale, schedule, comm, ops):
        fwd = ringx_dist.ringx_b_forward if schedule == "b" else ringx_dist.ringx_a_forward
        o, _lse, saved = fwd(q.contiguous(), k.contiguous(), v.contiguous(), scale, comm=comm, ops=ops)
        ctx.saved, ctx.schedule, ctx.comm, ctx.ops = saved, schedule, comm, ops
        return o

    @staticmethod
    def backward(ctx, dO):
        bwd = ringx_dist.ringx_b_backward if ctx.schedule == "b" else ringx_dist.ringx_a_backward
        dq, dk, dv = bwd(ctx.saved, dO.contiguous(), comm=ctx.comm, ops=ctx.ops)
        return dq, dk, dv, None, None, None, None


def ringx_sdpa(query, key, value, attn_mask=None, dropout_p: float = 0.0, is_causal: bool = False, scale=None,
               enable_gqa: bool = False, *, kv_chunk: int | None = None, schedule: str | None = None, comm=None, ops=None):
    """softmax(scale * Q K^T) V with the signature of torch's scaled_dot_product_attention.

    query [B,Hq,N,d], key/value [B,Hkv,N,d] (Hkv divides Hq: grouped-query attention needs enable_gqa=True, as in
    torch), bf16 or fp32 CUDA tensors, d in {64,128} -- or the multi-head-latent-attention widths query/key [.,192],
    value [.,128] (bf16, Hkv == Hq).  `scale` defaults to 1/sqrt(d).  `kv_chunk`: keys per pass.
    `schedule` = "b" or "a" runs the paper's RingX_b / RingX_a over `comm` (default: the torch.distributed world)
    with the arguments being the local sequence chunks."""
    if attn_mask is not None or dropout_p != 0.0 or is_causal:
        raise NotImplementedError("RingX attention is non-causal, unmasked and has no dropout (PAPER.md:174-179)")
    if query.shape[1] != key.shape[1] and not enable_gqa:
        raise ValueError("query and key have different head counts: pass enable_gqa=True")
    if query.shape[-1] != value.shape[-1] and query.shape[1] != key.shape[1]:
        raise NotImplementedError("the MLA widths (d_qk != d_v) are built for Hkv == Hq only")
    scale = 1.0 / math.sqrt(query.shape[-1]) if scale is None else float(scale)
    if schedule is not None:
        if schedule not in ("a", "b"):
            raise ValueError("schedule must be 'a', 'b' or None")
        return _RingXDistAttention.apply(query, key, value, scale, schedule, comm, ops)
    kv_chunk = _default_chunk(key.shape[2]) if kv_chunk is None else kv_chunk
    return _RingXAttention.apply(query, key, value, scale, kv_chunk)


class _RingXBlock(torch.autograd.Function):
    """The attention block of Table II as one autograd node: forward = ringx_attn_block_fwd (which keeps
    q, k, v, o, lse in its workspace), backward = ringx_attn_block_bwd reading that workspace."""

    @staticmethod
    def forward(ctx, x, w_qkv, w_o, H, kv_chunk, scale):
        x, w_qkv, w_o = x.contiguous(), w_qkv.contiguous(), w_o.contiguous()
        B, S, h = x.shape
        ws = torch.empty(max(256, ringx.ringx_attn_block_fwd_workspace_bytes(B, S, H, h // H, kv_chunk)), dtype=torch.uint8,
                         device=x.device)
        y = ringx.ringx_attn_block_fwd(x, w_qkv, w_o, H, kv_chunk, scale, workspace=ws)
        ctx.save_for_backward(x, w_qkv, w_o, ws)
        ctx.H, ctx.kv_chunk, ctx.scale = H, kv_chunk, scale
        return y

    @staticmethod
    def backward(ctx, dy):
        x, w_qkv, w_o, ws = ctx.saved_tensors
        dx, dw_qkv, dw_o = ringx.ringx_attn_block_bwd(x, w_qkv, w_o, dy.contiguous(), ws, ctx.H, ctx.kv_chunk, ctx.scale)
        return dx, dw_qkv.to(w_qkv.dtype), dw_o.to(w_o.dtype), None, None, None


def ringx_attention_block(x, w_qkv, w_o, num_heads: int, scale=None, kv_chunk: int | None = None):
    """y = W_o . attention(split_heads(W_qkv x)) for x [B,S,h] bf16, w_qkv [3h,h], w_o [h,h] (torch.nn.Linear layout, no
    bias), differentiable in x, w_qkv and w_o.  h = num_heads * d with d in {64,128}; h % 256 == 0 for the backward."""
    d = x.shape[-1] // num_heads
    scale = 1.0 / math.sqrt(d) if scale is None else float(scale)
    kv_chunk = _default_chunk(x.shape[1]) if kv_chunk is None else kv_chunk
    return _RingXBlock.apply(x, w_qkv, w_o, num_heads, kv_chunk, scale)
