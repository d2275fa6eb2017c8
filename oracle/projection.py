"""fp64 CPU oracle for the projection GEMMs either side of the attention kernel.
*** TEST INFRASTRUCTURE ONLY *** -- same rules as oracle/attention.py (no code shared with the CUDA path; only
`tests/`, `__graft_entry__.smoke()` and `bench.py`'s CPU legs may import it).

What the paper states (Table II): "Input to Q/K/V" is the GEMM `(b, S, h) x (h, h)` (three of them,
`6bSh^2` FLOPs), the attention kernel then works on the head-split layout `(b*a, S, h/a)`, and the "Linear
Projection" `(bS, h) x (h, h)` (`2bSh^2`) follows.  Nothing else is said, so (readings p1-p4):
  p1  weights are stored output-feature major, `W [out, in]`, and applied as `y = x W^T` (torch.nn.Linear's layout);
      the three input projections are stacked as `W_qkv = [W_q; W_k; W_v]`, shape `[3h, h]`.
  p2  head a owns the d = h/a consecutive features `[a*d, (a+1)*d)`: `q[b, a, s, c] = (x W_q^T)[b, s, a*d + c]`.
  p3  no bias (Table II counts none) and no activation.
  p4  the block is  x -> (q, k, v) -> Eq. 1 attention per head -> merge heads -> output projection.

Pins (tests/test_oracle_pins_projection.py): identity weights make the projections pure layout permutations;
one-hot inputs read single weights; brute-force Python loops; FLOP-free invariants (linearity, head independence);
torch.nn.functional.linear in fp64 as a library second opinion; the block against a per-head loop written out.
"""
from __future__ import annotations

import numpy as np

from . import attention as _att


def split_heads(y, H):
    """[B, S, h] -> [B, H, S, d]: head a = features [a*d, (a+1)*d) (reading p2; Table II's (b*a, S, h/a))."""
    B, S, h = y.shape
    d = h // H
    return y.reshape(B, S, H, d).transpose(0, 2, 1, 3)


def merge_heads(o):
    """[B, H, S, d] -> [B, S, h]: the inverse of split_heads."""
    B, H, S, d = o.shape
    return o.transpose(0, 2, 1, 3).reshape(B, S, H * d)


def qkv_projection(x, w_qkv, H):
    """"Input to Q/K/V": x [B,S,h], w_qkv [3h,h] = [W_q; W_k; W_v] -> q, k, v [B,H,S,d]."""
    x = np.asarray(x, dtype=np.float64)
    w = np.asarray(w_qkv, dtype=np.float64)
    h = x.shape[-1]
    y = x @ w.T                                               # [B, S, 3h]   (reading p1)
    return tuple(split_heads(y[..., i * h:(i + 1) * h], H) for i in range(3))


def out_projection(o, w_o):
    """"Linear Projection": o [B,H,S,d], w_o [h,h] -> y [B,S,h] = merge_heads(o) W_o^T."""
    return merge_heads(np.asarray(o, dtype=np.float64)) @ np.asarray(w_o, dtype=np.float64).T


def attention_block_fwd(x, w_qkv, w_o, H, scale):
    """The attention block of Table II (reading p4): projections, Eq. 1 attention per (batch, head), projection."""
    q, k, v = qkv_projection(x, w_qkv, H)
    B, _, S, d = q.shape
    o = np.empty_like(q)
    for b in range(B):
        for a in range(H):
            o[b, a], _ = _att.attention_fwd(q[b, a], k[b, a], v[b, a], scale)
    return out_projection(o, w_o)


# --------------------------------------------------------------------------------------------------------------------
# Backward of the projections and of the block: the derivative of the definitions above (the paper trains the model,
# PAPER.md:260-264, but prints no backward formulas; reading p5: plain calculus, loss L = sum dY * Y).
# --------------------------------------------------------------------------------------------------------------------
def out_projection_bwd(dy, o, w_o):
    """y = merge_heads(o) W_o^T  =>  dO = split_heads(dY W_o),  dW_o = dY^T merge_heads(o).
    dy [B,S,h], o [B,H,S,d], w_o [h,h] -> (dO [B,H,S,d], dW_o [h,h])."""
    dy = np.asarray(dy, dtype=np.float64)
    o = np.asarray(o, dtype=np.float64)
    w = np.asarray(w_o, dtype=np.float64)
    H = o.shape[1]
    om = merge_heads(o)                                         # [B, S, h]
    d_o = split_heads(dy @ w, H)
    dw = np.einsum("bsn,bsi->ni", dy, om)
    return d_o, dw


def qkv_projection_bwd(dq, dk, dv, x, w_qkv):
    """[q|k|v] = x W_qkv^T  =>  dX = [dQ|dK|dV]_merged W_qkv,  dW_qkv = [dQ|dK|dV]_merged^T x.
    dq,dk,dv [B,H,S,d], x [B,S,h], w_qkv [3h,h] -> (dX [B,S,h], dW_qkv [3h,h])."""
    x = np.asarray(x, dtype=np.float64)
    w = np.asarray(w_qkv, dtype=np.float64)
    g = np.concatenate([merge_heads(np.asarray(t, dtype=np.float64)) for t in (dq, dk, dv)], axis=-1)   # [B, S, 3h]
    dx = g @ w
    dw = np.einsum("bsn,bsi->ni", g, x)
    return dx, dw


def attention_block_bwd(x, w_qkv, w_o, dy, H, scale):
    """Gradients of L = sum dY * attention_block_fwd(x, ...): returns (dX, dW_qkv, dW_o)."""
    q, k, v = qkv_projection(x, w_qkv, H)
    B = q.shape[0]
    o = np.empty_like(q)
    for b in range(B):
        for a in range(H):
            o[b, a], _ = _att.attention_fwd(q[b, a], k[b, a], v[b, a], scale)
    d_o, dw_o = out_projection_bwd(dy, o, w_o)
    dq, dk, dv = np.empty_like(q), np.empty_like(k), np.empty_like(v)
    for b in range(B):
        for a in range(H):
            dq[b, a], dk[b, a], dv[b, a] = _att.attention_bwd(q[b, a], k[b, a], v[b, a], d_o[b, a], scale)
    dx, dw_qkv = qkv_projection_bwd(dq, dk, dv, x, w_qkv)
    return dx, dw_qkv, dw_o
