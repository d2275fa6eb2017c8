"""RingX_a / RingX_b schedules (paper_2507_16697_b200.ringx_dist) on CPU: world_size 2 and 3,
gloo backend.  The per-device kernel set is replaced by an fp64 stand-in built on the oracle, so what is checked
here is the host logic alone -- which chunk meets which, which collective carries what to whom, ping-pong buffer
reuse -- against the unchunked oracle attention of the concatenated sequence.  (The CUDA kernels behind the same
interface are checked against the oracle in the `-m gpu` tests.)"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import attention as orc
from paper_2507_16697_b200 import ringx_dist


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class OracleOps:
    """fp64 stand-in for ringx_dist.CudaOps (same method names and in/out conventions), test-only."""

    @staticmethod
    def _heads(*ts):
        B, H = ts[0].shape[:2]
        for b in range(B):
            for h in range(H):
                yield (b, h), [t[b, h].numpy() for t in ts]

    def acc_dtype(self, q):
        return torch.float64

    def attn_fwd(self, q, k, v, scale):
        return self.chunk_fwd(q, k, v, scale)

    def fwd_scratch(self, q, k):
        return None

    def bwd_scratch(self, q):
        return {"prepared_for": None}          # stands in for the D / lse2 workspace: records what it was prepared for

    def round_share(self, acc, like):
        return acc.clone()

    def chunk_fwd(self, q, k, v, scale, scratch=None):
        o = torch.empty(q.shape[:3] + (v.shape[3],), dtype=torch.float64)
        lse = torch.empty(q.shape[:3], dtype=torch.float64)
        for (b, h), (qq, kk, vv) in self._heads(q, k, v):
            a, l = orc.attention_fwd(qq, kk, vv, scale)
            o[b, h], lse[b, h] = torch.from_numpy(a), torch.from_numpy(l)
        return o, lse

    def chunk_fwd_fold(self, q, k, v, o_acc, lse_acc, scale, final, scratch=None):
        o_p, lse_p = self.chunk_fwd(q, k, v, scale)
        return self.lse_merge(o_acc, lse_acc, o_p, lse_p, o_acc.dtype, not final)

    def lse_merge(self, o_a, lse_a, o_b, lse_b, out_dtype, inplace):
        o, lse = orc.lse_merge(o_a.reshape(-1, o_a.shape[-1]).numpy(), lse_a.reshape(-1).numpy(),
                               o_b.reshape(-1, o_b.shape[-1]).numpy(), lse_b.reshape(-1).numpy())
        o, lse = torch.from_numpy(o).reshape(o_a.shape), torch.from_numpy(lse).reshape(lse_a.shape)
        if inplace:
            o_a.copy_(o)
            lse_a.copy_(lse)
            return o_a, lse_a
        return o, lse

    def eq5_scale(self, loc_out, loc_lse, lse_max):            # Eq. 5's summands
        w = torch.exp(loc_lse - lse_max)
        loc_out.mul_(w.unsqueeze(-1))
        return loc_out, w

    def eq5_finalize(self, num, den, lse_max, out_dtype):
        return num / den.unsqueeze(-1), lse_max + torch.log(den)

    def bwd_partial(self, q, k, v, o, lse, dO, scale, dq_acc, dk, dv, scratch, prepared):
        # the schedule must prepare (D, lse2) exactly once per backward, on its first step, and say so afterwards
        key = (o.data_ptr(), dO.data_ptr())
        assert prepared == (scratch["prepared_for"] == key), "D/lse2 preprocess: once per backward, first step only"
        scratch["prepared_for"] = key
        assert dk.dtype == self.acc_dtype(q) and dv.dtype == self.acc_dtype(q) or not prepared and dk.dtype == k.dtype
        for (b, h), (qq, kk, vv, oo, ll, dd) in self._heads(q, k, v, o, lse, dO):
            D = (dd * oo).sum(axis=1)
            a, bk, bv = orc.attention_bwd_partial(qq, kk, vv, dd, ll, D, scale)
            dq_acc[b, h] += torch.from_numpy(a)
            dk[b, h], dv[b, h] = torch.from_numpy(bk), torch.from_numpy(bv)
        return dq_acc, dk, dv

    def dq_finalize(self, dq_acc, like):
        return dq_acc.clone()


def _inputs(world, B=1, H=2, Nl=5, d=4, seed=3):
    g = np.random.default_rng(seed)
    shape = (B, H, world * Nl, d)
    return [g.standard_normal(shape) for _ in range(4)]          # q, k, v, dO of the whole sequence


def _worker(rank, world, port, variant, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        q, k, v, dO = _inputs(world)
        Nl = q.shape[2] // world
        sl = slice(rank * Nl, (rank + 1) * Nl)
        ql, kl, vl, dOl = (torch.from_numpy(np.ascontiguousarray(t[:, :, sl])) for t in (q, k, v, dO))
        fwd, bwd = ((ringx_dist.ringx_a_forward, ringx_dist.ringx_a_backward) if variant == "a" else
                    (ringx_dist.ringx_b_forward, ringx_dist.ringx_b_backward))
        ops = OracleOps()
        if variant.startswith("sdpa_"):          # the autograd drop-in over the same schedules
            from paper_2507_16697_b200.sdpa import ringx_sdpa
            ql, kl, vl = (t.requires_grad_() for t in (ql, kl, vl))
            o = ringx_sdpa(ql, kl, vl, scale=0.5, schedule=variant[-1], ops=ops)
            o.backward(dOl)
            lse = torch.from_numpy(orc.attention_fwd_bhnd(q, k, v, 0.5)[1][:, :, sl].copy())   # (sdpa returns o only)
            o, dq, dk, dv = o.detach(), ql.grad, kl.grad, vl.grad
        else:
            o, lse, ctx = fwd(ql, kl, vl, 0.5, ops=ops)
            dq, dk, dv = bwd(ctx, dOl, ops=ops)
        out.put((rank, [t.numpy().copy() for t in (o, lse, dq, dk, dv)]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("variant,world", [("a", 2), ("b", 2), ("a", 3), ("b", 3), ("sdpa_a", 2), ("sdpa_b", 2)])
def test_ringx_schedules_equal_the_unchunked_attention(variant, world):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, variant, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(out.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    q, k, v, dO = _inputs(world)
    Nl = q.shape[2] // world
    o_ref, lse_ref = orc.attention_fwd_bhnd(q, k, v, 0.5)
    grads_ref = orc.attention_bwd_bhnd(q, k, v, dO, 0.5)
    for r in range(world):
        sl = slice(r * Nl, (r + 1) * Nl)
        o, lse, dq, dk, dv = got[r]
        np.testing.assert_allclose(o, o_ref[:, :, sl], atol=1e-12)
        np.testing.assert_allclose(lse, lse_ref[:, :, sl], atol=1e-12)
        for g, ref in zip((dq, dk, dv), grads_ref):
            np.testing.assert_allclose(g, ref[:, :, sl], atol=1e-12)


def test_sdpa_drop_in_rejects_what_the_papers_attention_does_not_have():
    from paper_2507_16697_b200.sdpa import ringx_sdpa, _default_chunk
    t = torch.zeros(1, 2, 256, 64, dtype=torch.bfloat16)
    with pytest.raises(NotImplementedError):
        ringx_sdpa(t, t, t, is_causal=True)
    with pytest.raises(NotImplementedError):
        ringx_sdpa(t, t, t, attn_mask=torch.ones(256, 256, dtype=torch.bool))
    with pytest.raises(NotImplementedError):
        ringx_sdpa(t, t, t, dropout_p=0.1)
    with pytest.raises(ValueError, match="enable_gqa"):
        ringx_sdpa(t, t[:, :1], t[:, :1])
    with pytest.raises(ValueError, match="CUDA tensor"):          # no CPU fallback
        ringx_sdpa(t, t, t)
    assert _default_chunk(262144) == 32768 and _default_chunk(1280) == 256 and _default_chunk(384) == 128


def test_requires_a_process_group():
    t = torch.zeros(1, 1, 4, 4)
    with pytest.raises(RuntimeError, match="process group"):
        ringx_dist.ringx_b_forward(t, t, t, 1.0, ops=OracleOps())


def test_default_ops_have_no_cpu_fallback():
    """The product path drives the CUDA library only: CPU tensors are refused, not routed elsewhere."""
    ops = ringx_dist.CudaOps()
    t = torch.zeros(1, 1, 256, 64, dtype=torch.bfloat16)
    with pytest.raises(ValueError, match="CUDA tensor"):
        ops.chunk_fwd(t, t, t, 1.0)
