"""RingX_a and RingX_b over `torch.distributed`: the paper's two sequence-parallel
attention schedules (Fig. 2), one process per GPU, NCCL over NVLink/NVSwitch.

Every rank holds an equal sequence chunk `q, k, v [B,H,N/W,d]`.  All arithmetic of the method
runs in libringx kernels (`ringx_attn_chunk_fwd`, `ringx_attn_chunk_fwd_fold`, `ringx_eq5_scale/finalize`,
`ringx_attn_bwd_partial`, `ringx_dq_finalize`); this module only sequences them with the collectives the paper names:

  RingX_b   forward : all-gather(K,V) -> local chunk loop + running Eq. 5 merge
                           backward: local chunk loop (dQ accumulates) -> reduce-scatter(dK,dV)
  RingX_a forward, step t: broadcast(Q_t) -> local attention against the own (K,V) chunk
                           -> all-reduce(max) of loc_lse -> Eq. 5 weights -> reduce(num, den) to rank t
                           backward, step t: broadcast(K_t,V_t) -> dK_t,dV_t shares reduced to rank t,
                           dQ "accumulated for each rank over N steps"

Communication/computation overlap follows PAPER.md:147: the collective that feeds step t+1 is issued (async_op)
before the kernels of step t are enqueued, into the other of two ping-pong buffers; RingX_b starts on the chunk it
already owns while the all-gather is in flight.  On NVSwitch every peer is one hop away at full bandwidth, so the
all-gather form (RingX_b) is the natural default; RingX_a keeps per-rank memory at O(N/W).

Gradient shares cross the collectives in fp32: a device's dK,dV of a step are only its SHARE of a sum over devices
(PAPER.md:143, 145), so `ringx_attn_bwd_partial_ex` writes them unrounded, the reduce / reduce-scatter sums fp32, and
the owner rounds once to bf16 -- the accuracy of the single-device path, independent of the world size (bf16 shares
would be rounded W times and then added in bf16).  Scratch buffers are allocated once per schedule call, and
D_i = dO_i.O_i is formed once per backward, not once per step.

`ops` is the per-device kernel set; the default drives the CUDA library and has no CPU fallback.  `comm` is the
set of collectives (default: torch.distributed, NCCL on GPUs).  The CPU/gloo tests substitute an fp64 `ops` to check
the schedules themselves (which chunk meets which, what is reduced where) without a GPU; the one-GPU tests run the
real kernels for W simulated ranks through an in-process `comm`.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


class CudaOps:
    """The per-device steps, each one call into libringx (paper_2507_16697_b200.ringx)."""

    def __init__(self):
        from . import ringx
        self.rx = ringx

    def attn_fwd(self, q, k, v, scale):                       # single device, single pass
        return self.rx.ringx_attn_fwd(q, k, v, q.shape[2], scale)

    def fwd_scratch(self, q, k):                              # split-KV workspace of one chunk pass (None: not needed)
        if q.dtype != torch.bfloat16:
            return None
        B, H, Nq, d = q.shape
        n = self.rx.ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, k.shape[2], d, q.dtype)
        return torch.empty(n, dtype=torch.uint8, device=q.device) if n else None

    def chunk_fwd(self, q, k, v, scale, scratch=None):        # (loc_out fp32, loc_lse)
        if q.dtype == torch.bfloat16:                         # split-KV when the local chunk cannot fill the GPU
            return self.rx.ringx_attn_chunk_fwd_ex(q, k, v, scale, workspace=scratch)
        return self.rx.ringx_attn_chunk_fwd(q, k, v, scale)

    def chunk_fwd_fold(self, q, k, v, o_acc, lse_acc, scale, final, scratch=None):   # chunk pass + two-operand Eq. 5
        return self.rx.ringx_attn_chunk_fwd_ex(q, k, v, scale, o_acc=o_acc, lse_acc=lse_acc, final=final, workspace=scratch)

    def eq5_scale(self, loc_out, loc_lse, lse_max):           # num, den of one operand (in place on loc_out)
        return self.rx.ringx_eq5_scale(loc_out, loc_lse, lse_max, inplace=True)

    def eq5_finalize(self, num, den, lse_max, out_dtype):
        return self.rx.ringx_eq5_finalize(num, den, lse_max, out_dtype=out_dtype)

    def bwd_scratch(self, q):                                 # D, lse2 (+ fixed-point scratch in deterministic mode): allocated once
        B, H, Nq, d = q.shape
        n = max(256, self.rx.ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d))
        return torch.empty(n, dtype=torch.uint8, device=q.device)

    def bwd_partial(self, q, k, v, o, lse, dO, scale, dq_acc, dk, dv, scratch, prepared):
        """dq_acc += these keys' contribution; (dk, dv) = this device's share for these keys, in dk's dtype.  `prepared`:
        `scratch` holds D, lse2 of (o, lse, dO) from an earlier step of this backward."""
        return self.rx.ringx_attn_bwd_partial_ex(q, k, v, o, lse, dO, scale, dq_acc, dk, dv, scratch, prepared=prepared)

    def dq_finalize(self, dq_acc, like):
        return self.rx.ringx_dq_finalize(dq_acc)

    def round_share(self, acc, like):                         # the one rounding of a reduced fp32 gradient (same kernel)
        return self.rx.ringx_dq_finalize(acc)

    def acc_dtype(self, q):                                   # dtype of partials, accumulators and gradient shares
        return torch.float32


class MlaCudaOps(CudaOps):
    """The same steps for multi-head latent attention widths (q, k [.,192]; v, o, dO [.,128]): the MLA
    kernels of libringx.  The fp32 dQ accumulator is kept transposed by the kernel; the schedules only create, pass on and
    finalize it, so it stays a tensor of q's shape whose layout is the kernel's business."""

    def attn_fwd(self, q, k, v, scale):
        return self.rx.ringx_attn_fwd_mla(q, k, v, q.shape[2], scale)

    def fwd_scratch(self, q, k):
        return None

    def chunk_fwd(self, q, k, v, scale, scratch=None):
        return self.rx.ringx_attn_chunk_fwd_mla(q, k, v, scale)

    def chunk_fwd_fold(self, q, k, v, o_acc, lse_acc, scale, final, scratch=None):
        return self.rx.ringx_attn_chunk_fwd_mla(q, k, v, scale, o_acc=o_acc, lse_acc=lse_acc, final=final)

    def bwd_scratch(self, q):
        B, H, Nq, _ = q.shape
        n = max(256, self.rx.ringx_attn_bwd_partial_mla_workspace_bytes(B, H, Nq))
        return torch.empty(n, dtype=torch.uint8, device=q.device)

    def bwd_partial(self, q, k, v, o, lse, dO, scale, dq_acc, dk, dv, scratch, prepared):
        return self.rx.ringx_attn_bwd_partial_mla(q, k, v, o, lse, dO, scale, dq_acc, dk, dv, scratch, prepared=prepared)

    def dq_finalize(self, dq_acc, like):
        B, H, Nq, d_qk = like.shape
        return self.rx.ringx_dq_finalize_mla(dq_acc, B, H, Nq, d_qk)


def default_ops(q, v):
    """The CUDA kernel set for these widths: MHA / GQA-free d in {64,128}, or the MLA widths (d_qk != d_v)."""
    return MlaCudaOps() if q.shape[-1] != v.shape[-1] else CudaOps()


class _Done:
    def wait(self):
        return None


class TorchComm:
    """The collectives the paper names, on a torch.distributed group (NCCL on GPUs).
    Every method returns a handle with .wait(); the transfer is asynchronous to the caller's stream until then."""

    def __init__(self, group=None):
        if not dist.is_initialized():
            raise RuntimeError("ringx_dist needs an initialised torch.distributed process group (backend nccl on GPUs)")
        self.group = group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)

    def _global(self, r):
        return r if self.group is None else dist.get_global_rank(self.group, r)

    def broadcast(self, t, src):
        return dist.broadcast(t, src=self._global(src), group=self.group, async_op=True)

    def all_reduce_max(self, t):
        return dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group, async_op=True)

    def reduce_sum(self, t, dst):
        return dist.reduce(t, dst=self._global(dst), group=self.group, async_op=True)

    def all_gather(self, stacked, t):
        """stacked [W, *t.shape] <- every rank's t (the collective sees the concatenation along dim 0)."""
        return dist.all_gather_into_tensor(stacked.view((-1,) + tuple(t.shape[1:])), t.contiguous(), group=self.group,
                                           async_op=True)

    def reduce_scatter_sum(self, out, stacked):
        """out <- sum over ranks of their stacked[self.rank]."""
        if dist.get_backend(self.group) == "gloo":       # CPU tests: gloo has no reduce-scatter
            dist.all_reduce(stacked, group=self.group)
            out.copy_(stacked[self.rank])
            return _Done()
        return dist.reduce_scatter_tensor(out, stacked.view((-1,) + tuple(stacked.shape[2:])), group=self.group,
                                          async_op=True)


# ---------------------------------------------------------------------------------------------- RingX_b
def ringx_b_forward(q, k, v, scale, comm=None, ops=None):
    """All-gather(K,V), then the local chunk loop with the running Eq. 5 merge.
    Returns (o, lse, ctx); ctx keeps the gathered K,V for the backward."""
    ops = ops or default_ops(q, v)
    comm = comm or TorchComm()
    W, r = comm.world, comm.rank
    if W == 1:
        o, lse = ops.attn_fwd(q, k, v, scale)
        return o, lse, (q, k.unsqueeze(0), v.unsqueeze(0), o, lse, scale)
    kg = torch.empty((W,) + tuple(k.shape), dtype=k.dtype, device=k.device)
    vg = torch.empty((W,) + tuple(v.shape), dtype=v.dtype, device=v.device)
    works = [comm.all_gather(kg, k), comm.all_gather(vg, v)]
    scratch = ops.fwd_scratch(q, k)                           # one allocation for all W chunk passes
    o_acc, lse_acc = ops.chunk_fwd(q, k, v, scale, scratch)   # the chunk already here overlaps the gather
    for w in works:
        w.wait()
    o = lse = None
    for s in range(1, W):
        c = (r + s) % W                                       # ring order: every rank starts on a different chunk
        if s == W - 1:
            o, lse = ops.chunk_fwd_fold(q, kg[c], vg[c], o_acc, lse_acc, scale, True, scratch)     # last fold writes bf16
        else:
            o_acc, lse_acc = ops.chunk_fwd_fold(q, kg[c], vg[c], o_acc, lse_acc, scale, False, scratch)
    return o, lse, (q, kg, vg, o, lse, scale)


def ringx_b_backward(ctx, dO, comm=None, ops=None):
    """Local loop over the gathered chunks (dK_c, dV_c shares; dQ accumulates), then reduce-scatter(dK,dV)
    (PAPER.md:145).  Returns (dq, dk, dv) for the local sequence chunk."""
    q, kg, vg, o, lse, scale = ctx
    ops = ops or default_ops(q, vg)
    comm = comm or TorchComm()
    W, r = comm.world, comm.rank
    dq_acc = torch.zeros(q.shape, dtype=ops.acc_dtype(q), device=q.device)
    scratch = ops.bwd_scratch(q)
    if W == 1:
        dk, dv = torch.empty_like(kg[0]), torch.empty_like(vg[0])
        ops.bwd_partial(q, kg[0], vg[0], o, lse, dO, scale, dq_acc, dk, dv, scratch, False)
        return ops.dq_finalize(dq_acc, q), dk, dv
    share = ops.acc_dtype(q)                                  # the shares cross the reduce-scatter unrounded
    dkg = torch.empty(kg.shape, dtype=share, device=kg.device)
    dvg = torch.empty(vg.shape, dtype=share, device=vg.device)
    for s in range(W):
        c = (r + s) % W
        ops.bwd_partial(q, kg[c], vg[c], o, lse, dO, scale, dq_acc, dkg[c], dvg[c], scratch, s > 0)
    dq = ops.dq_finalize(dq_acc, q)
    dk, dv = torch.empty_like(dkg[0]), torch.empty_like(dvg[0])
    works = [comm.reduce_scatter_sum(dk, dkg), comm.reduce_scatter_sum(dv, dvg)]
    for w in works:
        w.wait()
    return dq, ops.round_share(dk, kg[0]), ops.round_share(dv, vg[0])


# ---------------------------------------------------------------------------------------------- RingX_a
def ringx_a_forward(q, k, v, scale, comm=None, ops=None):
    """Step t: broadcast(Q_t), every rank attends it against its own (K,V) chunk, all-reduce(max) of loc_lse,
    reduce(num, den) to rank t, which forms num/den.  The broadcast for step t+1 is issued
    before step t computes, into the other ping-pong buffer.  Returns (o, lse, ctx)."""
    ops = ops or default_ops(q, v)
    comm = comm or TorchComm()
    W, r = comm.world, comm.rank
    if W == 1:
        o, lse = ops.attn_fwd(q, k, v, scale)
        return o, lse, (q, k, v, o, lse, scale)
    bufs = [torch.empty_like(q), torch.empty_like(q)]

    def start_bcast(t):
        buf = q if t == r else bufs[t & 1]
        return buf, comm.broadcast(buf, t)

    nxt = start_bcast(0)
    scratch = ops.fwd_scratch(q, k)                           # one allocation for all W steps
    o = lse = None
    for t in range(W):
        q_t, work = nxt
        if t + 1 < W:
            nxt = start_bcast(t + 1)
        work.wait()
        loc_out, loc_lse = ops.chunk_fwd(q_t, k, v, scale, scratch)
        lse_max = loc_lse.clone()
        comm.all_reduce_max(lse_max).wait()
        num, den = ops.eq5_scale(loc_out, loc_lse, lse_max)
        works = [comm.reduce_sum(num, t), comm.reduce_sum(den, t)]
        for w in works:
            w.wait()
        if t == r:
            o, lse = ops.eq5_finalize(num, den, lse_max, q.dtype)
    return o, lse, (q, k, v, o, lse, scale)


def ringx_a_backward(ctx, dO, comm=None, ops=None):
    """Step t: broadcast(K_t, V_t); every rank computes its share of dK_t, dV_t from its local Q, dO (reduced to
    rank t) and adds these keys' contribution to its dQ accumulator.  Returns (dq, dk, dv)."""
    q, k, v, o, lse, scale = ctx
    ops = ops or default_ops(q, v)
    comm = comm or TorchComm()
    W, r = comm.world, comm.rank
    dq_acc = torch.zeros(q.shape, dtype=ops.acc_dtype(q), device=q.device)
    scratch = ops.bwd_scratch(q)
    if W == 1:
        dk, dv = torch.empty_like(k), torch.empty_like(v)
        ops.bwd_partial(q, k, v, o, lse, dO, scale, dq_acc, dk, dv, scratch, False)
        return ops.dq_finalize(dq_acc, q), dk, dv
    share = ops.acc_dtype(q)
    dkb = [torch.empty(k.shape, dtype=share, device=k.device) for _ in range(2)]     # ping-pong: step t's reduce may still
    dvb = [torch.empty(v.shape, dtype=share, device=v.device) for _ in range(2)]     # read one pair while t+1 writes the other
    kb = [torch.empty_like(k), torch.empty_like(k)]
    vb = [torch.empty_like(v), torch.empty_like(v)]

    def start_bcast(t):
        kt, vt = (k, v) if t == r else (kb[t & 1], vb[t & 1])
        return kt, vt, [comm.broadcast(kt, t), comm.broadcast(vt, t)]

    nxt = start_bcast(0)
    dk = dv = None
    for t in range(W):
        k_t, v_t, works = nxt
        if t + 1 < W:
            nxt = start_bcast(t + 1)
        for w in works:
            w.wait()
        dk_t, dv_t = dkb[t & 1], dvb[t & 1]
        ops.bwd_partial(q, k_t, v_t, o, lse, dO, scale, dq_acc, dk_t, dv_t, scratch, t > 0)
        works = [comm.reduce_sum(dk_t, t), comm.reduce_sum(dv_t, t)]
        for w in works:
            w.wait()
        if t == r:                                            # the fp32 sums over all ranks: round once
            dk, dv = ops.round_share(dk_t, k), ops.round_share(dv_t, v)
    return ops.dq_finalize(dq_acc, q), dk, dv
