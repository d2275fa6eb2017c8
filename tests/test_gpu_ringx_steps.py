"""GPU parity of the per-device RingX steps against the fp64 oracle:
  ringx_attn_bwd_partial / ringx_dq_finalize  (Nq != Nk, global LSE)
  ringx_eq5_scale / ringx_eq5_finalize        (Eq. 5 with N operands)
and of the RingX_a / RingX_b schedules of ringx_dist with the real kernels: W ranks simulated on ONE GPU (threads,
an in-process stand-in for the collectives -- the kernels of different ranks never wait on one another), plus the
torch.distributed/NCCL path itself at world size 1."""
import math
import os
import socket
import threading

import numpy as np
import pytest
import torch

from oracle import attention as orc
from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_GRAD = 2e-2      # BASELINE.json: gradients <= 2e-2 relative Frobenius
TOL_LSE = 1e-3


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


def relf(a, ref):
    return np.linalg.norm(a - ref) / np.linalg.norm(ref)


# ------------------------------------------------------------------------------------------------ bwd_partial
@pytest.mark.parametrize("d,Nq,chunks", [(64, 512, (512, 512)), (128, 256, (384, 640)), (64, 1024, (128, 256, 128)),
                                         (128, 384, (1024,)), (128, 300, (200, 333)), (64, 77, (1000,)),
                                         (64, 129, (1, 127, 130))])       # the last three: ragged Nq and Nk
def test_bwd_partial_steps_add_up_to_the_oracle_gradient(rx, d, Nq, chunks):
    """Nq query rows against Nk = sum(chunks) keys, one ringx_attn_bwd_partial call per key chunk (ragged chunk
    sizes, Nq != Nk).  dq accumulates over the calls; each call's dk, dv are complete for its keys."""
    B, H, Nk = 1, 3, sum(chunks)
    scale = 1.0 / math.sqrt(d)
    q = wl.make_tensor((B, H, Nq, d), "q", seed=71, dtype="bf16")
    do = wl.make_tensor((B, H, Nq, d), "do", seed=71, dtype="bf16")
    k = wl.make_tensor((B, H, Nk, d), "k", seed=71, dtype="bf16")
    v = wl.make_tensor((B, H, Nk, d), "v", seed=71, dtype="bf16")
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    bounds = np.concatenate([[0], np.cumsum(chunks)])
    q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
    o_ref, lse_ref = orc.attention_fwd_bhnd(q64, k64, v64, scale)
    # the saved global (o, lse) of these rows from the library itself: chunk partials + Eq. 5, bf16 at the end
    parts = [rx.ringx_attn_chunk_fwd(qd, kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous(), scale)
             for lo, hi in zip(bounds[:-1], bounds[1:])]
    o_acc, lse_acc = parts[0]
    for i, (o_p, lse_p) in enumerate(parts[1:]):
        last = i == len(parts) - 2
        o_acc, lse_acc = rx.ringx_lse_merge(o_acc, lse_acc, o_p, lse_p,
                                            out_dtype=torch.bfloat16 if last else torch.float32)
    o_dev, lse_dev = o_acc.to(torch.bfloat16), lse_acc
    assert np.abs(lse_dev.cpu().double().numpy() - lse_ref).max() <= 5e-5
    assert relf(f64(o_dev), o_ref) <= 1e-2
    dq_acc = torch.zeros((B, H, Nq, d), dtype=torch.float32, device="cuda")
    dq_ref, dk_ref, dv_ref = orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
    for lo, hi in zip(bounds[:-1], bounds[1:]):
        _, dk, dv = rx.ringx_attn_bwd_partial(qd, kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous(), o_dev,
                                              lse_dev, dod, scale, dq_acc=dq_acc)
        assert rx.ringx_last_launch_count() == 2 + (1 if Nq % 128 else 0)   # preprocess (+ pad of a ragged head) + chunk kernel
        assert relf(f64(dk), dk_ref[:, :, lo:hi]) <= TOL_GRAD
        assert relf(f64(dv), dv_ref[:, :, lo:hi]) <= TOL_GRAD
        assert relf(f64(dk), dk_ref[:, :, lo:hi]) <= 6e-3 and relf(f64(dv), dv_ref[:, :, lo:hi]) <= 6e-3
    dq = rx.ringx_dq_finalize(dq_acc)
    assert dq.dtype == torch.bfloat16
    assert relf(f64(dq), dq_ref) <= 6e-3
    # the accumulator itself holds the true gradient (scale included), before the bf16 rounding
    assert relf(dq_acc.cpu().double().numpy(), dq_ref) <= 6e-3
    if Nq % 128:
        # the same steps with ringx_set_deterministic (int32 scratch per step, added to the fp32 accumulator): reproducible
        accs = []
        rx.ringx_set_deterministic(True)
        try:
            for _ in range(2):
                acc = torch.zeros((B, H, Nq, d), dtype=torch.float32, device="cuda")
                for lo, hi in zip(bounds[:-1], bounds[1:]):
                    rx.ringx_attn_bwd_partial(qd, kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous(), o_dev, lse_dev,
                                              dod, scale, dq_acc=acc)
                accs.append(acc)
            torch.cuda.synchronize()
        finally:
            rx.ringx_set_deterministic(False)
        assert torch.equal(accs[0], accs[1])
        assert relf(accs[0].cpu().double().numpy(), dq_ref) <= 6e-3


@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("case", ["zero_local_v", "other_chunk_16x"])
def test_deterministic_partial_step_with_zero_and_small_local_v(rx, d, case):
    """Deterministic (int32 fixed-point) dQ in a per-device step whose own V says nothing about D_i = dO_i.O_i: O comes from
    the keys of ALL steps, so with this step's V all zero (padding) or another step's V 16x larger, |D_i| is far above
    ||dO_i|| max_local||V||.  A scale taken from the local V alone overflows the int32 (the advisor's finding on r02);
    the bound now carries |D_i| itself.  Two steps of 512 keys; dq must match the oracle, and the fp32 mode's result."""
    B, H, Nq, Nk = 1, 2, 384, 1024
    scale = 1.0 / math.sqrt(d)
    q = wl.make_tensor((B, H, Nq, d), "q", seed=73, dtype="bf16")
    do = wl.make_tensor((B, H, Nq, d), "do", seed=73, dtype="bf16")
    k = wl.make_tensor((B, H, Nk, d), "k", seed=73, dtype="bf16")
    v = wl.make_tensor((B, H, Nk, d), "v", seed=73, dtype="bf16").clone()
    if case == "zero_local_v":
        v[:, :, :512] = 0
    else:
        v[:, :, 512:] = (v[:, :, 512:].float() * 16).to(torch.bfloat16)
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
    o_dev, lse_dev = rx.ringx_attn_chunk_fwd_ex(qd, kd, vd, scale, final=True)
    dq_ref, dk_ref, dv_ref = orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
    results = {}
    for det in (False, True):
        rx.ringx_set_deterministic(det)
        try:
            acc = torch.zeros((B, H, Nq, d), dtype=torch.float32, device="cuda")
            for lo, hi in ((0, 512), (512, 1024)):
                _, dk, dv = rx.ringx_attn_bwd_partial(qd, kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous(), o_dev,
                                                      lse_dev, dod, scale, dq_acc=acc)
                assert relf(f64(dk), dk_ref[:, :, lo:hi]) <= TOL_GRAD
            torch.cuda.synchronize()
        finally:
            rx.ringx_set_deterministic(False)
        results[det] = acc.cpu().double().numpy()
    assert relf(results[False], dq_ref) <= 6e-3
    assert relf(results[True], dq_ref) <= 6e-3                     # r02: saturated integers, garbage
    assert np.abs(results[True] - results[False]).max() <= 1e-4 * np.abs(dq_ref).max()


def test_deterministic_mode_propagates_non_finite_gradients(rx):
    """The fp32 accumulator turns a NaN or Inf upstream gradient into a NaN row of dq; the integer accumulator would round it
    to 0 (float -> int of NaN is 0).  The per-row scale is NaN when its bound is not finite, so the row comes out NaN in
    deterministic mode too, and the other rows are untouched."""
    B, H, N, d = 1, 2, 512, 128
    scale = 1.0 / math.sqrt(d)
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=83, dtype="bf16")
    do = do.clone()
    do[0, 0, 5, 3] = float("nan")
    do[0, 1, 300, 0] = float("inf")
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, N, scale)
    rx.ringx_set_deterministic(True)
    try:
        dq, _, _ = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, N, scale)
        torch.cuda.synchronize()
    finally:
        rx.ringx_set_deterministic(False)
    dq = dq.float().cpu()
    assert torch.isnan(dq[0, 0, 5]).all() and torch.isnan(dq[0, 1, 300]).all()
    finite = torch.ones(B, H, N, dtype=torch.bool)
    finite[0, 0, 5] = finite[0, 1, 300] = False
    assert torch.isfinite(dq[finite]).all()
    do_clean = do.clone()
    do_clean[0, 0, 5] = 0
    do_clean[0, 1, 300] = 0
    dq_ref, _, _ = orc.attention_bwd_bhnd(f64(q), f64(k), f64(v), f64(do_clean), scale)
    assert relf(dq[finite].double().numpy(), dq_ref[finite.numpy()]) <= 6e-3


def test_bwd_partial_equals_full_backward_when_it_sees_everything(rx):
    """With Nq == Nk and one call, ringx_attn_bwd_partial + ringx_dq_finalize is ringx_attn_bwd (same kernels)."""
    B, H, N, d = 1, 2, 1024, 128
    scale = 1.0 / math.sqrt(d)
    q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=5, dtype="bf16"))
    o, lse = rx.ringx_attn_fwd(q, k, v, N, scale)
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do, N, scale)
    dq_acc, dk2, dv2 = rx.ringx_attn_bwd_partial(q, k, v, o, lse, do, scale)
    assert torch.equal(dk, dk2) and torch.equal(dv, dv2)        # atomic-free: bit-reproducible
    dq2 = rx.ringx_dq_finalize(dq_acc)
    assert relf(f64(dq2), f64(dq)) <= 1e-3                      # dQ: reduce-add order differs between runs


def test_bwd_partial_rejects_bad_arguments(rx):
    L = rx.lib()
    t = torch.zeros(1, 1, 256, 64, dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros(1, 1, 256, device="cuda")
    acc = torch.zeros(1, 1, 256, 64, device="cuda")
    ws = torch.empty(4096, dtype=torch.uint8, device="cuda")
    p = [x.data_ptr() for x in (t, t, t, t, lse, t, acc, t, t)]
    call = lambda Nq, Nk, d, dt, wsb: L.ringx_attn_bwd_partial(*p, 1, 1, Nq, Nk, d, 0.125, dt, ws.data_ptr(), wsb, None)
    assert call(256, 256, 64, 1, 4096) == 0
    assert call(200, 100, 64, 1, 4096) == 0       # any Nq, Nk (ragged tiles)
    assert call(0, 256, 64, 1, 4096) == 2         # BAD_SHAPE
    assert call(256, 0, 64, 1, 4096) == 2
    assert call(256, 256, 96, 1, 4096) == 2
    assert call(256, 256, 64, 0, 4096) == 3       # BAD_DTYPE: bf16 only
    assert call(256, 256, 64, 1, 16) == 5         # WORKSPACE_TOO_SMALL
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------------------------ fused fold
@pytest.mark.parametrize("d,Nq,chunks,gain", [(128, 512, (256, 128, 640), 1.0), (64, 256, (512, 512), 1.0),
                                              (128, 256, (128, 128, 128, 128), 3.0), (128, 300, (200, 333, 1), 1.0),
                                              (64, 1000, (77, 500), 1.0)])      # the last two: ragged Nq and Nk
def test_chunk_fwd_fold_equals_the_running_merge(rx, d, Nq, chunks, gain):
    """ringx_attn_chunk_fwd_fold = ringx_attn_chunk_fwd + two-operand Eq. 5 in one kernel: against the oracle's
    running merge over ragged chunks, and against the library's own two-kernel route (fp32 rounding apart)."""
    B, H, Nk = 2, 2, sum(chunks)
    scale = 1.0 / math.sqrt(d)
    q = wl.make_tensor((B, H, Nq, d), "q", seed=91, dtype="bf16", gain=gain)
    k = wl.make_tensor((B, H, Nk, d), "k", seed=91, dtype="bf16", gain=gain)
    v = wl.make_tensor((B, H, Nk, d), "v", seed=91, dtype="bf16")
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    bounds = np.concatenate([[0], np.cumsum(chunks)])
    ck = [(kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous()) for lo, hi in zip(bounds[:-1], bounds[1:])]
    o_acc, lse_acc = rx.ringx_attn_chunk_fwd(qd, *ck[0], scale)
    o_ref2, lse_ref2 = o_acc.clone(), lse_acc.clone()
    for kc, vc in ck[1:-1]:
        o_acc, lse_acc = rx.ringx_attn_chunk_fwd_fold(qd, kc, vc, o_acc, lse_acc, scale)
        assert rx.ringx_last_launch_count() == 1
        o_p, lse_p = rx.ringx_attn_chunk_fwd(qd, kc, vc, scale)
        o_ref2, lse_ref2 = rx.ringx_lse_merge(o_ref2, lse_ref2, o_p, lse_p)
        assert (o_acc - o_ref2).abs().max().item() <= 2e-6 * max(1.0, o_ref2.abs().max().item())
        assert (lse_acc - lse_ref2).abs().max().item() <= 1e-5
    keep_o, keep_l = o_acc.clone(), lse_acc.clone()
    o, lse = rx.ringx_attn_chunk_fwd_fold(qd, *ck[-1], o_acc, lse_acc, scale, final=True)
    assert o.dtype == torch.bfloat16
    assert torch.equal(keep_o, o_acc) and torch.equal(keep_l, lse_acc)          # final fold leaves the accumulators alone
    q64, k64, v64 = f64(q), f64(k), f64(v)
    o_ref, lse_ref = orc.attention_fwd_bhnd(q64, k64, v64, scale)
    for b in range(B):
        for h in range(H):
            a, l = orc.attention_fwd_running(q64[b, h], k64[b, h], v64[b, h], scale, [int(x) for x in bounds])
            np.testing.assert_allclose(a, o_ref[b, h], atol=1e-12)              # (oracle: running == unchunked)
    assert np.abs(f64(o) - o_ref).max() <= 1e-2 * np.abs(v64).max()
    assert relf(f64(o), o_ref) <= 1e-2
    assert np.abs(f64(lse) - lse_ref).max() <= 5e-5
    L = rx.lib()
    assert L.ringx_attn_chunk_fwd_fold(qd.data_ptr(), kd.data_ptr(), vd.data_ptr(), o_acc.data_ptr(), lse_acc.data_ptr(),
                                       o.data_ptr(), None, B, H, Nq, Nk, d, scale, 1, None) == 1     # one of the pair NULL
    assert L.ringx_attn_chunk_fwd_fold(qd.data_ptr(), kd.data_ptr(), vd.data_ptr(), o_acc.data_ptr(), lse_acc.data_ptr(),
                                       None, None, B, H, Nq, Nk, d, scale, 0, None) == 3             # bf16 only


# ------------------------------------------------------------------------------------------------ Eq. 5, N operands
@pytest.mark.parametrize("rows,d,n_ops", [(1, 8, 2), (777, 64, 3), (4099, 128, 5), (130, 1024, 4)])
def test_eq5_scale_and_finalize_match_oracle(rx, rows, d, n_ops):
    g = torch.Generator().manual_seed(rows + d + n_ops)
    outs = [torch.randn(rows, d, generator=g) for _ in range(n_ops)]
    lses = [torch.randn(rows, generator=g) * 6 for _ in range(n_ops)]
    lses[0][::7] = -math.inf                       # an empty chunk on some rows: weight 0, its loc_out ignored
    outs[0][::7] = math.nan
    if rows > 20:
        for l in lses:
            l[13] = -math.inf                      # a row with every operand empty: o = 0, lse = -inf
    lse_max = torch.stack(lses).max(dim=0).values.cuda()         # the all-reduce(max) of the schedule
    num = torch.zeros(rows, d, device="cuda")
    den = torch.zeros(rows, device="cuda")
    for o_i, l_i in zip(outs, lses):
        n_i, d_i = rx.ringx_eq5_scale(o_i.cuda(), l_i.cuda(), lse_max)
        num += n_i                                  # the reduce(num, den) of the schedule
        den += d_i
    # (the oracle multiplies by the zero weight, so the garbage behind an empty chunk is zeroed for it: reading g12)
    o_ref, lse_ref = orc.merge_partials([np.nan_to_num(f64(o), nan=0.0) for o in outs], [f64(l) for l in lses])
    for out_dtype, tol in ((torch.float32, 2e-6), (torch.bfloat16, 4e-3)):
        o, lse = rx.ringx_eq5_finalize(num, den, lse_max, out_dtype=out_dtype)
        og, lg = f64(o), f64(lse)
        assert np.isfinite(og).all()
        assert np.abs(og - o_ref).max() <= tol * max(1.0, np.abs(o_ref).max())
        fin = np.isfinite(lse_ref)
        assert (lg[~fin] == lse_ref[~fin]).all()
        assert np.abs(lg[fin] - lse_ref[fin]).max() <= 2e-6 * max(1.0, np.abs(lse_ref[fin]).max())
    # in place on loc_out
    a = outs[1].cuda()
    n_i, _ = rx.ringx_eq5_scale(a, lses[1].cuda(), lse_max, inplace=True)
    assert n_i.data_ptr() == a.data_ptr()
    assert rx.lib().ringx_eq5_scale(None, None, None, None, None, 0, 64, None) == 0      # rows == 0: no-op


# ------------------------------------------------------------------------------------------------ schedules, W ranks
class ThreadComm:
    """In-process stand-in for ringx_dist.TorchComm: W threads = W simulated ranks sharing one GPU and one stream.
    Every collective is "publish, barrier, combine, barrier"; combining uses plain torch copies and sums IN THE
    TENSOR'S OWN DTYPE, as NCCL does (the schedules hand it fp32 gradient shares, so that is an fp32 sum)."""

    class _Shared:
        def __init__(self, world):
            self.world = world
            self.barrier = threading.Barrier(world)
            self.slots = [None] * world

    class _Done:
        def wait(self):
            return None

    def __init__(self, shared, rank):
        self.sh, self.rank, self.world = shared, rank, shared.world

    def _exchange(self, t):
        self.sh.slots[self.rank] = t
        self.sh.barrier.wait()
        return list(self.sh.slots)

    def _finish(self):
        self.sh.barrier.wait()
        return self._Done()

    def broadcast(self, t, src):
        got = self._exchange(t)
        if self.rank != src:
            t.copy_(got[src])
        return self._finish()

    def all_reduce_max(self, t):
        got = self._exchange(t.clone())
        t.copy_(torch.stack(got).max(dim=0).values)
        return self._finish()

    def reduce_sum(self, t, dst):
        got = self._exchange(t.clone())
        if self.rank == dst:
            t.copy_(torch.stack(got).sum(dim=0))
        return self._finish()

    def all_gather(self, stacked, t):
        got = self._exchange(t)
        for i, g in enumerate(got):
            stacked[i].copy_(g)
        return self._finish()

    def reduce_scatter_sum(self, out, stacked):
        got = self._exchange(stacked)
        out.copy_(torch.stack([g[self.rank] for g in got]).sum(dim=0))
        return self._finish()


@pytest.mark.parametrize("variant", ["a", "b"])
@pytest.mark.parametrize("world,d,Nl", [(2, 128, 512), (4, 64, 256), (3, 128, 300)])   # the last: ragged per-rank chunks
def test_ringx_schedules_on_simulated_ranks(rx, variant, world, d, Nl):
    """RingX_a / RingX_b forward + backward with the real kernels, W sequence chunks of Nl tokens, against the
    oracle attention of the whole sequence and against the library's own single-device ringx_attn_fwd/bwd."""
    from paper_2507_16697_b200 import ringx_dist
    B, H, N = 1, 2, world * Nl
    scale = 1.0 / math.sqrt(d)
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=23 + world, dtype="bf16")
    fwd, bwd = ((ringx_dist.ringx_a_forward, ringx_dist.ringx_a_backward) if variant == "a" else
                (ringx_dist.ringx_b_forward, ringx_dist.ringx_b_backward))
    shared = ThreadComm._Shared(world)
    results, errors = [None] * world, []

    def rank_main(r):
        try:
            torch.cuda.set_device(0)
            comm = ThreadComm(shared, r)
            sl = slice(r * Nl, (r + 1) * Nl)
            ql, kl, vl, dol = (t[:, :, sl].contiguous().cuda() for t in (q, k, v, do))
            o, lse, ctx = fwd(ql, kl, vl, scale, comm=comm)
            dq, dk, dv = bwd(ctx, dol, comm=comm)
            torch.cuda.synchronize()
            results[r] = [t.cpu() for t in (o, lse, dq, dk, dv)]
        except Exception as e:                      # noqa: BLE001 -- surface it in the main thread
            errors.append(e)
            shared.barrier.abort()

    threads = [threading.Thread(target=rank_main, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not errors, errors
    q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
    o_ref, lse_ref = orc.attention_fwd_bhnd(q64, k64, v64, scale)
    dq_ref, dk_ref, dv_ref = orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
    for r in range(world):
        sl = slice(r * Nl, (r + 1) * Nl)
        o, lse, dq, dk, dv = results[r]
        assert o.dtype == torch.bfloat16 and dq.dtype == torch.bfloat16
        assert np.abs(f64(o) - o_ref[:, :, sl]).max() <= 1e-2 * np.abs(v64).max()
        assert relf(f64(o), o_ref[:, :, sl]) <= 1e-2
        assert np.abs(f64(lse) - lse_ref[:, :, sl]).max() <= 5e-5
        for g, ref in ((dq, dq_ref), (dk, dk_ref), (dv, dv_ref)):
            e = relf(f64(g), ref[:, :, sl])
            assert e <= TOL_GRAD and e <= 8e-3, e


def run_simulated(rx, variant, world, B, H, Nl, d, seed):
    """Both directions of one schedule on `world` simulated ranks; returns the per-rank results and the whole-sequence inputs."""
    from paper_2507_16697_b200 import ringx_dist
    N = world * Nl
    scale = 1.0 / math.sqrt(d)
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=seed, dtype="bf16")
    fwd, bwd = ((ringx_dist.ringx_a_forward, ringx_dist.ringx_a_backward) if variant == "a" else
                (ringx_dist.ringx_b_forward, ringx_dist.ringx_b_backward))
    shared = ThreadComm._Shared(world)
    results, errors = [None] * world, []

    def rank_main(r):
        try:
            torch.cuda.set_device(0)
            comm = ThreadComm(shared, r)
            sl = slice(r * Nl, (r + 1) * Nl)
            ql, kl, vl, dol = (t[:, :, sl].contiguous().cuda() for t in (q, k, v, do))
            o, lse, ctx = fwd(ql, kl, vl, scale, comm=comm)
            dq, dk, dv = bwd(ctx, dol, comm=comm)
            torch.cuda.synchronize()
            results[r] = [t.cpu() for t in (o, lse, dq, dk, dv)]
        except Exception as e:                      # noqa: BLE001 -- surface it in the main thread
            errors.append(e)
            shared.barrier.abort()

    threads = [threading.Thread(target=rank_main, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert not errors, errors
    return results, (q, k, v, do), scale


def test_gradient_error_does_not_grow_with_the_world_size(rx):
    """The gradient shares cross the collectives in fp32 and are rounded once (ringx_attn_bwd_partial_ex): the error of
    dK, dV against the oracle at W = 2, 4, 8, 16 ranks (same whole sequence, N = 4096) stays at the single-device level
    -- with bf16 shares it would grow with W (W roundings, then a bf16 sum)."""
    import grad_bounds as gb
    B, H, N, d = 1, 1, 4096, 64
    errs = {}
    for variant in ("b", "a"):
        for world in (2, 4, 8, 16):
            results, (q, k, v, do), scale = run_simulated(rx, variant, world, B, H, N // world, d, seed=31)
            q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
            if "ref" not in errs:
                errs["ref"] = orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
                qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
                o1, l1 = rx.ringx_attn_fwd(qd, kd, vd, N, scale)
                errs["single"] = [relf(f64(g), r) for g, r in zip(rx.ringx_attn_bwd(qd, kd, vd, o1, l1, dod, N, scale), errs["ref"])]
            got = [torch.cat([results[r][i] for r in range(world)], dim=2) for i in (2, 3, 4)]     # dq, dk, dv, whole sequence
            e = [relf(f64(g), r) for g, r in zip(got, errs["ref"])]
            errs[(variant, world)] = e
            for name, g, r in zip(("dq", "dk", "dv"), got, errs["ref"]):
                assert g.dtype == torch.bfloat16
                gb.check_grad(f"{name} RingX_{variant} W={world}", f64(g)[0, 0], r[0, 0])
    print("relative Frobenius error of (dq, dk, dv) vs W:", {k_: [f"{x:.2e}" for x in v_] for k_, v_ in errs.items() if k_ != "ref"})
    for key, e in errs.items():
        if key in ("ref", "single"):
            continue
        for x, x1 in zip(e, errs["single"]):
            assert x <= 1.5 * x1 + 5e-4, (key, e, errs["single"])       # no growth with W


def test_bwd_partial_ex_fp32_shares_and_prepared_workspace(rx):
    """ringx_attn_bwd_partial_ex: fp32 dk, dv are the accumulators the bf16 form rounds (so rounding them gives the bf16
    result bit for bit), and `prepared` reuses D / lse2 left in the workspace by the first step of the backward."""
    B, H, Nq, Nk, d = 1, 2, 512, 384, 128
    scale = 1.0 / math.sqrt(d)
    q = wl.make_tensor((B, H, Nq, d), "q", seed=61, dtype="bf16").cuda()
    do = wl.make_tensor((B, H, Nq, d), "do", seed=61, dtype="bf16").cuda()
    k = wl.make_tensor((B, H, 2 * Nk, d), "k", seed=61, dtype="bf16").cuda()
    v = wl.make_tensor((B, H, 2 * Nk, d), "v", seed=61, dtype="bf16").cuda()
    o, lse = rx.ringx_attn_fwd(q[:, :, :512].contiguous(), k[:, :, :512].contiguous(), v[:, :, :512].contiguous(), 512, scale)
    ws = torch.empty(rx.ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d), dtype=torch.uint8, device="cuda")
    ka, va = k[:, :, :Nk].contiguous(), v[:, :, :Nk].contiguous()
    kb, vb = k[:, :, Nk:].contiguous(), v[:, :, Nk:].contiguous()
    acc = torch.zeros(B, H, Nq, d, device="cuda")
    dk16, dv16 = torch.empty_like(ka), torch.empty_like(va)
    rx.ringx_attn_bwd_partial_ex(q, ka, va, o, lse, do, scale, acc, dk16, dv16, ws)
    assert rx.ringx_last_launch_count() == 2                     # preprocess + one backward pass
    acc2 = torch.zeros_like(acc)
    dk32 = torch.empty(ka.shape, device="cuda")
    dv32 = torch.empty(va.shape, device="cuda")
    rx.ringx_attn_bwd_partial_ex(q, ka, va, o, lse, do, scale, acc2, dk32, dv32, ws, prepared=True)
    assert rx.ringx_last_launch_count() == 1                     # the pass alone: D, lse2 reused
    assert torch.equal(dk32.to(torch.bfloat16), dk16) and torch.equal(dv32.to(torch.bfloat16), dv16)
    assert torch.equal(rx.ringx_dq_finalize(dk32), dk16)         # the library's own rounding kernel: the same bits
    # a second step on other keys with the prepared workspace, against the un-prepared call
    rx.ringx_attn_bwd_partial_ex(q, kb, vb, o, lse, do, scale, acc2, dk32, dv32, ws, prepared=True)
    ref = torch.zeros_like(acc)
    dkr, dvr = torch.empty_like(dk32), torch.empty_like(dv32)
    rx.ringx_attn_bwd_partial_ex(q, kb, vb, o, lse, do, scale, ref, dkr, dvr, ws, prepared=False)
    assert torch.equal(dkr, dk32) and torch.equal(dvr, dv32)
    L = rx.lib()
    p = [x.data_ptr() for x in (q, kb, vb, o, lse, do, ref, dkr, dvr)]
    assert L.ringx_attn_bwd_partial_ex(*p, B, H, Nq, Nk, d, scale, 1, 2, 0, ws.data_ptr(), ws.numel(), None) == 3   # dkv dtype
    torch.cuda.synchronize()


_NCCL_W2 = r"""
import math, os, sys, torch, torch.distributed as dist
sys.path.insert(0, {root!r})
from paper_2507_16697_b200 import ringx, ringx_dist, workloads as wl
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(rank)
dist.init_process_group("nccl", device_id=torch.device("cuda", rank))
B, H, Nl, d = 1, 2, 512, 128
N = world * Nl
scale = 1.0 / math.sqrt(d)
q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=47, dtype="bf16"))
o1, l1 = ringx.ringx_attn_fwd(q, k, v, N, scale)
g1 = ringx.ringx_attn_bwd(q, k, v, o1, l1, do, N, scale)
sl = slice(rank * Nl, (rank + 1) * Nl)
ql, kl, vl, dol = (t[:, :, sl].contiguous() for t in (q, k, v, do))
for fwd, bwd in ((ringx_dist.ringx_b_forward, ringx_dist.ringx_b_backward), (ringx_dist.ringx_a_forward, ringx_dist.ringx_a_backward)):
    o, lse, ctx = fwd(ql, kl, vl, scale)
    dq, dk, dv = bwd(ctx, dol)
    torch.cuda.synchronize()
    rel = lambda a, b: ((a.float() - b.float()).norm() / b.float().norm()).item()
    assert rel(o, o1[:, :, sl]) <= 5e-3 and (lse - l1[:, :, sl]).abs().max().item() <= 5e-5
    for g, r in zip((dq, dk, dv), g1):
        assert rel(g, r[:, :, sl]) <= 5e-3, rel(g, r[:, :, sl])
dist.barrier()
dist.destroy_process_group()
if rank == 0:
    print("NCCL_W2_OK")
"""


def test_ringx_schedules_over_nccl_two_gpus(rx, tmp_path):
    """RingX_a and RingX_b across two real devices over NCCL (one process per GPU), against the single-device library
    result of the whole sequence.  Skipped on a box with one GPU (every box of this project so far: no multi-GPU run of
    the schedules exists, and none is claimed)."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "nccl_w2.py"
    script.write_text(_NCCL_W2.format(root=root))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
                        "127.0.0.1", "--master-port", str(port), str(script)], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "NCCL_W2_OK" in r.stdout, (r.stdout[-2000:], r.stderr[-2000:])


def test_ringx_dist_over_nccl_world_size_one(rx):
    """The torch.distributed path itself (backend nccl, one rank on the one GPU): both schedules reduce to the
    single-device library calls."""
    import torch.distributed as dist
    from paper_2507_16697_b200 import ringx_dist
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        B, H, N, d = 1, 2, 512, 64
        scale = 1.0 / math.sqrt(d)
        q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=9, dtype="bf16"))
        o_ref, lse_ref = rx.ringx_attn_fwd(q, k, v, N, scale)
        for fwd, bwd in ((ringx_dist.ringx_a_forward, ringx_dist.ringx_a_backward),
                         (ringx_dist.ringx_b_forward, ringx_dist.ringx_b_backward)):
            o, lse, ctx = fwd(q, k, v, scale)
            dq, dk, dv = bwd(ctx, do)
            assert torch.equal(o, o_ref) and torch.equal(lse, lse_ref)
            dq_r, dk_r, dv_r = rx.ringx_attn_bwd(q, k, v, o, lse, do, N, scale)
            assert torch.equal(dk, dk_r) and torch.equal(dv, dv_r)
            assert relf(f64(dq), f64(dq_r)) <= 1e-3
        # the collectives themselves, on the one rank
        comm = ringx_dist.TorchComm()
        t = torch.arange(8, dtype=torch.float32, device="cuda")
        st = torch.zeros(1, 8, device="cuda")
        comm.all_gather(st, t).wait()
        comm.all_reduce_max(t).wait()
        comm.reduce_sum(t, 0).wait()
        comm.broadcast(t, 0).wait()
        out = torch.zeros(8, device="cuda")
        comm.reduce_scatter_sum(out, st).wait()
        torch.cuda.synchronize()
        assert torch.equal(out, t) and torch.equal(st[0], t)
    finally:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------ GQA (NEXT-3)
@pytest.mark.parametrize("Hq,Hkv,N,d,chunk", [(4, 2, 512, 64, 256), (6, 2, 256, 128, 128), (8, 1, 512, 64, 512),
                                              (4, 2, 333, 128, 128), (6, 3, 700, 64, 384)])   # the last two: ragged lengths
def test_gqa_forward_and_backward_match_oracle(rx, Hq, Hkv, N, d, chunk):
    """Hq query heads share Hkv kv heads (query head h attends kv head h // (Hq/Hkv)); the oracle is the plain
    attention of every query head against its kv head, dk/dv summed over the heads of the group."""
    B, G = 2, Hq // Hkv
    scale = 1.0 / math.sqrt(d)
    q = wl.make_tensor((B, Hq, N, d), "q", seed=41, dtype="bf16")
    do = wl.make_tensor((B, Hq, N, d), "do", seed=41, dtype="bf16")
    k = wl.make_tensor((B, Hkv, N, d), "k", seed=41, dtype="bf16")
    v = wl.make_tensor((B, Hkv, N, d), "v", seed=41, dtype="bf16")
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd_gqa(qd, kd, vd, chunk, scale)
    dq, dk, dv = rx.ringx_attn_bwd_gqa(qd, kd, vd, o, lse, dod, chunk, scale)
    q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
    k_rep, v_rep = np.repeat(k64, G, axis=1), np.repeat(v64, G, axis=1)      # kv head of every query head
    o_ref, lse_ref = orc.attention_fwd_bhnd(q64, k_rep, v_rep, scale)
    dq_ref, dk_rep, dv_rep = orc.attention_bwd_bhnd(q64, k_rep, v_rep, do64, scale)
    dk_ref = dk_rep.reshape(B, Hkv, G, N, d).sum(axis=2)
    dv_ref = dv_rep.reshape(B, Hkv, G, N, d).sum(axis=2)
    assert np.abs(f64(o) - o_ref).max() <= 1e-2 * np.abs(v64).max()
    assert relf(f64(o), o_ref) <= 1e-2
    assert np.abs(f64(lse) - lse_ref).max() <= 5e-5
    for g, ref in ((dq, dq_ref), (dk, dk_ref), (dv, dv_ref)):
        e = relf(f64(g), ref)
        assert e <= TOL_GRAD and e <= 6e-3, e
    # Hq == Hkv is the plain multi-head call, bit for bit
    o2, lse2 = rx.ringx_attn_fwd_gqa(qd[:, :Hkv].contiguous(), kd, vd, chunk, scale)
    o3, lse3 = rx.ringx_attn_fwd(qd[:, :Hkv].contiguous(), kd, vd, chunk, scale)
    assert torch.equal(o2, o3) and torch.equal(lse2, lse3)
    L = rx.lib()
    assert L.ringx_attn_fwd_gqa(qd.data_ptr(), kd.data_ptr(), vd.data_ptr(), o.data_ptr(), lse.data_ptr(), B, 5, 2, N, d,
                                chunk, scale, 1, None, 0, None) == 2          # Hq % Hkv != 0: BAD_SHAPE


# ------------------------------------------------------------------------------------------------ split-KV
@pytest.mark.parametrize("B,H,Nq,Nk,d", [(1, 2, 256, 4096, 128), (1, 4, 512, 8192, 64), (2, 1, 256, 3072, 128),
                                         (1, 8, 2048, 16384, 128)])
def test_chunk_fwd_ex_split_kv_matches_the_oracle(rx, B, H, Nq, Nk, d):
    """Few query tiles against many keys (the paper's per-device regime): the library splits the keys
    over groups of CTAs and combines the groups by Eq. 5 inside the pass.  All four result forms against the oracle:
    partial, final bf16, in-place fold with a running accumulator, final fold."""
    scale = 1.0 / math.sqrt(d)
    assert rx.ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, Nk, d, torch.bfloat16) > 0      # it does split here
    q = wl.make_tensor((B, H, Nq, d), "q", seed=5, dtype="bf16")
    k = wl.make_tensor((B, H, Nk, d), "k", seed=5, dtype="bf16")
    v = wl.make_tensor((B, H, Nk, d), "v", seed=5, dtype="bf16")
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    q64, k64, v64 = f64(q), f64(k), f64(v)
    o_ref = np.empty((B, H, Nq, d))
    l_ref = np.empty((B, H, Nq))
    for b in range(B):
        for h in range(H):
            o_ref[b, h], l_ref[b, h] = orc.attention_fwd(q64[b, h], k64[b, h], v64[b, h], scale)
    vmax = np.abs(v64).max()

    def check(o, lse, what):
        o = o.float().cpu().numpy()
        assert np.abs(o - o_ref).max() <= 1e-2 * vmax, what
        assert relf(o, o_ref) <= (1e-2 if o.dtype != np.float32 or what.endswith("bf16") else 5e-3), what
        assert np.abs(lse.cpu().numpy() - l_ref).max() <= 1e-3, what

    lo, ll = rx.ringx_attn_chunk_fwd_ex(qd, kd, vd, scale)
    assert rx.ringx_last_launch_count() == 2 and lo.dtype == torch.float32      # split chunk kernel + Eq. 5 kernel
    check(lo, ll, "partial")
    o, lse = rx.ringx_attn_chunk_fwd_ex(qd, kd, vd, scale, final=True)
    check(o, lse, "final bf16")
    # the unsplit kernel gives the same partials up to rounding (P is rounded to bf16 against a different running max)
    lo1, ll1 = rx.ringx_attn_chunk_fwd(qd, kd, vd, scale)
    assert (lo - lo1).abs().max().item() <= 1e-2 * lo1.abs().max().item() and (ll - ll1).abs().max().item() <= 1e-5
    # fold: first half of the keys as the running accumulator, second half folded in with split-KV
    half = Nk // 2
    ka, kb, va, vb = kd[:, :, :half].contiguous(), kd[:, :, half:].contiguous(), vd[:, :, :half].contiguous(), vd[:, :, half:].contiguous()
    acc_o, acc_l = rx.ringx_attn_chunk_fwd_ex(qd, ka, va, scale)
    o2, l2 = rx.ringx_attn_chunk_fwd_ex(qd, kb, vb, scale, o_acc=acc_o.clone(), lse_acc=acc_l.clone(), final=True)
    check(o2, l2, "fold final bf16")
    o3, l3 = rx.ringx_attn_chunk_fwd_ex(qd, kb, vb, scale, o_acc=acc_o, lse_acc=acc_l)
    assert o3.data_ptr() == acc_o.data_ptr() and l3.data_ptr() == acc_l.data_ptr()
    check(o3, l3, "fold in place")


def test_attn_fwd_uses_split_kv_when_the_pass_is_small(rx):
    """ringx_attn_fwd with few query tiles: same result as the oracle through the split path (single pass and chunked)."""
    B, H, N, d = 1, 2, 4096, 128
    scale = 1.0 / math.sqrt(d)
    q, k, v = wl.make_qkv((B, H, N, d), seed=9, dtype="bf16")
    q64, k64, v64 = f64(q), f64(k), f64(v)
    o_ref, l_ref = orc.attention_fwd_bhnd(q64, k64, v64, scale)
    for chunk, launches in ((4096, 2), (2048, 4)):
        o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), chunk, scale)
        assert rx.ringx_last_launch_count() == launches
        assert relf(o.float().cpu().numpy(), o_ref) <= 1e-2 and np.abs(lse.cpu().numpy() - l_ref).max() <= 1e-3
