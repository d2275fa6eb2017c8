"""Multi-head latent attention shapes (PAPER.md:376 names MLA among the layer designs RingX is
compatible with): d_qk = 192, d_v = 128, forward and backward.  The oracle is the same definition (oracle.attention takes
d != dv; pinned by tests/test_oracle_pins.py::test_brute_force_forward_nonsquare and, for the gradients, by
test_gradients_match_finite_differences, which runs with d = 3, dv = 4); tolerances are those of the bf16 d = 64 / 128 paths."""
import math

import numpy as np
import pytest
import torch

import grad_bounds as gb
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
                                              (1, 4, 1024, 512, 0.05),
                                              (1, 1, 1, 128, 1.0), (1, 2, 100, 128, 1.0), (2, 2, 1000, 384, 1.0),
                                              (1, 2, 1337, 512, 3.0), (1, 1, 640, 256, 1.0)])      # ragged lengths
def test_mla_forward_matches_oracle(rx, B, H, N, chunk, gain):
    q, k, v = make(B, H, N, seed=101, gain=gain)
    scale = 1.0 / math.sqrt(DQK)
    o, lse = rx.ringx_attn_fwd_mla(q.cuda(), k.cuda(), v.cuda(), chunk, scale)
    assert rx.ringx_last_launch_count() == -(-N // chunk) and o.shape == (B, H, N, DV)
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
    assert call(192, 128, 256, 200, 1) == 2       # kv_chunk % 128
    assert call(192, 128, 256, 512, 1) == 2       # kv_chunk longer than the sequence rounded up to a tile
    assert call(192, 128, 0, 128, 1) == 2
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------------------------ backward
def make_do(B, H, N, seed, device="cpu"):
    return wl.make_tensor((B, H, N, DV), "do", seed=seed, dtype="bf16", device=device)


def check_grads(dq, dk, dv, q64, k64, v64, do64, scale):
    """stated Frobenius tolerance (2e-2) and the element-wise bounds of tests/grad_bounds.py, head by head"""
    worst = 0.0
    for b in range(q64.shape[0]):
        for h in range(q64.shape[1]):
            q_, k_, v_, do_ = q64[b, h], k64[b, h], v64[b, h], do64[b, h]
            dq_ref, dk_ref, dv_ref = orc.attention_bwd(q_, k_, v_, do_, scale)
            E = gb.d_error_rows(q_, k_, v_, do_, scale)
            _, lse = orc.attention_fwd(q_, k_, v_, scale)
            worst = max(worst, gb.check_grad("dq", f64(dq[b, h]), dq_ref, gb.dq_dterm(q_, k_, v_, do_, scale)),
                        gb.check_grad("dk", f64(dk[b, h]), dk_ref, gb.dk_dterm(q_, k_, lse, E, scale)),
                        gb.check_grad("dv", f64(dv[b, h]), dv_ref, None))
    return worst


@pytest.mark.parametrize("B,H,N,chunk,gain", [(1, 1, 128, 128, 1.0), (1, 2, 512, 128, 1.0), (2, 3, 1280, 256, 1.0),
                                              (1, 2, 2304, 768, 1.0), (1, 1, 2048, 2048, 3.0), (1, 4, 1024, 512, 0.05),
                                              (1, 2, 100, 128, 1.0), (1, 1, 257, 128, 1.0), (2, 2, 1000, 384, 1.0),
                                              (1, 2, 1337, 512, 3.0)])                              # ragged lengths
def test_mla_backward_matches_oracle(rx, B, H, N, chunk, gain):
    """dq, dk [.,192], dv [.,128] against the derivative of the definition: several 64-query sub-tiles and key tiles,
    1-4 passes, peaked and near-uniform softmax; element by element."""
    q, k, v = make(B, H, N, seed=131, gain=gain)
    do = make_do(B, H, N, seed=131)
    scale = 1.0 / math.sqrt(DQK)
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd_mla(qd, kd, vd, chunk, scale)
    dq, dk, dv = rx.ringx_attn_bwd_mla(qd, kd, vd, o, lse, dod, chunk, scale)
    assert rx.ringx_last_launch_count() == -(-N // chunk) + 2 + (1 if N % 128 else 0)
    assert dq.shape == (B, H, N, DQK) and dk.shape == (B, H, N, DQK) and dv.shape == (B, H, N, DV)
    check_grads(dq, dk, dv, f64(q), f64(k), f64(v), f64(do), scale)


@pytest.mark.parametrize("B,H,N,chunk,gain", [(2, 3, 1280, 256, 1.0), (1, 8, 8192, 2048, 1.0), (1, 2, 2048, 512, 3.0),
                                              (2, 2, 777, 256, 1.0)])
def test_mla_backward_deterministic_mode(rx, B, H, N, chunk, gain):
    """ringx_set_deterministic with the MLA widths: the transposed dQ accumulator becomes int32 fixed point (per-query
    scales; integer reduce-adds are associative), so repeated runs agree bit for bit -- (1, 8, 8192, 2048) is 512 CTAs per
    pass, 3.5 waves, where the arrival order of the adds varies -- dk, dv are the default mode's, and the result still
    matches the oracle element by element."""
    q, k, v = make(B, H, N, seed=139, gain=gain)
    do = make_do(B, H, N, seed=139)
    scale = 1.0 / math.sqrt(DQK)
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd_mla(qd, kd, vd, chunk, scale)
    loose = rx.ringx_attn_bwd_mla(qd, kd, vd, o, lse, dod, chunk, scale)
    rx.ringx_set_deterministic(True)
    try:
        runs = [rx.ringx_attn_bwd_mla(qd, kd, vd, o, lse, dod, chunk, scale) for _ in range(3)]
        assert rx.ringx_last_launch_count() == -(-N // chunk) + 4 + (1 if N % 128 else 0)
        torch.cuda.synchronize()
    finally:
        rx.ringx_set_deterministic(False)
    for r in runs[1:]:
        for a, b in zip(runs[0], r):
            assert torch.equal(a, b)
    assert torch.equal(runs[0][1], loose[1]) and torch.equal(runs[0][2], loose[2])
    assert ((runs[0][0].float() - loose[0].float()).norm() / loose[0].float().norm()).item() <= 2e-3
    if N <= 2048:
        check_grads(*runs[0], f64(q), f64(k), f64(v), f64(do), scale)


def test_mla_backward_every_panel_matters_and_chunk_independent(rx):
    """Zeroing one 64-column panel of q (k, v, dO) in the ORACLE must break the agreement with the kernel's result: the
    kernel contracts over all three panels of q, k and both of v, dO.  dk, dv of a key tile are written once by one CTA
    whatever the chunking: bit-identical; dq is an fp32 reduce-add in arbitrary order: equal within rounding."""
    B, H, N = 1, 1, 512
    q, k, v = make(B, H, N, seed=137)
    do = make_do(B, H, N, seed=137)
    scale = 0.2
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd_mla(qd, kd, vd, N, scale)
    dq, dk, dv = rx.ringx_attn_bwd_mla(qd, kd, vd, o, lse, dod, N, scale)
    q64, k64, v64, do64 = (f64(t[0, 0]) for t in (q, k, v, do))
    full = orc.attention_bwd(q64, k64, v64, do64, scale)
    err = lambda g, r: np.linalg.norm(f64(g[0, 0]) - r) / np.linalg.norm(r)
    assert max(err(dq, full[0]), err(dk, full[1]), err(dv, full[2])) <= 2e-2
    for name, width in (("q", DQK), ("k", DQK), ("v", DV), ("do", DV)):
        for p in range(width // 64):
            args = {"q": q64.copy(), "k": k64.copy(), "v": v64.copy(), "do": do64.copy()}
            args[name][:, 64 * p:64 * p + 64] = 0.0
            cut = orc.attention_bwd(args["q"], args["k"], args["v"], args["do"], scale)
            assert max(err(dq, cut[0]), err(dk, cut[1]), err(dv, cut[2])) > 0.1, (name, p)
    for chunk in (128, 256):
        dq2, dk2, dv2 = rx.ringx_attn_bwd_mla(qd, kd, vd, o, lse, dod, chunk, scale)
        assert torch.equal(dk2, dk) and torch.equal(dv2, dv)
        assert ((dq2.float() - dq.float()).norm() / dq.float().norm()).item() <= 2e-3


def test_mla_backward_long_sequence_sampled(rx):
    """N = 16384, two passes: dq on sampled query rows (sub-tile, tile and chunk boundaries) against all keys; dk, dv on
    sampled key columns with the oracle's LSE and D of all rows of the head; sum_j dV_j = sum_i P^T dO invariants.
    192 CTAs per pass: more than one wave of the 148 SMs."""
    B, H, N, chunk = 1, 3, 16384, 8192
    q, k, v = make(B, H, N, seed=139, device="cuda")
    do = make_do(B, H, N, seed=139, device="cuda")
    scale = 1.0 / math.sqrt(DQK)
    o, lse = rx.ringx_attn_fwd_mla(q, k, v, chunk, scale)
    dq, dk, dv = rx.ringx_attn_bwd_mla(q, k, v, o, lse, do, chunk, scale)
    for t in (dq, dk, dv):
        assert torch.isfinite(t.float()).all()
    rng = np.random.default_rng(5)
    rows = np.array(sorted({0, 1, 63, 64, 65, 127, 128, 8191, 8192, N - 65, N - 64, N - 1} | set(rng.integers(0, N, 40).tolist())))
    cols = np.array(sorted({0, 1, 127, 128, 129, 8191, 8192, 8193, N - 129, N - 128, N - 1} | set(rng.integers(0, N, 40).tolist())))
    h = 2
    q64, k64, v64, do64 = (f64(t[0, h]) for t in (q, k, v, do))
    dq_ref, _, _ = orc.attention_bwd(q64[rows], k64, v64, do64[rows], scale)
    gb.check_grad("dq", f64(dq[0, h][rows]), dq_ref, gb.dq_dterm(q64[rows], k64, v64, do64[rows], scale))
    lse_all = np.empty(N)
    D_all = np.empty(N)
    for r0 in range(0, N, 2048):
        lse_all[r0:r0 + 2048], D_all[r0:r0 + 2048] = orc.row_stats(q64[r0:r0 + 2048], k64, v64, do64[r0:r0 + 2048], scale)
    dk_ref, dv_ref = orc.attention_bwd_cols(q64, k64[cols], v64[cols], do64, lse_all, D_all, scale)
    o_all = np.concatenate([orc.attention_fwd(q64[r0:r0 + 2048], k64, v64, scale)[0] for r0 in range(0, N, 2048)])
    E = gb.U_BF16 * (np.abs(do64) * np.abs(o_all)).sum(axis=1)
    gb.check_grad("dk", f64(dk[0, h][cols]), dk_ref, gb.dk_dterm(q64, k64[cols], lse_all, E, scale))
    gb.check_grad("dv", f64(dv[0, h][cols]), dv_ref, None)
    # sum_j dV_j = sum_i dO_i (rows of P sum to 1) and sum_j dK_j = 0 on every head, from the full outputs
    for hh in range(H):
        sv, sdo = f64(dv[0, hh]).sum(axis=0), f64(do[0, hh]).sum(axis=0)
        assert np.abs(sv - sdo).max() <= 2e-2 * np.abs(sdo).max() + 0.5
        assert np.abs(f64(dk[0, hh]).sum(axis=0)).max() <= 1.0


def test_mla_backward_errors(rx):
    L = rx.lib()
    t = torch.zeros(1, 1, 256, 192, dtype=torch.bfloat16, device="cuda")
    v = torch.zeros(1, 1, 256, 128, dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros(1, 1, 256, device="cuda")
    ws = torch.empty(rx.ringx_attn_bwd_mla_workspace_bytes(1, 1, 256, 192, 128, 256), dtype=torch.uint8, device="cuda")
    call = lambda dqk, dv_, N, chunk, dt, w, wb: L.ringx_attn_bwd_mla(
        t.data_ptr(), t.data_ptr(), v.data_ptr(), v.data_ptr(), lse.data_ptr(), v.data_ptr(), t.data_ptr(), t.data_ptr(),
        v.data_ptr(), 1, 1, N, dqk, dv_, chunk, 0.1, dt, w, wb, None)
    assert rx.ringx_attn_bwd_mla_workspace_bytes(1, 1, 256, 128, 128, 256) == 0
    assert call(192, 128, 256, 256, 1, ws.data_ptr(), ws.numel()) == 0
    assert call(128, 128, 256, 256, 1, ws.data_ptr(), ws.numel()) == 2      # only the 192 / 128 pair: BAD_SHAPE
    assert call(192, 128, 256, 256, 0, ws.data_ptr(), ws.numel()) == 3      # bf16 only
    assert call(192, 128, 256, 256, 1, None, 0) == 1                        # NULL_PTR
    assert call(192, 128, 256, 256, 1, ws.data_ptr(), 1024) == 5            # WORKSPACE_TOO_SMALL
    assert call(192, 128, 192, 192, 1, ws.data_ptr(), ws.numel()) == 2      # N % 128
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------------------------ per-device RingX steps
def test_mla_chunk_steps_are_the_papers_partials_and_fold(rx):
    """ringx_attn_chunk_fwd_mla with Nq != Nk: (loc_out, loc_lse) of a key chunk = the oracle's partials of that chunk
    (PAPER.md:135); folding chunk after chunk (in place, last fold to bf16) = the unchunked attention (Eq. 5)."""
    B, H, Nq, Nk = 1, 2, 256, 1024
    q = wl.make_tensor((B, H, Nq, DQK), "q", seed=151, dtype="bf16")
    k = wl.make_tensor((B, H, Nk, DQK), "k", seed=151, dtype="bf16")
    v = wl.make_tensor((B, H, Nk, DV), "v", seed=151, dtype="bf16")
    scale = 1.0 / math.sqrt(DQK)
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    bounds = [0, 384, 512, 1024]
    acc = None
    for i, (lo, hi) in enumerate(zip(bounds[:-1], bounds[1:])):
        kc, vc = kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous()
        if acc is None:
            acc = rx.ringx_attn_chunk_fwd_mla(qd, kc, vc, scale)
            for h in range(H):
                o_ref, l_ref = orc.attention_fwd(f64(q[0, h]), f64(k[0, h, lo:hi]), f64(v[0, h, lo:hi]), scale)
                assert np.abs(f64(acc[0][0, h]) - o_ref).max() <= 2e-2 * np.abs(o_ref).max()
                assert np.abs(f64(acc[1][0, h]) - l_ref).max() <= 5e-5
        elif i < len(bounds) - 2:
            got = rx.ringx_attn_chunk_fwd_mla(qd, kc, vc, scale, o_acc=acc[0], lse_acc=acc[1])
            assert got[0].data_ptr() == acc[0].data_ptr()
        else:
            keep_o, keep_l = acc[0].clone(), acc[1].clone()
            o, lse = rx.ringx_attn_chunk_fwd_mla(qd, kc, vc, scale, o_acc=acc[0], lse_acc=acc[1], final=True)
            assert torch.equal(keep_o, acc[0]) and torch.equal(keep_l, acc[1])
    assert o.dtype == torch.bfloat16
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    assert np.linalg.norm(f64(o) - o_ref) / np.linalg.norm(o_ref) <= 1e-2
    assert np.abs(f64(lse) - lse_ref).max() <= 5e-5


def test_mla_bwd_partial_steps_add_up_to_the_gradient(rx):
    """Two key chunks through ringx_attn_bwd_partial_mla (global LSE; dQ accumulates across the steps in the transposed
    fp32 accumulator, finalized once): dq = the oracle's, the chunks' dk, dv = the oracle's rows; fp32 shares round to the
    bf16 result bit for bit; `prepared` reuses D / lse2."""
    B, H, Nq, Nk = 1, 2, 384, 768
    q = wl.make_tensor((B, H, Nq, DQK), "q", seed=157, dtype="bf16")
    k = wl.make_tensor((B, H, Nk, DQK), "k", seed=157, dtype="bf16")
    v = wl.make_tensor((B, H, Nk, DV), "v", seed=157, dtype="bf16")
    do = wl.make_tensor((B, H, Nq, DV), "do", seed=157, dtype="bf16")
    scale = 1.0 / math.sqrt(DQK)
    q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
    o64, lse64 = orc.attention_fwd_bhnd(q64, k64, v64, scale)
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = torch.from_numpy(o64).to(torch.bfloat16).cuda(), torch.from_numpy(lse64).float().cuda()
    ws = torch.empty(rx.ringx_attn_bwd_partial_mla_workspace_bytes(B, H, Nq), dtype=torch.uint8, device="cuda")
    acc = torch.zeros((B, H, DQK, Nq), dtype=torch.float32, device="cuda")
    dk16, dv16 = torch.empty_like(kd), torch.empty_like(vd)
    dk32 = torch.empty(kd.shape, dtype=torch.float32, device="cuda")
    dv32 = torch.empty(vd.shape, dtype=torch.float32, device="cuda")
    for step, (lo, hi) in enumerate(((0, 256), (256, 768))):
        kc, vc = kd[:, :, lo:hi].contiguous(), vd[:, :, lo:hi].contiguous()
        a, b = torch.empty_like(kc), torch.empty_like(vc)
        rx.ringx_attn_bwd_partial_mla(qd, kc, vc, o, lse, dod, scale, acc, a, b, ws, prepared=step > 0)
        dk16[:, :, lo:hi], dv16[:, :, lo:hi] = a, b
        a32 = torch.empty(kc.shape, dtype=torch.float32, device="cuda")
        b32 = torch.empty(vc.shape, dtype=torch.float32, device="cuda")
        scratch_acc = torch.zeros_like(acc)
        rx.ringx_attn_bwd_partial_mla(qd, kc, vc, o, lse, dod, scale, scratch_acc, a32, b32, ws, prepared=True)
        dk32[:, :, lo:hi], dv32[:, :, lo:hi] = a32, b32
    dq = rx.ringx_dq_finalize_mla(acc, B, H, Nq)
    assert torch.equal(dk32.to(torch.bfloat16), dk16) and torch.equal(dv32.to(torch.bfloat16), dv16)
    check_grads(dq, dk16, dv16, q64, k64, v64, do64, scale)


@pytest.mark.parametrize("variant", ["a", "b"])
def test_mla_ringx_schedules_on_simulated_ranks(rx, variant):
    """RingX_a / RingX_b with the MLA kernels on W = 2 simulated ranks of 256 tokens, forward and
    backward, against the oracle attention of the whole sequence."""
    import threading
    from paper_2507_16697_b200 import ringx_dist
    from test_gpu_ringx_steps import ThreadComm
    world, Nl, B, H = 2, 256, 1, 2
    N = world * Nl
    scale = 1.0 / math.sqrt(DQK)
    q, k, v = make(B, H, N, seed=163)
    do = make_do(B, H, N, seed=163)
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
    rel = lambda a, r: np.linalg.norm(a - r) / np.linalg.norm(r)
    for r in range(world):
        sl = slice(r * Nl, (r + 1) * Nl)
        o, lse, dq, dk, dv = results[r]
        assert o.shape == (B, H, Nl, DV) and dq.shape == (B, H, Nl, DQK) and dq.dtype == torch.bfloat16
        assert rel(f64(o), o_ref[:, :, sl]) <= 1e-2 and np.abs(f64(lse) - lse_ref[:, :, sl]).max() <= 5e-5
        for g, ref in ((dq, dq_ref), (dk, dk_ref), (dv, dv_ref)):
            assert rel(f64(g), ref[:, :, sl]) <= 8e-3
