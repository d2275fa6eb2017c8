"""GPU parity at BASELINE.json's full sizes (C2..C5), in the launch configuration bench.py times.  The full
fp64 problem is 4e12..2e15 FLOPs, so the oracle is evaluated on sampled query rows of sampled heads against
ALL keys -- exact, because rows and heads are independent in non-causal attention -- plus
properties that hold at any size on the FULL GPU output (convex hull of V, LSE bounds, chunk independence).
Inputs are generated once on the GPU (same counter-based recipe) and the very same bits are copied to the
host for the oracle."""
import math

import numpy as np
import pytest
import torch

import grad_bounds as gb
from oracle import attention as orc
from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rx():
    from paper_2507_16697_b200 import ringx
    from paper_2507_16697_b200.build import build_library
    build_library()
    ringx.lib()
    return ringx


def sample_rows(N, n_random, seed):
    """Deliberate picks (tensor / 128-row tile / 256-row CTA boundaries) plus seeded random rows."""
    picks = [0, 1, 127, 128, 255, 256, 257, N // 2 - 1, N // 2, N - 257, N - 256, N - 129, N - 128, N - 1]
    rng = np.random.default_rng(seed)
    rows = sorted(set(picks) | set(rng.integers(0, N, n_random).tolist()))
    return np.array(rows)


def fwd_sampled_check(rx, cfg, heads, n_rows):
    q, k, v = wl.make_qkv(cfg, device="cuda")
    o, lse = rx.ringx_attn_fwd(q, k, v, cfg.kv_chunk, cfg.scale)
    torch.cuda.synchronize()
    n_c = cfg.N // cfg.kv_chunk
    assert rx.ringx_last_launch_count() == n_c        # one chunk kernel per pass; Eq. 5 is folded in its epilogue
    vmax = v.float().abs().max().item()
    worst = {"o": 0.0, "relf": 0.0, "lse": 0.0}
    for (b, h) in heads:
        rows = sample_rows(cfg.N, n_rows, seed=cfg.seed + 100 * b + h)
        k64, v64 = wl.to_f64_numpy(k[b, h]), wl.to_f64_numpy(v[b, h])
        q64 = wl.to_f64_numpy(q[b, h][rows])
        o_ref, lse_ref = orc.attention_fwd(q64, k64, v64, cfg.scale)
        og = o[b, h][rows].float().cpu().double().numpy()
        lg = lse[b, h][rows].cpu().double().numpy()
        worst["o"] = max(worst["o"], np.abs(og - o_ref).max())
        worst["relf"] = max(worst["relf"], np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref))
        worst["lse"] = max(worst["lse"], np.abs(lg - lse_ref).max())
        # LSE bounds from the definition: max_j s_ij <= LSE_i <= max_j s_ij + ln N
        smax = (cfg.scale * (q64 @ k64.T)).max(axis=1)
        assert np.all(lg >= smax - 1e-3) and np.all(lg <= smax + math.log(cfg.N) + 1e-3)
    assert worst["o"] <= 1e-2 * vmax, worst
    assert worst["relf"] <= 1e-2, worst
    assert worst["lse"] <= 1e-3, worst
    # full-output properties: finite, and O inside the per-column convex hull of V (up to bf16 rounding)
    assert torch.isfinite(o.float()).all() and torch.isfinite(lse).all()
    vmin_c = v.float().amin(dim=2, keepdim=True)
    vmax_c = v.float().amax(dim=2, keepdim=True)
    of = o.float()
    assert bool(((of >= vmin_c - 1e-2 * vmax) & (of <= vmax_c + 1e-2 * vmax)).all())
    return q, k, v, o, lse, worst


def test_C2_full_size(rx):
    cfg = wl.CONFIGS["C2"]
    q, k, v, o, lse, worst = fwd_sampled_check(rx, cfg, heads=[(0, 0), (0, 7), (0, 15)], n_rows=96)
    # chunk independence at full size: one pass (kv_chunk = N) agrees to bf16 rounding
    o1, lse1 = rx.ringx_attn_fwd(q, k, v, cfg.N, cfg.scale)
    assert (lse1 - lse).abs().max().item() <= 5e-5
    assert ((o1.float() - o.float()).norm() / o.float().norm()).item() <= 4e-3


def np64(t):
    return t.float().cpu().double().numpy()


def all_row_stats(q64, k64, v64, do64, scale, block=2048):
    """(LSE_i, D_i, E_i) of EVERY query row of a head from the oracle's forward (one full 4 N^2 d fp64 pass): what a
    key-column check of dK/dV needs.  D_i = dO_i . O_i (oracle.row_stats); E_i = 2^-9 sum_c |dO_ic| |O_ic| bounds the
    error of the kernel's D_i, which is formed from the saved bf16 O (tests/grad_bounds.py)."""
    N = q64.shape[0]
    lse, D, E = np.empty(N), np.empty(N), np.empty(N)
    for r0 in range(0, N, block):
        sl = slice(r0, r0 + block)
        o, lse[sl] = orc.attention_fwd(q64[sl], k64, v64, scale)
        D[sl] = (do64[sl] * o).sum(axis=1)
        E[sl] = gb.U_BF16 * (np.abs(do64[sl]) * np.abs(o)).sum(axis=1)
    return lse, D, E


def test_C3_full_size(rx):
    cfg = wl.CONFIGS["C3"]
    fwd_sampled_check(rx, cfg, heads=[(0, 0), (0, 5)], n_rows=64)


def test_C3_full_size_forward_and_backward(rx):
    """The configuration bench.py times (BASELINE.json configs[2] shape, fwd + bwd: B=1, H=8, N=262144, d=128,
    kv_chunk=32768), run exactly as bench.py runs it (ringx_attn_fwd then ringx_attn_bwd, caller-held workspaces).
    (1) dense dO, as in the bench: O, LSE, dQ on sampled query rows of two heads against ALL 262144 keys (exact per row);
        full-output invariants sum_j dV_j = sum_i dO_i, sum_j dK_j = 0 on every head.
    (2) sparse dO: dO is non-zero on 192 query rows only (spread over tile, CTA and chunk boundaries + random).  Rows
        with dO_i = 0 have dS_i = 0, so dK and dV of EVERY key of the head are sums over those 192 rows only -- which
        the oracle computes exactly in seconds.  The kernel still walks all 2048 query tiles with all 2048 key-tile CTAs
        of every pass, so every (key tile, chunk pass) of the d = 128 kernel is checked at full size, element by
        element, and dQ must be exactly zero outside the 192 rows."""
    cfg = wl.CONFIGS["C3"]
    B, H, N, d, C = cfg.B, cfg.H, cfg.N, cfg.d, cfg.kv_chunk
    q, k, v, do = wl.make_qkv(cfg, with_do=True, device="cuda")
    o = torch.empty_like(q)
    lse = torch.empty((B, H, N), dtype=torch.float32, device="cuda")
    ws_f = torch.empty(rx.ringx_attn_fwd_workspace_bytes(B, H, N, d, C, q.dtype), dtype=torch.uint8, device="cuda")
    ws_b = torch.empty(rx.ringx_attn_bwd_workspace_bytes(B, H, N, d, C, q.dtype), dtype=torch.uint8, device="cuda")
    rx.ringx_attn_fwd(q, k, v, C, cfg.scale, o=o, lse=lse, workspace=ws_f)
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do, C, cfg.scale, workspace=ws_b)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == N // C + 2
    for t in (dq, dk, dv):
        assert torch.isfinite(t.float()).all()
    heads = [(0, 2), (0, 7)]
    refs = []
    for (b, h) in heads:
        rows = sample_rows(N, 50, seed=cfg.seed + 7 * h)
        k64, v64 = wl.to_f64_numpy(k[b, h]), wl.to_f64_numpy(v[b, h])
        q64, do64 = wl.to_f64_numpy(q[b, h][rows]), wl.to_f64_numpy(do[b, h][rows])
        o_ref, lse_ref = orc.attention_fwd(q64, k64, v64, cfg.scale)
        dq_ref, _, _ = orc.attention_bwd(q64, k64, v64, do64, cfg.scale)
        og = np64(o[b, h][rows])
        assert np.abs(og - o_ref).max() <= 1e-2 * np.abs(v64).max()
        assert np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref) <= 1e-2
        assert np.abs(lse[b, h][rows].cpu().double().numpy() - lse_ref).max() <= 1e-3
        dterm = gb.dq_dterm(q64, k64, v64, do64, cfg.scale)
        gb.check_grad("dq", np64(dq[b, h][rows]), dq_ref, dterm)
        refs.append((b, h, rows, dq_ref, dterm))
    sum_dv, sum_do = dv.float().sum(dim=2), do.float().sum(dim=2)
    assert ((sum_dv - sum_do).norm() / sum_do.norm()).item() <= 1e-2
    assert (dk.float().sum(dim=2).norm() / dk.float().abs().sum(dim=2).norm()).item() <= 1e-2
    # ---- (1b) the same step with ringx_set_deterministic: dQ accumulated as int32 fixed point.  This shape is the worst
    # case for its resolution (diffuse rows over 262144 keys: |dQ| is ~2^-16 of the bound that sets the scale), so the
    # same element-wise bounds are checked here; two runs must agree bit for bit and dK, dV must not change at all.
    rx.ringx_set_deterministic(True)
    try:
        det = [rx.ringx_attn_bwd(q, k, v, o, lse, do, C, cfg.scale, workspace=ws_b) for _ in range(2)]
        torch.cuda.synchronize()
    finally:
        rx.ringx_set_deterministic(False)
    assert all(torch.equal(a, b_) for a, b_ in zip(det[0], det[1]))
    assert torch.equal(det[0][1], dk) and torch.equal(det[0][2], dv)
    for (b, h, rows, dq_ref, dterm) in refs:
        gb.check_grad("dq(deterministic)", np64(det[0][0][b, h][rows]), dq_ref, dterm)
    del dq, dk, dv, det
    # ---- (2) sparse dO: complete dK, dV of two heads, every key
    picks = [0, 127, 128, 255, 256, C - 1, C, 3 * C - 128, 3 * C + 5, N // 2 - 1, N // 2, N - C, N - 129, N - 128, N - 1]
    rows = np.array(sorted(set(picks) | set(np.random.default_rng(cfg.seed + 1).integers(0, N, 177).tolist())))
    idx = torch.from_numpy(rows).cuda()
    do_s = torch.zeros_like(do)
    do_s[:, :, idx] = do[:, :, idx]
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do_s, C, cfg.scale, workspace=ws_b)
    torch.cuda.synchronize()
    mask = torch.ones(N, dtype=torch.bool, device="cuda")
    mask[idx] = False
    assert not dq[:, :, mask].float().any()                     # dO_i = 0 => dQ_i = 0 exactly, every head
    for (b, h) in heads:
        k64, v64 = wl.to_f64_numpy(k[b, h]), wl.to_f64_numpy(v[b, h])
        q64, do64 = wl.to_f64_numpy(q[b, h][rows]), wl.to_f64_numpy(do[b, h][rows])
        dq_ref, dk_ref, dv_ref = orc.attention_bwd(q64, k64, v64, do64, cfg.scale)
        E = gb.d_error_rows(q64, k64, v64, do64, cfg.scale)
        _, lse_rows = orc.attention_fwd(q64, k64, v64, cfg.scale)
        gb.check_grad("dq(sparse)", np64(dq[b, h][rows]), dq_ref, gb.dq_dterm(q64, k64, v64, do64, cfg.scale))
        gb.check_grad("dk(all keys)", np64(dk[b, h]), dk_ref, gb.dk_dterm(q64, k64, lse_rows, E, cfg.scale))
        gb.check_grad("dv(all keys)", np64(dv[b, h]), dv_ref)


def test_C5_full_size_peaked(rx):
    cfg = wl.CONFIGS["C5"]
    q, k, v, o, lse, worst = fwd_sampled_check(rx, cfg, heads=[(0, 1), (0, 3)], n_rows=48)
    # the peaked config is the one where the stated O tolerance bites: |O| is O(1)
    assert o.float().abs().max().item() > 1.0


def test_voxel_order_is_metadata(rx):
    """C2's tokens are a 32^3 grid flattened x-fastest; any other flatten order is a joint permutation of the
    sequence axis and must give the permuted result (reading g15).  Checked on one head."""
    cfg = wl.CONFIGS["C2"]
    G = 32
    q, k, v = (t[:, :1].contiguous() for t in wl.make_qkv(cfg, device="cuda"))
    o, lse = rx.ringx_attn_fwd(q, k, v, cfg.kv_chunk, cfg.scale)
    idx = torch.tensor([wl.voxel_token_index(x, y, z, G) for x in range(G) for y in range(G) for z in range(G)],
                       device="cuda")            # z-fastest traversal expressed in x-fastest token ids
    assert idx[1].item() == G * G
    o2, lse2 = rx.ringx_attn_fwd(q[:, :, idx].contiguous(), k[:, :, idx].contiguous(), v[:, :, idx].contiguous(),
                                 cfg.kv_chunk, cfg.scale)
    assert (lse2 - lse[:, :, idx]).abs().max().item() <= 5e-5
    assert ((o2.float() - o.float()[:, :, idx]).norm() / o.float().norm()).item() <= 4e-3


def test_C4_full_size_forward_and_backward(rx):
    """BASELINE.json configs[3]: B=2,H=16,N=65536,d=64, kv_chunk=8192, fwd + bwd.  Oracle on sampled query rows
    (O, LSE, dQ -- exact per row) and on sampled key columns of one head (dK, dV -- needs LSE_i and D_i of ALL
    65536 rows of that head: one full 4*N^2*d fp64 pass), plus O(N d) invariants on the full GPU output."""
    cfg = wl.CONFIGS["C4"]
    q, k, v, do = wl.make_qkv(cfg, with_do=True, device="cuda")
    o, lse = rx.ringx_attn_fwd(q, k, v, cfg.kv_chunk, cfg.scale)
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do, cfg.kv_chunk, cfg.scale)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == cfg.N // cfg.kv_chunk + 2
    for t in (dq, dk, dv):
        assert torch.isfinite(t.float()).all()
    # ---- sampled rows: forward and dQ
    for (b, h) in [(0, 0), (1, 9)]:
        rows = sample_rows(cfg.N, 64, seed=cfg.seed + 100 * b + h)
        k64, v64 = wl.to_f64_numpy(k[b, h]), wl.to_f64_numpy(v[b, h])
        q64, do64 = wl.to_f64_numpy(q[b, h][rows]), wl.to_f64_numpy(do[b, h][rows])
        o_ref, lse_ref = orc.attention_fwd(q64, k64, v64, cfg.scale)
        dq_ref, _, _ = orc.attention_bwd(q64, k64, v64, do64, cfg.scale)
        og = o[b, h][rows].float().cpu().double().numpy()
        assert np.abs(og - o_ref).max() <= 1e-2 * np.abs(v64).max()
        assert np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref) <= 1e-2
        assert np.abs(lse[b, h][rows].cpu().double().numpy() - lse_ref).max() <= 1e-3
        gb.check_grad("dq", np64(dq[b, h][rows]), dq_ref, gb.dq_dterm(q64, k64, v64, do64, cfg.scale))
    # ---- sampled key columns of one head: dK, dV (tile / chunk boundaries + random)
    b, h = 1, 3
    q64, k64, v64, do64 = (wl.to_f64_numpy(t[b, h]) for t in (q, k, v, do))
    lse_all, D_all, E_all = all_row_stats(q64, k64, v64, do64, cfg.scale)
    assert np.abs(lse[b, h].cpu().double().numpy() - lse_all).max() <= 1e-3       # every row of the head
    C = cfg.kv_chunk
    cols = sorted(set([0, 127, 128, C - 1, C, C + 127, 3 * C - 1, 3 * C, cfg.N - 128, cfg.N - 1])
                  | set(np.random.default_rng(cfg.seed).integers(0, cfg.N, 54).tolist()))
    cols = np.array(cols)
    dk_ref, dv_ref = orc.attention_bwd_cols(q64, k64[cols], v64[cols], do64, lse_all, D_all, cfg.scale)
    dkg = dk[b, h][cols].float().cpu().double().numpy()
    dvg = dv[b, h][cols].float().cpu().double().numpy()
    gb.check_grad("dk(cols)", dkg, dk_ref, gb.dk_dterm(q64, k64[cols], lse_all, E_all, cfg.scale))
    gb.check_grad("dv(cols)", dvg, dv_ref)
    # ---- invariants on the full output (every head)
    sum_dv, sum_do = dv.float().sum(dim=2), do.float().sum(dim=2)
    assert ((sum_dv - sum_do).norm() / sum_do.norm()).item() <= 1e-2
    assert (dk.float().sum(dim=2).norm() / dk.float().abs().sum(dim=2).norm()).item() <= 1e-2


def test_C3_shape_backward_d128_sampled(rx):
    """d = 128 backward at a long sequence (one head of the C3 shape family, N = 65536): dQ rows vs the oracle."""
    B, H, N, d, chunk = 1, 2, 65536, 128, 16384
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=71, device="cuda")
    scale = 1.0 / math.sqrt(d)
    o, lse = rx.ringx_attn_fwd(q, k, v, chunk, scale)
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale)
    rows = sample_rows(N, 48, seed=5)
    k64, v64 = wl.to_f64_numpy(k[0, 1]), wl.to_f64_numpy(v[0, 1])
    dq_ref, _, _ = orc.attention_bwd(wl.to_f64_numpy(q[0, 1][rows]), k64, v64, wl.to_f64_numpy(do[0, 1][rows]), scale)
    gb.check_grad("dq", np64(dq[0, 1][rows]), dq_ref,
                  gb.dq_dterm(wl.to_f64_numpy(q[0, 1][rows]), k64, v64, wl.to_f64_numpy(do[0, 1][rows]), scale))
    sum_dv, sum_do = dv.float().sum(dim=2), do.float().sum(dim=2)
    assert ((sum_dv - sum_do).norm() / sum_do.norm()).item() <= 1e-2
    assert (dk.float().sum(dim=2).norm() / dk.float().abs().sum(dim=2).norm()).item() <= 1e-2
    # ---- dK, dV of the d = 128 kernel on sampled key columns, dense dO: needs LSE_i and D_i of ALL 65536 rows of the
    # head from the oracle (one full 4 N^2 d fp64 pass, ~2.2e12 FLOP), then the listed columns are cheap.  Columns at
    # key-tile and chunk boundaries plus random ones.
    b, h = 0, 0
    q64, k64, v64, do64 = (wl.to_f64_numpy(t[b, h]) for t in (q, k, v, do))
    lse_all, D_all, E_all = all_row_stats(q64, k64, v64, do64, scale)
    assert np.abs(lse[b, h].cpu().double().numpy() - lse_all).max() <= 1e-3       # every row of the head
    cols = sorted(set([0, 1, 127, 128, 129, chunk - 1, chunk, chunk + 127, 2 * chunk - 1, 2 * chunk, 3 * chunk + 64,
                       N - 129, N - 128, N - 1]) | set(np.random.default_rng(73).integers(0, N, 82).tolist()))
    cols = np.array(cols)
    dk_ref, dv_ref = orc.attention_bwd_cols(q64, k64[cols], v64[cols], do64, lse_all, D_all, scale)
    gb.check_grad("dk(cols)", np64(dk[b, h][cols]), dk_ref, gb.dk_dterm(q64, k64[cols], lse_all, E_all, scale))
    gb.check_grad("dv(cols)", np64(dv[b, h][cols]), dv_ref)


def test_C3_minus_one_token_ragged_full_size(rx):
    """C3's shape with one token fewer (N = 262143: every head ends one key short of a tile, the last of the 8 passes
    has 32767 keys).  Forward + backward at full size through the kTail instantiations: O, LSE, dQ on sampled rows
    (incl. the last rows of the ragged tile) against the oracle over all keys; the sum invariants on every head; then,
    with dO non-zero on the sampled rows only, dK and dV of every key of a head element by element."""
    cfg = wl.CONFIGS["C3"]
    B, H, N, d, C = cfg.B, cfg.H, cfg.N - 1, cfg.d, cfg.kv_chunk
    q, k, v, do = (wl.make_tensor((B, H, N, d), w, seed=cfg.seed + 3, dtype="bf16", device="cuda") for w in ("q", "k", "v", "do"))
    o, lse = rx.ringx_attn_fwd(q, k, v, C, cfg.scale)
    assert rx.ringx_last_launch_count() == 8
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do, C, cfg.scale)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == 8 + 3
    for t in (o, dq, dk, dv):
        assert torch.isfinite(t.float()).all()
    b, h = 0, 6
    rows = sample_rows(N, 180, seed=cfg.seed + 11)
    k64, v64 = wl.to_f64_numpy(k[b, h]), wl.to_f64_numpy(v[b, h])
    q64, do64 = wl.to_f64_numpy(q[b, h][rows]), wl.to_f64_numpy(do[b, h][rows])
    o_ref, lse_ref = orc.attention_fwd(q64, k64, v64, cfg.scale)
    dq_ref, _, _ = orc.attention_bwd(q64, k64, v64, do64, cfg.scale)
    og = np64(o[b, h][rows])
    assert np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref) <= 1e-2
    assert np.abs(lse[b, h][rows].cpu().double().numpy() - lse_ref).max() <= 1e-3
    gb.check_grad("dq", np64(dq[b, h][rows]), dq_ref, gb.dq_dterm(q64, k64, v64, do64, cfg.scale))
    sum_dv, sum_do = dv.float().sum(dim=2), do.float().sum(dim=2)
    assert ((sum_dv - sum_do).norm() / sum_do.norm()).item() <= 1e-2
    assert (dk.float().sum(dim=2).norm() / dk.float().abs().sum(dim=2).norm()).item() <= 1e-2
    del dq, dk, dv
    # sparse dO (as in test_C3_full_size_forward_and_backward): dO is non-zero on the sampled rows only, so dK, dV of EVERY key
    # are sums over those rows, which the oracle computes exactly -- all 2048 key tiles incl. the ragged one, element by element
    idx = torch.from_numpy(rows).cuda()
    do_s = torch.zeros_like(do)
    do_s[:, :, idx] = do[:, :, idx]
    dq, dk, dv = rx.ringx_attn_bwd(q, k, v, o, lse, do_s, C, cfg.scale)
    torch.cuda.synchronize()
    mask = torch.ones(N, dtype=torch.bool, device="cuda")
    mask[idx] = False
    assert not dq[:, :, mask].float().any()
    dq_ref, dk_ref, dv_ref = orc.attention_bwd(q64, k64, v64, do64, cfg.scale)
    E = gb.d_error_rows(q64, k64, v64, do64, cfg.scale)
    gb.check_grad("dq(sparse)", np64(dq[b, h][rows]), dq_ref, gb.dq_dterm(q64, k64, v64, do64, cfg.scale))
    gb.check_grad("dk(all keys)", np64(dk[b, h]), dk_ref, gb.dk_dterm(q64, k64, lse_ref, E, cfg.scale))
    gb.check_grad("dv(all keys)", np64(dv[b, h]), dv_ref)
