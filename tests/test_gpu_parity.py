"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 oracle on the
same seeded inputs, element by element.  Tolerances are BASELINE.json's (north_star):
  fp32 path  max|O - O_ref| <= 1e-5;   bf16  max|O - O_ref| <= 1e-2 * max|V|;   LSE <= 1e-3 abs;
  gradients  <= 2e-2 relative Frobenius error.
Because |O| is far below 1e-2*max|V| on the diffuse configs (an all-zero O would pass), every
bf16 check also imposes a scale-free bound: relative Frobenius error of O <= 1e-2 (expected ~2.3e-3: P and
the output are each rounded to bf16 once, unit roundoff 2^-8)."""
import math

import numpy as np
import pytest
import torch

import grad_bounds as gb
from oracle import attention as orc
from paper_2507_16697_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_F32_O = 1e-5
TOL_BF16_O_REL_V = 1e-2
TOL_LSE = 1e-3
TOL_GRAD = 2e-2
TOL_BF16_O_RELF = 1e-2     # self-imposed, scale-free


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


def check_fwd(o, lse, o_ref, lse_ref, v64, dtype):
    og = o.float().cpu().double().numpy()
    lg = lse.cpu().double().numpy()
    err_o = np.abs(og - o_ref).max()
    err_l = np.abs(lg - lse_ref).max()
    assert np.isfinite(og).all() and np.isfinite(lg).all()
    if dtype == "f32":
        assert err_o <= TOL_F32_O, err_o
        assert err_l <= 1e-5, err_l
    else:
        assert err_o <= TOL_BF16_O_REL_V * np.abs(v64).max(), err_o
        relf = np.linalg.norm(og - o_ref) / np.linalg.norm(o_ref)
        assert relf <= TOL_BF16_O_RELF, relf
        assert err_l <= TOL_LSE, err_l
        assert err_l <= 5e-5, err_l          # fp32 row sums: far tighter than the stated bar


# ------------------------------------------------------------------------------------------------
# ringx_lse_merge (Eq. 5, two operands)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rows,d", [(1, 8), (7, 64), (1000, 64), (4099, 128), (333, 24), (65, 1024), (5000, 256)])
@pytest.mark.parametrize("in_dt,out_dt", [("f32", "f32"), ("f32", "bf16"), ("bf16", "bf16"), ("bf16", "f32")])
def test_merge_matches_oracle(rx, rows, d, in_dt, out_dt):
    tdt = {"f32": torch.float32, "bf16": torch.bfloat16}
    g = torch.Generator().manual_seed(rows * 131 + d)
    o_a = torch.randn(rows, d, generator=g).to(tdt[in_dt])
    o_b = torch.randn(rows, d, generator=g).to(tdt[in_dt])
    lse_a = torch.randn(rows, generator=g) * 5
    lse_b = torch.randn(rows, generator=g) * 5
    o, lse = rx.ringx_lse_merge(o_a.cuda(), lse_a.cuda(), o_b.cuda(), lse_b.cuda(), out_dtype=tdt[out_dt])
    o_ref, lse_ref = orc.lse_merge(f64(o_a), f64(lse_a), f64(o_b), f64(lse_b))
    tol = 2e-6 * max(1.0, np.abs(o_ref).max()) if out_dt == "f32" else 2 ** -8 * np.abs(o_ref).max()
    assert np.abs(o.float().cpu().double().numpy() - o_ref).max() <= tol
    assert np.abs(lse.cpu().double().numpy() - lse_ref).max() <= 2e-6 * max(1.0, np.abs(lse_ref).max())


def test_merge_degenerate_operands(rx):
    """-inf operands get weight 0 even if the o behind them is garbage; both -inf -> (0, -inf); rows=0 no-op;
    merge with itself adds ln 2 (SURVEY.md §8c pins; reading g12)."""
    rows, d = 64, 64
    g = torch.Generator().manual_seed(5)
    o_a = torch.randn(rows, d, generator=g)
    o_b = torch.randn(rows, d, generator=g)
    lse_a = torch.randn(rows, generator=g)
    lse_b = torch.randn(rows, generator=g)
    lse_b[:16] = -math.inf
    o_b[:8] = float("nan")               # garbage behind an empty chunk must be ignored
    lse_a[16:32] = -math.inf
    lse_a[60:] = -math.inf
    lse_b[60:] = -math.inf
    o, lse = rx.ringx_lse_merge(o_a.cuda(), lse_a.cuda(), o_b.cuda(), lse_b.cuda())
    o, lse = o.cpu(), lse.cpu()
    assert torch.equal(o[:16], o_a[:16]) and torch.equal(lse[:16], lse_a[:16])
    assert torch.equal(o[16:32], o_b[16:32]) and torch.equal(lse[16:32], lse_b[16:32])
    assert torch.all(o[60:] == 0) and torch.all(lse[60:] == -math.inf)
    o_ref, lse_ref = orc.lse_merge(f64(o_a[32:60]), f64(lse_a[32:60]), f64(o_b[32:60]), f64(lse_b[32:60]))
    assert np.abs(o[32:60].double().numpy() - o_ref).max() <= 1e-5
    # self-merge: (o, lse + ln 2)
    o2, lse2 = rx.ringx_lse_merge(o_a.cuda(), lse_a.cuda(), o_a.cuda(), lse_a.cuda())
    fin = torch.isfinite(lse_a)
    assert torch.allclose(o2.cpu()[fin], o_a[fin], atol=1e-6)
    assert torch.allclose(lse2.cpu()[fin], lse_a[fin] + math.log(2.0), atol=1e-6)
    # rows == 0
    e = torch.empty(0, d, device="cuda")
    el = torch.empty(0, device="cuda")
    o0, _ = rx.ringx_lse_merge(e, el, e, el)
    assert o0.numel() == 0 and rx.ringx_last_launch_count() == 0
    # NaN propagates
    lse_n = lse_a.clone()
    lse_n[40] = float("nan")
    _, lse3 = rx.ringx_lse_merge(o_a.cuda(), lse_n.cuda(), o_b.cuda(), lse_b.cuda())
    assert math.isnan(lse3[40].item())


def test_merge_in_place_and_any_fold_order(rx):
    """Running left fold in place on operand a == one Eq. 5 over all chunks (associativity)."""
    rows, d, n = 777, 128, 5
    g = torch.Generator().manual_seed(9)
    outs = [torch.randn(rows, d, generator=g) for _ in range(n)]
    lses = [torch.randn(rows, generator=g) * 3 for _ in range(n)]
    o_ref, lse_ref = orc.merge_partials([f64(o) for o in outs], [f64(l) for l in lses])
    acc_o, acc_l = outs[0].cuda().clone(), lses[0].cuda().clone()
    for ob, lb in zip(outs[1:], lses[1:]):
        r_o, r_l = rx.ringx_lse_merge(acc_o, acc_l, ob.cuda(), lb.cuda(), inplace=True)
        assert r_o.data_ptr() == acc_o.data_ptr()
    assert np.abs(acc_o.cpu().double().numpy() - o_ref).max() <= 1e-5
    assert np.abs(acc_l.cpu().double().numpy() - lse_ref).max() <= 1e-5
    # reverse order
    acc_o, acc_l = outs[-1].cuda().clone(), lses[-1].cuda().clone()
    for ob, lb in zip(outs[-2::-1], lses[-2::-1]):
        rx.ringx_lse_merge(acc_o, acc_l, ob.cuda(), lb.cuda(), inplace=True)
    assert np.abs(acc_o.cpu().double().numpy() - o_ref).max() <= 1e-5


# ------------------------------------------------------------------------------------------------
# forward: fp32 path (config C1) and bf16 tcgen05 path at oracle-sized shapes
# ------------------------------------------------------------------------------------------------
def test_fwd_C1_fp32(rx):
    """BASELINE.json configs[0]: B=1,H=1,N=1024,d=64, 4 chunks of 256 merged by LSE; max abs err <= 1e-5."""
    cfg = wl.CONFIGS["C1"]
    q, k, v = wl.make_qkv(cfg)
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), cfg.kv_chunk, cfg.scale)
    assert rx.ringx_last_launch_count() == 4 + 3
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), cfg.scale)
    check_fwd(o, lse, o_ref, lse_ref, f64(v), "f32")


@pytest.mark.parametrize("B,H,N,d,chunk", [(1, 2, 512, 128, 128), (2, 1, 384, 64, 128), (1, 1, 128, 64, 128)])
def test_fwd_fp32_shapes(rx, B, H, N, d, chunk):
    q, k, v = wl.make_qkv((B, H, N, d), seed=3, dtype="f32")
    scale = 1.0 / math.sqrt(d)
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), chunk, scale)
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    check_fwd(o, lse, o_ref, lse_ref, f64(v), "f32")


BF16_SHAPES = [
    # B, H, N, d, kv_chunk, qk_gain        (several 256-row CTA tiles, ragged KV-tile counts, 1..16 passes)
    (1, 1, 256, 64, 256, 1.0),             # minimum size, single pass, one KV... two KV tiles
    (1, 1, 256, 128, 128, 1.0),            # two passes of one KV tile each
    (2, 3, 1280, 64, 256, 1.0),            # 5 passes, 5 CTAs per head
    (1, 2, 2304, 128, 768, 1.0),           # 3 passes of 6 KV tiles (ring wraps: 5 slots)
    (1, 2, 2048, 64, 2048, 1.0),           # single pass, 16 KV tiles (ring wraps: 8 slots)
    (1, 2, 2048, 128, 128, 3.0),           # 16 passes, peaked softmax (C5-like gain on Q and K)
    (1, 1, 4096, 128, 1024, 3.0),
    (1, 4, 1024, 64, 512, 0.05),           # nearly uniform softmax
]


@pytest.mark.parametrize("B,H,N,d,chunk,gain", BF16_SHAPES)
def test_fwd_bf16_matches_oracle(rx, B, H, N, d, chunk, gain):
    q, k, v = (wl.make_tensor((B, H, N, d), w, seed=17, dtype="bf16", gain=(gain if w != "v" else 1.0)) for w in "qkv")
    scale = 1.0 / math.sqrt(d)
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), chunk, scale)
    n_c = N // chunk
    # bf16: the Eq. 5 fold runs in the chunk kernel's epilogue; a pass too small to fill the GPU is split over the keys
    # (split-KV) and costs one more launch, the Eq. 5 kernel over the splits
    split = rx.ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, N, chunk, d, torch.bfloat16) > 0
    assert rx.ringx_last_launch_count() == n_c * (2 if split else 1)
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    check_fwd(o, lse, o_ref, lse_ref, f64(v), "bf16")


RAGGED_SHAPES = [
    # B, H, N, d, kv_chunk, qk_gain: sequence lengths that are no multiple of the 128-key / 256-row tiles
    (1, 1, 1, 64, 128, 1.0),               # one token: O = V, LSE = scale q.k
    (1, 2, 100, 128, 128, 1.0),            # less than one tile
    (1, 1, 257, 64, 128, 1.0),             # one row and one key past two tiles, 3 passes (the last of one key)
    (2, 3, 1000, 64, 256, 1.0),            # 4 passes, the last one 232 keys (one full and one ragged tile)
    (1, 2, 1337, 128, 512, 3.0),           # peaked softmax; last pass 313 keys
    (1, 2, 640, 128, 256, 1.0),            # N % 128 == 0 but not % 256: the second query tile of the last item is empty
    (1, 2, 2049, 64, 2176, 1.0),           # single pass of 17 key tiles, the last with one key
    (1, 1, 3000, 128, 3072, 0.05),         # single pass, nearly uniform softmax
]


@pytest.mark.parametrize("B,H,N,d,chunk,gain", RAGGED_SHAPES)
def test_fwd_bf16_ragged_lengths_match_oracle(rx, B, H, N, d, chunk, gain):
    """Any sequence length: tiles that run past the end of a head read zeros (3-D tensor maps), the keys past the end
    are masked to -inf in the pass's last key tile, rows past the end are never stored.  The tensors sit in the middle
    of a sentinel-filled buffer so that a store past the end of a head (into the next head or past the tensor) shows."""
    q, k, v = (wl.make_tensor((B, H, N, d), w, seed=19, dtype="bf16", gain=(gain if w != "v" else 1.0)) for w in "qkv")
    scale = 1.0 / math.sqrt(d)
    guard_o = torch.full((B * H * N * d + 4096,), 555.0, dtype=torch.bfloat16, device="cuda")
    o = guard_o[2048:2048 + B * H * N * d].view(B, H, N, d)
    guard_l = torch.full((B * H * N + 2048,), 555.0, dtype=torch.float32, device="cuda")
    lse = guard_l[1024:1024 + B * H * N].view(B, H, N)
    rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), chunk, scale, o=o, lse=lse)
    torch.cuda.synchronize()
    assert rx.ringx_last_launch_count() == -(-N // chunk)
    assert (guard_o[:2048] == 555.0).all() and (guard_o[2048 + B * H * N * d:] == 555.0).all()
    assert (guard_l[:1024] == 555.0).all() and (guard_l[1024 + B * H * N:] == 555.0).all()
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    check_fwd(o, lse, o_ref, lse_ref, f64(v), "bf16")


def test_fwd_bf16_chunk_partials_and_merge_are_the_papers_quantities(rx):
    """ringx_attn_chunk_fwd returns (loc_out_i, loc_lse_i) of PAPER.md:135 with Nq != Nk; merging them with
    ringx_lse_merge reproduces the oracle's Eq. 5 result."""
    B, H, Nq, Nk, d = 1, 2, 512, 768, 128
    q = wl.make_tensor((B, H, Nq, d), "q", seed=23)
    k = wl.make_tensor((B, H, Nk, d), "k", seed=23)
    v = wl.make_tensor((B, H, Nk, d), "v", seed=23)
    scale = 0.1
    bounds = [0, 256, 768]
    parts = []
    for lo, hi in zip(bounds[:-1], bounds[1:]):
        lo_o, lo_l = rx.ringx_attn_chunk_fwd(q.cuda(), k[:, :, lo:hi].contiguous().cuda(),
                                             v[:, :, lo:hi].contiguous().cuda(), scale)
        parts.append((lo_o, lo_l))
        for h in range(H):
            outs, lses = orc.chunk_partials(f64(q[0, h]), f64(k[0, h]), f64(v[0, h]), scale, bounds)
            i = len(parts) - 1
            assert np.abs(lo_l[0, h].cpu().double().numpy() - lses[i]).max() <= 5e-5
            rel = np.linalg.norm(lo_o[0, h].cpu().double().numpy() - outs[i]) / np.linalg.norm(outs[i])
            assert rel <= 5e-3, rel
    o, lse = rx.ringx_lse_merge(parts[0][0], parts[0][1], parts[1][0], parts[1][1], out_dtype=torch.bfloat16)
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    check_fwd(o, lse, o_ref, lse_ref, f64(v), "bf16")


def test_fwd_bf16_result_is_independent_of_kv_chunk(rx):
    """Several results are correct up to rounding (reading g5): every chunking agrees to bf16 rounding."""
    B, H, N, d = 1, 2, 2048, 128
    q, k, v = wl.make_qkv((B, H, N, d), seed=29)
    qd, kd, vd = q.cuda(), k.cuda(), v.cuda()
    scale = 1.0 / math.sqrt(d)
    o_ref, lse_ref = rx.ringx_attn_fwd(qd, kd, vd, N, scale)
    for chunk in (128, 256, 512, 1024):
        o, lse = rx.ringx_attn_fwd(qd, kd, vd, chunk, scale)
        assert (lse - lse_ref).abs().max().item() <= 2e-5
        rel = ((o.float() - o_ref.float()).norm() / o_ref.float().norm()).item()
        assert rel <= 4e-3, (chunk, rel)


def test_fwd_bf16_one_hot_v_reads_P(rx):
    """V = identity block over d chosen keys => O[:, c] = P[:, key(c)]: checks individual probabilities,
    which localises any tile-layout / swizzle / transposition error."""
    B, H, N, d = 1, 1, 512, 64
    q, k, _ = wl.make_qkv((B, H, N, d), seed=31)
    keys = np.array([0, 1, 63, 64, 127, 128, 129, 255, 256, 300, 383, 384, 450, 500, 510, 511] * 4)[:d]
    keys = (keys + np.arange(d) // 16 * 3) % N
    keys = np.unique(keys)
    v = torch.zeros(B, H, N, d, dtype=torch.bfloat16)
    for c, j in enumerate(keys):
        v[0, 0, j, c] = 1.0
    scale = 0.35
    o, _ = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), 256, scale)
    P = orc.softmax_probs(f64(q[0, 0]), f64(k[0, 0]), scale)
    og = o[0, 0].float().cpu().double().numpy()
    for c, j in enumerate(keys):
        assert np.abs(og[:, c] - P[:, j]).max() <= 2 ** -7 * max(P[:, j].max(), 1e-3) + 1e-6, (c, j)   # two bf16 roundings
    assert np.abs(og[:, len(keys):]).max() == 0.0


def test_fwd_closed_forms(rx):
    """Identical keys => O = mean(V), LSE = s + ln N;  Q = 0 => same with s = 0."""
    B, H, N, d = 1, 1, 512, 64
    q, _, v = wl.make_qkv((B, H, N, d), seed=37)
    k1 = wl.make_tensor((1, 1, 1, d), "k", seed=37)
    k = k1.expand(B, H, N, d).contiguous()
    scale = 0.125
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), 128, scale)
    mean_v = f64(v)[0, 0].mean(axis=0)
    s = scale * f64(q)[0, 0] @ f64(k1)[0, 0, 0]
    assert np.abs(o[0, 0].float().cpu().double().numpy() - mean_v[None, :]).max() <= 2 ** -8 * np.abs(mean_v).max() + 1e-4
    assert np.abs(lse[0, 0].cpu().double().numpy() - (s + math.log(N))).max() <= 1e-4
    q0 = torch.zeros_like(q)
    o, lse = rx.ringx_attn_fwd(q0.cuda(), wl.make_tensor((B, H, N, d), "k", seed=38).cuda(), v.cuda(), 256, scale)
    assert np.abs(o[0, 0].float().cpu().double().numpy() - mean_v[None, :]).max() <= 2 ** -8 * np.abs(mean_v).max() + 1e-4
    assert np.abs(lse.cpu().double().numpy() - math.log(N)).max() <= 1e-5


def test_fwd_large_magnitude_scores_do_not_overflow(rx):
    """Row maxima that keep growing across KV tiles exercise the lazy-rescale branch on every tile."""
    B, H, N, d = 1, 1, 1024, 64
    q, k, v = wl.make_qkv((B, H, N, d), seed=41)
    ramp = torch.linspace(0.2, 6.0, N).view(1, 1, N, 1)
    k = (k.float() * ramp).to(torch.bfloat16)         # later keys have larger norms
    scale = 1.0
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), 512, scale)
    o_ref, lse_ref = orc.attention_fwd_bhnd(f64(q), f64(k), f64(v), scale)
    og = o.float().cpu().double().numpy()
    assert np.isfinite(og).all()
    assert np.abs(og - o_ref).max() <= TOL_BF16_O_REL_V * np.abs(f64(v)).max()
    assert np.abs(lse.cpu().double().numpy() - lse_ref).max() <= TOL_LSE


def test_fwd_permutation_invariances(rx):
    """Jointly permuting (K,V) rows leaves (O,LSE) unchanged, and permuting Q rows permutes the outputs, both up
    to rounding (the lazy running max is decided per warp of 32 rows, so a row's rounding depends on its
    neighbours) -- the voxel flatten order is metadata only (reading g15)."""
    B, H, N, d = 1, 1, 1024, 128
    q, k, v = wl.make_qkv((B, H, N, d), seed=43)
    scale = 1.0 / math.sqrt(d)
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), 256, scale)
    g = torch.Generator().manual_seed(1)
    pq = torch.randperm(N, generator=g)
    o2, lse2 = rx.ringx_attn_fwd(q[:, :, pq].contiguous().cuda(), k.cuda(), v.cuda(), 256, scale)
    assert (lse2.cpu() - lse.cpu()[:, :, pq]).abs().max().item() <= 2e-5
    assert ((o2.cpu().float() - o.cpu().float()[:, :, pq]).norm() / o.float().norm()).item() <= 4e-3
    pk = torch.randperm(N, generator=g)
    o3, lse3 = rx.ringx_attn_fwd(q.cuda(), k[:, :, pk].contiguous().cuda(), v[:, :, pk].contiguous().cuda(), 256, scale)
    assert (lse3 - lse).abs().max().item() <= 2e-5
    assert ((o3.float() - o.float()).norm() / o.float().norm()).item() <= 4e-3


@pytest.mark.parametrize("B,H,N,d,chunk", [(1, 2, 1024, 64, 256), (2, 2, 900, 128, 256)])
def test_fwd_host_entry_matches_device_entry(rx, B, H, N, d, chunk):
    q, k, v = wl.make_qkv((B, H, N, d), seed=47)
    scale = 0.125
    o, lse = rx.ringx_attn_fwd(q.cuda(), k.cuda(), v.cuda(), chunk, scale)
    oh, lh = rx.ringx_attn_fwd_host(q.pin_memory(), k.pin_memory(), v.pin_memory(), chunk, scale)
    assert torch.equal(oh, o.cpu()) and torch.equal(lh, lse.cpu())


def test_errors_on_the_gpu_box(rx):
    q = torch.zeros(1, 1, 512, 64, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_attn_fwd(q, q, q, 200, 0.125)            # kv_chunk must be a multiple of the 128-key tile
    assert e.value.status == 2
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_attn_fwd(q, q, q, 640, 0.125)            # ... and no longer than the sequence rounded up to a tile
    assert e.value.status == 2
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_attn_fwd(q, q, q, 256, 0.125, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 5
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_attn_fwd(q, q, q, 256, -1.0)
    assert e.value.status == 2


# ------------------------------------------------------------------------------------------------
# backward: dQ, dK, dV against the oracle's derivative of the definition (reading g8)
# ------------------------------------------------------------------------------------------------
def rel_f(g, ref):
    return np.linalg.norm(g.float().cpu().double().numpy() - ref) / np.linalg.norm(ref)


def to64(t):
    return t.float().cpu().double().numpy()


def check_grads_full(dq, dk, dv, q64, k64, v64, do64, scale, refs=None):
    """dq, dk, dv [B,H,N,d] (GPU) against the oracle, head by head: stated Frobenius tolerance and the element-wise
    bound of tests/grad_bounds.py (with the D_i-from-bf16-O terms).  Returns the worst Frobenius error per tensor."""
    dq_ref, dk_ref, dv_ref = refs if refs is not None else orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
    worst = {"dq": 0.0, "dk": 0.0, "dv": 0.0}
    B, H = q64.shape[:2]
    for b in range(B):
        for h in range(H):
            q_, k_, v_, do_ = q64[b, h], k64[b, h], v64[b, h], do64[b, h]
            E = gb.d_error_rows(q_, k_, v_, do_, scale)
            _, lse = orc.attention_fwd(q_, k_, v_, scale)
            dqD = gb.dq_dterm(q_, k_, v_, do_, scale)
            dkD = gb.dk_dterm(q_, k_, lse, E, scale)
            worst["dq"] = max(worst["dq"], gb.check_grad("dq", to64(dq[b, h]), dq_ref[b, h], dqD, TOL_GRAD))
            worst["dk"] = max(worst["dk"], gb.check_grad("dk", to64(dk[b, h]), dk_ref[b, h], dkD, TOL_GRAD))
            worst["dv"] = max(worst["dv"], gb.check_grad("dv", to64(dv[b, h]), dv_ref[b, h], None, TOL_GRAD))
    return worst


BWD_SHAPES = [
    # B, H, N, d, kv_chunk, qk_gain
    (1, 1, 128, 64, 128, 1.0),             # one tile pair: minimum size (backward needs N % 128 only)
    (1, 1, 256, 128, 256, 1.0),
    (2, 2, 1152, 64, 384, 1.0),            # 9 query tiles (ring of 3 wraps), 3 passes of 3 key tiles
    (1, 2, 1280, 128, 256, 1.0),           # d = 128: dQ overlays dP^T in TMEM, ring of 2
    (1, 1, 2048, 64, 2048, 3.0),           # peaked softmax, single pass
    (1, 2, 1024, 128, 128, 3.0),           # 8 passes
    (1, 1, 1024, 64, 512, 0.05),           # nearly uniform softmax
]


@pytest.mark.parametrize("B,H,N,d,chunk,gain", BWD_SHAPES)
def test_bwd_bf16_matches_oracle(rx, B, H, N, d, chunk, gain):
    q, k, v, do = (wl.make_tensor((B, H, N, d), w, seed=53, dtype="bf16", gain=(gain if w in "qk" else 1.0))
                   for w in ("q", "k", "v", "do"))
    scale = 1.0 / math.sqrt(d)
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, chunk, scale)
    dq, dk, dv = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale)
    assert rx.ringx_last_launch_count() == N // chunk + 2
    worst = check_grads_full(dq, dk, dv, f64(q), f64(k), f64(v), f64(do), scale)
    assert max(worst.values()) <= 8e-3, worst        # expected ~2.4e-3 (bf16 P, dS and outputs); 5e-3 when peaked


BWD_RAGGED_SHAPES = [
    # B, H, N, d, kv_chunk, qk_gain: sequence lengths that are no multiple of the 128-row tile
    (1, 1, 1, 64, 128, 1.0),               # one token: dq = dk = 0, dv = dO
    (1, 2, 100, 128, 128, 1.0),            # less than one tile
    (1, 1, 257, 64, 128, 1.0),             # one row and one key past two tiles; the last pass has one key
    (2, 3, 1000, 64, 256, 1.0),            # 4 passes, the last one 232 keys
    (1, 2, 1337, 128, 512, 3.0),           # peaked softmax
    (1, 2, 2049, 128, 2176, 1.0),          # single pass of 17 key tiles, the last with one key
]


@pytest.mark.parametrize("B,H,N,d,chunk,gain", BWD_RAGGED_SHAPES)
def test_bwd_bf16_ragged_lengths_match_oracle(rx, B, H, N, d, chunk, gain):
    """Forward + backward of any sequence length: query rows and keys past the end of a head are read as zeros, get
    P = 0 (lse2 = +inf in the padding of the per-head statistics; a select on the key rows of the ragged key tile) and
    are neither stored nor reduce-added.  Gradients sit in sentinel-guarded buffers; the default and the deterministic
    mode (fixed-point dQ) are both checked element by element."""
    q, k, v, do = (wl.make_tensor((B, H, N, d), w, seed=59, dtype="bf16", gain=(gain if w in "qk" else 1.0))
                   for w in ("q", "k", "v", "do"))
    scale = 1.0 / math.sqrt(d)
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, chunk, scale)
    n = B * H * N * d
    refs = orc.attention_bwd_bhnd(f64(q), f64(k), f64(v), f64(do), scale)
    for det in (False, True):
        guards = [torch.full((n + 4096,), 555.0, dtype=torch.bfloat16, device="cuda") for _ in range(3)]
        dq, dk, dv = (g[2048:2048 + n].view(B, H, N, d) for g in guards)
        rx.ringx_set_deterministic(det)
        try:
            rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale, dq=dq, dk=dk, dv=dv)
            torch.cuda.synchronize()
            assert rx.ringx_last_launch_count() == -(-N // chunk) + 2 + (1 if N % 128 else 0) + (2 if det else 0)
            if det:
                dq2, _, _ = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale)
                assert torch.equal(dq2, dq)
        finally:
            rx.ringx_set_deterministic(False)
        for g in guards:
            assert (g[:2048] == 555.0).all() and (g[2048 + n:] == 555.0).all()
        if N == 1:
            assert not dq.float().any() and not dk.float().any() and torch.equal(dv, dod)
        else:
            check_grads_full(dq, dk, dv, f64(q), f64(k), f64(v), f64(do), scale, refs=refs)


@pytest.mark.parametrize("d", [64, 128])
def test_bwd_one_hot_probe_reads_single_P_and_dS(rx, d):
    """The backward twin of test_fwd_bf16_one_hot_v_reads_P.  dO has ONE non-zero row per probe, a unit vector e_c, so
    dV[j, c] = P[i_c, j]: a single probability lands in a single output element, for every key j -- a swizzle, tile
    or transposition error in S^T / P^T / dV cannot hide in a norm.  V has unit rows at chosen keys, so that
    dS[i_c, j] = P[i_c, j] (V[j, c] - O[i_c, c]) is read back through dQ[i_c, :] = scale * sum_j dS[i_c, j] K[j, :] with
    K = unit vectors as well (dQ[i_c, m] = scale * sum_{j: key j has unit m} dS[i_c, j]) and through
    dK[j, :] = scale * sum_c dS[i_c, j] Q[i_c, :].  Compared element by element with the oracle."""
    B, H, N = 1, 1, 512
    rows = np.array([0, 1, 31, 32, 127, 128, 129, 255, 256, 300, 383, 384, 450, 509, 510, 511])   # query rows probed
    cols = (np.arange(len(rows)) * 5 + 3) % d                                                    # distinct columns c
    assert len(set(cols.tolist())) == len(rows)
    q = wl.make_tensor((B, H, N, d), "q", seed=83)
    do = torch.zeros(B, H, N, d, dtype=torch.bfloat16)
    for i, c in zip(rows, cols):
        do[0, 0, i, c] = 1.0
    g = torch.Generator().manual_seed(7)
    # K: every key is a signed unit vector (so scores are single elements of q, well spread); V likewise
    kk = torch.zeros(B, H, N, d)
    vv = torch.zeros(B, H, N, d)
    ku = torch.randint(0, d, (N,), generator=g)
    vu = torch.randint(0, d, (N,), generator=g)
    kk[0, 0, torch.arange(N), ku] = (torch.randint(0, 2, (N,), generator=g) * 2 - 1).float() * 2.0
    vv[0, 0, torch.arange(N), vu] = 1.0
    k, v = kk.to(torch.bfloat16), vv.to(torch.bfloat16)
    scale = 0.5
    q64, k64, v64, do64 = f64(q), f64(k), f64(v), f64(do)
    o64, lse64 = orc.attention_fwd_bhnd(q64, k64, v64, scale)
    # (o, lse) from the oracle (rounded as the forward would), so that this test probes the backward alone
    o, lse = torch.from_numpy(o64).to(torch.bfloat16).cuda(), torch.from_numpy(lse64).float().cuda()
    for chunk in (N, 128):
        dq, dk, dv = rx.ringx_attn_bwd(q.cuda(), k.cuda(), v.cuda(), o, lse, do.cuda(), chunk, scale)
        P = orc.softmax_probs(q64[0, 0], k64[0, 0], scale)
        dvg = dv[0, 0].float().cpu().double().numpy()
        for i, c in zip(rows, cols):
            ref = P[i]                                        # dV[:, c] = P[i_c, :]
            assert np.abs(dvg[:, c] - ref).max() <= 2 ** -7 * ref.max() + 1e-7, ("dV", chunk, i, c)
        untouched = np.setdiff1d(np.arange(d), cols)
        assert np.abs(dvg[:, untouched]).max() == 0.0         # columns no probe wrote stay exactly zero
        dq_ref, dk_ref, dv_ref = orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
        dqg = dq[0, 0].float().cpu().double().numpy()
        others = np.setdiff1d(np.arange(N), rows)
        assert np.abs(dqg[others]).max() == 0.0               # dO_i = 0 => dS_i = 0 => dQ_i = 0 exactly
        # element by element: bf16 roundings of P, dS and of the output; the D_i the kernel uses comes from bf16 O
        for name, gg, rr in (("dq", dqg[rows], dq_ref[0, 0][rows]), ("dk", dk[0, 0].float().cpu().double().numpy(), dk_ref[0, 0])):
            tol = 2 ** -6 * np.abs(rr) + 2 ** -7 * np.abs(rr).max()
            assert (np.abs(gg - rr) <= tol).all(), (name, chunk, float((np.abs(gg - rr) / tol).max()))


def test_bwd_is_independent_of_kv_chunk_and_repeatable_within_rounding(rx):
    """dK/dV of a key tile are written once by one CTA -> bit-identical across chunkings; dQ is an fp32
    reduce-add in arbitrary order -> equal up to fp32 rounding before the final bf16 cast."""
    B, H, N, d = 1, 2, 1024, 64
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=59)
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    scale = 0.125
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, N, scale)
    ref = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, N, scale)
    for chunk in (128, 256, 512):
        dq, dk, dv = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale)
        assert torch.equal(dk, ref[1]) and torch.equal(dv, ref[2])
        assert ((dq.float() - ref[0].float()).norm() / ref[0].float().norm()).item() <= 2e-3


def test_bwd_invariants_and_degenerate_dO(rx):
    """sum_j dV_j = sum_i dO_i; sum_j dK_j = 0; dO = 0 => all gradients 0; linear in dO."""
    B, H, N, d = 1, 2, 1024, 64
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=61)
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    scale = 0.125
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, 256, scale)
    dq, dk, dv = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, 256, scale)
    sum_dv = dv.float().sum(dim=2)
    sum_do = dod.float().sum(dim=2)
    assert ((sum_dv - sum_do).norm() / sum_do.norm()).item() <= 1e-2
    assert (dk.float().sum(dim=2).norm() / dk.float().abs().sum(dim=2).norm()).item() <= 1e-2
    z = torch.zeros_like(dod)
    dq0, dk0, dv0 = rx.ringx_attn_bwd(qd, kd, vd, o, lse, z, 256, scale)
    assert not dq0.float().any() and not dk0.float().any() and not dv0.float().any()
    dq2, dk2, dv2 = rx.ringx_attn_bwd(qd, kd, vd, o, lse, (dod.float() * 2).to(torch.bfloat16), 256, scale)
    for a, b_ in ((dq2, dq), (dk2, dk), (dv2, dv)):
        assert ((a.float() - 2 * b_.float()).norm() / (2 * b_.float()).norm()).item() <= 5e-3


def test_bwd_errors(rx):
    q = torch.zeros(1, 1, 256, 64, dtype=torch.float32, device="cuda")
    lse = torch.zeros(1, 1, 256, device="cuda")
    with pytest.raises(KeyError):
        rx.ringx_attn_bwd(q.half(), q.half(), q.half(), q.half(), lse, q.half(), 256, 0.125)   # fp16 unsupported
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_attn_bwd(q, q, q, q, lse, q, 256, 0.125)                                      # f32 backward
    assert e.value.status == 3
    qb = q.to(torch.bfloat16)
    with pytest.raises(rx.RingxError) as e:
        rx.ringx_attn_bwd(qb, qb, qb, qb, lse, qb, 256, 0.125,
                          workspace=torch.empty(512, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 5


@pytest.mark.parametrize("B,H,N,d,chunk", [(1, 2, 1024, 64, 256), (2, 3, 512, 128, 512), (1, 2, 2048, 128, 1024),
                                           (1, 1, 16640, 64, 128), (2, 2, 1000, 128, 384), (1, 3, 77, 64, 128)])
def test_fwd_bwd_host_entry_matches_device_entries(rx, B, H, N, d, chunk):
    """The end-to-end entry (copies pipelined chunk by chunk on a side stream; one chunk and > 64 chunks take the
    plain path) gives exactly what the device entries give, twice in a row (the events are reused)."""
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=67)
    scale = 0.125
    qd, kd, vd, dod = q.cuda(), k.cuda(), v.cuda(), do.cuda()
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, chunk, scale)
    dq, dk, dv = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale)
    for _ in range(2):
        oh, lh, dqh, dkh, dvh = rx.ringx_attn_fwd_bwd_host(q.pin_memory(), k.pin_memory(), v.pin_memory(),
                                                           do.pin_memory(), chunk, scale)
        n_c = -(-N // chunk)                      # (the last two shapes: ragged lengths, a short last chunk)
        assert rx.ringx_last_launch_count() == n_c + (n_c + 2 + (1 if N % 128 else 0))
        assert torch.equal(oh, o.cpu()) and torch.equal(lh, lse.cpu())
        assert torch.equal(dkh, dk.cpu()) and torch.equal(dvh, dv.cpu())
        assert ((dqh.float() - dq.cpu().float()).norm() / dq.float().norm()).item() <= 2e-3   # fp32 red order


# ------------------------------------------------------------------------------------------------ deterministic dQ
@pytest.mark.parametrize("B,H,N,d,chunk", [(1, 2, 4096, 128, 1024), (2, 3, 2048, 64, 512)])
def test_deterministic_mode_gives_bit_identical_dq(rx, B, H, N, d, chunk):
    """NEXT-2: with ringx_set_deterministic(1) dQ is accumulated as int32 fixed point (integer adds are associative), so
    repeated runs agree bit for bit whatever order the CTAs' reduce-adds arrive in (dk, dv always do); the result still
    matches the oracle."""
    scale = 1.0 / math.sqrt(d)
    q, k, v, do = wl.make_qkv((B, H, N, d), with_do=True, seed=77, dtype="bf16")
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, chunk, scale)
    rx.ringx_set_deterministic(True)
    try:
        assert rx.ringx_get_deterministic()
        runs = [rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale) for _ in range(4)]
        torch.cuda.synchronize()
        acc = [rx.ringx_attn_bwd_partial(qd, kd, vd, o, lse, dod, scale)[0] for _ in range(3)]
        torch.cuda.synchronize()
    finally:
        rx.ringx_set_deterministic(False)
    assert not rx.ringx_get_deterministic()
    for r in runs[1:]:
        for a, b in zip(runs[0], r):
            assert torch.equal(a, b)
    for a in acc[1:]:
        assert torch.equal(acc[0], a)                      # the fp32 accumulator itself is reproducible
    q64, k64, v64, do64 = (wl.to_f64_numpy(t) for t in (q, k, v, do))
    check_grads_full(*runs[0], q64, k64, v64, do64, scale)


_MULTIWAVE_DET = r"""
import math, sys, torch
sys.path.insert(0, {root!r})
from paper_2507_16697_b200 import ringx as rx, workloads as wl
B, H, N, d, chunk = {shape}
scale = 1.0 / math.sqrt(d)
q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=79, dtype="bf16"))
o, lse = rx.ringx_attn_fwd(q, k, v, chunk, scale)
rx.ringx_set_deterministic(True)
runs = [rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale) for _ in range(3)]
torch.cuda.synchronize()
rx.ringx_set_deterministic(False)
loose = rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale)
torch.cuda.synchronize()
for r in runs[1:]:
    for a, b in zip(runs[0], r):
        assert torch.equal(a, b), "deterministic mode is not bit-reproducible"
rel = ((runs[0][0].float() - loose[0].float()).norm() / loose[0].float().norm()).item()
assert rel <= 2e-3, rel
assert torch.equal(runs[0][1], loose[1]) and torch.equal(runs[0][2], loose[2])
print("MULTIWAVE_DET_OK", B * H * (chunk // 128), "CTAs per pass")
"""


@pytest.mark.parametrize("shape", [(1, 8, 16384, 128, 16384), (2, 8, 8192, 64, 4096), (1, 8, 16384, 128, 4096)])
def test_deterministic_mode_multi_wave_grid(rx, shape):
    """Deterministic mode on grids of several waves -- 1024 / 512 / 256 CTAs per pass (7 / 3.5 / 1.7 waves of the 148
    resident CTAs), where the arrival order of the reduce-adds into a dQ tile differs from run to run: three runs,
    bit-identical dq, dk/dv identical to the default mode's.  (Run in a child process with a timeout: the first
    implementation ordered the adds with tickets and could have deadlocked; the fixed-point accumulator cannot.)"""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = _MULTIWAVE_DET.format(root=root, shape=repr(shape))
    try:
        r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300)
    except subprocess.TimeoutExpired:
        pytest.fail("deterministic-dQ backward did not finish in 300 s on a multi-wave grid")
    assert r.returncode == 0 and "MULTIWAVE_DET_OK" in r.stdout, (r.stdout[-2000:], r.stderr[-2000:])


def test_deterministic_mode_at_its_overflow_bound(rx):
    """The fixed-point scale of row i comes from |dQ_ic| <= scale (||dO_i|| max_j||V_j|| + |D_i|) max_jc|K_jc|.  Inputs
    that REACH that bound: Q = 0, so P is uniform; keys are +kvec / -kvec with values +vvec / -vvec, so
    dP_ij = +-(dO_i . vvec), D_i = 0 and dQ_i = scale (dO_i . vvec) kvec; dO_i parallel to vvec makes Cauchy-Schwarz tight
    (r02's bound used 2 ||dO_i|| max||V|| in place of ||dO_i|| max||V|| + |D_i| and these inputs reached half of it).  The
    int32 accumulator must hold 1.5e9 / 1.016 -- 2^30.5 -- without wrapping and the result must match the oracle to bf16
    accuracy."""
    B, H, N, d, chunk = 1, 2, 2048, 128, 512
    scale = 1.0 / math.sqrt(d)
    g = torch.Generator().manual_seed(5)
    kvec = torch.randn(d, generator=g).to(torch.bfloat16)
    vvec = torch.randn(d, generator=g).to(torch.bfloat16)
    sign = torch.where(torch.arange(N) % 2 == 0, 1.0, -1.0).view(1, 1, N, 1)
    k = (sign * kvec.float()).expand(B, H, N, d).to(torch.bfloat16).contiguous()
    v = (sign * vvec.float()).expand(B, H, N, d).to(torch.bfloat16).contiguous()
    q = torch.zeros(B, H, N, d, dtype=torch.bfloat16)
    amp = torch.linspace(0.25, 4.0, N).view(1, 1, N, 1)           # rows of very different ||dO_i||
    do = (amp * vvec.float()).expand(B, H, N, d).to(torch.bfloat16).contiguous()
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    o, lse = rx.ringx_attn_fwd(qd, kd, vd, chunk, scale)
    rx.ringx_set_deterministic(True)
    try:
        dq, dk, dv = rx.ringx_attn_bwd(qd, kd, vd, o, lse, dod, chunk, scale)
        torch.cuda.synchronize()
    finally:
        rx.ringx_set_deterministic(False)
    q64, k64, v64, do64 = (wl.to_f64_numpy(t) for t in (q, k, v, do))
    dq_ref, _, _ = orc.attention_bwd_bhnd(q64, k64, v64, do64, scale)
    bound = scale * np.linalg.norm(do64, axis=-1, keepdims=True) * np.linalg.norm(v64[0, 0, 0]) * np.abs(k64).max()
    assert (np.abs(dq_ref) / bound).max() >= 0.9                  # the inputs do reach the bound (D_i = 0 here)
    got = dq.float().cpu().numpy()
    assert np.abs(got - dq_ref).max() <= 2.0 ** -7 * np.abs(dq_ref).max()
    assert np.linalg.norm(got - dq_ref) / np.linalg.norm(dq_ref) <= 5e-3


# ------------------------------------------------------------------------------------------------ CUDA graphs
def test_forward_backward_capture_into_a_cuda_graph(rx):
    """Every entry point only enqueues work on the caller's stream (no allocation, no synchronisation), so a whole
    forward + backward -- 4 + 6 launches here -- can be captured once into a CUDA graph and replayed on new data."""
    B, H, N, d, chunk = 1, 2, 1024, 64, 256
    scale = 0.125
    q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=71))
    o = torch.empty_like(q)
    lse = torch.empty((B, H, N), dtype=torch.float32, device="cuda")
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(v)
    wf = torch.empty(max(256, rx.ringx_attn_fwd_workspace_bytes(B, H, N, d, chunk, q.dtype)), dtype=torch.uint8, device="cuda")
    wb = torch.empty(rx.ringx_attn_bwd_workspace_bytes(B, H, N, d, chunk, q.dtype), dtype=torch.uint8, device="cuda")

    def step():
        rx.ringx_attn_fwd(q, k, v, chunk, scale, o=o, lse=lse, workspace=wf)
        rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale, workspace=wb, dq=dq, dk=dk, dv=dv)

    step()                                   # warm-up outside the capture (function attributes are set on first use)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    for seed in (72, 73):
        q2, k2, v2, do2 = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=seed))
        for dst, src in ((q, q2), (k, k2), (v, v2), (do, do2)):
            dst.copy_(src)
        g.replay()
        torch.cuda.synchronize()
        got = [t.clone() for t in (o, lse, dk, dv, dq)]
        step()                               # eager, same buffers
        torch.cuda.synchronize()
        for a, b in zip(got[:4], (o, lse, dk, dv)):
            assert torch.equal(a, b)
        assert ((got[4].float() - dq.float()).norm() / dq.float().norm()).item() <= 2e-3      # fp32 reduce order


_FIRST_BWD_UNDER_CAPTURE = r"""
import sys, torch
sys.path.insert(0, {root!r})
from paper_2507_16697_b200 import ringx as rx, workloads as wl
B, H, N, d, chunk = 1, 2, 512, 128, 256
scale = d ** -0.5
q, k, v, do = (t.cuda() for t in wl.make_qkv((B, H, N, d), with_do=True, seed=91, dtype="bf16"))
o, lse = rx.ringx_attn_fwd(q, k, v, chunk, scale)
dq, dk, dv = (torch.empty_like(t) for t in (q, k, v))
wb = torch.empty(rx.ringx_attn_bwd_workspace_bytes(B, H, N, d, chunk, torch.bfloat16), dtype=torch.uint8, device="cuda")
torch.cuda.synchronize()
side = torch.cuda.Stream()
g = torch.cuda.CUDAGraph()
status = None
with torch.cuda.stream(side):
    g.capture_begin()
    try:
        rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale, workspace=wb, dq=dq, dk=dk, dv=dv)
    except rx.RingxError as e:
        status = e.status
    g.capture_end()                      # the capture is still valid: ending it does not raise
assert status == 7, status               # RINGX_ERR_CUDA: the first d = 128 backward on a device is refused under capture
# a pending event on the caller's stream must not be waited for by the one-time set-up (no synchronisation of `stream`)
s2 = torch.cuda.Stream()
with torch.cuda.stream(s2):
    torch.cuda._sleep(2_000_000_000)     # ~1 s of GPU time queued on s2
    rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale, workspace=wb, dq=dq, dk=dk, dv=dv)
    returned_while_busy = not s2.query()
torch.cuda.synchronize()
assert returned_while_busy, "the first backward waited for the caller's stream"
ref = rx.ringx_attn_bwd(q, k, v, o, lse, do, chunk, scale)
torch.cuda.synchronize()
assert torch.equal(dk, ref[1]) and torch.equal(dv, ref[2]) and torch.isfinite(dq.float()).all()
print("FIRST_BWD_OK")
"""


def test_first_backward_on_a_device_neither_synchronises_the_stream_nor_breaks_a_capture(rx):
    """The d = 128 backward checks the alignment of its shared memory once per device with a one-warp launch.  That launch
    runs on a stream of the library's own: a caller's stream with a second of work queued is not waited for, and when the
    caller's stream is being captured the call is refused (RINGX_ERR_CUDA) with the capture left valid.  Needs a process in
    which no backward has run yet, hence the child."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    # eager module loading: with the default lazy loading the DRIVER may wait for running kernels when it loads the backward
    # kernel on its first launch, which would hide what this test looks at (whether the LIBRARY waits for the caller's stream)
    env = dict(os.environ, CUDA_MODULE_LOADING="EAGER")
    r = subprocess.run([sys.executable, "-c", _FIRST_BWD_UNDER_CAPTURE.format(root=root)], capture_output=True, text=True,
                       timeout=300, env=env)
    assert r.returncode == 0 and "FIRST_BWD_OK" in r.stdout, (r.stdout[-2000:], r.stderr[-2000:])


# ------------------------------------------------------------------------------------------------ seeded random shapes
def _random_shapes(n, seed=20250716):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        N = int(rng.choice([rng.integers(1, 300), rng.integers(300, 1800), 128 * rng.integers(1, 12)]))
        chunk = 128 * int(rng.integers(1, (N + 127) // 128 + 1))
        out.append((int(rng.choice([1, 2])), int(rng.choice([1, 2, 3])), int(rng.choice([1, 1, 2, 4])), N,
                    int(rng.choice([64, 128])), chunk, float(rng.choice([1.0, 1.0, 3.0, 0.05])), bool(rng.random() < 0.3)))
    return out


@pytest.mark.parametrize("B,Hkv,G,N,d,chunk,gain,det", _random_shapes(12))
def test_seeded_random_shapes_match_oracle(rx, B, Hkv, G, N, d, chunk, gain, det):
    """Twelve shapes drawn from a seeded generator -- any length, any chunk that is a multiple of 128, MHA and GQA,
    diffuse and peaked softmax, default and deterministic mode -- forward and backward against the oracle (query head h
    attends kv head h // G; dk, dv summed over the heads of a group)."""
    Hq = Hkv * G
    scale = 1.0 / math.sqrt(d)
    q = wl.make_tensor((B, Hq, N, d), "q", seed=N, dtype="bf16", gain=gain)
    do = wl.make_tensor((B, Hq, N, d), "do", seed=N, dtype="bf16")
    k = wl.make_tensor((B, Hkv, N, d), "k", seed=N, dtype="bf16", gain=gain)
    v = wl.make_tensor((B, Hkv, N, d), "v", seed=N, dtype="bf16")
    qd, kd, vd, dod = (t.cuda() for t in (q, k, v, do))
    rx.ringx_set_deterministic(det)
    try:
        o, lse = rx.ringx_attn_fwd_gqa(qd, kd, vd, chunk, scale)
        dq, dk, dv = rx.ringx_attn_bwd_gqa(qd, kd, vd, o, lse, dod, chunk, scale)
        torch.cuda.synchronize()
    finally:
        rx.ringx_set_deterministic(False)
    q64, k64, v64, do64 = (f64(t) for t in (q, k, v, do))
    k_rep, v_rep = np.repeat(k64, G, axis=1), np.repeat(v64, G, axis=1)
    o_ref, lse_ref = orc.attention_fwd_bhnd(q64, k_rep, v_rep, scale)
    check_fwd(o, lse, o_ref, lse_ref, v64, "bf16")
    dq_ref, dk_rep, dv_rep = orc.attention_bwd_bhnd(q64, k_rep, v_rep, do64, scale)
    dk_ref = dk_rep.reshape(B, Hkv, G, N, d).sum(axis=2)
    dv_ref = dv_rep.reshape(B, Hkv, G, N, d).sum(axis=2)
    for name, g, ref in (("dq", dq, dq_ref), ("dk", dk, dk_ref), ("dv", dv, dv_ref)):
        nr = np.linalg.norm(ref)
        if nr == 0.0:                      # N = 1: dq = dk = 0 exactly
            assert not g.float().any(), name
        else:
            assert np.linalg.norm(to64(g) - ref) / nr <= TOL_GRAD, name
