"""Pins for the fp64 oracle (`oracle/attention.py`) -- CPU only.

The oracle is pinned to things other than itself: hand-derived fixtures (tests/golden/), closed
forms, invariants, brute-force Python loops, finite differences and a library second opinion.
Each test is chosen so that a plausible mistake (dropped term, wrong sign/index, transposed
operand, unscaled score, wrong log base) fails at least one of them.
"""
import json
import math
import os

import numpy as np
import pytest
import torch

from oracle import attention as orc

RNG = np.random.default_rng(20250716)


def rnd(*shape):
    return RNG.standard_normal(shape)


def load(golden_dir, name):
    with open(os.path.join(golden_dir, name)) as f:
        return json.load(f)


# ------------------------------------------------------------------ hand fixtures (tests/golden)
def test_golden_two_keys_d1(golden_dir):
    g = load(golden_dir, "two_keys_d1.json")
    q, v, dO = np.array(g["q"]), np.array(g["v"]), np.array(g["dO"])
    k = np.log(np.array(g["k_log_of"]))
    o, lse = orc.attention_fwd(q, k, v, g["scale"])
    np.testing.assert_allclose(orc.softmax_probs(q, k, g["scale"]), g["P"], atol=1e-15)
    np.testing.assert_allclose(o, g["O"], atol=1e-14)
    np.testing.assert_allclose(lse, np.log(g["LSE_log_of"]), atol=1e-15)
    dq, dk, dv = orc.attention_bwd(q, k, v, dO, g["scale"])
    np.testing.assert_allclose(dv, g["dV"], atol=1e-15)
    np.testing.assert_allclose(dk, g["dK"], atol=1e-14)
    np.testing.assert_allclose(dq, np.array(g["dQ_times_inv_ln3"]) * math.log(3.0), atol=1e-14)


def test_golden_three_keys_d2(golden_dir):
    g = load(golden_dir, "three_keys_d2.json")
    q, v, dO = np.array(g["q"]), np.array(g["v"]), np.array(g["dO"])
    k = np.stack([np.log(np.array(g["k0_log_of"])), np.array(g["k1"])], axis=1)
    sc = g["scale"]
    o, lse = orc.attention_fwd(q, k, v, sc)
    np.testing.assert_allclose(orc.softmax_probs(q, k, sc), g["P"], atol=1e-15)
    np.testing.assert_allclose(o, g["O"], atol=1e-14)
    np.testing.assert_allclose(lse, np.log(g["LSE_log_of"]), atol=1e-15)
    dq, dk, dv = orc.attention_bwd(q, k, v, dO, sc)
    dS = np.array(g["dS"])
    np.testing.assert_allclose(dv, g["dV"], atol=1e-15)
    np.testing.assert_allclose(dk, sc * dS.T @ q, atol=1e-14)
    np.testing.assert_allclose(dk[:, 1], 0.0, atol=1e-15)          # q[1] = 0
    np.testing.assert_allclose(dq, sc * dS @ k, atol=1e-13)
    # Eq. (5) on the fixture's chunks
    outs, lses = orc.chunk_partials(q, k, v, sc, g["chunk_bounds"])
    np.testing.assert_allclose(np.stack(lses)[:, 0], np.log(g["loc_lse_log_of"]), atol=1e-15)
    np.testing.assert_allclose(np.stack(outs), g["loc_out"], atol=1e-14)
    om, lm = orc.merge_partials(outs, lses)
    np.testing.assert_allclose(om, g["O"], atol=1e-14)
    np.testing.assert_allclose(lm, np.log(g["LSE_log_of"]), atol=1e-15)


# ------------------------------------------------------------------ brute force, tiny inputs
def brute_forward(q, k, v, scale):
    """Eq. (1)/(3)/(4) with Python loops and math.exp only -- no matmul, no numpy reductions."""
    Nq, d = len(q), len(q[0])
    Nk, dv = len(k), len(v[0])
    O = [[0.0] * dv for _ in range(Nq)]
    L = [0.0] * Nq
    for s in range(Nq):
        e = [scale * sum(q[s][c] * k[i][c] for c in range(d)) for i in range(Nk)]
        z = sum(math.exp(x) for x in e)
        L[s] = math.log(z)
        for i in range(Nk):
            w = math.exp(e[i]) / z
            for c in range(dv):
                O[s][c] += w * v[i][c]
    return np.array(O), np.array(L)


def test_brute_force_forward_nonsquare():
    # Nq != Nk != d != dv so that any transposed operand changes shapes or values
    q, k, v = rnd(5, 3), rnd(7, 3), rnd(7, 4)
    o, lse = orc.attention_fwd(q, k, v, 0.37)
    ob, lb = brute_forward(q.tolist(), k.tolist(), v.tolist(), 0.37)
    np.testing.assert_allclose(o, ob, atol=1e-13)
    np.testing.assert_allclose(lse, lb, atol=1e-13)


# ------------------------------------------------------------------ closed forms
def test_rows_of_p_sum_to_one():
    p = orc.softmax_probs(rnd(33, 16), rnd(257, 16), 0.25)
    assert np.abs(p.sum(axis=1) - 1.0).max() <= 1e-14
    assert (p >= 0).all()


def test_identical_keys_give_mean_of_v():
    N, d = 50, 8
    q, v = rnd(6, d), rnd(N, d)
    k = np.tile(rnd(1, d), (N, 1))
    o, lse = orc.attention_fwd(q, k, v, 0.5)
    np.testing.assert_allclose(o, np.tile(v.mean(axis=0), (6, 1)), atol=1e-13)
    np.testing.assert_allclose(lse, 0.5 * (q @ k[0]) + math.log(N), atol=1e-13)


def test_zero_query_gives_mean_and_log_n():
    N = 31
    k, v = rnd(N, 4), rnd(N, 4)
    o, lse = orc.attention_fwd(np.zeros((3, 4)), k, v, 1.0)
    np.testing.assert_allclose(o, np.tile(v.mean(axis=0), (3, 1)), atol=1e-14)
    np.testing.assert_allclose(lse, math.log(N), atol=1e-14)


def test_single_key():
    q, k, v = rnd(4, 5), rnd(1, 5), rnd(1, 3)
    o, lse = orc.attention_fwd(q, k, v, 0.7)
    np.testing.assert_allclose(o, np.tile(v, (4, 1)), atol=1e-15)
    np.testing.assert_allclose(lse, 0.7 * (q @ k[0]), atol=1e-14)


def test_two_keys_is_logistic():
    q, k, v = rnd(9, 6), rnd(2, 6), rnd(2, 6)
    s = 0.3 * q @ k.T
    sig = 1.0 / (1.0 + np.exp(-(s[:, 1] - s[:, 0])))
    o, lse = orc.attention_fwd(q, k, v, 0.3)
    np.testing.assert_allclose(o, sig[:, None] * v[1] + (1 - sig)[:, None] * v[0], atol=1e-14)
    np.testing.assert_allclose(lse, np.logaddexp(s[:, 0], s[:, 1]), atol=1e-14)


def test_one_hot_v_reads_p():
    q, k = rnd(7, 8), rnd(20, 8)
    keys = [3, 11, 19, 0]
    v = np.zeros((20, 4))
    for c, j in enumerate(keys):
        v[j, c] = 1.0
    o, _ = orc.attention_fwd(q, k, v, 0.4)
    np.testing.assert_allclose(o, orc.softmax_probs(q, k, 0.4)[:, keys], atol=1e-15)


def test_large_scores_are_stable():
    q = np.full((1, 2), 30.0)
    k = np.array([[30.0, 30.0], [0.0, 0.0], [29.0, 30.0]])      # scores 1800, 0, 1770
    o, lse = orc.attention_fwd(q, k, np.eye(3), 1.0)
    assert np.isfinite(o).all() and np.isfinite(lse).all()
    np.testing.assert_allclose(lse, 1800.0 + math.log1p(math.exp(-30.0)), rtol=1e-15)


# ------------------------------------------------------------------ invariances
def test_key_shift_moves_lse_only():
    q, k, v, c = rnd(5, 8), rnd(40, 8), rnd(40, 8), rnd(8)
    o0, l0 = orc.attention_fwd(q, k, v, 0.35)
    o1, l1 = orc.attention_fwd(q, k + c, v, 0.35)
    np.testing.assert_allclose(o1, o0, atol=1e-13)
    np.testing.assert_allclose(l1, l0 + 0.35 * q @ c, atol=1e-13)


def test_permutations_and_voxel_order():
    q, k, v = rnd(27, 4), rnd(27, 4), rnd(27, 4)
    o0, l0 = orc.attention_fwd(q, k, v, 0.5)
    pk, pq = RNG.permutation(27), RNG.permutation(27)
    o1, l1 = orc.attention_fwd(q, k[pk], v[pk], 0.5)           # keys: invariant
    np.testing.assert_allclose(o1, o0, atol=1e-14)
    np.testing.assert_allclose(l1, l0, atol=1e-14)
    o2, l2 = orc.attention_fwd(q[pq], k, v, 0.5)               # queries: equivariant (g15)
    np.testing.assert_allclose(o2, o0[pq], atol=1e-15)
    np.testing.assert_allclose(l2, l0[pq], atol=1e-15)


def test_convex_hull_and_lse_bounds():
    q, k, v = rnd(16, 8), rnd(100, 8), rnd(100, 8)
    o, lse = orc.attention_fwd(q, k, v, 0.35)
    assert (o <= v.max(axis=0) + 1e-15).all() and (o >= v.min(axis=0) - 1e-15).all()
    smax = (0.35 * q @ k.T).max(axis=1)
    assert (lse >= smax).all() and (lse <= smax + math.log(100) + 1e-14).all()


def test_scale_is_applied_to_scores():
    q, k, v = rnd(4, 8), rnd(12, 8), rnd(12, 8)
    o0, l0 = orc.attention_fwd(q, k, v, 0.125)
    o1, l1 = orc.attention_fwd(0.125 * q, k, v, 1.0)
    np.testing.assert_allclose(o0, o1, atol=1e-14)
    np.testing.assert_allclose(l0, l1, atol=1e-14)


# ------------------------------------------------------------------ Eq. (5): chunk merge
@pytest.mark.parametrize("bounds", [[0, 16, 32, 48, 64], [0, 1, 64], [0, 63, 64], [0, 5, 6, 40, 64], [0, 64]])
def test_chunked_equals_unchunked(bounds):
    q, k, v = rnd(10, 8), rnd(64, 8), rnd(64, 8)
    o0, l0 = orc.attention_fwd(q, k, v, 0.35)
    for fn in (orc.attention_fwd_chunked, orc.attention_fwd_running):
        o1, l1 = fn(q, k, v, 0.35, bounds)
        assert np.abs(o1 - o0).max() <= 1e-13
        assert np.abs(l1 - l0).max() <= 1e-13


def test_merge_any_tree_and_order():
    q, k, v = rnd(6, 4), rnd(40, 4), 3.0 * rnd(40, 4)
    o0, l0 = orc.attention_fwd(q, k, v, 1.3)
    outs, lses = orc.chunk_partials(q, k, v, 1.3, [0, 7, 8, 21, 33, 40])
    order = RNG.permutation(5)
    parts = [(outs[i], lses[i]) for i in order]
    while len(parts) > 1:                                       # random binary tree
        i = int(RNG.integers(0, len(parts) - 1))
        (oa, la), (ob, lb) = parts[i], parts[i + 1]
        parts[i:i + 2] = [orc.lse_merge(oa, la, ob, lb)]
    assert np.abs(parts[0][0] - o0).max() <= 1e-13
    assert np.abs(parts[0][1] - l0).max() <= 1e-13


def test_merge_special_cases():
    o, l = rnd(5, 3), rnd(5)
    om, lm = orc.lse_merge(o, l, o, l)                          # merge with itself
    np.testing.assert_allclose(om, o, atol=1e-15)
    np.testing.assert_allclose(lm, l + math.log(2.0), atol=1e-15)
    ninf = np.full(5, -np.inf)
    om, lm = orc.lse_merge(o, l, rnd(5, 3), ninf)               # empty operand = identity (g12)
    np.testing.assert_array_equal(om, o)
    np.testing.assert_array_equal(lm, l)
    om, lm = orc.lse_merge(rnd(5, 3), ninf, o, l)
    np.testing.assert_array_equal(om, o)
    om, lm = orc.lse_merge(o, ninf, o, ninf)                    # both empty
    assert (om == 0).all() and np.isneginf(lm).all()
    # weights follow exp(lse): lse_b = lse_a + ln 3 => o = (o_a + 3 o_b)/4
    ob = rnd(5, 3)
    om, lm = orc.lse_merge(o, l, ob, l + math.log(3.0))
    np.testing.assert_allclose(om, 0.25 * o + 0.75 * ob, atol=1e-15)
    np.testing.assert_allclose(lm, l + math.log(4.0), atol=1e-15)


# ------------------------------------------------------------------ gradients
def loss(q, k, v, dO, scale):
    return float((orc.attention_fwd(q, k, v, scale)[0] * dO).sum())


def finite_diff(fn, x, h=1e-5):
    g = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp, xm = x.copy(), x.copy()
        xp[idx] += h
        xm[idx] -= h
        g[idx] = (fn(xp) - fn(xm)) / (2 * h)
    return g


def test_gradients_match_finite_differences():
    q, k, v, dO = rnd(5, 3), rnd(9, 3), rnd(9, 4), rnd(5, 4)
    sc = 0.6
    dq, dk, dv = orc.attention_bwd(q, k, v, dO, sc)
    for got, fd in ((dq, finite_diff(lambda x: loss(x, k, v, dO, sc), q)),
                    (dk, finite_diff(lambda x: loss(q, x, v, dO, sc), k)),
                    (dv, finite_diff(lambda x: loss(q, k, x, dO, sc), v))):
        assert np.abs(got - fd).max() <= 1e-8 * max(1.0, np.abs(fd).max())


def test_gradient_identities():
    q, k, v, dO = rnd(12, 8), rnd(30, 8), rnd(30, 8), rnd(12, 8)
    dq, dk, dv = orc.attention_bwd(q, k, v, dO, 0.35)
    np.testing.assert_allclose(dv.sum(axis=0), dO.sum(axis=0), atol=1e-13)   # rows of P sum to 1
    np.testing.assert_allclose(dk.sum(axis=0), 0.0, atol=1e-13)              # sum_j dS_ij = 0
    z = orc.attention_bwd(q, k, v, np.zeros_like(dO), 0.35)
    assert all((g == 0).all() for g in z)
    dO2 = rnd(12, 8)                                                         # linear in dO
    a = orc.attention_bwd(q, k, v, 2.0 * dO - 3.0 * dO2, 0.35)
    b = orc.attention_bwd(q, k, v, dO2, 0.35)
    for ga, g1, g2 in zip(a, (dq, dk, dv), b):
        np.testing.assert_allclose(ga, 2.0 * g1 - 3.0 * g2, atol=1e-12)


def test_row_and_column_sampled_backward_are_exact():
    q, k, v, dO = rnd(24, 8), rnd(40, 8), rnd(40, 8), rnd(24, 8)
    sc = 0.35
    dq, dk, dv = orc.attention_bwd(q, k, v, dO, sc)
    rows = [0, 5, 23]
    dq_r, _, _ = orc.attention_bwd(q[rows], k, v, dO[rows], sc)
    np.testing.assert_allclose(dq_r, dq[rows], atol=1e-14)
    # contributions of disjoint row sets add up to dK, dV ("reduced over N ranks")
    _, dk_a, dv_a = orc.attention_bwd(q[:10], k, v, dO[:10], sc)
    _, dk_b, dv_b = orc.attention_bwd(q[10:], k, v, dO[10:], sc)
    np.testing.assert_allclose(dk_a + dk_b, dk, atol=1e-13)
    np.testing.assert_allclose(dv_a + dv_b, dv, atol=1e-13)
    cols = [0, 7, 39]
    lse, D = orc.row_stats(q, k, v, dO, sc)
    dk_c, dv_c = orc.attention_bwd_cols(q, k[cols], v[cols], dO, lse, D, sc)
    np.testing.assert_allclose(dk_c, dk[cols], atol=1e-13)
    np.testing.assert_allclose(dv_c, dv[cols], atol=1e-13)


def test_partial_backward_steps_add_up_to_the_gradient():
    """attention_bwd_partial (one device's step of the RingX backward) against the pinned full
    gradient: dQ shares over any partition of the keys sum to dQ; dK/dV of a key subset from a partition of the
    query rows sum to those rows of dK/dV; and against finite differences directly (ragged 2 x 3 grid of blocks)."""
    q, k, v, dO = rnd(7, 3), rnd(11, 3), rnd(11, 4), rnd(7, 4)
    sc = 0.45
    lse, D = orc.row_stats(q, k, v, dO, sc)
    fd_q = finite_diff(lambda x: loss(x, k, v, dO, sc), q)
    fd_k = finite_diff(lambda x: loss(q, x, v, dO, sc), k)
    fd_v = finite_diff(lambda x: loss(q, k, x, dO, sc), v)
    dq, dk, dv = np.zeros_like(q), np.zeros_like(k), np.zeros_like(v)
    for r0, r1 in ((0, 3), (3, 7)):                       # two "devices" holding query rows
        for c0, c1 in ((0, 1), (1, 6), (6, 11)):          # three key chunks (ragged)
            a, b, c = orc.attention_bwd_partial(q[r0:r1], k[c0:c1], v[c0:c1], dO[r0:r1], lse[r0:r1], D[r0:r1], sc)
            dq[r0:r1] += a
            dk[c0:c1] += b
            dv[c0:c1] += c
    for got, fd in ((dq, fd_q), (dk, fd_k), (dv, fd_v)):
        assert np.abs(got - fd).max() <= 1e-8 * max(1.0, np.abs(fd).max())
    full = orc.attention_bwd(q, k, v, dO, sc)
    for got, ref in zip((dq, dk, dv), full):
        np.testing.assert_allclose(got, ref, atol=1e-13)
    # a transposed operand would survive neither: shapes differ (Nq != Nk, d != dv)


# ------------------------------------------------------------------ library second opinion
def test_against_torch_fp64():
    q, k, v, dO = rnd(40, 16), rnd(70, 16), rnd(70, 16), rnd(40, 16)
    sc = 0.25
    tq, tk, tv = (torch.tensor(x, requires_grad=True) for x in (q, k, v))
    s = sc * tq @ tk.T
    to = torch.softmax(s, dim=1) @ tv
    tl = torch.logsumexp(s, dim=1)
    (to * torch.tensor(dO)).sum().backward()
    o, lse = orc.attention_fwd(q, k, v, sc)
    dq, dk, dv = orc.attention_bwd(q, k, v, dO, sc)
    np.testing.assert_allclose(o, to.detach().numpy(), atol=1e-12)
    np.testing.assert_allclose(lse, tl.detach().numpy(), atol=1e-12)
    np.testing.assert_allclose(dq, tq.grad.numpy(), atol=1e-12)
    np.testing.assert_allclose(dk, tk.grad.numpy(), atol=1e-12)
    np.testing.assert_allclose(dv, tv.grad.numpy(), atol=1e-12)


def test_bhnd_wrappers_match_per_head_calls():
    q, k, v, dO = rnd(2, 3, 20, 4), rnd(2, 3, 20, 4), rnd(2, 3, 20, 4), rnd(2, 3, 20, 4)
    o, lse = orc.attention_fwd_bhnd(q, k, v, 0.5, block_rows=7)
    dq, dk, dv = orc.attention_bwd_bhnd(q, k, v, dO, 0.5, block_rows=7)
    for b in range(2):
        for h in range(3):
            o1, l1 = orc.attention_fwd(q[b, h], k[b, h], v[b, h], 0.5)
            g = orc.attention_bwd(q[b, h], k[b, h], v[b, h], dO[b, h], 0.5)
            np.testing.assert_allclose(o[b, h], o1, atol=1e-15)
            np.testing.assert_allclose(lse[b, h], l1, atol=1e-15)
            for got, exp in zip((dq[b, h], dk[b, h], dv[b, h]), g):
                np.testing.assert_allclose(got, exp, atol=1e-13)
