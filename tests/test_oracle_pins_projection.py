"""Pins for `oracle/projection.py` (Table II's projection GEMMs, NEXT-4) -- CPU only."""
import numpy as np
import torch

from oracle import attention as orc
from oracle import projection as proj

RNG = np.random.default_rng(20250723)


def test_identity_weights_are_a_layout_permutation():
    B, S, H, d = 2, 5, 3, 4
    h = H * d
    x = RNG.standard_normal((B, S, h))
    w = np.concatenate([np.eye(h), 2.0 * np.eye(h), -np.eye(h)], axis=0)
    q, k, v = proj.qkv_projection(x, w, H)
    for b in range(B):
        for a in range(H):
            for s in range(S):
                for c in range(d):
                    assert q[b, a, s, c] == x[b, s, a * d + c]
                    assert k[b, a, s, c] == 2.0 * x[b, s, a * d + c]
                    assert v[b, a, s, c] == -x[b, s, a * d + c]
    np.testing.assert_array_equal(proj.out_projection(q, np.eye(h)), x)       # merge_heads inverts split_heads


def test_one_hot_input_reads_single_weights():
    H, d = 2, 3
    h = H * d
    w = RNG.standard_normal((3 * h, h))
    for f in (0, 4):
        x = np.zeros((1, 2, h))
        x[0, 1, f] = 1.0
        q, k, v = proj.qkv_projection(x, w, H)
        for a in range(H):
            for c in range(d):
                assert q[0, a, 1, c] == w[a * d + c, f]              # y = x W^T: W[out, in]  (a transposed W fails)
                assert k[0, a, 1, c] == w[h + a * d + c, f]
                assert v[0, a, 1, c] == w[2 * h + a * d + c, f]
        assert not q[0, :, 0].any()
    wo = RNG.standard_normal((h, h))
    o = np.zeros((1, H, 2, d))
    o[0, 1, 0, 2] = 1.0                                              # head 1, feature 1*d + 2 = 5
    y = proj.out_projection(o, wo)
    np.testing.assert_array_equal(y[0, 0], wo[:, 5])
    assert not y[0, 1].any()


def test_brute_force_loops():
    B, S, H, d = 1, 3, 2, 2
    h = H * d
    x, w, wo = RNG.standard_normal((B, S, h)), RNG.standard_normal((3 * h, h)), RNG.standard_normal((h, h))
    q, k, v = proj.qkv_projection(x, w, H)
    for t, off in ((q, 0), (k, h), (v, 2 * h)):
        for a in range(H):
            for s in range(S):
                for c in range(d):
                    acc = sum(x[0, s, i] * w[off + a * d + c, i] for i in range(h))
                    assert abs(t[0, a, s, c] - acc) < 1e-14
    o = RNG.standard_normal((B, H, S, d))
    y = proj.out_projection(o, wo)
    for s in range(S):
        for f in range(h):
            acc = sum(o[0, i // d, s, i % d] * wo[f, i] for i in range(h))
            assert abs(y[0, s, f] - acc) < 1e-14


def test_library_second_opinion_linear():
    B, S, H, d = 2, 7, 4, 8
    h = H * d
    x, w, wo = RNG.standard_normal((B, S, h)), RNG.standard_normal((3 * h, h)), RNG.standard_normal((h, h))
    y = torch.nn.functional.linear(torch.from_numpy(x), torch.from_numpy(w))
    ref = [t.reshape(B, S, H, d).permute(0, 2, 1, 3).numpy() for t in y.chunk(3, dim=-1)]
    for got, r in zip(proj.qkv_projection(x, w, H), ref):
        np.testing.assert_allclose(got, r, atol=1e-13)
    o = RNG.standard_normal((B, H, S, d))
    ref = torch.nn.functional.linear(torch.from_numpy(o).permute(0, 2, 1, 3).reshape(B, S, h), torch.from_numpy(wo)).numpy()
    np.testing.assert_allclose(proj.out_projection(o, wo), ref, atol=1e-13)


def test_block_equals_per_head_loop_and_library():
    B, S, H, d = 2, 6, 2, 4
    h = H * d
    scale = d ** -0.5
    x, w, wo = RNG.standard_normal((B, S, h)), RNG.standard_normal((3 * h, h)) * 0.5, RNG.standard_normal((h, h))
    y = proj.attention_block_fwd(x, w, wo, H, scale)
    # written out: per batch, per head, softmax(q k^T scale) v, concatenated over heads, times W_o^T
    for b in range(B):
        cat = np.zeros((S, h))
        for a in range(H):
            rows = slice(a * d, (a + 1) * d)
            qh, kh, vh = x[b] @ w[0:h][rows].T, x[b] @ w[h:2 * h][rows].T, x[b] @ w[2 * h:][rows].T
            cat[:, rows] = orc.softmax_probs(qh, kh, scale) @ vh
        np.testing.assert_allclose(y[b], cat @ wo.T, atol=1e-13)
    # library: torch multi-head attention functional in fp64 (no bias), batch_first
    xt = torch.from_numpy(x)
    ref, _ = torch.nn.functional.multi_head_attention_forward(
        xt.transpose(0, 1), xt.transpose(0, 1), xt.transpose(0, 1), h, H, torch.from_numpy(w), None, None, None, False, 0.0,
        torch.from_numpy(wo), None, need_weights=False)
    np.testing.assert_allclose(y, ref.transpose(0, 1).numpy(), atol=1e-12)


def test_linearity_and_head_independence():
    B, S, H, d = 1, 4, 2, 3
    h = H * d
    x1, x2, w = RNG.standard_normal((B, S, h)), RNG.standard_normal((B, S, h)), RNG.standard_normal((3 * h, h))
    a = proj.qkv_projection(2.0 * x1 - x2, w, H)
    b1, b2 = proj.qkv_projection(x1, w, H), proj.qkv_projection(x2, w, H)
    for t, u, v in zip(a, b1, b2):
        np.testing.assert_allclose(t, 2.0 * u - v, atol=1e-13)
    w2 = w.copy()
    w2[d:2 * d] += 1.0                                               # rows of W_q that feed head 1 only
    q2 = proj.qkv_projection(x1, w2, H)[0]
    np.testing.assert_array_equal(q2[:, 0], b1[0][:, 0])
    assert np.abs(q2[:, 1] - b1[0][:, 1]).max() > 0


# ------------------------------------------------------------------------------------------------ backward (reading p5)
def _block_loss(x, w, wo, dy, H, scale):
    return float((dy * proj.attention_block_fwd(x, w, wo, H, scale)).sum())


def test_block_backward_by_central_finite_differences():
    B, S, H, d = 1, 5, 2, 3
    h = H * d
    scale = 0.7
    x, w, wo, dy = (RNG.standard_normal(s) for s in ((B, S, h), (3 * h, h), (h, h), (B, S, h)))
    w *= 0.4
    dx, dw, dwo = proj.attention_block_bwd(x, w, wo, dy, H, scale)
    eps = 1e-6
    for arr, grad, idxs in ((x, dx, [(0, 0, 0), (0, 3, 4), (0, 4, 5)]), (w, dw, [(0, 0), (7, 2), (13, 5), (17, 1)]),
                            (wo, dwo, [(0, 0), (2, 5), (5, 3)])):
        for idx in idxs:
            old = arr[idx]
            arr[idx] = old + eps
            lp = _block_loss(x, w, wo, dy, H, scale)
            arr[idx] = old - eps
            lm = _block_loss(x, w, wo, dy, H, scale)
            arr[idx] = old
            fd = (lp - lm) / (2 * eps)
            assert abs(fd - grad[idx]) <= 1e-6 * max(1.0, abs(fd)), (idx, fd, grad[idx])


def test_projection_backward_against_torch_autograd():
    B, S, H, d = 2, 6, 2, 4
    h = H * d
    x, w, wo = RNG.standard_normal((B, S, h)), RNG.standard_normal((3 * h, h)), RNG.standard_normal((h, h))
    dq, dk, dv, o = (RNG.standard_normal((B, H, S, d)) for _ in range(4))
    dy = RNG.standard_normal((B, S, h))
    xt, wt = torch.from_numpy(x).requires_grad_(), torch.from_numpy(w).requires_grad_()
    y = torch.nn.functional.linear(xt, wt)
    g = torch.cat([torch.from_numpy(t).permute(0, 2, 1, 3).reshape(B, S, h) for t in (dq, dk, dv)], dim=-1)
    y.backward(g)
    dx, dw = proj.qkv_projection_bwd(dq, dk, dv, x, w)
    np.testing.assert_allclose(dx, xt.grad.numpy(), atol=1e-12)
    np.testing.assert_allclose(dw, wt.grad.numpy(), atol=1e-12)
    ot, wot = torch.from_numpy(o).requires_grad_(), torch.from_numpy(wo).requires_grad_()
    yo = torch.nn.functional.linear(ot.permute(0, 2, 1, 3).reshape(B, S, h), wot)
    yo.backward(torch.from_numpy(dy))
    d_o, dwo = proj.out_projection_bwd(dy, o, wo)
    np.testing.assert_allclose(d_o, ot.grad.numpy(), atol=1e-12)
    np.testing.assert_allclose(dwo, wot.grad.numpy(), atol=1e-12)


def test_projection_backward_one_hot_reads():
    """dY one-hot at (s, n): dO row s = column... W_o[n, :] split into heads; dW_o row n = merged o row s."""
    B, S, H, d = 1, 3, 2, 2
    h = H * d
    o, wo = RNG.standard_normal((B, H, S, d)), RNG.standard_normal((h, h))
    dy = np.zeros((B, S, h))
    dy[0, 1, 2] = 1.0
    d_o, dwo = proj.out_projection_bwd(dy, o, wo)
    for a in range(H):
        for c in range(d):
            assert d_o[0, a, 1, c] == wo[2, a * d + c] and d_o[0, a, 0, c] == 0.0
            assert dwo[2, a * d + c] == o[0, a, 1, c]
    assert not dwo[[0, 1, 3]].any()
