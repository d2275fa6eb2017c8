"""fp64 CPU oracle for the RingX chunked-attention hot path.  *** TEST INFRASTRUCTURE ONLY ***

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` leg
may import this package.  The product path (`paper_2507_16697_b200`) never does, shares no code,
tables or helpers with it, and fails loudly when its CUDA library is missing.

What is written here is the *definition*, in numpy float64, because the method reaches exactly
(up to rounding order) a result that has a plain definition: "Our RingX methods calculate the
exact attention as defined by Eq. (1) (within numerical rounding for low precision arithmetic)"
(PAPER.md:211).  A matmul / exp / log from numpy serves as a step; there is no key blocking, no
online rescaling and no fusion.  Rows (and heads) are independent in non-causal attention, so every
function takes "some query rows against ALL keys"; callers that cannot hold an [Nq, Nk] score
matrix pass fewer rows at a time -- that is a subset of the definition, not a reordering of it.

Shapes: q [Nq,d], k [Nk,d], v [Nk,dv], dO [Nq,dv]; everything float64.  `scale` is explicit
(Eq. 1/4 print no 1/sqrt(d); reading g1).

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): hand-derived fixture under tests/golden/,
closed forms (identical keys, Q=0, one key, two keys = logistic), one-hot V reads P, invariances,
brute-force Python loops on tiny inputs, chunked == unchunked for equal / ragged / random
partitions and any merge tree, central finite differences for every gradient, and a library second
opinion (torch fp64 logsumexp/softmax).  Every function below is pinned; none is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


# --------------------------------------------------------------------------------------------
# Forward: Eq. (1), evaluated stably through the LSE of Eq. (3)-(4)
# --------------------------------------------------------------------------------------------
def scores(q, k, scale):
    """e_i^s = Q_s . K_i^T (Eq. 4), times the explicit `scale` (reading g1)."""
    return scale * (q @ k.T)


def attention_fwd(q, k, v, scale):
    """A^s = sum_i Softmax(Q_s . K_i^T) V_i (Eq. 1) and LSE_s = log sum_i exp(e_i^s)
    (Eq. 3).  Eq. 2 is garbled in the source; the standard stable evaluation --
    subtract the row max of the scores -- is used (reading g2).  Returns (O [Nq,dv], LSE [Nq])."""
    s = scores(q, k, scale)                                   # [Nq, Nk]
    m = s.max(axis=1)                                         # row max over keys
    l = np.exp(s - m[:, None]).sum(axis=1)
    lse = m + np.log(l)                                       # natural log, scaled scores (g6)
    p = np.exp(s - lse[:, None])                              # Softmax rows, sum to 1
    return p @ v, lse


def softmax_probs(q, k, scale):
    """The matrix P_ij = Softmax_j(scale q_i.k_j) itself (for tests that inspect it)."""
    s = scores(q, k, scale)
    m = s.max(axis=1, keepdims=True)
    e = np.exp(s - m)
    return e / e.sum(axis=1, keepdims=True)


# --------------------------------------------------------------------------------------------
# Chunked forward + merge: Eq. (5)
# --------------------------------------------------------------------------------------------
def chunk_partials(q, k, v, scale, bounds):
    """(loc_out_i, loc_lse_i) of every key chunk S_i = [bounds[i], bounds[i+1]) -- "the local
    attention output and LSE on the sequence chunk S_i".  `bounds` is an increasing
    list starting at 0 and ending at Nk; chunks may be ragged (reading g11)."""
    outs, lses = [], []
    for lo, hi in zip(bounds[:-1], bounds[1:]):
        o, lse = attention_fwd(q, k[lo:hi], v[lo:hi], scale)
        outs.append(o)
        lses.append(lse)
    return outs, lses


def merge_partials(outs, lses):
    """Eq. (5): num = sum_i loc_out_i exp(loc_lse_i - lse_max),
    den = sum_i exp(loc_lse_i - lse_max), with lse_max the maximum over chunks;
    "num/den gives the corresponding attention".  The merged LSE, which the paper
    never writes down, is lse_max + log(den) -- forced by Eq. (3) (reading g4).
    A chunk with loc_lse = -inf (no keys) gets weight 0; all -inf gives O = 0, LSE = -inf (g12)."""
    lses = np.stack(lses, axis=0)                             # [n_chunks, Nq]
    outs = np.stack(outs, axis=0)                             # [n_chunks, Nq, dv]
    lse_max = lses.max(axis=0)
    safe_max = np.where(np.isfinite(lse_max), lse_max, 0.0)
    w = np.exp(lses - safe_max[None, :])                      # exp(-inf) = 0
    den = w.sum(axis=0)
    num = (outs * w[:, :, None]).sum(axis=0)
    with np.errstate(divide="ignore", invalid="ignore"):
        o = np.where(den[:, None] > 0, num / den[:, None], 0.0)
        lse = np.where(den > 0, safe_max + np.log(den), -np.inf)
    return o, lse


def lse_merge(o_a, lse_a, o_b, lse_b):
    """The two-operand form of Eq. (5): what one `ringx_lse_merge` call computes."""
    return merge_partials([o_a, o_b], [lse_a, lse_b])


def attention_fwd_chunked(q, k, v, scale, bounds):
    """Chunked attention: partials per chunk, then one Eq. (5) merge over all chunks."""
    outs, lses = chunk_partials(q, k, v, scale, bounds)
    return merge_partials(outs, lses)


def attention_fwd_running(q, k, v, scale, bounds):
    """Same, merged left to right two at a time ("running" merge, north_star).  Mathematically
    identical to `attention_fwd_chunked` -- the sums are associative (reading g5)."""
    outs, lses = chunk_partials(q, k, v, scale, bounds)
    o, lse = outs[0], lses[0]
    for ob, lb in zip(outs[1:], lses[1:]):
        o, lse = lse_merge(o, lse, ob, lb)
    return o, lse


# --------------------------------------------------------------------------------------------
# Backward: the derivative of the definition (the paper gives only the data-flow, PAPER.md:143;
# reading g8).  Loss L = sum_ic dO_ic O_ic.
# --------------------------------------------------------------------------------------------
def attention_bwd(q, k, v, dO, scale):
    """Returns (dQ [Nq,d], dK [Nk,d], dV [Nk,dv]) for the given query rows against all keys.
    P_ij = exp(s_ij - LSE_i); dV_j = sum_i P_ij dO_i; dP_ij = dO_i . v_j;
    D_i = sum_j P_ij dP_ij; dS_ij = P_ij (dP_ij - D_i); dQ_i = scale sum_j dS_ij k_j;
    dK_j = scale sum_i dS_ij q_i.  With a subset of rows, dQ is complete for those rows and
    (dK, dV) are those rows' contributions (the paper's "reduced over N ranks" sum)."""
    s = scores(q, k, scale)
    m = s.max(axis=1)
    lse = m + np.log(np.exp(s - m[:, None]).sum(axis=1))
    p = np.exp(s - lse[:, None])
    dv = p.T @ dO
    dp = dO @ v.T
    D = (p * dp).sum(axis=1)
    ds = p * (dp - D[:, None])
    dq = scale * (ds @ k)
    dk = scale * (ds.T @ q)
    return dq, dk, dv


def row_stats(q, k, v, dO, scale):
    """(LSE_i, D_i) for the given rows: what a key-column check of dK/dV needs for ALL rows."""
    o, lse = attention_fwd(q, k, v, scale)
    return lse, (dO * o).sum(axis=1)          # D_i = sum_j P_ij dP_ij = dO_i . O_i


def attention_bwd_cols(q, k_cols, v_cols, dO, lse, D, scale):
    """dK, dV for a subset of key columns, given LSE_i and D_i of every query row of the head
    (from `row_stats`).  Exact, because column j of P only needs s_ij and LSE_i."""
    p = np.exp(scores(q, k_cols, scale) - lse[:, None])       # [Nq, ncols]
    dv = p.T @ dO
    ds = p * (dO @ v_cols.T - D[:, None])
    dk = scale * (ds.T @ q)
    return dk, dv


def attention_bwd_partial(q, k_cols, v_cols, dO, lse, D, scale):
    """One device's step of the RingX backward (reading g8): with the *global* LSE_i and D_i
    of the given query rows, the key subset (k_cols, v_cols) yields its complete share of those rows' dQ,
    dQ_i += scale sum_{j in cols} dS_ij k_j, and these rows' share of dK_j, dV_j for j in cols.
    Summing the dQ shares over a partition of the keys gives `attention_bwd`'s dQ."""
    p = np.exp(scores(q, k_cols, scale) - lse[:, None])       # [Nq, ncols]
    ds = p * (dO @ v_cols.T - D[:, None])
    return scale * (ds @ k_cols), scale * (ds.T @ q), p.T @ dO


# --------------------------------------------------------------------------------------------
# [B,H,N,d] conveniences (loops over heads; block_rows bounds the [rows, N] score matrix)
# --------------------------------------------------------------------------------------------
def attention_fwd_bhnd(q, k, v, scale, block_rows=4096):
    B, H, N, _ = q.shape
    o = np.empty(q.shape[:3] + (v.shape[3],), dtype=np.float64)
    lse = np.empty((B, H, N), dtype=np.float64)
    for b in range(B):
        for h in range(H):
            for r0 in range(0, N, block_rows):
                r1 = min(N, r0 + block_rows)
                o[b, h, r0:r1], lse[b, h, r0:r1] = attention_fwd(q[b, h, r0:r1], k[b, h], v[b, h], scale)
    return o, lse


def attention_bwd_bhnd(q, k, v, dO, scale, block_rows=4096):
    B, H, N, _ = q.shape
    dq, dk, dv = np.zeros_like(q), np.zeros_like(k), np.zeros_like(v)
    for b in range(B):
        for h in range(H):
            for r0 in range(0, N, block_rows):
                r1 = min(N, r0 + block_rows)
                a, bk, bv = attention_bwd(q[b, h, r0:r1], k[b, h], v[b, h], dO[b, h, r0:r1], scale)
                dq[b, h, r0:r1] = a
                dk[b, h] += bk
                dv[b, h] += bv
    return dq, dk, dv
