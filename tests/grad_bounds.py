"""Element-wise error bounds for the bf16 gradients (test helper; uses only oracle/ and numpy).

The stated tolerance for gradients is a relative Frobenius norm (BASELINE.json: <= 2e-2), which cannot see one bad row
in 65536.  Beside it every gradient check applies, element by element,

    |g_e - ref_e|  <=  2^-7 |ref_e|  +  8 * 2^-8 * rms(ref)  +  Dterm_e

* 2^-7 |ref_e|: the bf16 output rounding (2^-9 |ref_e|) with margin.
* 8 * 2^-8 * rms(ref): a gradient element is a sum of n products of bf16-rounded factors (P, dS: unit roundoff 2^-9
  each, signs independent), accumulated in fp32, so its error is ~2^-9 * rms(ref) * O(1) -- not n times a term; 8 * 2^-8
  is ~16x that.  A misplaced or missing element is off by O(rms(ref)), thirty times the bound.
* Dterm_e: the kernel forms D_i = dO_i . O_i from the SAVED bf16 O (last bullet of the tolerance analysis;
  DESIGN.md reading g8), the oracle from the exact O.  |delta D_i| <= 2^-9 sum_c |dO_ic| |O_ic| =: E_i, and since
  dS_ij = P_ij (dP_ij - D_i), this moves  dQ_ic by scale * |sum_j P_ij k_jc| * E_i  and  dK_jc by
  scale * sum_i P_ij |q_ic| E_i  (dV does not depend on D).  It is negligible for diffuse softmax rows and the leading term
  for sharply peaked ones, where dS is a small difference of O(1) quantities (measured: up to 1.8x the first two terms on
  a Q,K x 3 config; 0.57 of Dterm itself).
"""
import numpy as np

from oracle import attention as orc

U_BF16 = 2.0 ** -9


def d_error_rows(q_rows, k, v, dO_rows, scale):
    """E_i = 2^-9 sum_c |dO_ic| |O_ic| for the given query rows (O from the oracle's forward)."""
    o, _ = orc.attention_fwd(q_rows, k, v, scale)
    return U_BF16 * (np.abs(dO_rows) * np.abs(o)).sum(axis=1)


def dq_dterm(q_rows, k, v, dO_rows, scale):
    """scale * |sum_j P_ij k_jc| * E_i -- the attention-averaged key is the oracle's forward with V := K."""
    kbar, _ = orc.attention_fwd(q_rows, k, k, scale)
    return scale * np.abs(kbar) * d_error_rows(q_rows, k, v, dO_rows, scale)[:, None]


def dk_dterm(q_rows, k_cols, lse_rows, E_rows, scale):
    """scale * sum_i P_ij |q_ic| E_i for the key columns given; P from the rows' LSE (as attention_bwd_cols does)."""
    p = np.exp(orc.scores(q_rows, k_cols, scale) - lse_rows[:, None])        # [rows, cols]
    return scale * (p.T @ (np.abs(q_rows) * E_rows[:, None]))


def excess(g, ref, dterm=None):
    """max_e |g_e - ref_e| / bound_e (must be <= 1)."""
    g = np.asarray(g, dtype=np.float64)
    rms = np.sqrt(np.mean(ref * ref))
    bound = 2.0 ** -7 * np.abs(ref) + 8.0 * 2.0 ** -8 * rms
    if dterm is not None:
        bound = bound + dterm
    return float((np.abs(g - ref) / bound).max())


def check_grad(name, g, ref, dterm=None, tol=2e-2):
    """relative Frobenius error <= tol (the stated bar) AND the element-wise bound; returns the Frobenius error."""
    g = np.asarray(g, dtype=np.float64)
    assert np.isfinite(g).all(), name
    e = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    assert e <= tol, (name, "relative Frobenius error", e)
    x = excess(g, ref, dterm)
    assert x <= 1.0, (name, "element-wise bound exceeded", x)
    return e
