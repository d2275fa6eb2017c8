"""fp64 CPU oracle for the Turbulence-Transformer tokeniser.
*** TEST INFRASTRUCTURE ONLY *** -- same rules as oracle/attention.py: only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s CPU legs may import it; it shares no code with the CUDA path.

What the paper states: the state is `Y in R^{D x H x W x 4}` (three velocity
components and pressure); a fidelity mode is a sub-domain selection `C_i(.)` of size
`D_i x H_i x W_i` "centered at [x_ci, y_ci, z_ci]" followed by a Gaussian filter `F_i(.)` "of kernel
size k_i^3 ... via convolution", the result lying in `R^{D_i/k_i x H_i/k_i x W_i/k_i x 4}`
(low fidelity: no crop; high fidelity: no filter, i.e. k = 1).  Each filtered voxel is a token
(patch size 1), and M input states are concatenated along the sequence.

The definition written out: with `(z0, y0, x0)` the crop origin and `G` a normalised k^3 Gaussian,

    T[m, z', y', x', c] = sum_{a,b,e = 0}^{k-1} G[a,b,e] * Y[m, z0 + k z' + a, y0 + k y' + b, x0 + k x' + e, c]

Readings where the paper is silent (t1-t6):
  t1  output size D_i/k_i  =>  the convolution has stride k (windows tile the crop, no overlap, no padding).
  t2  G[a,b,e] = g[a] g[b] g[e] / (sum g)^3,  g[a] = exp(-(a - (k-1)/2)^2 / (2 sigma^2)); sigma is an
      explicit argument; the default sigma = k / sqrt(12) is the LES Gaussian filter of width
      Delta = k grid spacings (G(r) ~ exp(-6 r^2 / Delta^2)), the paper's own analogy.
  t3  the crop must lie inside the domain (no periodic wrap); D_i, H_i, W_i are multiples of k.
  t4  F(C(Y)): crop first, then filter; with t1 the order does not matter.
  t5  layout: Y [M, D, H, W, 4], channels fastest (the paper's R^{D x H x W x 4}); tokens
      [M, D_i/k, H_i/k, W_i/k, 4] = [L, 4] with x' fastest (the order of BASELINE.json's C2).
  t6  "centered at": origin = centre - size/2 (integer division); the functions below take the origin.

Pins (tests/test_oracle_pins_fidelity.py): constant field -> the constant; k = 1 -> the crop itself;
unit impulse reads G[a,b,e]; k = 2 -> box filter (all eight weights 1/8 by symmetry); affine field
-> its value at the window centre (G symmetric, sums to 1); a hand fixture for k = 3 under
tests/golden/; brute-force Python loops; a library second opinion (torch conv3d fp64, stride k).
"""
from __future__ import annotations

import math

import numpy as np


def default_sigma(k: int) -> float:
    """LES Gaussian filter of width Delta = k: variance Delta^2 / 12 (reading t2)."""
    return k / math.sqrt(12.0)


def gaussian_weights_1d(k: int, sigma: float):
    """g[a] / sum(g), a = 0..k-1, centred on (k-1)/2 (reading t2)."""
    a = np.arange(k, dtype=np.float64)
    g = np.exp(-((a - 0.5 * (k - 1)) ** 2) / (2.0 * sigma * sigma))
    return g / g.sum()


def gaussian_kernel_3d(k: int, sigma: float):
    """G[a,b,e] = w[a] w[b] w[e]: the normalised k^3 Gaussian kernel."""
    w = gaussian_weights_1d(k, sigma)
    return w[:, None, None] * w[None, :, None] * w[None, None, :]


def crop_origin(centre, size):
    """"centered at [x_c, y_c, z_c]" -> origin = centre - size // 2 (reading t6)."""
    return tuple(int(c) - int(s) // 2 for c, s in zip(centre, size))


def fidelity_tokens(y, origin, size, k, sigma=None):
    """F_k(C(Y)).  y [M, D, H, W, C] float64; origin (z0,y0,x0); size (Dc,Hc,Wc).
    Returns T [M, Dc/k, Hc/k, Wc/k, C] float64."""
    y = np.asarray(y, dtype=np.float64)
    z0, y0, x0 = origin
    Dc, Hc, Wc = size
    M, D, H, W, C = y.shape
    if min(z0, y0, x0) < 0 or z0 + Dc > D or y0 + Hc > H or x0 + Wc > W:
        raise ValueError("crop outside the domain (reading t3)")
    if Dc % k or Hc % k or Wc % k:
        raise ValueError("crop size must be a multiple of k (reading t3)")
    sigma = default_sigma(k) if sigma is None else sigma
    G = gaussian_kernel_3d(k, sigma)
    c = y[:, z0:z0 + Dc, y0:y0 + Hc, x0:x0 + Wc, :]          # C(Y)
    out = np.zeros((M, Dc // k, Hc // k, Wc // k, C), dtype=np.float64)
    for a in range(k):                                        # the triple sum of the definition
        for b in range(k):
            for e in range(k):
                out += G[a, b, e] * c[:, a::k, b::k, e::k, :]
    return out
