#!/usr/bin/env python
"""Writes tests/golden/bf16_ragged_expected.txt: the fp64 oracle's O, LSE, dQ, dK, dV for a ragged bf16 problem
(B=1, H=2, N=333, d=128, scale 1/sqrt(128); q, k, v, dO the seeded N(0,1) bf16 tensors of
paper_2507_16697_b200/workloads.py, seed 20250731) on a sample of entries.  Calls only `oracle/` and the seeded input
generator -- never the CUDA path.  Read by tests/c_abi/ringx_bf16_ragged.c.

    python tests/golden/make_bf16_ragged_golden.py

Sample: LSE of every row; O, dQ (query rows) and dK, dV (key rows) of rows {0, 127, 128, 256, 331, 332} of
both heads, all 128 columns -- the rows either side of every 128-row tile boundary and the last rows of the ragged tile.
Lines are "<tensor> <flat index into [2,333,128] (or [2,333] for lse)> <value>".  Eq. 1 / Eq. 3 and
the derivative of Eq. 1 (reading g8).
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import attention as orc                      # noqa: E402
from paper_2507_16697_b200 import workloads as wl        # noqa: E402

SHAPE = (1, 2, 333, 128)
SEED = 20250731
ROWS = (0, 127, 128, 256, 331, 332)


def inputs():
    return tuple(wl.make_tensor(SHAPE, w, seed=SEED, dtype="bf16") for w in ("q", "k", "v", "do"))


def expected():
    """[(tensor, flat index, value)] in file order."""
    q, k, v, do = (wl.to_f64_numpy(t) for t in inputs())
    _, H, N, d = SHAPE
    scale = d ** -0.5
    o, lse = orc.attention_fwd_bhnd(q, k, v, scale)
    dq, dk, dv = orc.attention_bwd_bhnd(q, k, v, do, scale)
    out = []
    for h in range(H):
        for n in range(N):
            out.append(("lse", h * N + n, lse[0, h, n]))
    for name, t in (("o", o), ("dq", dq), ("dk", dk), ("dv", dv)):
        for h in range(H):
            for n in ROWS:
                for c in range(d):
                    out.append((name, (h * N + n) * d + c, t[0, h, n, c]))
    return out


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "bf16_ragged_expected.txt")
    vals = expected()
    with open(path, "w") as f:
        f.write("# ragged bf16 forward + backward (B=1 H=2 N=333 d=128): expected values from oracle.attention "
                "(attention_fwd_bhnd, attention_bwd_bhnd; fp64), written by tests/golden/make_bf16_ragged_golden.py; seed %d\n" % SEED)
        for name, idx, val in vals:
            f.write("%s %d %.10g\n" % (name, idx, val))
    print(path, len(vals), "values")


if __name__ == "__main__":
    main()
