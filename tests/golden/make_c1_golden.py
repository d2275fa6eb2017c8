#!/usr/bin/env python
"""Writes tests/golden/c1_expected.txt: the fp64 oracle's O and LSE for BASELINE.json configs[0] (C1: fp32, B=1, H=1,
N=1024, d=64, scale 1/8; Q,K,V the seeded N(0,1) tensors of paper_2507_16697_b200/workloads.py) on a sample of entries.
Calls only `oracle/` and the seeded input generator -- never the CUDA path.  Read by tests/c_abi/ringx_c1.c.

    python tests/golden/make_c1_golden.py

Sample: LSE of every 8th row plus the last row; O of rows {0, 1, 127, 128, 255, 256, 511, 512, 767, 768, 1000, 1023} plus
every 64th row, all 64 columns.  The oracle evaluates Eq. 1 / Eq. 3 unchunked; the program under test
runs the four-chunk forms, which must agree to rounding (Eq. 5).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import attention as orc                      # noqa: E402
from paper_2507_16697_b200 import workloads as wl        # noqa: E402


def main():
    cfg = wl.CONFIGS["C1"]
    q, k, v = wl.make_qkv(cfg)
    o, lse = orc.attention_fwd(wl.to_f64_numpy(q[0, 0]), wl.to_f64_numpy(k[0, 0]), wl.to_f64_numpy(v[0, 0]), cfg.scale)
    lse_rows = sorted(set(range(0, cfg.N, 8)) | {cfg.N - 1})
    o_rows = sorted({0, 1, 127, 128, 255, 256, 511, 512, 767, 768, 1000, 1023} | set(range(0, cfg.N, 64)))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_expected.txt")
    with open(out, "w") as f:
        f.write("# C1 (BASELINE.json configs[0]) expected values from oracle.attention.attention_fwd (fp64), Eq. 1 / Eq. 3 "
                "(PAPER.md:89, 124); written by tests/golden/make_c1_golden.py; seed %d\n" % cfg.seed)
        for r in lse_rows:
            f.write("lse %d %.17g\n" % (r, lse[r]))
        for r in o_rows:
            for c in range(cfg.d):
                f.write("o %d %d %.17g\n" % (r, c, o[r, c]))
    print(out, len(lse_rows), "lse values,", len(o_rows) * cfg.d, "o values")


if __name__ == "__main__":
    main()
