"""Writes tests/golden/configs0_oracle.txt: sampled outputs of the oracle (brute-force DFT
mode) on BASELINE.json configs[0].  Calls only oracle/ and the seeded input generators;
nothing here comes from the CUDA path.  Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import afno_oracle  # noqa: E402
from paper_2208_05419_b200 import inputs  # noqa: E402

wl = inputs.WORKLOADS["tiny"]
d = inputs.make_inputs(wl)
cfg = afno_oracle.Config(wl.B, wl.H, wl.W, wl.C, wl.num_blocks, lam=float(np.float32(wl.lam)),
                         naive_dft=True)
y = afno_oracle.forward(cfg, d["x"], d["w1"], d["b1"], d["w2"], d["b2"])
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "configs0_oracle.txt")
with open(out, "w") as f:
    f.write("# BASELINE.json configs[0] (B=1, 8x16, C=16, 2 blocks, lambda=0.01, kept 1.0)\n")
    f.write("# oracle forward, brute-force O(N^2) DFT, fp64.  Columns: h w c y[0,h,w,c]\n")
    f.write("# written by tests/golden/make_golden.py (calls only oracle/)\n")
    for (h, w, c) in [(0, 0, 0), (1, 2, 3), (3, 7, 8), (7, 15, 15), (4, 9, 5), (2, 11, 12)]:
        f.write(f"{h} {w} {c} {float(y[0, h, w, c])!r}\n")
print(open(out).read())
