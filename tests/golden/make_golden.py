"""Writes tests/golden/config1_oracle_snr.txt — oracle-written regression values (NOT paper values:
PAPER.md prints no worked LLOID example).  Calls only oracle/ and the seeded input generator.
Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import lloid_oracle as oc                      # noqa: E402
from paper_2410_16416_b200 import workloads as wl          # noqa: E402

w = wl.config1()
b = w.bins[0]
x = w.strain[0].astype(np.float64)
points = [(0, 0), (5, 1), (64, 19209), (65, 19209), (64, 19208), (17, 8191), (100, 12345), (127, 32767),
          (3, 1024 + 95), (40, 20480)]
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle_snr.txt")
with open(out, "w") as f:
    f.write("# oracle regression values, config 1 (workloads.config1(), strain seed 20241016 + 1000): row i, sample k, rho_i[k]\n")
    f.write("# written by tests/golden/make_golden.py from oracle/lloid_oracle.py; not from the paper, not from CUDA\n")
    for i, k in points:
        v = oc.snr_series(x, b.slices, b.basis, b.recon, k, k + 1, wl.K_DOWN, wl.K_UP)[i, 0]
        f.write(f"{i} {k} {v:.15e}\n")
print("wrote", out)
