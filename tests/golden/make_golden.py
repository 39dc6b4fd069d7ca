"""Writes tests/golden/config0_oracle_samples.txt: sampled entries of the FP64 oracle result for
BASELINE.json configs[0] (M=64, N=256, K=256, A and B FP32 N(0,1), seed 0).  Calls only oracle/ and
the seeded input generator; nothing here touches the CUDA path.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2606_21023_b200 import inputs  # noqa: E402

A = inputs.activations(64, 256, seed=0)
B = inputs.weights_f32(256, 256, seed=0, dist="normal")
C = oracle.gemm_f64(A, B)
pts = [(0, 0), (0, 255), (63, 0), (63, 255), (31, 128), (32, 127), (1, 64), (17, 200), (40, 3), (62, 254)]
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle_samples.txt"), "w") as f:
    f.write("# i j Cref[i][j] -- oracle.gemm_f64 on configs[0] inputs (seed 0); written by make_golden.py\n")
    for i, j in pts:
        f.write(f"{i} {j} {float(C[i, j])!r}\n")
