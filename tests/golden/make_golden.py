"""Writes tests/golden/config0_extended.txt.  Calls ONLY oracle/ and the input generator.

The paper prints no worked numeric example (Figs. 3, 4, 6 are images), so
there is no paper value to store.  What is stored instead is the DEFINITION (PAPER.md:56-58,
Eqs. 1-2) evaluated by 80-bit extended-precision dense Gauss-Jordan inversion on
BASELINE.json:configs[0] with the Sigma_B of the fp64 decimation, sampled at fixed entries.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import dense, pipeline  # noqa: E402
from paper_2602_03438_b200 import workloads as W  # noqa: E402

SAMPLES = [(0, 0, 0), (0, 3, 7), (3, 15, 2), (7, 9, 9), (5, 0, 15)]   # (block, row, col)


def main():
    wl = W.make_workload(0)
    out = pipeline.solve_energy(wl, 0)
    d = dense.dense_green(*out["A"], B_list=[out["BL"]], extended=True)
    lines = ["# family block row col re im   (80-bit dense definition, configs[0], E=0.3, eta=1e-6)"]
    fams = {"GR_diag": d["GR"][0], "GR_upper": d["GR"][1], "GR_lower": d["GR"][2],
            "GL_diag": d["GX"][0][0], "GL_upper": d["GX"][0][1]}
    for name, arr in fams.items():
        for (i, r, c) in SAMPLES:
            if i >= arr.shape[0]:
                continue
            v = complex(arr[i, r, c])
            lines.append(f"{name} {i} {r} {c} {v.real:.17e} {v.imag:.17e}")
    with open(os.path.join(os.path.dirname(__file__), "config0_extended.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
