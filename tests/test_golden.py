"""configs[0] fp64 oracle (decimation + RGF) against the stored extended-precision definition
(tests/golden/config0_extended.txt, written by tests/golden/make_golden.py from oracle/ only)."""
import os

import numpy as np

from oracle import pipeline
from paper_2602_03438_b200 import workloads as W


def test_config0_against_stored_extended_values():
    wl = W.make_workload(0)
    out = pipeline.solve_energy(wl, 0)
    fams = {"GR_diag": out["ret"]["GR_diag"], "GR_upper": out["ret"]["GR_upper"],
            "GR_lower": out["ret"]["GR_lower"], "GL_diag": out["les"]["GX_diag"],
            "GL_upper": out["les"]["GX_upper"]}
    path = os.path.join(os.path.dirname(__file__), "golden", "config0_extended.txt")
    count = 0
    for line in open(path):
        if line.startswith("#"):
            continue
        name, i, r, c, re, im = line.split()
        ref = complex(float(re), float(im))
        got = fams[name][int(i), int(r), int(c)]
        scale = np.abs(fams[name][int(i)]).max()
        assert abs(got - ref) < 1e-10 * scale, (name, i, r, c, got, ref)
        count += 1
    assert count == 22  # 5 samples x 2 diagonal families + 4 x 3 off-diagonal families (block 7 absent there)
