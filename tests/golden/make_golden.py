"""Writes tests/golden/config1_cg.txt from the oracle alone (never from the CUDA path)."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
from oracle import nko                                    # noqa: E402
from workloads import config_mesh, config_rhs, CONFIGS    # noqa: E402

m = config_mesh("config1")
o = nko.Oracle.from_mesh(m)
x, hist = o.cg(config_rhs("config1", m), CONFIGS["config1"]["niter"])
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_cg.txt")
with open(out, "w") as f:
    f.write("# oracle residual history, config 1 (E=8, N=3, a=0.05, seed 1001, 20 iterations), then max|x|\n")
    for h in hist:
        f.write(f"{h:.17e}\n")
    f.write(f"{np.max(np.abs(x)):.17e}\n")
print(out)
