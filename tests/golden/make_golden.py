"""Writes tests/golden/oracle_config1_samples.txt from the C oracle ONLY (never from the CUDA
path): BASELINE config 1 (32^3, nu = eta = 5e-3, non-helical forcing k_f = 3, f0 = 0.02, fixed
dt = 1e-3), sampled state values after 1 and 10 steps plus the diagnostics.  It is a drift guard
for the oracle, not a pin (the pins are tests/test_oracle_*.py).

Run from the repo root:  python tests/golden/make_golden.py
"""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import forcing as of, mhd_c                      # noqa: E402
from paper_2012_08758_b200 import inputs                      # noqa: E402

SEED = 1001
L3 = (2 * math.pi,) * 3
SAMPLES = [(0, 0, 0), (31, 31, 31), (5, 17, 29), (16, 0, 31), (30, 2, 1), (13, 13, 13)]    # (z, y, x)


def main():
    state = inputs.gaussian_state(32, SEED)
    st = mhd_c.Stepper(state, L3, 5e-3, 5e-3, 1.0)
    lines = ["# written by tests/golden/make_golden.py from oracle/mhd_oracle.c; step field z y x value"]
    for step in range(10):
        u = inputs.counter_uniforms(SEED + 7, step)
        f = of.forcing_from_draws(*u, 3, 0.0, 1e-3, 0.02, 1.0)
        st.step(1e-3, f)
        if step in (0, 9):
            for q in range(7):
                for (z, y, x) in SAMPLES:
                    lines.append("%d %d %d %d %d %.17e" % (step + 1, q, z, y, x, st.state[q, z, y, x]))
            d = st.diagnostics()
            for key in ("urms", "umax", "brms", "bmax"):
                lines.append("%d diag %s %.17e" % (step + 1, key, d[key]))
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_config1_samples.txt"), "w") as fh:
        fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
