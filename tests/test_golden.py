"""Golden fixtures: constants the paper prints, and a drift guard for the oracle."""
import math
import os

import numpy as np

from oracle import forcing as of, mhd_c
from paper_2012_08758_b200 import inputs

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def paper_constants():
    out = {}
    for line in open(os.path.join(HERE, "paper_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_paper_constants_are_what_the_code_uses():
    c = paper_constants()
    # k_f = 5 shell of the paper: every vector lies in the printed range, both ends are reached
    norms = [math.sqrt(a * a + b * b + cc * cc) for a, b, cc in of.shell(5)]
    assert min(norms) >= c["shell_lo_kf5"] and max(norms) <= c["shell_hi_kf5"]
    assert min(norms) < 4.6 and max(norms) > 5.4
    assert c["box_side_over_pi"] * math.pi == 2 * math.pi
    # the paper's 35x is its two per-cell times
    assert abs(c["pencil_ns_per_cell_step_40cores"] / c["astaroth_ns_per_cell_step_4xV100"] - c["speedup"]) < 1.0
    # 1.19209e-7 is 2^-23 (single-precision epsilon), to the printed digits
    assert abs(c["benchmark_dt"] - 2.0 ** -23) < 5e-13


def test_oracle_drift_guard_config1():
    L3 = (2 * math.pi,) * 3
    seed = 1001
    st = mhd_c.Stepper(inputs.gaussian_state(32, seed), L3, 5e-3, 5e-3, 1.0)
    want = {}
    for line in open(os.path.join(HERE, "oracle_config1_samples.txt")):
        if line.startswith("#"):
            continue
        p = line.split()
        if p[1] == "diag":
            want[(int(p[0]), p[2])] = float(p[3])
        else:
            want[(int(p[0]), int(p[1]), int(p[2]), int(p[3]), int(p[4]))] = float(p[5])
    for step in range(10):
        u = inputs.counter_uniforms(seed + 7, step)
        st.step(1e-3, of.forcing_from_draws(*u, 3, 0.0, 1e-3, 0.02, 1.0))
        if step in (0, 9):
            d = st.diagnostics()
            scale = {0: 1e-3, 1: 1e-3, 2: 1e-3, 3: 1e-3, 4: 1e-5, 5: 1e-5, 6: 1e-5}
            for key, val in want.items():
                if key[0] != step + 1:
                    continue
                if isinstance(key[1], str):
                    assert abs(d[key[1]] - val) <= 1e-12 * abs(val)
                else:
                    _, q, z, y, x = key
                    assert abs(st.state[q, z, y, x] - val) <= 1e-12 * scale[q]
