"""NEXT-2: the whole step against numbers the paper prints.  Tables 1-2
 give, for N = 64, eta = nu = 5e-3, k_f = 5, the magnetic Reynolds number and the
exponential growth rate lambda of B_rms (Eq. 8) under helical (sigma = 1: a dynamo, lambda > 0) and
non-helical (sigma = 0: decay, lambda < 0) forcing, from a weak delta-correlated Gaussian seed field,
uniform density and zero velocity.  About 2 x 10^4 RK3 steps per case: only the GPU
path can run it (the oracle needs more than an hour), so this pins the CUDA path directly to the paper.

Reading G23: with f0 = 0.08 in Eq. 5 as printed the flow settles at u_rms = 0.22
(Re_M = 8.8), not at the Re_M = 3.5-3.6 of the tables - the paper's amplitude convention is at odds
with its own Eq. 5.  Re_M, not f0, is what the tables are indexed by, so the run calibrates f0 on a
short precursor (the flow at Re = 3.6 is almost linear in f0) until u_rms matches the printed Re_M,
and then compares lambda."""
import math
import os

import numpy as np
import pytest

from paper_2012_08758_b200 import binding

pytestmark = pytest.mark.gpu
HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def paper_constants():
    out = {}
    for line in open(os.path.join(HERE, "paper_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def shell_mean_k(k_f):
    r = int(k_f + 1)
    ks = [math.sqrt(a * a + b * b + c * c) for a in range(-r, r + 1) for b in range(-r, r + 1) for c in range(-r, r + 1)
          if (k_f - 0.5) ** 2 <= a * a + b * b + c * c <= (k_f + 0.5) ** 2]
    return sum(ks) / len(ks)


def run(ctx, n, f0, dt, t_end, seed, every=100):
    rng = np.random.default_rng(42)
    st = np.zeros((7, n, n, n))
    st[4:7] = rng.standard_normal((3, n, n, n)) * 1e-5
    ctx.ac_load_state(st.astype(ctx.np_dtype))
    log = []
    for s in range(int(t_end / dt)):
        ctx.ac_step(dt, ctx.ac_make_forcing(seed, s, dt, f0))
        if s % every == every - 1:
            d = ctx.ac_reduce()
            assert d["nonfinite"] == 0
            log.append(((s + 1) * dt, d["urms"], d["brms"]))
    return np.array(log)


@pytest.mark.parametrize("dtype,upwind", [(binding.AC_F64, False), (binding.AC_F32, False), (binding.AC_F64, True)])
@pytest.mark.parametrize("sigma,table", [(1.0, "table1"), (0.0, "table2")])
def test_growth_rate_of_brms_matches_tables_1_and_2(sigma, table, dtype, upwind):
    c = paper_constants()
    n, eta, k_f = 64, c["table1_N64_eta"], int(c["kf_paper"])
    lam_paper, rem_paper = c[table + "_N64_lambda"], c[table + "_N64_ReM"]
    kbar = shell_mean_k(k_f)                               # "k_f is the average wave number of the forcing"
    u_target = rem_paper * eta * kbar
    ctx = binding.Context((n, n, n), dtype=dtype, nu=eta, eta=eta, cs=1.0, k_f=k_f, helicity=sigma)
    ctx.ac_set_upwind(upwind)                              # the paper's production runs used upwinding
    h = 2 * math.pi / n
    dt = 0.4 * h / 1.4
    f0 = 0.03
    for _ in range(2):                                     # precursor runs: u_rms is nearly linear in f0
        pre = run(ctx, n, f0, dt, 80.0, seed=7)
        f0 *= u_target / pre[pre[:, 0] > 30.0, 1].mean()
    log = run(ctx, n, f0, dt, 600.0, seed=7)
    ctx.ac_free()
    grow = log[log[:, 0] >= 150.0]                         # past the decay of the small-scale part of the seed
    rem = grow[:, 1].mean() / (eta * kbar)
    lam = np.polyfit(grow[:, 0], np.log(grow[:, 2]), 1)[0]
    print("dtype %s upwind %s" % ("f64" if dtype == binding.AC_F64 else "f32", upwind), end=" ")
    print("sigma %.0f: f0 %.4f Re_M %.3f (paper %.2f) lambda %.4e (paper %.2e)" % (sigma, f0, rem, rem_paper, lam, lam_paper))
    # CALIBRATION check, not a comparison: f0 was tuned on the precursor runs until u_rms gives the printed Re_M
    # (reading G23: Eq. 5 as printed, with f0 = 0.08, gives Re_M = 8.8, not the tables' 3.6), so this only says that
    # the tuning converged.  The amplitude of Eq. 5 on the GPU path is pinned by parity with the oracle, whose own pin
    # is P12 (box mean of |f|^2 = N^2 / 2).  The comparison with the paper is the growth rate below.
    assert abs(rem - rem_paper) <= 0.05 * rem_paper, "f0 calibration did not converge"
    # the paper's own rows for this eta differ by 7 % between resolutions; one forcing realisation adds scatter
    assert abs(lam - lam_paper) <= 0.25 * abs(lam_paper)
    assert (lam > 0) == (sigma == 1.0)
