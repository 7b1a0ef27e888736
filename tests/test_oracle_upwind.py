"""Pins of the upwinded continuity equation (NEXT-1, reading G17; PAPER.md:172 names the method of
Dobler et al. 2006 but prints no formula, so the reading itself is unpinned by the paper).  What the
mathematics fixes: central D1 minus sign(u) delta6/(60 h) is the unique 5th-order stencil on the six
points biased against the flow; it differentiates polynomials of degree <= 5 exactly; its error falls
32 x per halving of h; the C oracle (central + |u| delta6) equals the numpy restatement that picks
the one-sided stencil by the sign of u."""
import math
from fractions import Fraction

import numpy as np

from oracle import mhd_c, mhd_numpy
from paper_2012_08758_b200 import inputs

L3 = (2 * math.pi,) * 3


def solve_rational(A, b):
    n = len(b)
    M = [row[:] + [bb] for row, bb in zip(A, b)]
    for i in range(n):
        piv = next(r for r in range(i, n) if M[r][i] != 0)
        M[i], M[piv] = M[piv], M[i]
        M[i] = [v / M[i][i] for v in M[i]]
        for r in range(n):
            if r != i and M[r][i] != 0:
                M[r] = [vr - M[r][i] * vi for vr, vi in zip(M[r], M[i])]
    return [M[i][n] for i in range(n)]


def test_upwind_stencil_is_the_unique_5th_order_one_on_its_six_points():
    # weights w_m on m = -3 .. +2 with sum w_m m^p = delta_{p,1}, p = 0 .. 5  (h = 1)
    pts = [-3, -2, -1, 0, 1, 2]
    A = [[Fraction(m) ** p for m in pts] for p in range(6)]
    w = solve_rational(A, [Fraction(int(p == 1)) for p in range(6)])
    assert [x * 60 for x in w] == [-2, 15, -60, 20, 30, -3]
    assert tuple(float(x * 60) for x in w) == mhd_numpy.UPW5
    # the C oracle's operators on a unit impulse: central D1 - delta6/60 reproduces those weights
    n = 16
    f = np.zeros((n, n, n))
    f[5, 6, 7] = 1.0
    lengths = (float(n),) * 3                                  # h = 1
    for a, idx in ((0, lambda m: (5, 6, 7 - m)), (1, lambda m: (5, 6 - m, 7)), (2, lambda m: (5 - m, 6, 7))):
        comb = mhd_c.der1_field(f, a, lengths) - mhd_c.der6_upwind_field(f, a, lengths)
        got = [comb[idx(m)] * 60 for m in pts] + [comb[idx(3)] * 60]
        assert np.allclose(got, [-2, 15, -60, 20, 30, -3, 0], atol=1e-13)
        mirror = mhd_c.der1_field(f, a, lengths) + mhd_c.der6_upwind_field(f, a, lengths)
        got = [mirror[idx(-m)] * 60 for m in pts] + [mirror[idx(-3)] * 60]
        assert np.allclose(got, [2, -15, 60, -20, -30, 3, 0], atol=1e-13)


def test_upwind_derivative_is_5th_order_on_a_sine():
    errs = []
    for n in (16, 32, 64):
        x = np.arange(n) * (2 * math.pi / n)
        f = np.broadcast_to(np.sin(2 * x), (4, 4, n)).copy()
        d = mhd_c.der1_field(f, 0, (2 * math.pi,) * 3) - mhd_c.der6_upwind_field(f, 0, (2 * math.pi,) * 3)
        errs.append(np.abs(d[0, 0] - 2 * np.cos(2 * x)).max())
    assert 25 < errs[0] / errs[1] < 40 and 28 < errs[1] / errs[2] < 36          # 2^5 = 32


def test_upwind_rhs_c_equals_numpy_and_only_touches_continuity():
    shape = (12, 10, 14)
    state = inputs.smooth_strong_state(shape, 3)
    state[0] += 0.05 * inputs.uniform_state(shape, 9)[0]       # rough ln rho: delta6 is far from zero
    lengths = (2 * math.pi, 1.7 * math.pi, 2.3 * math.pi)
    f = ((1.0, 2.0, 0.0), 0.4, (0.01, 0.0, 0.02), (0.0, 0.03, 0.0))
    r_c = mhd_c.rhs(state, lengths, 1e-2, 2e-2, 1.1, f, upwind=True)
    r_n = mhd_numpy.rhs(state, lengths, 1e-2, 2e-2, 1.1, f, upwind=True)
    r_0 = mhd_c.rhs(state, lengths, 1e-2, 2e-2, 1.1, f, upwind=False)
    scale = np.abs(r_0[0]).max()
    assert np.abs(r_c[0] - r_n[0]).max() <= 1e-12 * scale
    assert np.abs(r_c[0] - r_0[0]).max() > 1e-3 * scale        # the correction is there
    assert np.array_equal(r_c[1:], r_0[1:])                    # momentum and induction untouched
    # the correction is dissipative: it has the sign of |u| delta6, i.e. it damps the grid-scale mode
    n = 16
    st = np.zeros((7, n, n, n))
    st[0] = 1e-3 * (-1.0) ** np.arange(n)[None, None, :]       # Nyquist mode in x
    st[1] = 0.5
    r = mhd_c.rhs(st, L3, 0.0, 0.0, 1.0, None, upwind=True)[0]
    assert np.all(r * st[0] < 0)                               # d ln rho/dt opposes the mode
    assert np.abs(mhd_c.rhs(st, L3, 0.0, 0.0, 1.0, None, upwind=False)[0]).max() < 1e-15   # central D1 is blind to it


def test_upwind_step_c_equals_numpy():
    state = inputs.smooth_strong_state(12, 4)
    a = mhd_c.step(state, 1e-3, L3, 5e-3, 5e-3, 1.0, None, upwind=True)
    b = mhd_numpy.step(state, 1e-3, L3, 5e-3, 5e-3, 1.0, None, upwind=True)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()
    c = mhd_c.step(state, 1e-3, L3, 5e-3, 5e-3, 1.0, None, upwind=False)
    assert np.abs(a[0] - c[0]).max() > 0
