"""Pins added in round 2 (none of them re-types the oracle's formulas):

P19  extended diagnostics (Eq. 11): on a Beltrami mode the kinetic helicity, the current helicity and
     the largest Alfven speed have closed forms in the modified wavenumbers; sign flips with the handedness;
     C against numpy on a random state; the Alfven form of the CFL rule (G15).
P20  the 2N-RK3 coefficients (G7) satisfy ALL four third-order conditions (Butcher tableau rebuilt from alpha, beta in
     exact rationals: b = (1/6, 3/10, 8/15), c = (0, 1/3, 3/4)), and the full NON-LINEAR step converges with order 3
     (error ratio ~8 under dt halving against a dt/16 run): the condition sum b_i c_i^2 = 1/3 never enters a
     linear test.
P22  the alternative reading of G8 (forcing as one impulse per step, oracle flag kick=True): from a zero state the
     step returns exactly u = dt f(x) (Eq. 4 evaluated directly, nothing else touched); on a moving state the two
     readings differ, at O(dt^2) (the coupling of f with the other terms inside the substeps); C against numpy.
P21  the tensor-product reading of the mixed derivative (oracle flag mixed="tensor", G2) has the symbol
     -k1~(a) k1~(b) on a Fourier mode.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import mhd_c, mhd_numpy as mn
from paper_2012_08758_b200 import inputs
from test_oracle_operators import modified_k1, modified_k2sq

L3 = (2 * math.pi,) * 3


def ext(impl):
    return mhd_c.diagnostics_ext if impl == "c" else mn.diagnostics_ext


@pytest.mark.parametrize("impl", ["c", "numpy"])
@pytest.mark.parametrize("hand", [+1, -1])
def test_p19_helicities_of_a_beltrami_mode(impl, hand):
    n, k, a0, u0 = 16, 3.0, 1e-2, 0.3
    shape = (n, 6, 8)
    lengths = (2 * math.pi * 8 / n, 2 * math.pi * 6 / n, 2 * math.pi)
    h = 2 * math.pi / n
    z = np.arange(n) * h
    state = np.zeros((7,) + shape)
    # (sin kz, hand cos kz, 0): curl = hand k (itself); the same mode in u and in A, ln rho = const
    for base, amp in ((1, u0), (4, a0)):
        state[base] = amp * np.sin(k * z)[:, None, None]
        state[base + 1] = hand * amp * np.cos(k * z)[:, None, None]
    state[0] = 0.5
    k1, k2 = modified_k1(k, h), modified_k2sq(k, h)
    d = ext(impl)(state, lengths)
    # omega = hand k1~ u and |u|^2 = u0^2 everywhere; j = k2~ A (div A = 0, the bidiagonal mixed stencil vanishes on
    # a function of z alone), B = hand k1~ A
    assert abs(d["kin_hel"] - hand * k1 * u0 * u0) < 1e-14 * k1 * u0 * u0
    assert abs(d["cur_hel"] - hand * k2 * k1 * a0 * a0) < 1e-13 * k2 * k1 * a0 * a0
    assert abs(d["va_max"] - k1 * a0 * math.exp(-0.25)) < 1e-14 * k1 * a0
    # a uniform external field adds nothing to <j.B> (<j> = 0 in a periodic box) but raises the Alfven speed
    bext = (0.0, 0.0, 0.2)
    db = ext(impl)(state, lengths, bext=bext)
    assert abs(db["cur_hel"] - d["cur_hel"]) < 1e-13 * abs(d["cur_hel"])
    assert abs(db["va_max"] - math.sqrt((k1 * a0) ** 2 + 0.04) * math.exp(-0.25)) < 1e-14


def test_p19_c_matches_numpy_on_a_random_state_and_alfven_cfl():
    shape = (10, 12, 16)
    lengths = (2.0, 1.5, 1.0)
    state = inputs.smooth_strong_state(shape, 77)
    state += np.random.default_rng(77).normal(size=state.shape) * 1e-3       # all wavenumbers present
    for mixed in ("bidiagonal", "tensor"):
        a = mhd_c.diagnostics_ext(state, lengths, bext=(0.01, -0.02, 0.03), mixed=mixed)
        b = mn.diagnostics_ext(state, lengths, bext=(0.01, -0.02, 0.03), mixed=mixed)
        for key in a:
            assert abs(a[key] - b[key]) <= 1e-12 * max(1.0, abs(b[key])), (mixed, key, a[key], b[key])
    # G15 with the Alfven term: c_s -> sqrt(c_s^2 + v_A^2); never larger than the plain rule, equal for v_A = 0
    plain = mn.cfl_dt(0.3, shape, lengths, 1e-3, 2e-3, 1.0)
    assert mn.cfl_dt_alfven(0.3, 0.0, shape, lengths, 1e-3, 2e-3, 1.0) == plain
    hmin = min(l / s for l, s in zip(lengths, shape[::-1]))
    got = mn.cfl_dt_alfven(0.3, 2.0, shape, lengths, 0.0, 0.0, 1.0)
    assert abs(got - 0.4 * hmin / (0.3 + math.sqrt(5.0))) < 1e-15


def test_p20_butcher_tableau_of_the_2n_scheme_in_rationals():
    """w_s = alpha_s w_{s-1} + dt F(y_{s-1}); y_s = y_{s-1} + beta_s w_s  (G7).  Unrolled: the
    coefficient of dt F_j in y_s is a_{s+1, j}; the last row is b; c_i = sum_j a_ij."""
    al = [Fraction(0), Fraction(-5, 9), Fraction(-153, 128)]
    be = [Fraction(1, 3), Fraction(15, 16), Fraction(8, 15)]
    assert [float(x) for x in al] == list(mn.RK_ALPHA) and [float(x) for x in be] == list(mn.RK_BETA)
    wcoef = [Fraction(0)] * 3               # w as a combination of F_0, F_1, F_2
    ycoef = [Fraction(0)] * 3
    rows = []
    for s in range(3):
        rows.append(list(ycoef))            # stage s is evaluated at y_{s-1}
        wcoef = [al[s] * v for v in wcoef]
        wcoef[s] += 1
        ycoef = [ycoef[j] + be[s] * wcoef[j] for j in range(3)]
    b = ycoef
    A = rows
    c = [sum(r) for r in A]
    assert b == [Fraction(1, 6), Fraction(3, 10), Fraction(8, 15)]
    assert c == [Fraction(0), Fraction(1, 3), Fraction(3, 4)]
    assert sum(b) == 1
    assert sum(bi * ci for bi, ci in zip(b, c)) == Fraction(1, 2)
    assert sum(bi * ci * ci for bi, ci in zip(b, c)) == Fraction(1, 3)
    assert sum(b[i] * A[i][j] * c[j] for i in range(3) for j in range(3)) == Fraction(1, 6)


def test_p20_full_nonlinear_step_is_third_order_in_dt():
    n = 12
    state = inputs.smooth_strong_state((n, n, n), 5)
    state[1:4] *= 3.0                                   # u ~ 0.3: the advection terms matter
    T = 0.08

    def run(nsteps):
        st = mhd_c.Stepper(state, L3, 2e-2, 3e-2, 1.0)
        for _ in range(nsteps):
            st.step(T / nsteps, None)
        return st.state.copy()

    ref = run(64)
    errs = [np.abs(run(m) - ref).max() for m in (4, 8, 16)]
    assert errs[2] > 1e-13                              # above round-off: the ratios mean something
    assert 6.5 < errs[0] / errs[1] < 9.5 and 6.5 < errs[1] / errs[2] < 9.5, errs


@pytest.mark.parametrize("impl", ["c", "numpy"])
@pytest.mark.parametrize("a,b", [(0, 1), (0, 2), (1, 2)])
def test_p21_tensor_product_mixed_derivative_symbol(impl, a, b):
    shape = (12, 16, 20)                                # (nz, ny, nx)
    lengths = (2 * math.pi, 2 * math.pi * 0.8, 2 * math.pi * 1.25)   # (lx, ly, lz)
    nn = shape[::-1]
    h = [lengths[i] / nn[i] for i in range(3)]
    kk = [2 * math.pi / lengths[0] * 2, 2 * math.pi / lengths[1] * 3, 2 * math.pi / lengths[2] * 1]
    x = [np.arange(nn[i]) * h[i] for i in range(3)]
    phase = kk[0] * x[0][None, None, :] + kk[1] * x[1][None, :, None] + kk[2] * x[2][:, None, None] + 0.3
    f = np.cos(phase)
    if impl == "c":
        got = mhd_c.dermix_field(f, a, b, lengths, mixed="tensor")
    else:
        got = mn.dermix(f, a, b, h, mixed="tensor")
    want = -modified_k1(kk[a], h[a]) * modified_k1(kk[b], h[b]) * f
    assert np.abs(got - want).max() < 1e-13 * modified_k1(kk[a], h[a]) * modified_k1(kk[b], h[b])
    # and it is NOT the bidiagonal symbol (the two readings differ at this resolution)
    if impl == "numpy":
        bid = mn.dermix(f, a, b, h)
        assert np.abs(bid - want).max() > 1e-6


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p22_forcing_as_one_impulse_per_step(impl):
    from oracle import forcing as of
    shape = (8, 10, 12)
    lengths = (2 * math.pi, 1.5 * math.pi, 2.5 * math.pi)
    dt = 2e-3
    f = of.forcing_from_draws(0.37, 0.81, 0.12, 3, 1.0, dt, 0.05, 1.0, lengths)
    step = mhd_c.step if impl == "c" else mn.step
    zero = np.zeros((7,) + shape)
    got = step(zero, dt, lengths, 1e-2, 1e-2, 1.0, f, kick=True)
    # Eq. 4 written out here: f_i = re_i cos(k.x + phase) - im_i sin(k.x + phase)
    k, phase, re, im = f
    nz, ny, nx = shape
    x = np.arange(nx) * (lengths[0] / nx)
    y = np.arange(ny) * (lengths[1] / ny)
    z = np.arange(nz) * (lengths[2] / nz)
    th = k[0] * x[None, None, :] + k[1] * y[None, :, None] + k[2] * z[:, None, None] + phase
    amp = max(np.abs(re).max(), np.abs(im).max())
    for i in range(3):
        assert np.abs(got[1 + i] - dt * (re[i] * np.cos(th) - im[i] * np.sin(th))).max() <= 1e-15 * dt * amp
    assert np.abs(got[0]).max() == 0.0 and np.abs(got[4:]).max() == 0.0
    # on a moving state the readings differ, but only at second order in dt
    state = inputs.smooth_strong_state(shape, 9)
    a = step(state, dt, lengths, 1e-2, 1e-2, 1.0, f)
    b = step(state, dt, lengths, 1e-2, 1e-2, 1.0, f, kick=True)
    gap = np.abs(a[1:4] - b[1:4]).max()
    assert 0.0 < gap < 20 * dt * dt * amp
    if impl == "c":
        assert np.abs(b - mn.step(state, dt, lengths, 1e-2, 1e-2, 1.0, f, kick=True)).max() < 1e-15
