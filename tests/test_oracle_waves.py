"""Pins P4, P7-P11, P17: the oracle's time step against closed forms.  For a single Fourier
mode the discrete step is exactly y_{n+1} = R(dt M) y_n with R(z) = 1 + z + z^2/2 + z^3/6 (any
3-stage 3rd-order Runge-Kutta scheme) and M built from the modified wavenumbers of the 6th-order
stencils; both facts are textbook results, independent of the oracle's code."""
import math

import numpy as np
import pytest

from oracle import mhd_c, mhd_numpy as mn
from test_oracle_operators import modified_k1, modified_k2sq, modified_kxy

L3 = (2 * math.pi,) * 3
IMPLS = ["c", "numpy"]


def stepper(impl):
    return mhd_c.step if impl == "c" else mn.step


def R(z):
    """Stability polynomial of a 3-stage 3rd-order RK scheme; z scalar or matrix."""
    if np.ndim(z) == 0:
        return 1 + z + z * z / 2 + z * z * z / 6
    I = np.eye(z.shape[0])
    return I + z + z @ z / 2 + z @ z @ z / 6


@pytest.mark.parametrize("impl", IMPLS)
def test_p8_shear_wave_decays_with_stability_polynomial_and_p4_third_order(impl):
    n, k, nu, eps = 16, 2.0, 5e-2, 1e-3
    shape = (8, 8, n)
    lengths = (2 * math.pi, 2 * math.pi * 8 / n, 2 * math.pi * 8 / n)
    h = 2 * math.pi / n
    x = np.arange(n) * h
    state = np.zeros((7,) + shape)
    state[2] = eps * np.cos(k * x)[None, None, :]
    k2 = modified_k2sq(k, h)
    dt = 0.05
    s = state
    for _ in range(4):
        s = stepper(impl)(s, dt, lengths, nu, 0.0, 1.0)
    expect = R(-nu * k2 * dt) ** 4 * state[2]
    assert np.abs(s[2] - expect).max() < 1e-14 * eps
    assert np.abs(s[[0, 1, 3, 4, 5, 6]]).max() < 1e-18
    # P4: third order in dt against the exact solution of the semi-discrete ODE
    errs = []
    T = 0.8
    lam = -nu * k2 * 10.0          # |lam dt| = 0.4, 0.2, 0.1: asymptotic and well above round-off
    for nsteps in (4, 8, 16):
        dt = T / nsteps
        s = state
        for _ in range(nsteps):
            s = stepper(impl)(s, dt, lengths, nu * 10.0, 0.0, 1.0)
        errs.append(abs(s[2, 0, 0, 0] - math.exp(lam * T) * eps))
    assert 7.0 < errs[0] / errs[1] < 10.5 and 7.4 < errs[1] / errs[2] < 9.0


@pytest.mark.parametrize("impl", IMPLS)
def test_p7_beltrami_mode_resistive_decay(impl):
    n, k, eta, a0 = 16, 3.0, 2e-2, 1e-2
    shape = (n, 6, 8)
    lengths = (2 * math.pi * 8 / n, 2 * math.pi * 6 / n, 2 * math.pi)
    h = 2 * math.pi / n
    z = np.arange(n) * h
    state = np.zeros((7,) + shape)
    state[4] = a0 * np.sin(k * z)[:, None, None]
    state[5] = a0 * np.cos(k * z)[:, None, None]
    k2 = modified_k2sq(k, h)
    dt = 0.02
    s = state
    for _ in range(5):
        s = stepper(impl)(s, dt, lengths, 1e-2, eta, 1.0)
    fac = R(-eta * k2 * dt) ** 5
    assert np.abs(s[4] - fac * state[4]).max() < 2e-15 * a0
    assert np.abs(s[5] - fac * state[5]).max() < 2e-15 * a0
    # discretely force free: the velocity stays at round-off of j x B (|j||B| ~ k^3 a0^2 ~ 3e-3)
    roundoff = 100 * 2.2e-16 * (k ** 3 * a0 * a0) * (5 * dt)
    assert np.abs(s[1:4]).max() < roundoff
    assert np.abs(s[0]).max() < roundoff
    # B = k1~ A and |B| diagnostics
    d = (mhd_c.diagnostics if impl == "c" else mn.diagnostics)(state, lengths)
    assert abs(d["brms"] - modified_k1(k, h) * a0) < 1e-15


@pytest.mark.parametrize("impl", IMPLS)
def test_p9_sound_wave(impl):
    n, k, nu, cs, eps = 16, 2.0, 1e-2, 1.3, 1e-9
    shape = (6, 6, n)
    lengths = (2 * math.pi, 2 * math.pi * 6 / n, 2 * math.pi * 6 / n)
    h = 2 * math.pi / n
    x = np.arange(n) * h
    state = np.zeros((7,) + shape)
    state[0] = eps * np.cos(k * x)[None, None, :]
    k1, k2 = modified_k1(k, h), modified_k2sq(k, h)
    M = np.array([[0.0, -1j * k1], [-1j * cs * cs * k1, -(4.0 / 3.0) * nu * k2]])
    dt, nsteps = 0.05, 6
    s = state
    for _ in range(nsteps):
        s = stepper(impl)(s, dt, lengths, nu, 0.0, cs)
    amp = np.linalg.matrix_power(R(dt * M), nsteps) @ np.array([eps, 0.0], dtype=complex)
    e = np.exp(1j * k * x)
    assert np.abs(s[0][0, 0] - (amp[0] * e).real).max() < 1e-6 * eps
    assert np.abs(s[1][0, 0] - (amp[1] * e).real).max() < 1e-6 * eps
    assert abs(amp[1]) > 0.3 * eps                       # the wave actually moved energy into u
    # frequency: the inviscid eigenvalue of M is +- i c_s k1~
    ev = np.linalg.eigvals(np.array([[0.0, -1j * k1], [-1j * cs * cs * k1, 0.0]]))
    assert np.allclose(sorted(ev.imag), [-cs * k1, cs * k1])


@pytest.mark.parametrize("impl", IMPLS)
def test_p10_diagonal_sound_wave_exercises_mixed_stencil(impl):
    n, nu, cs, eps = 16, 5e-2, 1.0, 1e-9
    shape = (6, n, n)
    lengths = (2 * math.pi, 2 * math.pi, 2 * math.pi * 6 / n)
    h = 2 * math.pi / n
    x = np.arange(n) * h
    ph = x[None, :] + x[:, None]                         # [y, x] -> x + y
    state = np.zeros((7,) + shape)
    state[0] = eps * np.cos(ph)[None, :, :]
    k1, k2, kxy = modified_k1(1.0, h), modified_k2sq(1.0, h), modified_kxy(1.0, 1.0, h, h)
    M = np.array([[0.0, -2j * k1], [-1j * cs * cs * k1, -nu * (2 * k2 + (k2 + kxy) / 3.0)]])
    dt, nsteps = 0.1, 5
    s = state
    for _ in range(nsteps):
        s = stepper(impl)(s, dt, lengths, nu, 0.0, cs)
    amp = np.linalg.matrix_power(R(dt * M), nsteps) @ np.array([eps, 0.0], dtype=complex)
    e = np.exp(1j * ph)
    assert np.abs(s[0][0] - (amp[0] * e).real).max() < 1e-6 * eps
    assert np.abs(s[1][0] - (amp[1] * e).real).max() < 1e-6 * eps
    assert np.abs(s[2][0] - (amp[1] * e).real).max() < 1e-6 * eps
    # the mixed-derivative term matters at this tolerance: dropping it must break the match
    M_bad = np.array([[0.0, -2j * k1], [-1j * cs * cs * k1, -nu * (2 * k2 + k2 / 3.0)]])
    amp_bad = np.linalg.matrix_power(R(dt * M_bad), nsteps) @ np.array([eps, 0.0], dtype=complex)
    assert abs(amp_bad[1] - amp[1]) > 1e-4 * eps


@pytest.mark.parametrize("impl", IMPLS)
def test_p11_alfven_wave_with_external_field(impl):
    n, k, nu, eta, b0, eps = 16, 2.0, 1e-2, 2e-2, 0.7, 1e-9
    shape = (6, 6, n)
    lengths = (2 * math.pi, 2 * math.pi * 6 / n, 2 * math.pi * 6 / n)
    h = 2 * math.pi / n
    x = np.arange(n) * h
    state = np.zeros((7,) + shape)
    state[2] = eps * np.cos(k * x)[None, None, :]
    k2 = modified_k2sq(k, h)
    M = np.array([[-nu * k2, b0 * k2], [-b0, -eta * k2]])
    dt, nsteps = 0.05, 6
    s = state
    for _ in range(nsteps):
        s = stepper(impl)(s, dt, lengths, nu, eta, 1.0, None, (b0, 0.0, 0.0))
    amp = np.linalg.matrix_power(R(dt * M), nsteps) @ np.array([eps, 0.0])
    c = np.cos(k * x)
    assert np.abs(s[2][0, 0] - amp[0] * c).max() < 1e-6 * eps
    assert np.abs(s[6][0, 0] - amp[1] * c).max() < 1e-6 * eps
    assert abs(amp[1]) > 0.1 * eps
    # nu = eta: eigenvalues -nu k2~ +- i B0 sqrt(k2~)  (k2~, not k1~: j comes from second derivatives)
    ev = np.linalg.eigvals(np.array([[-nu * k2, b0 * k2], [-b0, -nu * k2]]))
    assert np.allclose(sorted(ev.imag), [-b0 * math.sqrt(k2), b0 * math.sqrt(k2)])
    assert np.allclose(ev.real, -nu * k2)


def test_p17_difference_form_of_the_2n_update_equals_explicit_register():
    """The GPU path stores no register w: it recovers w_{s-1} = (f_{s-1} - f_{s-2}) / beta_{s-1}
    from the two state buffers (storage S8).  Restated here with the oracle's rhs."""
    rng = np.random.default_rng(17)
    shape = (12, 12, 12)
    state = rng.standard_normal((7,) + shape) * 0.05
    k = np.array([1.0, 2.0, -2.0])
    forcing = (k, 0.7, np.array([0.1, 0.0, -0.1]), np.array([0.0, 0.1, 0.05]))
    dt, nu, eta, cs = 5e-3, 1e-2, 1e-2, 1.0
    ref = state
    for _ in range(3):
        ref = mhd_c.step(ref, dt, L3, nu, eta, cs, forcing)
    al, be = mn.RK_ALPHA, mn.RK_BETA
    cur = state.copy()
    for _ in range(3):
        prev = None
        for s in range(3):
            r = mhd_c.rhs(cur, L3, nu, eta, cs, forcing)
            if s == 0:
                new = cur + be[0] * dt * r
            else:
                new = cur + be[s] * (al[s] * (cur - prev) / be[s - 1] + dt * r)
            prev, cur = cur, new
    assert np.abs(cur - ref).max() < 1e-13 * np.abs(ref).max()
