"""Pins P12-P13 for the forcing (Eq. 4-6)."""
import math

import numpy as np
import pytest

from oracle import forcing as of, mhd_c, mhd_numpy as mn
from paper_2012_08758_b200 import inputs

L3 = (2 * math.pi,) * 3


def test_shell_counts_by_brute_force():
    for kf, count in ((3, 98), (5, 350)):
        sh = of.shell(kf)
        brute = sum(1 for kx in range(-9, 10) for ky in range(-9, 10) for kz in range(-9, 10)
                    if kf - 0.5 <= math.sqrt(kx * kx + ky * ky + kz * kz) <= kf + 0.5)
        assert len(sh) == brute == count
        assert sh == sorted(sh)
        assert all((-a, -b, -c) in sh for (a, b, c) in sh)
    mean5 = np.mean([math.sqrt(a * a + b * b + c * c) for a, b, c in of.shell(5)])
    assert abs(mean5 - 5.0976) < 1e-3            # "k_f is the average wave number of the forcing"


@pytest.mark.parametrize("sigma", [0.0, 0.5, 1.0])
def test_p12_eigenfunction_properties(sigma):
    rng = np.random.default_rng(12)
    for k in [(3, 0, 0), (1, -2, 2), (0, 2, -2), (2, 2, 1), (-1, 0, 3)]:
        kv = np.array(k, dtype=float)
        kabs = math.sqrt(kv @ kv)
        e1, e2 = of.e_basis(kv)
        assert abs(e1 @ kv) < 1e-14 and abs(e2 @ kv) < 1e-14 and abs(e1 @ e2) < 1e-14
        for _ in range(3):
            psi = rng.uniform(0, 2 * math.pi)
            ehat = math.cos(psi) * e1 + math.sin(psi) * e2
            fk = of.f_k(kv, ehat, sigma)
            assert abs(np.vdot(fk, fk).real - 1.0) < 1e-14              # |f_k| = 1
            assert abs(kv @ fk) < 1e-14                                 # solenoidal
            if sigma == 1.0:                                            # eigenfunction of the curl
                assert np.abs(1j * np.cross(kv, fk) - kabs * fk).max() < 1e-14
            # perpendicular e-hat: closed form (-e - i sigma k^ x e)/sqrt(1 + sigma^2)
            closed = (-ehat - 1j * sigma * np.cross(kv / kabs, ehat)) / math.sqrt(1 + sigma * sigma)
            assert np.abs(fk - closed).max() < 1e-14
        # Eq. 6 in full also normalises an oblique e-hat (reading G9)
        eo = ehat + 0.4 * kv / kabs
        eo /= math.sqrt(eo @ eo)
        fo = of.f_k(kv, eo, sigma)
        assert abs(np.vdot(fo, fo).real - 1.0) < 1e-13 and abs(kv @ fo) < 1e-13


def test_p12_box_mean_and_normalisation():
    u = inputs.counter_uniforms(7, 3)
    dt, f0, cs, sigma = 2e-3, 0.02, 1.0, 1.0
    k, phase, re, im = of.forcing_from_draws(*u, 3, sigma, dt, f0, cs)
    kabs = math.sqrt(k @ k)
    assert 2.5 <= kabs <= 3.5 and -math.pi <= phase < math.pi
    N = f0 * cs * math.sqrt(kabs * cs / dt)                              # Eq. 5
    assert abs(math.sqrt(re @ re + im @ im) - N) < 1e-12 * N
    shape = (16, 16, 16)
    h = mn.grid_spacing(shape, L3)
    f = mn.forcing_field(shape, h, (k, phase, re, im))
    mean_f2 = sum((c ** 2).mean() for c in f)
    assert abs(mean_f2 - N * N / 2) < 1e-12 * N * N
    # f is solenoidal: k . Re{amp e^{i theta}} = 0 pointwise
    assert np.abs(k[0] * f[0] + k[1] * f[1] + k[2] * f[2]).max() < 1e-12 * N


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p13_first_substep_from_zero_state(impl):
    shape = (8, 10, 12)
    u = inputs.counter_uniforms(11, 0)
    dt = 1e-3
    forcing = of.forcing_from_draws(*u, 3, 0.0, dt, 0.02, 1.0)
    zero = np.zeros((7,) + shape)
    if impl == "c":
        st = mhd_c.Stepper(zero, L3, 5e-3, 5e-3, 1.0)
        st.substep(0, dt, forcing)
        s = st.state
    else:
        s, _ = mn.substep(zero, np.zeros_like(zero), 0, dt, L3, 5e-3, 5e-3, 1.0, forcing)
    h = mn.grid_spacing(shape, L3)
    k, phase, re, im = forcing
    X = (np.arange(12) * h[0])[None, None, :]
    Y = (np.arange(10) * h[1])[None, :, None]
    Z = (np.arange(8) * h[2])[:, None, None]
    th = k[0] * X + k[1] * Y + k[2] * Z + phase
    for i in range(3):
        expect = (dt / 3.0) * (re[i] * np.cos(th) - im[i] * np.sin(th))
        assert np.abs(s[1 + i] - expect).max() < 1e-15 * np.abs(expect).max() + 1e-20
    assert np.abs(s[0]).max() == 0.0 and np.abs(s[4:7]).max() == 0.0


def test_counter_generator_is_uniform_and_reproducible():
    d = inputs.forcing_draws(1001, 2000)
    assert d.shape == (2000, 3) and (d >= 0).all() and (d < 1).all()
    assert np.abs(d.mean(axis=0) - 0.5).max() < 0.03
    assert (inputs.forcing_draws(1001, 5) == d[:5]).all()
    assert (inputs.forcing_draws(1002, 5) != d[:5]).all()
    # SplitMix64 reference value: first output for state 0 (Steele, Lea & Flood 2014 generator)
    assert inputs.splitmix64(0) == 0xE220A8397B1DCDAF
