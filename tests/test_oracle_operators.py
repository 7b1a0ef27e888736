"""Pins P1-P3, P5, P6, P15, P18 for the derivative operators of the oracle (both the C code and
the numpy restatement).  None of these retypes the oracle's formula: the stencil weights are read
off the oracle's impulse response and compared with an exact rational solve of the moment
equations; accuracy is checked against the analytic derivative."""
from fractions import Fraction
import math

import numpy as np
import pytest

from oracle import mhd_c, mhd_numpy as mn

L3 = (2 * math.pi,) * 3


def solve_rational(A, b):
    """Gaussian elimination in exact rationals."""
    n = len(b)
    M = [[Fraction(A[i][j]) for j in range(n)] + [Fraction(b[i])] for i in range(n)]
    for c in range(n):
        p = next(r for r in range(c, n) if M[r][c] != 0)
        M[c], M[p] = M[p], M[c]
        M[c] = [v / M[c][c] for v in M[c]]
        for r in range(n):
            if r != c and M[r][c] != 0:
                M[r] = [vr - M[r][c] * vc for vr, vc in zip(M[r], M[c])]
    return [M[i][n] for i in range(n)]


def moment_weights():
    """Unique maximal-order central weights on offsets -3..3 (reading G1) and the bidiagonal
    mixed weights (reading G2), from the Taylor moment equations."""
    # first derivative: sum_m a_m (f(+m) - f(-m)) = h f' + O(h^7):  2 sum a_m m^p = [p == 1], p = 1, 3, 5
    a = solve_rational([[2 * m ** p for m in (1, 2, 3)] for p in (1, 3, 5)], [1, 0, 0])
    # second derivative: sum_m b_m (f(+m) + f(-m)) + b0 f = h^2 f'' + O(h^8)
    b = solve_rational([[m ** p for m in (1, 2, 3)] for p in (2, 4, 6)], [1, 0, 0])
    b0 = -2 * sum(b)
    # mixed: sum_m c_m [f(m,m) + f(-m,-m) - f(m,-m) - f(-m,m)] = h^2 f_xy + O(h^8)
    c = solve_rational([[4 * m ** 2 for m in (1, 2, 3)],
                        [m ** 4 for m in (1, 2, 3)],
                        [m ** 6 for m in (1, 2, 3)]], [1, 0, 0])
    return a, b0, b, c


def impulse(shape, at):
    f = np.zeros(shape)
    f[at] = 1.0
    return f


def operators(impl):
    if impl == "c":
        return (lambda f, a, L: mhd_c.der1_field(f, a, L),
                lambda f, a, L: mhd_c.der2_field(f, a, L),
                lambda f, a, b, L: mhd_c.dermix_field(f, a, b, L))
    def h(f, L):
        return mn.grid_spacing(f.shape, L)
    return (lambda f, a, L: mn.der1(f, a, h(f, L)),
            lambda f, a, L: mn.der2(f, a, h(f, L)),
            lambda f, a, b, L: mn.dermix(f, a, b, h(f, L)))


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p1_impulse_response_equals_rational_weights(impl):
    d1, d2, dm = operators(impl)
    a, b0, b, c = moment_weights()
    assert a == [Fraction(3, 4), Fraction(-3, 20), Fraction(1, 60)]
    assert (b0, b) == (Fraction(-49, 18), [Fraction(3, 2), Fraction(-3, 20), Fraction(1, 90)])
    assert c == [Fraction(3, 8), Fraction(-3, 80), Fraction(1, 360)]
    n = 12
    shape = (n, n, n)
    lengths = (float(n), float(n), float(n))            # h = 1 on every axis
    ctr = (5, 6, 7)                                      # (z, y, x)
    f = impulse(shape, ctr)
    for axis in range(3):
        npax = 2 - axis
        r1 = d1(f, axis, lengths)
        r2 = d2(f, axis, lengths)
        expect1 = np.zeros(shape)
        expect2 = np.zeros(shape)
        expect2[ctr] = float(b0)
        for m in (1, 2, 3):
            for sgn in (1, -1):
                idx = list(ctr)
                # output cell at ctr - sgn*m sees the impulse at offset +sgn*m
                idx[npax] = ctr[npax] - sgn * m
                expect1[tuple(idx)] = sgn * float(a[m - 1])
                expect2[tuple(idx)] = float(b[m - 1])
        assert np.abs(r1 - expect1).max() < 1e-15
        assert np.abs(r2 - expect2).max() < 1e-15
    for (pa, pb) in ((0, 1), (0, 2), (1, 2), (1, 0)):
        r = dm(f, pa, pb, lengths)
        expect = np.zeros(shape)
        for m in (1, 2, 3):
            for sa in (1, -1):
                for sb in (1, -1):
                    idx = list(ctr)
                    idx[2 - pa] -= sa * m
                    idx[2 - pb] -= sb * m
                    expect[tuple(idx)] = sa * sb * float(c[m - 1])
        assert np.abs(r - expect).max() < 1e-15
        assert np.count_nonzero(r) == 12


def modified_k1(k, h):
    return (1.5 * math.sin(k * h) - 0.3 * math.sin(2 * k * h) + math.sin(3 * k * h) / 30.0) / h


def modified_k2sq(k, h):
    return (49.0 / 18.0 - 3.0 * math.cos(k * h) + 0.3 * math.cos(2 * k * h) - math.cos(3 * k * h) / 45.0) / (h * h)


def modified_kxy(ka, kb, ha, hb):
    c = (3.0 / 8.0, -3.0 / 80.0, 1.0 / 360.0)
    return 4.0 / (ha * hb) * sum(c[m - 1] * math.sin(m * ka * ha) * math.sin(m * kb * hb) for m in (1, 2, 3))


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p2_modified_wavenumber_and_sixth_order(impl):
    d1, d2, dm = operators(impl)
    k = 3.0
    errs1, errs2 = [], []
    for n in (16, 32, 64):
        for axis in range(3):
            shp = [8, 8, 8]
            shp[2 - axis] = n
            lengths = [2 * math.pi * shp[2] / 8.0, 2 * math.pi * shp[1] / 8.0, 2 * math.pi * shp[0] / 8.0]
            lengths[axis] = 2 * math.pi
            h = lengths[axis] / n
            idx = np.arange(n) * h
            bshape = [1, 1, 1]
            bshape[2 - axis] = n
            f = np.broadcast_to(np.sin(k * idx + 0.3).reshape(bshape), shp).copy()
            fc = np.broadcast_to(np.cos(k * idx + 0.3).reshape(bshape), shp).copy()
            r1 = d1(f, axis, tuple(lengths))
            r2 = d2(f, axis, tuple(lengths))
            assert np.abs(r1 - modified_k1(k, h) * fc).max() < 5e-14 * k
            assert np.abs(r2 + modified_k2sq(k, h) * f).max() < 5e-14 * k * k * (n / 16) ** 2
            if axis == 0:
                errs1.append(np.abs(r1 - k * fc).max())
                errs2.append(np.abs(r2 + k * k * f).max())
    # sixth order: error falls ~64x per halving of h
    assert 45 < errs1[0] / errs1[1] < 80 and 55 < errs1[1] / errs1[2] < 70
    assert 45 < errs2[0] / errs2[1] < 80 and 55 < errs2[1] / errs2[2] < 70


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p3_mixed_modified_wavenumber_symmetry_and_order(impl):
    d1, d2, dm = operators(impl)
    ka, kb = 2.0, 3.0
    errs = []
    for n in (32, 64, 128):
        shape = (4, n, n)
        nz, ny, nx = shape
        lengths = (2 * math.pi, 2 * math.pi, 2 * math.pi * nz / n)
        h = 2 * math.pi / n
        x = np.arange(nx) * h
        y = np.arange(ny) * h
        f = np.sin(ka * x + 0.2)[None, None, :] * np.sin(kb * y - 0.4)[None, :, None] * np.ones((nz, 1, 1))
        exact_shape = np.cos(ka * x + 0.2)[None, None, :] * np.cos(kb * y - 0.4)[None, :, None] * np.ones((nz, 1, 1))
        r = dm(f, 0, 1, lengths)
        r_t = dm(f, 1, 0, lengths)
        assert np.abs(r - r_t).max() < 1e-13
        assert np.abs(r - modified_kxy(ka, kb, h, h) * exact_shape).max() < 1e-12
        errs.append(np.abs(r - ka * kb * exact_shape).max())
    assert 55 < errs[0] / errs[1] < 70 and 60 < errs[1] / errs[2] < 66
    # the other two planes, on a non-cubic grid with different spacings
    shape = (20, 24, 16)
    lengths = (2 * math.pi, 3.0, 5.0)
    nz, ny, nx = shape
    hx, hy, hz = lengths[0] / nx, lengths[1] / ny, lengths[2] / nz
    X = (np.arange(nx) * hx)[None, None, :]
    Y = (np.arange(ny) * hy)[None, :, None]
    Z = (np.arange(nz) * hz)[:, None, None]
    kx, ky, kz = 2 * math.pi / lengths[0], 2 * 2 * math.pi / lengths[1], 3 * 2 * math.pi / lengths[2]
    f = np.sin(kx * X) * np.sin(ky * Y) * np.sin(kz * Z)
    cxz = np.cos(kx * X) * np.sin(ky * Y) * np.cos(kz * Z)
    cyz = np.sin(kx * X) * np.cos(ky * Y) * np.cos(kz * Z)
    assert np.abs(dm(f, 0, 2, lengths) - modified_kxy(kx, kz, hx, hz) * cxz).max() < 1e-12
    assert np.abs(dm(f, 2, 1, lengths) - modified_kxy(kz, ky, hz, hy) * cyz).max() < 1e-12


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p5_div_curl_is_zero_to_roundoff(impl):
    d1, _, _ = operators(impl)
    rng = np.random.default_rng(5)
    shape = (12, 14, 16)
    lengths = (2 * math.pi, 5.0, 4.0)
    A = rng.standard_normal((3,) + shape)
    bx = d1(A[2], 1, lengths) - d1(A[1], 2, lengths)
    by = d1(A[0], 2, lengths) - d1(A[2], 0, lengths)
    bz = d1(A[1], 0, lengths) - d1(A[0], 1, lengths)
    div = d1(bx, 0, lengths) + d1(by, 1, lengths) + d1(bz, 2, lengths)
    hmin = min(lengths[0] / 16, lengths[1] / 14, lengths[2] / 12)
    bmag = np.sqrt(bx ** 2 + by ** 2 + bz ** 2).max()
    assert np.abs(div).max() < 2e-14 * bmag / hmin
    # and the oracle's own B (through the diagnostics path) is that curl
    state = np.zeros((7,) + shape)
    state[4:7] = A
    diag = (mhd_c.diagnostics if impl == "c" else mn.diagnostics)(state, lengths)
    assert abs(diag["bmax"] - bmag) < 1e-12 * bmag
    assert abs(diag["brms"] - math.sqrt((bx ** 2 + by ** 2 + bz ** 2).mean())) < 1e-12 * bmag


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p6_sum_of_divergence_vanishes_and_mass_after_substep(impl):
    rng = np.random.default_rng(6)
    shape = (10, 12, 14)
    state = np.zeros((7,) + shape)
    state[1:4] = rng.standard_normal((3,) + shape) * 0.1
    rhs = (mhd_c.rhs if impl == "c" else mn.rhs)(state, L3, 1e-3, 1e-3, 1.0)
    # ln rho = 0 => d ln rho/dt = -div u, whose sum over the periodic box is zero
    scale = np.abs(rhs[0]).max()
    assert abs(rhs[0].sum()) < 1e-13 * scale * rhs[0].size ** 0.5 * 10


@pytest.mark.parametrize("impl", ["c", "numpy"])
def test_p15_axis_permutation_covariance(impl):
    rng = np.random.default_rng(15)
    shape = (10, 12, 14)                       # nz, ny, nx
    lengths = (2 * math.pi, 5.0, 4.0)          # lx, ly, lz
    state = rng.standard_normal((7,) + shape) * 0.1
    k = np.array([1.0, -2.0, 3.0]) * 2 * math.pi / np.array(lengths)
    forcing = (k, 0.4, np.array([0.1, -0.2, 0.3]), np.array([0.05, 0.15, -0.1]))
    bext = (0.3, -0.2, 0.1)
    fn = mhd_c.rhs if impl == "c" else mn.rhs
    r = fn(state, lengths, 2e-2, 3e-2, 1.3, forcing, bext)

    # proper rotation: new (x', y', z') = old (y, z, x)
    def rot_scalar(f):
        return np.ascontiguousarray(np.transpose(f, (2, 0, 1)))

    def rot_state(s):
        out = np.empty((7,) + rot_scalar(s[0]).shape)
        out[0] = rot_scalar(s[0])
        for base in (1, 4):
            out[base + 0] = rot_scalar(s[base + 1])     # v'_x' = v_y
            out[base + 1] = rot_scalar(s[base + 2])     # v'_y' = v_z
            out[base + 2] = rot_scalar(s[base + 0])     # v'_z' = v_x
        return out

    def rot_vec(v):
        return (v[1], v[2], v[0])

    lengths_r = rot_vec(lengths)
    forcing_r = (np.array(rot_vec(k)), 0.4, np.array(rot_vec(forcing[2])), np.array(rot_vec(forcing[3])))
    r_rot = fn(rot_state(state), lengths_r, 2e-2, 3e-2, 1.3, forcing_r, rot_vec(bext))
    assert np.abs(r_rot - rot_state(r)).max() < 1e-12 * np.abs(r).max()


def test_p18_c_oracle_equals_numpy_oracle_all_terms_on():
    rng = np.random.default_rng(18)
    for shape, lengths in (((16, 16, 16), L3), ((12, 20, 16), (2 * math.pi, 7.0, 3.0))):
        state = rng.standard_normal((7,) + shape) * 0.1
        k = np.array([2.0, -1.0, 2.0]) * 2 * math.pi / np.array(lengths)
        forcing = (k, -1.1, np.array([0.3, 0.1, -0.2]), np.array([0.0, 0.25, 0.1]))
        for mixed in ("bidiagonal", "tensor"):
            a = mhd_c.rhs(state, lengths, 5e-3, 7e-3, 1.0, forcing, (0.1, 0.0, -0.2), mixed)
            b = mn.rhs(state, lengths, 5e-3, 7e-3, 1.0, forcing, (0.1, 0.0, -0.2), mixed)
            assert np.abs(a - b).max() < 1e-13 * np.abs(b).max()
        a = state
        b = state
        for _ in range(3):
            a = mhd_c.step(a, 2e-3, lengths, 5e-3, 7e-3, 1.0, forcing)
            b = mn.step(b, 2e-3, lengths, 5e-3, 7e-3, 1.0, forcing)
        assert np.abs(a - b).max() < 1e-13 * np.abs(b).max()
        da, db = mhd_c.diagnostics(a, lengths), mn.diagnostics(b, lengths)
        for key in ("urms", "umax", "brms", "bmax"):
            assert abs(da[key] - db[key]) < 1e-13 * db[key]
    # the two readings of the mixed derivative differ at truncation level, not round-off (G2)
    a = mhd_c.rhs(state, lengths, 5e-3, 7e-3, 1.0, None, (0, 0, 0), "bidiagonal")
    b = mhd_c.rhs(state, lengths, 5e-3, 7e-3, 1.0, None, (0, 0, 0), "tensor")
    assert np.abs(a - b).max() > 1e-6 * np.abs(b).max()
