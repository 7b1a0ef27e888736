"""GPU tests added in round 2: the extended diagnostics (NEXT-4) against the oracle, the ordering rules of
ac_substep, and full-field parity at 256^3 in both precisions."""
import math

import numpy as np
import pytest

from oracle import mhd_c
from paper_2012_08758_b200 import binding, inputs
import helpers
from helpers import TWO_PI3

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
@pytest.mark.parametrize("shape", [(8, 8, 8), (40, 9, 72), (34, 64, 28)])
def test_next4_extended_diagnostics_match_the_oracle(variant, dtype, shape):
    """<omega.u>, <j.B>, max Alfven speed and the Alfven CFL step (Eq. 11; G15) on ragged grids with
    an external field; fp32 runs on the packed-pair layout (variant 0) and on the plain one (variant 1)."""
    lengths = (2 * math.pi, 1.3 * math.pi, 2.9 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 21).astype(npdt)
    bext = (0.01, -0.02, 0.03)
    ctx = binding.Context(shape, lengths, dtype, nu=3e-3, eta=1e-3)
    ctx.ac_set_variant(variant)
    ctx.ac_set_bext(bext)
    ctx.ac_load_state(state)
    d1, d2 = ctx.ac_reduce_ext(), ctx.ac_reduce_ext()
    base = ctx.ac_reduce()
    ctx.ac_free()
    assert d1 == d2                                           # deterministic
    s64 = state.astype(np.float64)
    want = mhd_c.diagnostics_ext(s64, lengths, bext)
    dw = mhd_c.diagnostics(s64, lengths, bext)
    # the helicities are signed sums with cancellation: scale by the rms product of the factors
    sk = dw["urms"] ** 2 * 4.0                                # |omega| ~ k |u|, k <= 4
    sc = dw["brms"] ** 2 * 4.0
    tol = 1e-12 if dtype == binding.AC_F64 else 2e-5
    assert abs(d1["kin_hel"] - want["kin_hel"]) <= tol * sk, (d1, want)
    assert abs(d1["cur_hel"] - want["cur_hel"]) <= tol * sc * 10, (d1, want)
    assert abs(d1["va_max"] - want["va_max"]) <= tol * want["va_max"]
    nz, ny, nx = shape
    h = min(lengths[0] / nx, lengths[1] / ny, lengths[2] / nz)
    dt = min(0.4 * h / (dw["umax"] + math.sqrt(1.0 + want["va_max"] ** 2)), 0.25 * h * h / 3e-3)
    assert abs(d1["dt_cfl_alfven"] - dt) <= max(tol, 1e-12) * dt * 2
    assert d1["dt_cfl_alfven"] <= base["dt_cfl"] * (1 + 1e-12)
    assert d1["nonfinite"] == 0


def test_substep_order_and_stores_between_substeps():
    """between substeps the idle buffer holds the previous state.  ac_substep must come in order;
    host-staged stores, field loads, ac_step and ac_reduce_ext are refused inside a step; a device-destination
    store and ac_reduce are allowed and leave the result of the step untouched."""
    import torch
    shape = (16, 24, 32)
    state = inputs.gaussian_state(shape, 3, u_amp=0.1, a_amp=0.01)
    dt = 1e-3
    ctx = binding.Context(shape, TWO_PI3, binding.AC_F64, nu=1e-2, eta=1e-2, k_f=3, helicity=1.0)
    f = ctx.ac_make_forcing(5, 0, dt, 0.02)
    ctx.ac_load_state(state)
    ctx.ac_step(dt, f)
    want = ctx.ac_store_state()
    ctx.ac_load_state(state)
    with pytest.raises(binding.AcError):
        ctx.ac_substep(1, dt, f)                               # out of order
    ctx.ac_substep(0, dt, f)
    with pytest.raises(binding.AcError):
        ctx.ac_substep(0, dt, f)
    with pytest.raises(binding.AcError):
        ctx.ac_store_state()                                   # host destination: stages in the idle buffer
    with pytest.raises(binding.AcError):
        ctx.ac_step(dt, f)
    with pytest.raises(binding.AcError):
        ctx.ac_reduce_ext()
    with pytest.raises(binding.AcError):
        ctx.ac_load_field(0, state[0])
    bad = binding.AcForcing.from_tuple(f.as_tuple())
    bad.phase = float("nan")
    with pytest.raises(binding.AcError):
        ctx.ac_substep(1, dt, bad)                             # non-finite forcing is refused like in ac_step
    snap = torch.empty((7,) + shape, dtype=torch.float64, device="cuda")
    ctx.ac_store_state(snap)                                   # device destination: allowed
    ctx.ac_reduce()
    ctx.ac_substep(1, dt, f)
    ctx.ac_store_state(snap)
    ctx.ac_substep(2, dt, f)
    got = ctx.ac_store_state()                                 # the step is complete: host stores work again
    ctx.ac_free()
    assert np.array_equal(got, want)


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_config3_256cubed_full_field_one_step(dtype):
    """BASELINE config 3 (256^3, nu = eta = 1e-3, non-helical forcing at k_f = 3, f0 = 0.02): EVERY cell of all
    7 fields after one CFL step against the oracle (about 15 s of oracle), fp64 <= 1e-12, fp32 <= 1e-5."""
    n = 256
    nu, seed = 1e-3, 1003
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.solenoidal_state(n, seed).astype(npdt)
    ctx = binding.Context((n, n, n), TWO_PI3, dtype, nu=nu, eta=nu, cs=1.0, k_f=3, helicity=0.0)
    ctx.ac_load_state(state)
    dt = ctx.ac_reduce()["dt_cfl"]
    ctx.ac_step(dt, ctx.ac_make_forcing(seed + 7, 0, dt, 0.02))
    got = ctx.ac_store_state()
    ctx.ac_free()
    f = helpers.oracle_forcing(seed + 7, 0, 3, 0.0, dt, 0.02, 1.0)
    want = mhd_c.step(state.astype(np.float64), dt, TWO_PI3, nu, nu, 1.0, f)
    err = helpers.group_errors(got, want)
    print("256^3 full field", npdt.__name__, err)
    assert max(err.values()) <= (1e-12 if dtype == binding.AC_F64 else 1e-5)


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_forcing_as_one_impulse_per_step(variant, dtype):
    """the alternative reading of G8 (ac_set_forcing_mode("kick")) against the oracle's kick=True,
    two steps on a moving state; and it is not the default reading."""
    shape = (24, 40, 32)
    lengths = (2 * math.pi, 1.6 * math.pi, 2.2 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 33).astype(npdt)
    nu, eta, dt = 2e-2, 1e-2, 2e-3
    ctx = binding.Context(shape, lengths, dtype, nu=nu, eta=eta, k_f=3, helicity=1.0)
    ctx.ac_set_variant(variant)
    ctx.ac_set_forcing_mode("kick")
    ctx.ac_load_state(state)
    want = state.astype(np.float64)
    other = want
    for s in range(2):
        f = helpers.oracle_forcing(9, s, 3, 1.0, dt, 0.05, 1.0, lengths)
        ctx.ac_step(dt, ctx.ac_make_forcing(9, s, dt, 0.05))
        want = mhd_c.step(want, dt, lengths, nu, eta, 1.0, f, kick=True)
        other = mhd_c.step(other, dt, lengths, nu, eta, 1.0, f)
    got = ctx.ac_store_state()
    ctx.ac_free()
    err = helpers.max_group_error(got, want)
    gap = helpers.max_group_error(other, want)
    print("kick reading", variant, npdt.__name__, err, "kick vs rhs", gap)
    assert err <= (2e-12 if dtype == binding.AC_F64 else 1e-5)
    assert gap > 100 * err or dtype == binding.AC_F32


def test_config3_256cubed_ten_steps_fp64():
    """north_star: fp64 within 1e-9 of the oracle after 10 steps on the same seeded inputs, on EVERY cell of the
    256^3 box of BASELINE config 3 (about two minutes of oracle on 16 cores); forcing redrawn every step."""
    n = 256
    nu, seed = 1e-3, 1003
    state = inputs.solenoidal_state(n, seed)
    ctx = binding.Context((n, n, n), TWO_PI3, binding.AC_F64, nu=nu, eta=nu, cs=1.0, k_f=3, helicity=0.0)
    ctx.ac_load_state(state)
    h = 2 * math.pi / n
    umax = float(np.sqrt((state[1:4] ** 2).sum(axis=0).max()))
    dt = 0.8 * min(0.4 * h / (umax + 1.0), 0.25 * h * h / nu)       # fixed, from the oracle side
    st = mhd_c.Stepper(state, TWO_PI3, nu, nu, 1.0)
    for s in range(10):
        ctx.ac_step(dt, ctx.ac_make_forcing(seed + 7, s, dt, 0.02))
        st.step(dt, helpers.oracle_forcing(seed + 7, s, 3, 0.0, dt, 0.02, 1.0))
    got = ctx.ac_store_state()
    ctx.ac_free()
    err = helpers.group_errors(got, st.state)
    print("256^3, 10 steps, fp64:", err)
    assert max(err.values()) <= 1e-9


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_degenerate_states_are_fixed_points(variant, dtype):
    """Degenerate cases of the method: a uniform state (constant ln rho, u, A; no forcing) has an exactly vanishing
    right-hand side - every stencil sums differences of equal numbers - so the step must return it BITWISE, with
    viscosity and resistivity on, on a ragged grid; and with A = 0 the magnetic part stays exactly zero while the
    hydrodynamic part moves."""
    shape = (24, 9, 40)
    lengths = (2 * math.pi, 1.3 * math.pi, 2.9 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    ctx = binding.Context(shape, lengths, dtype, nu=1e-2, eta=2e-2, cs=1.3)
    ctx.ac_set_variant(variant)
    state = np.empty((7,) + shape, dtype=npdt)
    for q, v in enumerate((0.3, 0.2, -0.1, 0.05, 1e-3, -2e-3, 3e-3)):
        state[q] = v
    ctx.ac_load_state(state)
    for _ in range(3):
        ctx.ac_step(1e-3, None)
    assert np.array_equal(ctx.ac_store_state(), state)
    d = ctx.ac_reduce()
    assert d["brms"] == 0.0 and d["bmax"] == 0.0 and d["lnrho_min"] == d["lnrho_max"] == float(npdt(0.3))
    moving = inputs.smooth_strong_state(shape, 7).astype(npdt)
    moving[4:7] = 0.0
    ctx.ac_load_state(moving)
    ctx.ac_step(1e-3, None)
    out = ctx.ac_store_state()
    ctx.ac_free()
    assert np.all(out[4:7] == 0.0) and not np.array_equal(out[1:4], moving[1:4])
