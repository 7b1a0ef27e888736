"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json's: fp64 <= 1e-12 after 1 step and <= 1e-9 after
10 steps, fp32 <= 1e-5 after 1 step, in the group-scaled max norm of DESIGN.md reading G14."""
import math

import numpy as np
import pytest

from oracle import mhd_c
from paper_2012_08758_b200 import binding, inputs
import helpers
from helpers import TWO_PI3

pytestmark = pytest.mark.gpu

VARIANTS = [0, 1, 2]          # 0 = pair-march (default), 1 = direct, 2 = scatter-march with a ghost-zone kernel


def make_ctx(shape, dtype=binding.AC_F64, lengths=TWO_PI3, variant=0, **kw):
    ctx = binding.Context(shape, lengths, dtype, **kw)
    ctx.ac_set_variant(variant)
    return ctx


@pytest.mark.parametrize("variant", VARIANTS)
def test_config1_32cubed_fp64_1_and_10_steps(variant):
    seed, n, dt = 1001, 32, 1e-3
    state = inputs.gaussian_state(n, seed)
    ctx = make_ctx((n, n, n), nu=5e-3, eta=5e-3, cs=1.0, k_f=3, helicity=0.0, variant=variant)
    ctx.ac_load_state(state)
    assert np.array_equal(ctx.ac_store_state(), state)              # load/store round trip is exact
    ff = lambda s: helpers.oracle_forcing(seed + 7, s, 3, 0.0, dt, 0.02, 1.0)
    want = helpers.oracle_run(state, 10, dt, TWO_PI3, 5e-3, 5e-3, 1.0, ff)
    for s in range(10):
        f = ctx.ac_make_forcing(seed + 7, s, dt, 0.02)
        ctx.ac_step(dt, f)
        if s == 0:
            err1 = helpers.group_errors(ctx.ac_store_state(), want[0])
    err10 = helpers.group_errors(ctx.ac_store_state(), want[9])
    print("config1 variant", variant, "1 step", err1, "10 steps", err10)
    assert max(err1.values()) <= 1e-12
    assert max(err10.values()) <= 1e-9
    ctx.ac_free()


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("sigma", [0.0, 0.5, 1.0])
def test_noncubic_strong_field_all_terms(variant, sigma):
    shape = (64, 48, 32)                                # nz, ny, nx; different spacing per axis
    lengths = (2 * math.pi, 2 * math.pi, 2 * math.pi)
    state = inputs.smooth_strong_state(shape, 77)
    dt, nu, eta, cs = 2e-3, 3e-3, 4e-3, 1.1
    ctx = make_ctx(shape, lengths=lengths, nu=nu, eta=eta, cs=cs, k_f=3, helicity=sigma, variant=variant)
    ctx.ac_load_state(state)
    ff = lambda s: helpers.oracle_forcing(5, s, 3, sigma, dt, 0.02, cs, lengths)
    want = helpers.oracle_run(state, 2, dt, lengths, nu, eta, cs, ff)
    for s in range(2):
        ctx.ac_step(dt, ctx.ac_make_forcing(5, s, dt, 0.02))
    err = helpers.group_errors(ctx.ac_store_state(), want[1], cs)
    print("noncubic sigma", sigma, err)
    assert max(err.values()) <= 2e-12
    ctx.ac_free()


@pytest.mark.parametrize("variant", VARIANTS)
def test_inviscid_ideal_and_external_field(variant):
    shape = (24, 20, 16)
    state = inputs.smooth_strong_state(shape, 9)
    dt = 1e-3
    for nu, eta, bext in ((0.0, 0.0, (0.0, 0.0, 0.0)), (1e-2, 0.0, (0.3, -0.1, 0.2))):
        ctx = make_ctx(shape, nu=nu, eta=eta, variant=variant)
        ctx.ac_set_bext(bext)
        ctx.ac_load_state(state)
        ctx.ac_step(dt, None)
        want = helpers.oracle_run(state, 1, dt, TWO_PI3, nu, eta, 1.0, None, bext)[0]
        assert helpers.max_group_error(ctx.ac_store_state(), want) <= 1e-12
        d = ctx.ac_reduce()
        dw = mhd_c.diagnostics(want, TWO_PI3, bext)
        for key in ("urms", "umax", "brms", "bmax", "lnrho_min", "lnrho_max"):
            assert abs(d[key] - dw[key]) <= 1e-12 * max(abs(dw[key]), 1e-30), key
        ctx.ac_free()


@pytest.mark.parametrize("variant", VARIANTS)
def test_fp32_one_step(variant):
    n = 48
    state64 = inputs.solenoidal_state(n, 1003)
    state32 = state64.astype(np.float32)
    dt, nu = 5e-3, 1e-3
    ctx = make_ctx((n, n, n), dtype=binding.AC_F32, nu=nu, eta=nu, k_f=3, helicity=0.0, variant=variant)
    ctx.ac_load_state(state32)
    f = ctx.ac_make_forcing(1010, 0, dt, 0.02)
    ctx.ac_step(dt, f)
    got = ctx.ac_store_state()
    assert got.dtype == np.float32
    # the oracle starts from the fp32-rounded inputs (reading G14)
    want = helpers.oracle_run(state32.astype(np.float64), 1, dt, TWO_PI3, nu, nu, 1.0,
                              lambda s: helpers.oracle_forcing(1010, s, 3, 0.0, dt, 0.02, 1.0))[0]
    err = helpers.group_errors(got, want)
    print("fp32 one step", err)
    assert max(err.values()) <= 1e-5
    ctx.ac_free()


def test_config2_cfl_loop_and_reductions_fp64():
    """BASELINE config 2 scaled to what the oracle finishes in seconds: 64^3, helical forcing,
    CFL dt from ac_reduce every step; diagnostics within 1e-12 of the oracle's."""
    n, seed, nu = 64, 1002, 2e-3
    state = inputs.gaussian_state(n, seed)
    ctx = make_ctx((n, n, n), nu=nu, eta=nu, k_f=3, helicity=1.0)
    ctx.ac_load_state(state)
    st = mhd_c.Stepper(state, TWO_PI3, nu, nu, 1.0)
    for s in range(4):
        d = ctx.ac_reduce()
        dw = st.diagnostics()
        for key in ("urms", "umax", "brms", "bmax"):
            assert abs(d[key] - dw[key]) <= 1e-12 * dw[key], (s, key, d[key], dw[key])
        h = 2 * math.pi / n
        dt_want = min(0.4 * h / (dw["umax"] + 1.0), 0.25 * h * h / nu)
        assert abs(d["dt_cfl"] - dt_want) <= 1e-12 * dt_want and d["nonfinite"] == 0
        dt = d["dt_cfl"]
        ctx.ac_step(dt, ctx.ac_make_forcing(seed + 7, s, dt, 0.02))
        st.step(dt, helpers.oracle_forcing(seed + 7, s, 3, 1.0, dt, 0.02, 1.0))
    assert helpers.max_group_error(ctx.ac_store_state(), st.state) <= 1e-11
    ctx.ac_free()


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
@pytest.mark.parametrize("variant", VARIANTS)
def test_p14_translation_invariance_is_bitwise(dtype, variant):
    """Roll every input by (sz, sy, sx) cells, step, roll back: bitwise equal, because the per-cell
    arithmetic does not depend on position.  Catches tile seams, halo wrap and races."""
    shape = (40, 36, 64)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 21).astype(npdt)
    ctx = make_ctx(shape, dtype=dtype, nu=2e-3, eta=3e-3, variant=variant)
    outs = []
    for shift in ((0, 0, 0), (7, 5, 13), (-3, 17, 31)):
        rolled = np.ascontiguousarray(np.roll(state, shift, axis=(1, 2, 3)))
        ctx.ac_load_state(rolled)
        for _ in range(2):
            ctx.ac_step(1e-3, None)
        outs.append(np.roll(ctx.ac_store_state(), tuple(-s for s in shift), axis=(1, 2, 3)))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    ctx.ac_free()


@pytest.mark.parametrize("variant", VARIANTS)
def test_ragged_and_minimum_grids(variant):
    for shape in ((8, 8, 8), (12, 20, 36), (9, 11, 44)):
        state = inputs.gaussian_state(shape, 4, u_amp=1e-2, a_amp=1e-3)
        state[0] = 0.1 * inputs.uniform_state(shape, 5)[0]
        ctx = make_ctx(shape, nu=1e-2, eta=1e-2, helicity=1.0, variant=variant)
        ctx.ac_load_state(state)
        dt = 1e-3
        f = ctx.ac_make_forcing(3, 0, dt, 0.02)
        ctx.ac_step(dt, f)
        want = helpers.oracle_run(state, 1, dt, TWO_PI3, 1e-2, 1e-2, 1.0,
                                  lambda s: helpers.oracle_forcing(3, s, 3, 1.0, dt, 0.02, 1.0))[0]
        assert helpers.max_group_error(ctx.ac_store_state(), want) <= 1e-12, shape
        ctx.ac_free()


def test_variants_agree_and_run_to_run_determinism():
    shape = (32, 32, 64)
    state = inputs.smooth_strong_state(shape, 31)
    res = []
    for variant in VARIANTS + VARIANTS[:1]:
        ctx = make_ctx(shape, nu=1e-3, eta=1e-3, variant=variant)
        ctx.ac_load_state(state)
        for s in range(3):
            ctx.ac_step(1e-3, ctx.ac_make_forcing(1, s, 1e-3, 0.02))
        res.append((ctx.ac_store_state(), ctx.ac_reduce()))
        ctx.ac_free()
    assert np.array_equal(res[0][0], res[-1][0]) and res[0][1] == res[-1][1]       # same variant twice: bitwise
    for other in res[1:-1]:
        assert helpers.max_group_error(other[0], res[0][0]) <= 1e-13


def test_state_errors_and_device_buffers():
    import torch
    shape = (16, 16, 16)
    ctx = make_ctx(shape, nu=1e-3, eta=1e-3)
    with pytest.raises(binding.AcError):
        ctx.ac_step(1e-3, None)                       # AC_ESTATE: nothing loaded
    with pytest.raises(binding.AcError):
        ctx.ac_reduce()
    state = inputs.gaussian_state(shape, 2)
    dev = torch.from_numpy(state).cuda()
    ctx.ac_load_state(dev)                            # device source
    with pytest.raises(binding.AcError):
        ctx.ac_step(0.0, None)                        # AC_EINVAL
    with pytest.raises(binding.AcError):
        ctx.ac_step(float("nan"), None)
    out = torch.empty_like(dev)
    ctx.ac_store_state(out)                           # device destination
    ctx.synchronize()
    assert torch.equal(out, dev)
    n0 = ctx.ac_launch_count()
    ctx.ac_step(1e-3, None)
    assert ctx.ac_launch_count() - n0 == 6            # three fused substep kernels + three ghost-zone kernels, nothing else
    ctx.ac_step(1e-3, ctx.ac_make_forcing(1, 0, 1e-3, 0.02))
    assert ctx.ac_launch_count() - n0 == 13           # + the same and ONE forcing table kernel for the step
    # a NaN in the state is reported
    bad = state.copy()
    bad[5, 3, 3, 3] = np.nan
    ctx.ac_load_state(bad)
    assert ctx.ac_reduce()["nonfinite"] == 1
    ctx.ac_free()


@pytest.mark.parametrize("dtype,n", [(binding.AC_F64, 256), (binding.AC_F32, 256), (binding.AC_F64, 512),
                                     (binding.AC_F32, 512)])
def test_sampled_parity_at_baseline_sizes(dtype, n):
    """BASELINE configs 3 (256^3) and 4 (512^3), in the launch configuration bench.py times:
    one step, checked at sampled cells (corners, faces, interior) that the oracle computes one
    by one on 24^3 periodic-extracted sub-boxes."""
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    cfg = {256: dict(seed=1003, nu=1e-3, sigma=0.0), 512: dict(seed=1004, nu=5e-4, sigma=1.0)}[n]
    state = inputs.solenoidal_state(n, cfg["seed"]).astype(npdt)
    ctx = make_ctx((n, n, n), dtype=dtype, nu=cfg["nu"], eta=cfg["nu"], k_f=3, helicity=cfg["sigma"])
    ctx.ac_load_state(state)
    # dt and forcing for the oracle come from the oracle side, never from the CUDA path
    h = 2 * math.pi / n
    umax = float(np.sqrt((state[1:4].astype(np.float64) ** 2).sum(axis=0).max()))
    dt = min(0.4 * h / (umax + 1.0), 0.25 * h * h / cfg["nu"])
    d = ctx.ac_reduce()
    assert abs(d["dt_cfl"] - dt) <= (1e-12 if dtype == binding.AC_F64 else 1e-6) * dt
    assert abs(d["urms"] - 0.1) < 1e-6
    f_oracle = helpers.oracle_forcing(cfg["seed"] + 7, 0, 3, cfg["sigma"], dt, 0.02, 1.0)
    ctx.ac_step(dt, ctx.ac_make_forcing(cfg["seed"] + 7, 0, dt, 0.02))
    got = ctx.ac_store_state()
    ctx.ac_free()
    rng = np.random.default_rng(n)
    cells = [(0, 0, 0), (n - 1, n - 1, n - 1), (0, n - 1, 5), (n // 2, 0, n - 2), (3, n - 3, n // 2)]
    cells += [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(7)]
    # the seams: last / first column and row of a 16 x 16 tile (and of the 16 x 8 tiles of variant 2), both cells of
    # a y-pair, the planes where the packed fp32 halves meet (z = n/2 - 1, n/2) and the first planes of the march
    cells += [(n // 2 - 1, 15, 15), (n // 2, 16, 16), (2, 31, 32), (n - 4, 8, 47), (3, 7, 16), (n // 2 + 2, 240, 255)]
    s_u = float(np.abs(state[1:4]).max())
    s_a = float(np.abs(state[4:7]).max())
    scale = np.array([s_u, s_u, s_u, s_u, s_a, s_a, s_a])
    tol = 1e-12 if dtype == binding.AC_F64 else 1e-5
    worst = 0.0
    state64 = state.astype(np.float64) if dtype == binding.AC_F32 else state
    for c in cells:
        want = helpers.subbox_oracle_step(state64, c, dt, TWO_PI3, cfg["nu"], cfg["nu"], 1.0, f_oracle)
        err = np.abs(got[:, c[0], c[1], c[2]].astype(np.float64) - want) / scale
        worst = max(worst, float(err.max()))
    print("sampled parity", n, npdt.__name__, worst)
    assert worst <= tol


def test_config2_full_grid_ten_steps_with_logged_diagnostics():
    """BASELINE config 2 at its own grid (128^3, nu = eta = 2e-3, helical forcing, CFL dt from ac_reduce every
    step, rms(u) and rms(B) logged each step), for the 10 steps the oracle finishes in ~15 s on the GPU box's
    cores: logged diagnostics within 1e-12, state within 1e-9 after 10 steps (north_star's bounds)."""
    n, seed, nu = 128, 1002, 2e-3
    state = inputs.gaussian_state(n, seed)
    ctx = make_ctx((n, n, n), nu=nu, eta=nu, k_f=3, helicity=1.0)
    ctx.ac_load_state(state)
    st = mhd_c.Stepper(state, TWO_PI3, nu, nu, 1.0)
    log = []
    for s in range(10):
        d = ctx.ac_reduce()
        dw = st.diagnostics()
        log.append((d["urms"], d["brms"]))
        assert abs(d["urms"] - dw["urms"]) <= 1e-12 * dw["urms"] and abs(d["brms"] - dw["brms"]) <= 1e-12 * dw["brms"]
        dt = d["dt_cfl"]
        ctx.ac_step(dt, ctx.ac_make_forcing(seed + 7, s, dt, 0.02))
        st.step(dt, helpers.oracle_forcing(seed + 7, s, 3, 1.0, dt, 0.02, 1.0))
    err = helpers.max_group_error(ctx.ac_store_state(), st.state)
    ctx.ac_free()
    print("config 2, 10 steps: error", err, "urms", log[0][0], "->", log[-1][0], "brms", log[0][1], "->", log[-1][1])
    assert err <= 1e-9
    assert log[-1][0] > log[0][0]                         # the forcing is stirring the flow


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_p16_periodic_replication_1024cubed(dtype):
    """P16, BASELINE config 5 size: a 128^3 state tiled 8 x per axis on a 1024^3
    grid (box 2 pi) must evolve exactly like the 128^3 state in a box of side 2 pi / 8, which is
    all the oracle ever runs.  Forcing wavevector (8, 16, -8): a multiple of 8 per axis, so the
    forcing has the tile's period too.  Pins indexing, chunking and ghost zones at 122.6 GB.
    Fields are streamed through ac_load_field / ac_store_field (8.6 GB each)."""
    import torch
    n, t, rep = 1024, 128, 8
    f64 = dtype == binding.AC_F64
    tdt = torch.float64 if f64 else torch.float32
    need = binding.ac_workspace_bytes((n, n, n), TWO_PI3, dtype) + 3 * (8 if f64 else 4) * n ** 3
    import gc
    gc.collect()
    torch.cuda.empty_cache()                               # give back what earlier tests' contexts cached
    free, _total = torch.cuda.mem_get_info()
    if free < need:
        pytest.skip("needs %.0f GB of free device memory" % (need / 1e9))
    nu = 2.5e-4
    tile = inputs.solenoidal_state(t, 1005, kmax=4)
    tile[0] = 0.05 * inputs.solenoidal_velocity(t, 77, 1.0, 3)[1]
    tile[4:7] *= 1e3                                        # A rms 1e-2: the Lorentz force takes part
    small = (2 * math.pi / rep,) * 3
    h = 2 * math.pi / n
    dt = 0.4 * h / (float(np.sqrt((tile[1:4] ** 2).sum(axis=0).max())) + 1.0)
    forcing = ((8.0, 16.0, -8.0), 0.3, (0.5, -0.25, 0.125), (0.1, 0.2, 0.5))
    if not f64:
        tile = tile.astype(np.float32).astype(np.float64)     # the oracle starts from the fp32-rounded inputs (G14)
    want = helpers.oracle_run(tile, 1, dt, small, nu, nu, 1.0, lambda s: forcing)[0]

    ctx = make_ctx((n, n, n), dtype=dtype, nu=nu, eta=nu, k_f=3, helicity=0.0)
    for q in range(7):
        dev = torch.from_numpy(tile[q]).to(tdt).cuda().repeat(rep, rep, rep).contiguous()
        ctx.ac_load_field(q, dev)
        ctx.synchronize()
        del dev
    d0 = ctx.ac_reduce()
    dwant = mhd_c.diagnostics(tile, small)
    assert abs(d0["urms"] - dwant["urms"]) <= (1e-12 if f64 else 1e-6) * dwant["urms"]
    assert abs(d0["bmax"] - dwant["bmax"]) <= (1e-11 if f64 else 1e-4) * dwant["bmax"]
    ctx.ac_step(dt, forcing)
    out = torch.empty((n, n, n), dtype=tdt, device="cuda")
    s_u, s_a = np.abs(want[1:4]).max(), np.abs(want[4:7]).max()
    scale = [max(np.abs(want[0]).max(), s_u), s_u, s_u, s_u, s_a, s_a, s_a]
    worst = 0.0
    for q in range(7):
        ctx.ac_store_field(q, out)
        ctx.synchronize()
        ref = torch.from_numpy(want[q]).to(tdt).cuda()
        # every one of the 512 tiles against the oracle field
        blocks = out.view(rep, t, rep, t, rep, t)
        err = (blocks - ref.view(1, t, 1, t, 1, t)).abs().max().item()
        worst = max(worst, err / scale[q])
    ctx.ac_free()
    del ctx, out, ref, blocks
    print("P16 worst group-scaled error", worst)
    assert worst <= (1e-12 if f64 else 1e-5)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_next1_upwinded_continuity_equation(variant, dtype):
    """NEXT-1 (reading G17): ac_set_upwind(1) against the oracle's upwind flag, on a state
    whose ln rho is rough enough for the sixth differences to matter, non-cubic grid, 1 and 5 steps."""
    shape = (40, 24, 36)
    lengths = (2 * math.pi, 1.5 * math.pi, 2.5 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 21)
    state[0] += 0.02 * (inputs.uniform_state(shape, 22)[0] - 0.5)
    state[1:4] *= 3.0                                           # |u| up to ~1: the correction is O(1) of the advection term
    state = state.astype(npdt)
    nu, dt = 5e-3, 2e-3
    ctx = make_ctx(shape, dtype=dtype, lengths=lengths, nu=nu, eta=nu, k_f=3, helicity=0.5, variant=variant)
    ctx.ac_set_upwind(True)
    ctx.ac_load_state(state)
    st = mhd_c.Stepper(state.astype(np.float64), lengths, nu, nu, 1.0, upwind=True)
    plain = mhd_c.Stepper(state.astype(np.float64), lengths, nu, nu, 1.0, upwind=False)
    nsteps = 5 if dtype == binding.AC_F64 else 1
    for s in range(nsteps):
        f = helpers.oracle_forcing(5, s, 3, 0.5, dt, 0.02, 1.0, lengths)
        ctx.ac_step(dt, ctx.ac_make_forcing(5, s, dt, 0.02))
        st.step(dt, f)
        plain.step(dt, f)
        if s == 0:
            err1 = helpers.max_group_error(ctx.ac_store_state(), st.state)
    errn = helpers.max_group_error(ctx.ac_store_state(), st.state)
    ctx.ac_free()
    differs = helpers.max_group_error(plain.state, st.state)
    print("upwind parity", variant, npdt.__name__, err1, errn, "upwind vs central", differs)
    assert differs > 1e-6                                       # the flag does something
    if dtype == binding.AC_F64:
        assert err1 <= 1e-12 and errn <= 1e-11
    else:
        assert err1 <= 1e-5


@pytest.mark.parametrize("shape", [(8, 8, 8), (12, 20, 36), (9, 11, 44), (34, 17, 52)])
def test_fp32_ragged_grids_packed_and_unpacked(shape):
    """fp32 on grids that are not multiples of the 16 x 8 tile; odd nz cannot be stored as (z, z + nz/2)
    pairs and runs the direct kernel, even nz runs the packed march kernel (nz/2 as small as 4 planes)."""
    state = inputs.gaussian_state(shape, 4, u_amp=1e-2, a_amp=1e-3)
    state[0] = 0.1 * inputs.uniform_state(shape, 5)[0]
    state32 = state.astype(np.float32)
    dt = 1e-3
    ctx = make_ctx(shape, dtype=binding.AC_F32, nu=1e-2, eta=1e-2, helicity=1.0)
    ctx.ac_load_state(state32)
    ctx.ac_step(dt, ctx.ac_make_forcing(3, 0, dt, 0.02))
    got = ctx.ac_store_state()
    d = ctx.ac_reduce()
    ctx.ac_free()
    want = helpers.oracle_run(state32.astype(np.float64), 1, dt, TWO_PI3, 1e-2, 1e-2, 1.0,
                              lambda s: helpers.oracle_forcing(3, s, 3, 1.0, dt, 0.02, 1.0))[0]
    assert helpers.max_group_error(got, want) <= 1e-5, shape
    dw = mhd_c.diagnostics(want, TWO_PI3)
    for key in ("urms", "umax", "brms", "bmax"):
        assert abs(d[key] - dw[key]) <= 2e-5 * dw[key], (shape, key)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("shape", [(8, 8, 8), (40, 9, 72), (33, 64, 28), (96, 40, 24)])
def test_s9_reductions_match_the_oracle_on_ragged_grids(variant, shape):
    """S9: rms/max of |u| and |B| (B_ext included), min/max of ln rho and the CFL dt on grids that are
    not multiples of the reduction kernel's 32 x 8 x 32 work items; run twice: deterministic bits."""
    lengths = (2 * math.pi, 1.3 * math.pi, 2.9 * math.pi)
    state = inputs.gaussian_state(shape, 11, u_amp=0.2, a_amp=0.05)
    state[0] = 0.3 * (inputs.uniform_state(shape, 12)[0] - 0.5)
    bext = (0.01, -0.02, 0.03)
    ctx = make_ctx(shape, lengths=lengths, nu=3e-3, eta=1e-3, variant=variant)
    ctx.ac_set_bext(bext)
    ctx.ac_load_state(state)
    d1, d2 = ctx.ac_reduce(), ctx.ac_reduce()
    ctx.ac_free()
    assert d1 == d2
    dw = mhd_c.diagnostics(state, lengths, bext)
    for key in ("urms", "umax", "brms", "bmax"):
        assert abs(d1[key] - dw[key]) <= 1e-12 * dw[key], (shape, key)
    assert d1["lnrho_min"] == dw["lnrho_min"] and d1["lnrho_max"] == dw["lnrho_max"]
    nz, ny, nx = shape
    h = min(lengths[0] / nx, lengths[1] / ny, lengths[2] / nz)
    dt = min(0.4 * h / (dw["umax"] + 1.0), 0.25 * h * h / 3e-3)
    assert abs(d1["dt_cfl"] - dt) <= 1e-12 * dt


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("upwind", [False, True])
@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_next4_tensor_product_mixed_reading(dtype, upwind, variant):
    """NEXT-4 (reading G2's alternative): ac_set_mixed("tensor") against the oracle's mixed="tensor" flag, in the
    pair-march kernel (variant 0: staged in-plane first derivatives, the performance variant) and in the direct
    kernel; the two readings differ at truncation level, far above the parity tolerance, so the flag is shown to take
    effect.  Three steps: every substep kind, the previous-state ring and the staging barriers over many planes; the
    grid is ragged in y (40 = 2.5 tiles)."""
    shape = (24, 40, 32)
    lengths = (2 * math.pi, 1.6 * math.pi, 2.2 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 31).astype(npdt)
    nu, eta, dt = 2e-2, 1e-2, 2e-3
    ctx = make_ctx(shape, dtype=dtype, lengths=lengths, nu=nu, eta=eta, k_f=3, helicity=1.0, variant=variant)
    ctx.ac_set_mixed("tensor")
    ctx.ac_set_upwind(upwind)
    ctx.ac_load_state(state)
    want = state.astype(np.float64)
    other = want
    n0 = ctx.ac_launch_count()
    for s in range(3):
        f = helpers.oracle_forcing(9, s, 3, 1.0, dt, 0.02, 1.0, lengths)
        ctx.ac_step(dt, ctx.ac_make_forcing(9, s, dt, 0.02))
        want = mhd_c.step(want, dt, lengths, nu, eta, 1.0, f, mixed="tensor", upwind=upwind)
        other = mhd_c.step(other, dt, lengths, nu, eta, 1.0, f, mixed="bidiagonal", upwind=upwind)
        if s == 0:
            n1 = ctx.ac_launch_count()
            err1 = helpers.max_group_error(ctx.ac_store_state(), want)
    got = ctx.ac_store_state()
    ctx.ac_free()
    err = helpers.max_group_error(got, want)
    gap = helpers.max_group_error(other, want)
    print("tensor-product mixed parity", npdt.__name__, "variant", variant, "upwind", upwind, "1 step", err1, "3 steps", err,
          "tensor vs bidiagonal", gap)
    assert err1 <= (1e-12 if dtype == binding.AC_F64 else 1e-5)
    assert err <= (3e-12 if dtype == binding.AC_F64 else 3e-5)
    assert gap > 100 * err or dtype == binding.AC_F32
    if variant == 0:
        assert n1 - n0 == 7               # the march path: forcing tables + 3 x (substep + ghost zones)


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_next4_tensor_product_translation_invariance_is_bitwise(dtype):
    """P14 for the staged tensor-product build of the pair-march kernel: a staged derivative has the same bits
    whether a tile's owner thread or a neighbour tile's halo thread formed it."""
    shape = (40, 36, 64)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 22).astype(npdt)
    ctx = make_ctx(shape, dtype=dtype, nu=2e-3, eta=3e-3, variant=0)
    ctx.ac_set_mixed("tensor")
    outs = []
    for shift in ((0, 0, 0), (7, 5, 13), (-3, 17, 31)):
        rolled = np.ascontiguousarray(np.roll(state, shift, axis=(1, 2, 3)))
        ctx.ac_load_state(rolled)
        for s in range(2):
            ctx.ac_step(1e-3, None)
        outs.append(np.roll(ctx.ac_store_state(), tuple(-s for s in shift), axis=(1, 2, 3)))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    ctx.ac_free()


def test_per_field_load_store_and_option_errors():
    """ac_load_field / ac_store_field: the context counts as loaded only after all 7 fields; results equal the
    whole-state calls; bad arguments are refused; ac_set_mixed / ac_set_variant drop a loaded state."""
    import torch
    shape = (16, 24, 32)
    state = inputs.gaussian_state(shape, 8, u_amp=1e-2, a_amp=1e-3)
    ctx = make_ctx(shape, nu=1e-2, eta=1e-2)
    out = np.empty(shape)
    for q in range(7):
        with pytest.raises(binding.AcError):
            ctx.ac_store_field(q, out)                     # AC_ESTATE: not all fields loaded yet
        with pytest.raises(binding.AcError):
            ctx.ac_step(1e-3, None)
        if q % 2:
            ctx.ac_load_field(q, torch.from_numpy(state[q]).cuda())
        else:
            ctx.ac_load_field(q, np.ascontiguousarray(state[q]))
    for bad_q in (-1, 7):
        with pytest.raises(binding.AcError):
            ctx._lib and binding._check(ctx._lib.ac_load_field(ctx._ctx, bad_q, out.ctypes.data, 0), "ac_load_field")
    got = np.stack([ctx.ac_store_field(q, np.empty(shape)) for q in range(7)])
    assert np.array_equal(got, state)
    ctx.ac_step(1e-3, None)
    a = ctx.ac_store_state()
    ctx2 = make_ctx(shape, nu=1e-2, eta=1e-2)
    ctx2.ac_load_state(state)
    ctx2.ac_step(1e-3, None)
    assert np.array_equal(a, ctx2.ac_store_state())
    dev = torch.empty(shape, dtype=torch.float64, device="cuda")
    ctx2.ac_store_field(3, dev)
    ctx2.synchronize()
    assert np.array_equal(dev.cpu().numpy(), a[3])
    with pytest.raises(binding.AcError):
        ctx2.ac_set_mixed(2)
    with pytest.raises(binding.AcError):
        ctx2.ac_set_variant(5)
    ctx2.ac_set_mixed("tensor")                            # reconfigures: the loaded state is gone
    with pytest.raises(binding.AcError):
        ctx2.ac_step(1e-3, None)
    ctx.ac_free()
    ctx2.ac_free()
