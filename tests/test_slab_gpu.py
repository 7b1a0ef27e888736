"""NEXT-3: the z-slab decomposition, emulated on ONE GPU as p contexts driven by one process (the
profiling guide's advice for fewer GPUs than ranks: no kernel waits on another rank).  The decomposed run must equal
the single-context run: bitwise without forcing (per-cell arithmetic does not depend on where a cell sits), to
round-off of the forcing phase with forcing; the combined reductions must equal ac_reduce of the whole box."""
import math

import numpy as np
import pytest

from paper_2012_08758_b200 import binding, inputs, slab
import helpers

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
@pytest.mark.parametrize("world", [2, 3])
def test_slabs_equal_single_context(world, dtype):
    shape = (48, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 41).astype(npdt)
    kw = dict(nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=1.0)
    one = binding.Context(shape, lengths, dtype, **kw)
    if dtype == binding.AC_F32:
        one.ac_set_variant(1)                      # same kernel as the slabs use in fp32
    grp = slab.SlabGroupInProcess(shape, lengths, world, dtype, **kw)
    one.ac_load_state(state)
    grp.load_state(state)
    dt = 2e-3
    # two steps without forcing: bitwise
    for _ in range(2):
        one.ac_step(dt, None)
        grp.step(dt, None)
    a, b = one.ac_store_state(), grp.store_state()
    assert np.array_equal(a, b)
    d1, dg = one.ac_reduce(), grp.reduce()
    for key in ("urms", "umax", "brms", "bmax", "dt_cfl"):
        assert abs(d1[key] - dg[key]) <= 1e-13 * abs(d1[key]), key
    assert d1["lnrho_min"] == dg["lnrho_min"] and d1["lnrho_max"] == dg["lnrho_max"]
    # two more with forcing: the slabs' phase k_z z0 is added in floating point
    for s in range(2):
        f = one.ac_make_forcing(17, s, dt, 0.02)
        one.ac_step(dt, f)
        grp.step(dt, f)
    err = helpers.max_group_error(grp.store_state(), one.ac_store_state())
    print("slabs", world, npdt.__name__, "with forcing:", err)
    assert err <= (1e-13 if dtype == binding.AC_F64 else 1e-6)
    one.ac_free()
    grp.free()


def test_three_substeps_equal_one_step():
    shape = (16, 24, 32)
    state = inputs.smooth_strong_state(shape, 5)
    a = binding.Context(shape, nu=1e-2, eta=1e-2)
    b = binding.Context(shape, nu=1e-2, eta=1e-2)
    a.ac_load_state(state)
    b.ac_load_state(state)
    f = a.ac_make_forcing(3, 0, 1e-3, 0.02)
    a.ac_step(1e-3, f)
    for s in range(3):
        b.ac_substep(s, 1e-3, f)
    assert np.array_equal(a.ac_store_state(), b.ac_store_state())
    with pytest.raises(binding.AcError):
        b.ac_substep(3, 1e-3, f)
    a.ac_free()
    b.ac_free()
