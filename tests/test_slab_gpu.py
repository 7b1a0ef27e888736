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


@pytest.mark.parametrize("overlap", [True, False])
@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
@pytest.mark.parametrize("world", [2, 3])
def test_slabs_equal_single_context(world, dtype, variant, overlap):
    """Every kernel variant, both precisions (fp32 variants 0 and 2 on the packed-pair layout, whose halo lanes
    ac_halo_pack / ac_halo_unpack pick), with the inner / outer split of the paper's schedule and without it."""
    shape = (48, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 41).astype(npdt)
    kw = dict(nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=1.0)
    one = binding.Context(shape, lengths, dtype, **kw)
    one.ac_set_variant(variant)
    grp = slab.SlabGroupInProcess(shape, lengths, world, dtype, variant=variant, overlap=overlap, **kw)
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


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_slabs_with_the_tensor_product_reading(dtype):
    """The NEXT-4 build of the pair-march kernel (ac_set_mixed("tensor")) through the inner / outer split: its staged
    planes and their barriers must not care where a launch starts and ends along z."""
    shape = (48, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 43).astype(npdt)
    kw = dict(nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=1.0)

    def tensor_context(*a, **k):
        ctx = binding.Context(*a, **k)
        ctx.ac_set_mixed("tensor")
        return ctx

    one = tensor_context(shape, lengths, dtype, **kw)
    grp = slab.SlabGroupInProcess(shape, lengths, 2, dtype, variant=0, overlap=True, context_factory=tensor_context, **kw)
    one.ac_load_state(state)
    grp.load_state(state)
    n0 = one.ac_launch_count()
    for _ in range(2):
        one.ac_step(2e-3, None)
        grp.step(2e-3, None)
    assert one.ac_launch_count() - n0 == 12           # the march path (substep + ghost zones), not the direct kernel
    assert np.array_equal(one.ac_store_state(), grp.store_state())
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
    # and so do inner + outer parts (an ordinary box: the ghost planes are the box's own periodic images)
    c = binding.Context(shape, nu=1e-2, eta=1e-2)
    c.ac_load_state(state)
    for s in range(3):
        with pytest.raises(binding.AcError):
            c.ac_substep_part(s, 1e-3, f, binding.AC_PART_OUTER)          # outer before inner
        c.ac_substep_part(s, 1e-3, f, binding.AC_PART_INNER)
        with pytest.raises(binding.AcError):
            c.ac_substep_part(s, 1e-3, f, binding.AC_PART_INNER)          # twice
        with pytest.raises(binding.AcError):
            c.ac_substep(s, 1e-3, f)
        c.ac_substep_part(s, 1e-3, f, binding.AC_PART_OUTER)
    assert np.array_equal(a.ac_store_state(), c.ac_store_state())
    a.ac_free()
    b.ac_free()
    c.ac_free()


def test_slab_ranks_as_processes(tmp_path):
    """The multi-process path (slab.SlabRank under torchrun, world_size 2) end to end.  Both ranks share the one GPU
    and exchange through gloo with host staging; with NCCL on two GPUs only the transport differs."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29551", os.path.join(root, "tests", "slab_worker.py"), str(tmp_path)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=root)
    assert r.returncode == 0, r.stderr[-3000:]
    got = np.concatenate([np.load(tmp_path / ("slab_%d.npy" % k)) for k in range(2)], axis=1)
    shape = (32, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    one = binding.Context(shape, lengths, binding.AC_F64, nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=1.0)
    one.ac_load_state(inputs.smooth_strong_state(shape, 41))
    dt = 2e-3
    for s in range(2):
        one.ac_step(dt, one.ac_forcing_from_draws(0.3 + 0.1 * s, 0.6, 0.2, dt, 0.02))
    err = helpers.max_group_error(got, one.ac_store_state())
    d = one.ac_reduce()
    diag = np.load(tmp_path / "diag.npy")
    one.ac_free()
    print("2 processes:", err)
    assert err <= 1e-13
    for v, key in zip(diag, ("urms", "brms", "umax", "bmax", "dt_cfl")):
        assert abs(v - d[key]) <= 1e-12 * abs(d[key]), key


def test_slab_rank_over_nccl_with_one_rank(tmp_path):
    """The NCCL transport on one GPU: a single rank is its own neighbour above and below, so slab.SlabRank sends its
    halo buffers to itself through ncclSend / ncclRecv on the communication stream, overlapped with the inner part,
    exactly as between GPUs.  Must equal the ordinary periodic context."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "1", "--master-addr",
           "127.0.0.1", "--master-port", "29553", os.path.join(root, "tests", "slab_worker.py"), str(tmp_path), "nccl"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=root)
    assert r.returncode == 0, r.stderr[-3000:]
    got = np.load(tmp_path / "slab_0.npy")
    shape = (32, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    one = binding.Context(shape, lengths, binding.AC_F64, nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=1.0)
    one.ac_load_state(inputs.smooth_strong_state(shape, 41))
    dt = 2e-3
    for s in range(2):
        one.ac_step(dt, one.ac_forcing_from_draws(0.3 + 0.1 * s, 0.6, 0.2, dt, 0.02))
    want = one.ac_store_state()
    d = one.ac_reduce()
    diag = np.load(tmp_path / "diag.npy")
    one.ac_free()
    assert np.array_equal(got, want)
    for v, key in zip(diag, ("urms", "brms", "umax", "bmax", "dt_cfl")):
        assert abs(v - d[key]) <= 1e-13 * abs(d[key]), key


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
@pytest.mark.parametrize("world", [2, 3])
def test_slabs_with_the_pull_kernel_equal_single_context(world, dtype):
    """transport="pull": the ghost planes come straight out of the neighbours' state arrays (ac_halo_pull, one kernel,
    no staging buffers), here between contexts of one process; packed fp32 lanes included."""
    shape = (48, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    state = inputs.smooth_strong_state(shape, 43).astype(npdt)
    kw = dict(nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=0.5)
    one = binding.Context(shape, lengths, dtype, **kw)
    grp = slab.SlabGroupInProcess(shape, lengths, world, dtype, transport="pull", **kw)
    one.ac_load_state(state)
    grp.load_state(state)
    dt = 2e-3
    for _ in range(3):
        one.ac_step(dt, None)
        grp.step(dt, None)
    assert np.array_equal(one.ac_store_state(), grp.store_state())
    d1, dg = one.ac_reduce(), grp.reduce()
    for key in ("urms", "umax", "brms", "bmax", "dt_cfl"):
        assert abs(d1[key] - dg[key]) <= 1e-13 * abs(d1[key]), key
    one.ac_free()
    grp.free()


def test_slab_ranks_pull_over_cuda_ipc(tmp_path):
    """Two ranks as separate processes whose pull kernels read each other's workspace through CUDA IPC mappings,
    ordered by interprocess events (both processes share the one GPU here; between GPUs the same mappings are peer
    memory over NVLink).  No kernel waits on another rank: the ordering is stream waits on events."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29555", os.path.join(root, "tests", "slab_worker.py"), str(tmp_path), "gloo",
           "pull"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=root)
    assert r.returncode == 0, r.stderr[-3000:]
    got = np.concatenate([np.load(tmp_path / ("slab_%d.npy" % k)) for k in range(2)], axis=1)
    shape = (32, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    one = binding.Context(shape, lengths, binding.AC_F64, nu=5e-3, eta=4e-3, cs=1.0, k_f=3, helicity=1.0)
    one.ac_load_state(inputs.smooth_strong_state(shape, 41))
    dt = 2e-3
    for s in range(2):
        one.ac_step(dt, one.ac_forcing_from_draws(0.3 + 0.1 * s, 0.6, 0.2, dt, 0.02))
    err = helpers.max_group_error(got, one.ac_store_state())
    one.ac_free()
    print("2 processes, pull over CUDA IPC:", err)
    assert err <= 1e-13
