"""ac_reduce_dense_noalloc (include/ac_mhd.h): the S9 reductions of a dense device state through the one entry point
that allocates nothing (its scratch is a fixed static __device__ array inside the library), against the existing path
(a context's ac_reduce_raw) on the same seeded inputs, on two calls in a row that share the scratch array.

Collected last on purpose (the file name sorts after every other test file): the suite runs with pytest -x."""
import ctypes
import math

import numpy as np
import pytest

from paper_2012_08758_b200 import binding, inputs

pytestmark = pytest.mark.gpu

KEYS = ("sum_u2", "max_u2", "sum_b2", "max_b2", "lnrho_min", "lnrho_max")


def existing_path(state, lengths, dtype, variant, bext):
    """ac_reduce_raw of a context that holds `state` (numpy (7, nz, ny, nx))."""
    ctx = binding.Context(state.shape[1:], lengths, dtype, nu=1e-3, eta=1e-3, cs=1.0, k_f=3, helicity=1.0)
    ctx.ac_set_variant(variant)
    if bext is not None:
        ctx.ac_set_bext(bext)
    ctx.ac_load_state(state)
    raw = np.array(ctx.ac_reduce_raw(), dtype=np.float64)
    ctx.ac_free()
    return raw


def check(got, want, want_stage1, dtype):
    # tolerance of the suite's reduction tests (tests/test_parity_gpu.py): 1e-12 relative in fp64, 1e-6 in fp32
    tol = 1e-12 if dtype == binding.AC_F64 else 1e-6
    for i, key in enumerate(KEYS):
        assert abs(got[i] - want[i]) <= tol * max(abs(want[i]), 1e-30), (key, got[i], want[i])
    # against reduce_stage1_kernel (variant 1), whose per-cell arithmetic the dense kernel repeats: the maxima and the
    # ln rho extrema bit for bit, the sums to summation order
    for i in (1, 3, 4, 5):
        assert got[i] == want_stage1[i], (KEYS[i], got[i], want_stage1[i])
    for i in (0, 2):
        assert abs(got[i] - want_stage1[i]) <= 1e-13 * abs(want_stage1[i]), (KEYS[i], got[i], want_stage1[i])


@pytest.mark.parametrize("dtype", [binding.AC_F64, binding.AC_F32])
def test_no_alloc_entry_point_equals_the_context_path_on_two_calls_in_a_row(dtype):
    import torch
    torch.cuda.set_device(0)
    npdt = np.float64 if dtype == binding.AC_F64 else np.float32
    lengths_a = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    lengths_b = (2 * math.pi,) * 3
    bext = (0.01, -0.02, 0.03)
    # call 1: ragged, several blocks with a partly filled last one (40 * 36 * 64 = 45 blocks of 2048 cells);
    # call 2: a smaller box (the scratch array still holds call 1's partials beyond the ones call 2 writes)
    a = inputs.smooth_strong_state((40, 36, 64), 51).astype(npdt)
    a += (np.random.default_rng(51).normal(size=a.shape) * 1e-3).astype(npdt)
    b = inputs.smooth_strong_state((12, 20, 16), 52).astype(npdt)
    b[1:4] *= 2.5
    want_a = existing_path(a, lengths_a, dtype, 0, bext)
    want_b = existing_path(b, lengths_b, dtype, 0, None)
    stage1_a = existing_path(a, lengths_a, dtype, 1, bext)
    stage1_b = existing_path(b, lengths_b, dtype, 1, None)
    da, db = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    out = torch.full((3, 6), float("nan"), dtype=torch.float64, device="cuda")
    binding.ac_reduce_dense_noalloc(da, lengths_a, out[0], bext=bext)        # warm-up: loads the kernels
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    out[0].fill_(float("nan"))
    # two calls in a row on one stream, no synchronisation between them
    binding.ac_reduce_dense_noalloc(da, lengths_a, out[0], bext=bext)
    binding.ac_reduce_dense_noalloc(db, lengths_b, out[1])
    binding.ac_reduce_dense_noalloc(da, lengths_a, out[2], bext=bext)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before                       # nothing was allocated on the device
    got = out.cpu().numpy()
    check(got[0], want_a, stage1_a, dtype)
    check(got[1], want_b, stage1_b, dtype)
    assert np.array_equal(got[0], got[2])                                    # deterministic; call 2 left no trace
    print("no-alloc reductions", npdt.__name__, got[0], "context path", want_a)


def test_no_alloc_entry_point_limits_and_bad_arguments():
    import torch
    torch.cuda.set_device(0)
    lib = binding.load_library()
    assert binding.ac_noalloc_max_cells() == 2 ** 27
    small = torch.zeros((7, 8, 8, 8), dtype=torch.float64, device="cuda")
    out = torch.zeros(6, dtype=torch.float64, device="cuda")

    def call(state_ptr, grid, out_ptr, dtype=binding.AC_F64):
        return lib.ac_reduce_dense_noalloc(ctypes.c_void_p(state_ptr), dtype, ctypes.byref(grid), None,
                                           ctypes.c_void_p(out_ptr), None)

    # one plane more than 512^3: refused before anything is launched or read, with its own status and text
    too_big = binding.AcGrid(512, 512, 513, 1.0, 1.0, 1.0)
    rc = call(small.data_ptr(), too_big, out.data_ptr())
    assert rc == -5 and b"512^3" in lib.ac_strerror(rc)
    with pytest.raises(binding.AcError, match="larger than the fixed scratch array"):
        binding._check(rc, "ac_reduce_dense_noalloc")
    ok = binding.AcGrid(8, 8, 8, 1.0, 1.0, 1.0)
    host = np.zeros((7, 8, 8, 8))
    assert call(host.ctypes.data, ok, out.data_ptr()) == -1                  # a host pointer is not a device address
    assert call(small.data_ptr(), ok, host.ctypes.data) == -1
    assert call(0, ok, out.data_ptr()) == -1
    assert call(small.data_ptr(), ok, out.data_ptr() + 4) == -1              # misaligned result
    assert call(small.data_ptr(), binding.AcGrid(8, 8, 4, 1.0, 1.0, 1.0), out.data_ptr()) == -1
    assert call(small.data_ptr(), ok, out.data_ptr(), dtype=7) == -1
    torch.cuda.synchronize()
    assert call(small.data_ptr(), ok, out.data_ptr()) == 0                   # and the library still works
    torch.cuda.synchronize()
    assert out.cpu().numpy().tolist() == [0.0, 0.0, 0.0, 0.0, 0.0, 0.0]
