"""CPU-side checks of the boundary: the library builds for sm_100a, loads without a GPU, exports
every symbol include/ac_mhd.h declares, and its host-only logic (workspace sizing, argument
validation, Eq. 4-6 helper) agrees with the oracle.  No compute call is made here."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from oracle import forcing as of
from paper_2012_08758_b200 import binding, build, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def test_header_symbols_are_exported(lib):
    text = open(os.path.join(ROOT, "include", "ac_mhd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(ac_[a-z_]+)\s*\(", text))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.ac_version()


def test_workspace_bytes_and_grid_validation(lib):
    two_pi = (2 * math.pi,) * 3
    # 14 padded fields: (n + 2*gx rounded) x (n + 6) x (n + 6)
    n = 64
    b64 = binding.ac_workspace_bytes((n, n, n), two_pi, binding.AC_F64)
    b32 = binding.ac_workspace_bytes((n, n, n), two_pi, binding.AC_F32)
    lo64 = 14 * (n + 6) ** 3 * 8
    assert lo64 <= b64 <= 1.12 * lo64 + (1 << 20)
    assert 14 * (n + 6) ** 3 * 4 <= b32 <= b64
    # 1024^3 fp64 must fit one B200 (BASELINE config 5: "about 120 GB")
    big = binding.ac_workspace_bytes((1024, 1024, 1024), two_pi, binding.AC_F64)
    assert 120e9 < big < 126e9
    # invalid grids
    assert binding.ac_workspace_bytes((4, 64, 64), two_pi, binding.AC_F64) == 0          # nz < 8
    assert binding.ac_workspace_bytes((64, 64, 66), two_pi, binding.AC_F64) == 0          # nx % 4 != 0
    assert binding.ac_workspace_bytes((64, 64, 64), (0.0, 1.0, 1.0), binding.AC_F64) == 0
    assert binding.ac_workspace_bytes((64, 64, 64), two_pi, 7) == 0


def test_status_strings(lib):
    assert lib.ac_strerror(0) == b"ok"
    for code in (-1, -2, -4):
        assert len(lib.ac_strerror(code)) > 3
    assert lib.ac_launch_count(None) == 0
    lib.ac_free(None)                       # documented no-op


def test_init_fails_loudly_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    g = binding.AcGrid(32, 32, 32, 1.0, 1.0, 1.0)
    ctx = ctypes.c_void_p()
    rc = lib.ac_init(ctypes.byref(ctx), ctypes.byref(g), binding.AC_F64, 1e-3, 1e-3, 1.0, 3.0, 0.0, None, None)
    assert rc == -3 and not ctx.value
    assert b"CUDA" in lib.ac_strerror(rc)
    with pytest.raises(binding.AcError):
        binding.Context((32, 32, 32))


def test_null_and_bad_arguments(lib):
    g = binding.AcGrid(32, 32, 32, 1.0, 1.0, 1.0)
    assert lib.ac_init(None, ctypes.byref(g), 1, 0.0, 0.0, 1.0, 3.0, 0.0, None, None) == -1
    ctx = ctypes.c_void_p()
    assert lib.ac_init(ctypes.byref(ctx), ctypes.byref(g), 1, -1.0, 0.0, 1.0, 3.0, 0.0, None, None) == -1   # nu < 0
    assert lib.ac_init(ctypes.byref(ctx), ctypes.byref(g), 1, 0.0, 0.0, 0.0, 3.0, 0.0, None, None) == -1    # cs = 0
    assert lib.ac_init(ctypes.byref(ctx), ctypes.byref(g), 1, 0.0, 0.0, 1.0, 3.0, 1.5, None, None) == -1    # sigma > 1
    assert lib.ac_step(None, 1e-3, None) == -1
    assert lib.ac_reduce(None, None) == -1
    f = binding.AcForcing()
    assert lib.ac_forcing_params(3.0, 0.0, 1.0, ctypes.byref(g), 1.0, 0.5, 0.5, 1e-3, 0.02, ctypes.byref(f)) == -1
    assert lib.ac_forcing_params(3.0, 0.0, 1.0, ctypes.byref(g), 0.5, 0.5, 0.5, 0.0, 0.02, ctypes.byref(f)) == -1


@pytest.mark.parametrize("sigma", [0.0, 0.5, 1.0])
@pytest.mark.parametrize("k_f", [3.0, 5.0])
def test_forcing_helper_matches_oracle(lib, sigma, k_f):
    lengths = (2 * math.pi, 2 * math.pi, 2 * math.pi)
    shape = (32, 32, 32)
    for step in range(40):
        u = inputs.counter_uniforms(1008, step)
        dt = 1e-3 * (1 + step)
        got = binding.ac_forcing_params(k_f, sigma, 1.0, shape, lengths, *u, dt, 0.02).as_tuple()
        want = of.forcing_from_draws(*u, k_f, sigma, dt, 0.02, 1.0, lengths)
        assert np.array_equal(got[0], want[0])
        assert abs(got[1] - want[1]) < 1e-15
        amp = math.sqrt(want[2] @ want[2] + want[3] @ want[3])
        assert np.abs(got[2] - want[2]).max() < 1e-14 * amp
        assert np.abs(got[3] - want[3]).max() < 1e-14 * amp
    # non-2pi box: wavevector scaled to periods per box side
    got = binding.ac_forcing_params(3.0, sigma, 1.3, (16, 24, 32), (1.0, 2.0, 4.0), 0.3, 0.6, 0.9, 1e-2, 0.05).as_tuple()
    want = of.forcing_from_draws(0.3, 0.6, 0.9, 3.0, sigma, 1e-2, 0.05, 1.3, (1.0, 2.0, 4.0))
    assert np.abs(got[0] - want[0]).max() < 1e-13
    assert np.abs(got[2] - want[2]).max() < 1e-13 and np.abs(got[3] - want[3]).max() < 1e-13
