"""ctypes binding and build step for the plain-C oracle (oracle/mhd_oracle.c).

TEST INFRASTRUCTURE ONLY (see the header of mhd_oracle.c).  Argument marshalling only:
every number comes out of the C code.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mhd_oracle.c")
_LIB = os.path.join(_HERE, "libmhd_oracle.so")
_lib = None


class OrcParams(ctypes.Structure):
    _fields_ = [
        ("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
        ("lx", ctypes.c_double), ("ly", ctypes.c_double), ("lz", ctypes.c_double),
        ("nu", ctypes.c_double), ("eta", ctypes.c_double), ("cs", ctypes.c_double),
        ("bext", ctypes.c_double * 3),
        ("mixed_mode", ctypes.c_int), ("has_forcing", ctypes.c_int),
        ("fk", ctypes.c_double * 3), ("fphase", ctypes.c_double),
        ("fre", ctypes.c_double * 3), ("fim", ctypes.c_double * 3),
        ("upwind", ctypes.c_int), ("forcing_kick", ctypes.c_int),
    ]


def build(force=False):
    """Compile the oracle with gcc (-O2 -ffp-contract=off, OpenMP over z planes)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c99", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        pp = ctypes.POINTER(OrcParams)
        L.orc_rhs.argtypes = [dp, dp, pp]
        L.orc_substep.argtypes = [dp, dp, dp, ctypes.c_int, ctypes.c_double, pp]
        L.orc_step.argtypes = [dp, dp, dp, ctypes.c_double, pp]
        L.orc_diag.argtypes = [dp, pp, dp]
        L.orc_der1_field.argtypes = [dp, dp, pp, ctypes.c_int]
        L.orc_der2_field.argtypes = [dp, dp, pp, ctypes.c_int]
        L.orc_dermix_field.argtypes = [dp, dp, pp, ctypes.c_int, ctypes.c_int]
        L.orc_der6_upwind_field.argtypes = [dp, dp, pp, ctypes.c_int]
        L.orc_der6_upwind_field.restype = None
        L.orc_max_threads.restype = ctypes.c_int
        L.orc_set_threads.argtypes = [ctypes.c_int]
        for f in (L.orc_rhs, L.orc_substep, L.orc_step, L.orc_diag, L.orc_der1_field, L.orc_der2_field,
                  L.orc_dermix_field, L.orc_set_threads):
            f.restype = None
        _lib = L
    return _lib


def _ptr(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def make_params(shape, lengths, nu=0.0, eta=0.0, cs=1.0, forcing=None, bext=(0.0, 0.0, 0.0), mixed="bidiagonal",
                upwind=False, kick=False):
    nz, ny, nx = shape
    p = OrcParams()
    p.nx, p.ny, p.nz = nx, ny, nz
    p.lx, p.ly, p.lz = lengths
    p.nu, p.eta, p.cs = nu, eta, cs
    p.bext[:] = bext
    p.mixed_mode = {"bidiagonal": 0, "tensor": 1}[mixed]
    p.upwind = 1 if upwind else 0
    p.forcing_kick = 1 if kick else 0
    if forcing is None:
        p.has_forcing = 0
    else:
        k, phase, re, im = forcing
        p.has_forcing = 1
        p.fk[:] = [float(v) for v in k]
        p.fphase = float(phase)
        p.fre[:] = [float(v) for v in re]
        p.fim[:] = [float(v) for v in im]
    return p


def rhs(state, lengths, nu, eta, cs, forcing=None, bext=(0.0, 0.0, 0.0), mixed="bidiagonal", upwind=False):
    state = np.ascontiguousarray(state, dtype=np.float64)
    p = make_params(state.shape[1:], lengths, nu, eta, cs, forcing, bext, mixed, upwind)
    out = np.empty_like(state)
    lib().orc_rhs(_ptr(state), _ptr(out), ctypes.byref(p))
    return out


def step(state, dt, lengths, nu, eta, cs, forcing=None, bext=(0.0, 0.0, 0.0), mixed="bidiagonal", upwind=False,
         kick=False):
    """One full RK3 step; returns a new array.  kick=True: the alternative reading of G8 (forcing as one impulse
    u += dt f after the last substep instead of a term of the RHS in all three)."""
    state = np.array(state, dtype=np.float64, order="C", copy=True)
    p = make_params(state.shape[1:], lengths, nu, eta, cs, forcing, bext, mixed, upwind, kick)
    w = np.empty_like(state)
    scratch = np.empty_like(state)
    lib().orc_step(_ptr(state), _ptr(w), _ptr(scratch), float(dt), ctypes.byref(p))
    return state


class Stepper:
    """Keeps the work arrays so that repeated steps (and the timed baseline) do not reallocate."""

    def __init__(self, state, lengths, nu, eta, cs, bext=(0.0, 0.0, 0.0), mixed="bidiagonal", upwind=False):
        self.state = np.array(state, dtype=np.float64, order="C", copy=True)
        self.w = np.zeros_like(self.state)
        self.scratch = np.empty_like(self.state)
        self.args = (lengths, nu, eta, cs, bext, mixed)
        self.upwind = upwind

    def step(self, dt, forcing=None):
        lengths, nu, eta, cs, bext, mixed = self.args
        p = make_params(self.state.shape[1:], lengths, nu, eta, cs, forcing, bext, mixed, self.upwind)
        lib().orc_step(_ptr(self.state), _ptr(self.w), _ptr(self.scratch), float(dt), ctypes.byref(p))

    def substep(self, s, dt, forcing=None):
        lengths, nu, eta, cs, bext, mixed = self.args
        p = make_params(self.state.shape[1:], lengths, nu, eta, cs, forcing, bext, mixed, self.upwind)
        lib().orc_substep(_ptr(self.state), _ptr(self.w), _ptr(self.scratch), int(s), float(dt), ctypes.byref(p))

    def diagnostics(self):
        lengths, nu, eta, cs, bext, mixed = self.args
        return diagnostics(self.state, lengths, bext)


def diagnostics(state, lengths, bext=(0.0, 0.0, 0.0)):
    state = np.ascontiguousarray(state, dtype=np.float64)
    p = make_params(state.shape[1:], lengths, bext=bext)
    out = np.zeros(7)
    lib().orc_diag(_ptr(state), ctypes.byref(p), _ptr(out))
    return {"urms": out[0], "umax": out[1], "brms": out[2], "bmax": out[3],
            "lnrho_min": out[4], "lnrho_max": out[5], "nonfinite": int(out[6])}


def diagnostics_ext(state, lengths, bext=(0.0, 0.0, 0.0), mixed="bidiagonal"):
    """<omega.u>, <j.B> (Eq. 11) and the largest Alfven speed (G15): orc_diag_ext."""
    state = np.ascontiguousarray(state, dtype=np.float64)
    p = make_params(state.shape[1:], lengths, bext=bext, mixed=mixed)
    out = np.zeros(3)
    lib().orc_diag_ext(_ptr(state), ctypes.byref(p), _ptr(out))
    return {"kin_hel": out[0], "cur_hel": out[1], "va_max": out[2]}


def der1_field(f, a, lengths):
    f = np.ascontiguousarray(f, dtype=np.float64)
    p = make_params(f.shape, lengths)
    out = np.empty_like(f)
    lib().orc_der1_field(_ptr(f), _ptr(out), ctypes.byref(p), a)
    return out


def der2_field(f, a, lengths):
    f = np.ascontiguousarray(f, dtype=np.float64)
    p = make_params(f.shape, lengths)
    out = np.empty_like(f)
    lib().orc_der2_field(_ptr(f), _ptr(out), ctypes.byref(p), a)
    return out


def der6_upwind_field(f, a, lengths):
    """delta6_a f / (60 h_a) (reading G17)."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    p = make_params(f.shape, lengths)
    out = np.empty_like(f)
    lib().orc_der6_upwind_field(_ptr(f), _ptr(out), ctypes.byref(p), a)
    return out


def dermix_field(f, a, b, lengths, mixed="bidiagonal"):
    f = np.ascontiguousarray(f, dtype=np.float64)
    p = make_params(f.shape, lengths, mixed=mixed)
    out = np.empty_like(f)
    lib().orc_dermix_field(_ptr(f), _ptr(out), ctypes.byref(p), a, b)
    return out


def max_threads():
    return lib().orc_max_threads()


def set_threads(n):
    lib().orc_set_threads(int(n))
