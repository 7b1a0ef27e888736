"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no stencils, no right-hand sides, no
Runge-Kutta, no Eq. 4-6): it only produces initial fields and raw random numbers.  It imports
neither oracle/ nor the CUDA binding.  The recipes are stated in DESIGN.md ("Input recipe")
and stand in for the paper's snapshot datasets, which are not available.

State arrays have shape (7, nz, ny, nx), C order, x fastest; field order
lnrho, ux, uy, uz, ax, ay, az.
"""
import math

import numpy as np

FIELDS = ("lnrho", "ux", "uy", "uz", "ax", "ay", "az")
TWO_PI = 2.0 * math.pi


def _shape(n):
    if isinstance(n, int):
        return (n, n, n)
    nz, ny, nx = n
    return (int(nz), int(ny), int(nx))


def gaussian_state(n, seed, u_amp=1e-3, a_amp=1e-5):
    """BASELINE configs 1-2: ln rho = 0; u i.i.d. N(0, u_amp^2); A i.i.d. N(0, a_amp^2).
    Draw order ux, uy, uz, ax, ay, az from numpy.random.default_rng(seed)."""
    shape = _shape(n)
    rng = np.random.default_rng(seed)
    s = np.zeros((7,) + shape)
    for i in (1, 2, 3):
        s[i] = rng.standard_normal(shape) * u_amp
    for i in (4, 5, 6):
        s[i] = rng.standard_normal(shape) * a_amp
    return s


def solenoidal_modes(seed, kmax=4):
    """The 128 integer wavevectors with 0 < |k| <= kmax in the half space (kx,ky,kz) > (0,0,0)
    (tuple order), lexicographic, each with a complex Gaussian amplitude projected
    perpendicular to k (flat spectrum)."""
    rng = np.random.default_rng(seed)
    ks = []
    r = int(kmax)
    for kx in range(-r, r + 1):
        for ky in range(-r, r + 1):
            for kz in range(-r, r + 1):
                k2 = kx * kx + ky * ky + kz * kz
                if 0 < k2 <= kmax * kmax and (kx, ky, kz) > (0, 0, 0):
                    ks.append((kx, ky, kz))
    ks.sort()
    amps = []
    for k in ks:
        kv = np.array(k, dtype=np.float64)
        a = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        a = a - kv * (kv @ a) / (kv @ kv)
        amps.append(a)
    return ks, amps


def _solenoidal_components(n, seed, kmax):
    """Generator of the three unscaled components (nz, ny, nx) of the mode sum, one at a time."""
    nz, ny, nx = _shape(n)
    ks, amps = solenoidal_modes(seed, kmax)
    r = int(kmax)
    nk = 2 * r + 1
    coef = np.zeros((3, nk, nk, nk), dtype=np.complex128)       # [comp, kx, ky, kz]
    for k, a in zip(ks, amps):
        coef[:, k[0] + r, k[1] + r, k[2] + r] = a
    kk = np.arange(-r, r + 1, dtype=np.float64)
    # wavenumber k_a means exp(i k_a 2 pi i_a / n_a): k counts periods per box (k1 = 1)
    ex = np.exp(1j * np.outer(kk, TWO_PI * np.arange(nx) / nx))        # [kx, x]
    ey = np.exp(1j * np.outer(kk, TWO_PI * np.arange(ny) / ny))
    ez = np.exp(1j * np.outer(kk, TWO_PI * np.arange(nz) / nz))
    for c in range(3):
        t1 = np.einsum("abc,cz->abz", coef[c], ez)                     # [kx, ky, z]
        t2 = np.einsum("abz,by->azy", t1, ey)                          # [kx, z, y]
        t2 = np.ascontiguousarray(t2.reshape(nk, nz * ny).T)           # [(z,y), kx]
        # real part of t2 @ ex without forming the complex product
        yield (t2.real @ ex.real - t2.imag @ ex.imag).reshape(nz, ny, nx)


def _sum_sq(a):
    return float(np.einsum("i,i->", a.ravel(), a.ravel()))


def solenoidal_velocity(n, seed, urms=0.1, kmax=4, lengths=(TWO_PI, TWO_PI, TWO_PI)):
    """Sum over the modes of Re{a exp(i k.x)}, x_a = i_a L_a / n_a, rescaled so that
    sqrt(mean |u|^2) = urms.  Evaluated with per-axis tables exp(i k_a x_a) contracted axis by
    axis (a separable sum, no FFT).  Returns (3, nz, ny, nx)."""
    nz, ny, nx = _shape(n)
    u = np.empty((3, nz, ny, nx))
    ssq = 0.0
    for c, comp in enumerate(_solenoidal_components(n, seed, kmax)):
        u[c] = comp
        ssq += _sum_sq(comp)
    u *= urms / math.sqrt(ssq / (nz * ny * nx))
    return u


def solenoidal_state_fields(n, seed, urms=0.1, a_amp=1e-5, kmax=4):
    """The 7 fields of solenoidal_state(n, seed), one (nz, ny, nx) array at a time and with the
    same values, holding at most two fields in memory (1024^3: 8.6 GB per field).  The velocity
    is generated twice: once for its rms, once scaled."""
    shape = _shape(n)
    ssq = sum(_sum_sq(comp) for comp in _solenoidal_components(n, seed, kmax))
    scale = urms / math.sqrt(ssq / (shape[0] * shape[1] * shape[2]))
    yield np.zeros(shape)
    for comp in _solenoidal_components(n, seed, kmax):
        comp *= scale
        yield comp
    rng = np.random.default_rng(seed + 1)
    for _ in range(3):
        yield rng.standard_normal(shape) * a_amp


def solenoidal_state(n, seed, urms=0.1, a_amp=1e-5, kmax=4):
    """BASELINE configs 3-5: ln rho = 0; u = seeded solenoidal field of rms `urms` at |k| <= kmax;
    A i.i.d. N(0, a_amp^2) (draw order ax, ay, az from default_rng(seed + 1))."""
    shape = _shape(n)
    s = np.zeros((7,) + shape)
    s[1:4] = solenoidal_velocity(shape, seed, urms, kmax)
    rng = np.random.default_rng(seed + 1)
    for i in (4, 5, 6):
        s[i] = rng.standard_normal(shape) * a_amp
    return s


def uniform_state(n, seed):
    """The paper's own benchmark inputs: all 7 fields uniform random in [0, 1)."""
    shape = _shape(n)
    rng = np.random.default_rng(seed)
    return rng.random((7,) + shape)


def smooth_strong_state(n, seed, a_rms=1e-2, lnrho_amp=0.3, urms=0.1):
    """Extra parity input: smooth fields at |k| <= 4 with a strong magnetic field
    (A rms 1e-2, so j x B / rho is O(1e-2)) and ln rho of amplitude `lnrho_amp` (exercises
    exp(-ln rho) and S.grad ln rho)."""
    shape = _shape(n)
    s = np.zeros((7,) + shape)
    s[1:4] = solenoidal_velocity(shape, seed, urms, 4)
    a = solenoidal_velocity(shape, seed + 11, 1.0, 4)
    a *= a_rms / math.sqrt(float((a ** 2).sum(axis=0).mean()))
    s[4:7] = a
    l = solenoidal_velocity(shape, seed + 23, 1.0, 3)[0]
    s[0] = l * (lnrho_amp / np.abs(l).max())
    return s


# ---------------------------------------------------------------------------------------------
# raw random numbers for the forcing: three uniforms in [0, 1) per time step
# ---------------------------------------------------------------------------------------------
_M64 = (1 << 64) - 1


def splitmix64(x):
    """One round of the SplitMix64 output function on a 64-bit counter (public-domain generator)."""
    x = (x + 0x9E3779B97F4A7C15) & _M64
    z = x
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def counter_uniforms(seed, step):
    """The counter-based generator that ac_make_forcing implements on its side:
    u_i = (splitmix64(splitmix64(seed) ^ (3*step + i)) >> 11) * 2^-53, i = 0, 1, 2."""
    key = splitmix64(int(seed) & _M64)
    out = []
    for i in range(3):
        ctr = (3 * int(step) + i) & _M64
        out.append((splitmix64(key ^ ctr) >> 11) * (1.0 / 9007199254740992.0))
    return tuple(out)


def forcing_draws(seed, nsteps):
    """(nsteps, 3) array of the counter-based uniforms for steps 0..nsteps-1."""
    return np.array([counter_uniforms(seed, s) for s in range(nsteps)], dtype=np.float64)
