"""Host side of the forcing (Eq. 4-6), fp64 numpy.

TEST INFRASTRUCTURE ONLY (see oracle/mhd_numpy.py header).  Shares no code with
the C-ABI library's ac_make_forcing / ac_forcing_from_draws.

The random numbers are INPUTS: three uniforms u1, u2, u3 in [0, 1) per time step
(one wavevector, one phase, one direction e-hat per step).

* shell ("4.5 <= |k| <= 5.5, such that kx, ky, kz are integers";
  reading G11): all integer vectors with k_f - 1/2 <= |k| <= k_f + 1/2, sorted
  lexicographically; index = floor(u1 * len).
* phase phi = -pi + 2 pi u2 ("random phase in range [-pi, pi]").
* e-hat ("random unit vector perpendicular to k"): reading G9,
  e-hat = cos(psi) e1 + sin(psi) e2, psi = 2 pi u3, e1 = normalise(k x a) with a the
  coordinate unit vector of the smallest |k_a| (ties: lowest axis), e2 = k-hat x e1.
* f_k: Eq. 6 written out in full, including the factor
  sqrt(1 - (k.e)^2/k^2) that equals 1 for perpendicular e-hat.
* N = f0 c_s sqrt(|k| c_s / dt)  (Eq. 5; readings G10, G12).

Pins (tests/test_oracle_forcing.py, P12-P13): |f_k| = 1, k.f_k = 0,
i k x f_k = |k| f_k for sigma = 1, box mean of |f|^2 = N^2/2, brute-force shell counts.
"""
import math
import numpy as np


def shell(k_f):
    """Sorted list of integer wavevectors with k_f - 1/2 <= |k| <= k_f + 1/2."""
    lo2, hi2 = (k_f - 0.5) ** 2, (k_f + 0.5) ** 2
    r = int(math.floor(k_f + 0.5))
    out = []
    for kx in range(-r, r + 1):
        for ky in range(-r, r + 1):
            for kz in range(-r, r + 1):
                k2 = kx * kx + ky * ky + kz * kz
                if lo2 <= k2 <= hi2:
                    out.append((kx, ky, kz))
    out.sort()
    return out


def e_basis(k):
    k = np.asarray(k, dtype=np.float64)
    absk = np.abs(k)
    a_idx = int(np.argmin(absk))            # argmin returns the lowest index on ties
    a = np.zeros(3)
    a[a_idx] = 1.0
    e1 = np.cross(k, a)
    e1 = e1 / np.sqrt(e1 @ e1)
    khat = k / np.sqrt(k @ k)
    e2 = np.cross(khat, e1)
    return e1, e2


def f_k(k, ehat, sigma):
    """Eq. 6.  Returns a complex 3-vector."""
    k = np.asarray(k, dtype=np.float64)
    ehat = np.asarray(ehat, dtype=np.float64)
    k2 = k @ k
    kabs = math.sqrt(k2)
    kxe = np.cross(k, ehat)
    kxkxe = np.cross(k, kxe)
    num = kxkxe - 1j * sigma * kabs * kxe
    kde = k @ ehat
    den = math.sqrt(1.0 + sigma * sigma) * k2 * math.sqrt(1.0 - kde * kde / k2)
    return num / den


def normalisation(kabs, dt, f0, cs):
    """Eq. 5."""
    return f0 * cs * math.sqrt(kabs * cs / dt)


def forcing_from_draws(u1, u2, u3, k_f, sigma, dt, f0, cs, lengths=(2.0 * math.pi,) * 3):
    """(k[3], phase, re[3], im[3]) with re + i im = N f_k, for the three uniforms of this step.
    The integer shell vector counts periods per box side; the returned k is in radians per unit
    length, k_a * 2 pi / L_a (equal to the integers for the paper's L = 2 pi)."""
    sh = shell(k_f)
    idx = min(int(math.floor(u1 * len(sh))), len(sh) - 1)
    k = np.array(sh[idx], dtype=np.float64)
    phase = -math.pi + 2.0 * math.pi * u2
    psi = 2.0 * math.pi * u3
    e1, e2 = e_basis(k)
    ehat = math.cos(psi) * e1 + math.sin(psi) * e2
    fk = f_k(k, ehat, sigma)
    n = normalisation(math.sqrt(k @ k), dt, f0, cs)
    amp = n * fk
    k_phys = k * (2.0 * math.pi / np.asarray(lengths, dtype=np.float64))
    return (k_phys, phase, amp.real.copy(), amp.imag.copy())
