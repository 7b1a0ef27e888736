"""Shared pieces of the parity tests: the group-scaled error norm (reading G14), the
sub-box trick that lets the oracle check sampled cells of a large grid, and forcing plumbing."""
import math

import numpy as np

from oracle import forcing as of, mhd_c
from paper_2012_08758_b200 import inputs

TWO_PI3 = (2 * math.pi,) * 3


def group_errors(got, want, cs=1.0):
    """max |got - want| / S_g per group g in (lnrho, u, A); S_u = max|u_i|, S_A = max|A_i|,
    S_lnrho = max(max|lnrho|, max|u|/cs), all from the oracle values (reading G14)."""
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    s_u = np.abs(want[1:4]).max()
    s_a = np.abs(want[4:7]).max()
    s_l = max(np.abs(want[0]).max(), s_u / cs)
    tiny = 1e-300
    return {
        "lnrho": np.abs(got[0] - want[0]).max() / max(s_l, tiny),
        "u": np.abs(got[1:4] - want[1:4]).max() / max(s_u, tiny),
        "A": np.abs(got[4:7] - want[4:7]).max() / max(s_a, tiny),
    }


def max_group_error(got, want, cs=1.0):
    return max(group_errors(got, want, cs).values())


def oracle_forcing(seed, step, k_f, sigma, dt, f0, cs, lengths=TWO_PI3):
    u = inputs.counter_uniforms(seed, step)
    return of.forcing_from_draws(*u, k_f, sigma, dt, f0, cs, lengths)


def oracle_run(state, nsteps, dt, lengths, nu, eta, cs, forcing_fn=None, bext=(0.0, 0.0, 0.0)):
    """nsteps oracle steps; forcing_fn(step) -> forcing tuple or None.  Returns list of states."""
    st = mhd_c.Stepper(state, lengths, nu, eta, cs, bext)
    out = []
    for s in range(nsteps):
        st.step(dt, forcing_fn(s) if forcing_fn else None)
        out.append(st.state.copy())
    return out


def subbox_oracle_step(state, centre, dt, lengths, nu, eta, cs, forcing=None, half=12, nsteps=1):
    """Oracle value of all 7 fields at cell `centre` = (z, y, x) after `nsteps` steps (same dt and
    forcing each step), computed on the periodic-extracted (2*half)^3 neighbourhood.  One step
    has a dependency radius of 9 cells (3 substeps x stencil radius 3), so the centre of a
    24^3 sub-box is exact for nsteps = 1 regardless of what happens at the sub-box faces."""
    assert half >= 9 * nsteps + 3
    nz, ny, nx = state.shape[1:]
    cz, cy, cx = centre
    iz = (np.arange(cz - half, cz + half)) % nz
    iy = (np.arange(cy - half, cy + half)) % ny
    ix = (np.arange(cx - half, cx + half)) % nx
    sub = np.ascontiguousarray(state[:, iz][:, :, iy][:, :, :, ix], dtype=np.float64)
    h = (lengths[0] / nx, lengths[1] / ny, lengths[2] / nz)
    sub_lengths = (h[0] * 2 * half, h[1] * 2 * half, h[2] * 2 * half)
    f = None
    if forcing is not None:
        k, phase, re, im = forcing
        origin = np.array([(cx - half) * h[0], (cy - half) * h[1], (cz - half) * h[2]])
        f = (k, phase + float(np.dot(k, origin)), re, im)
    cur = sub
    for _ in range(nsteps):
        cur = mhd_c.step(cur, dt, sub_lengths, nu, eta, cs, f)
    return cur[:, half, half, half]
