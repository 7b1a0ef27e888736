"""Plain numpy fp64 oracle for one 2N-RK3 step of isothermal resistive MHD.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (the package, the C-ABI
library, bench.py's GPU legs) may import this module; only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs do.
It shares no code with the CUDA path.

What it computes, step by step, in the paper's order and notation
(citations are /root/reference/PAPER.md line numbers):

* state: ln rho, u = (ux, uy, uz), A = (ax, ay, az) on a triply periodic grid
  (Eq. 1-3; periodic cube of side 2*pi).
* spatial derivatives: "6th-order finite difference scheme",
  stencil radius r = 3 (Fig. 1).  The paper prints no
  coefficients; they are the unique maximal-order central stencils (DESIGN.md
  reading G1) and the bidiagonal 12-point mixed stencil (reading G2).  The
  tests re-derive them from the moment equations in exact rationals.
* right-hand sides: Eq. 1 (continuity, ln rho form), Eq. 2 (momentum with
  c_s^2 grad ln rho, j x B / rho, nu[lap u + 1/3 grad div u + 2 S.grad ln rho],
  forcing f), Eq. 3 (dA/dt = u x B + eta lap A), with
  B = curl A, j = curl B / mu0, mu0 = 1.
* forcing: f(x) = Re{N f_k exp[i k.x + i phi]}  (Eq. 4).
* time integration: "3rd-order 2N-Runge-Kutta"; coefficients are
  Williamson's (reading G7).  The register w is kept explicitly.

Arrays: state has shape (7, nz, ny, nx), C order, x fastest; field order
lnrho, ux, uy, uz, ax, ay, az.  Axis numbering below: 0 = x, 1 = y, 2 = z,
which is numpy axis 2, 1, 0 of a (nz, ny, nx) array.

Every neighbour access is a numpy roll, i.e. periodic index wrap.  No
blocking, fusion or reordering beyond the formulas as written.

Pins (tests/test_oracle_*.py): P1 rational re-derivation of the coefficients,
P2/P3 modified wavenumbers and 6th-order convergence, P4 stability polynomial
and 3rd-order convergence, P5 div B = 0, P6 sum of div u = 0, P7-P11 linear
waves with the discrete modified wavenumber, P12-P13 forcing, P15 axis
permutation covariance, P18 agreement with the independent C oracle.
Parity unpinned by the paper (fixed by DESIGN.md readings): choice of the
bidiagonal mixed stencil (G2), forcing applied in all three substeps (G8).
"""
import numpy as np

# DESIGN.md reading G1: maximal-order central 7-point stencils.
D1 = (3.0 / 4.0, -3.0 / 20.0, 1.0 / 60.0)              # first derivative, weights of f(+m) - f(-m)
D2_0 = -49.0 / 18.0                                     # second derivative, centre weight
D2 = (3.0 / 2.0, -3.0 / 20.0, 1.0 / 90.0)              # second derivative, weights of f(+m) + f(-m)
# DESIGN.md reading G2: bidiagonal mixed stencil, weights of the 4-point corner sums.
DMIX = (270.0 / 720.0, -27.0 / 720.0, 2.0 / 720.0)

# DESIGN.md reading G7: Williamson (1980) 2N-storage RK3.
RK_ALPHA = (0.0, -5.0 / 9.0, -153.0 / 128.0)
RK_BETA = (1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0)

LNRHO, UX, UY, UZ, AX, AY, AZ = range(7)


def _np_axis(a):
    """grid axis a (0 = x, 1 = y, 2 = z) -> numpy axis of a (nz, ny, nx) array."""
    return 2 - a


def shift(f, a, m):
    """f evaluated at index + m along grid axis a, periodic."""
    return np.roll(f, -m, axis=_np_axis(a))


def grid_spacing(shape, lengths):
    nz, ny, nx = shape
    lx, ly, lz = lengths
    return (lx / nx, ly / ny, lz / nz)


def der1(f, a, h):
    """D_a f, 6th order."""
    s = 0.0
    for m in (1, 2, 3):
        s = s + D1[m - 1] * (shift(f, a, m) - shift(f, a, -m))
    return s / h[a]


def der2(f, a, h):
    """D_aa f, 6th order."""
    s = D2_0 * f
    for m in (1, 2, 3):
        s = s + D2[m - 1] * (shift(f, a, m) + shift(f, a, -m))
    return s / (h[a] * h[a])


# 5th-order upwind-biased first derivative on points -3 .. +2 (flow towards +a); the mirror image
# serves flow towards -a.  Textbook weights (Dobler et al. 2006's upwinding, reading G17), over 60 h.
UPW5 = (-2.0, 15.0, -60.0, 20.0, 30.0, -3.0)


def der1_upwind(f, a, h, vel):
    """First derivative of f along a taken on the side the flow `vel` comes from."""
    plus = 0.0      # vel > 0: points -3 .. +2
    minus = 0.0     # vel < 0: points -2 .. +3 with mirrored, negated weights
    for w, m in zip(UPW5, (-3, -2, -1, 0, 1, 2)):
        plus = plus + w * shift(f, a, m)
        minus = minus - w * shift(f, a, -m)
    return np.where(vel >= 0.0, plus, minus) / (60.0 * h[a])


def dermix(f, a, b, h, mixed="bidiagonal"):
    """D_ab f, a != b.  Default: bidiagonal 12-point stencil (reading G2).
    mixed="tensor" is the alternative reading D_a(D_b f) (36 points), kept as a flag."""
    assert a != b
    if mixed == "tensor":
        return der1(der1(f, b, h), a, h)
    s = 0.0
    for m in (1, 2, 3):
        pp = shift(shift(f, a, m), b, m)
        mm = shift(shift(f, a, -m), b, -m)
        pm = shift(shift(f, a, m), b, -m)
        mp = shift(shift(f, a, -m), b, m)
        s = s + DMIX[m - 1] * (pp + mm - pm - mp)
    return s / (h[a] * h[b])


def curl_a(state, h):
    """B = curl A with first-derivative stencils."""
    ax, ay, az = state[AX], state[AY], state[AZ]
    bx = der1(az, 1, h) - der1(ay, 2, h)
    by = der1(ax, 2, h) - der1(az, 0, h)
    bz = der1(ay, 0, h) - der1(ax, 1, h)
    return [bx, by, bz]


def forcing_field(shape, h, forcing):
    """f_i(x) = re_i cos(theta) - im_i sin(theta), theta = k.x + phase, x_a = i_a h_a
    (Eq. 4; re + i im = N f_k).  forcing = (k[3], phase, re[3], im[3]) or None."""
    nz, ny, nx = shape
    if forcing is None:
        z = np.zeros(shape)
        return [z, z, z]
    k, phase, re, im = forcing
    x = np.arange(nx) * h[0]
    y = np.arange(ny) * h[1]
    z = np.arange(nz) * h[2]
    theta = (k[0] * x)[None, None, :] + (k[1] * y)[None, :, None] + (k[2] * z)[:, None, None] + phase
    c, s = np.cos(theta), np.sin(theta)
    return [re[i] * c - im[i] * s for i in range(3)]


def rhs(state, lengths, nu, eta, cs, forcing=None, bext=(0.0, 0.0, 0.0), mixed="bidiagonal", upwind=False):
    """Right-hand sides of Eq. 1-3, SURVEY 8(c) steps 2-5."""
    shape = state.shape[1:]
    h = grid_spacing(shape, lengths)
    lnrho = state[LNRHO]
    u = [state[UX], state[UY], state[UZ]]
    A = [state[AX], state[AY], state[AZ]]

    # step 2: gradients of ln rho and u
    g = [der1(lnrho, a, h) for a in range(3)]
    G = [[der1(u[i], j, h) for j in range(3)] for i in range(3)]          # G[i][j] = d_j u_i
    divu = G[0][0] + G[1][1] + G[2][2]
    lapu = [der2(u[i], 0, h) + der2(u[i], 1, h) + der2(u[i], 2, h) for i in range(3)]
    graddivu = []
    for i in range(3):
        s = der2(u[i], i, h)
        for j in range(3):
            if j != i:
                s = s + dermix(u[j], i, j, h, mixed)
        graddivu.append(s)
    S = [[0.5 * (G[i][j] + G[j][i]) - (divu / 3.0 if i == j else 0.0) for j in range(3)] for i in range(3)]

    # step 3: B, lap A, j = grad div A - lap A (mu0 = 1)
    B = curl_a(state, h)
    B = [B[i] + bext[i] for i in range(3)]
    lapA = [der2(A[i], 0, h) + der2(A[i], 1, h) + der2(A[i], 2, h) for i in range(3)]
    jj = []
    for i in range(3):
        s = der2(A[i], i, h)
        for j in range(3):
            if j != i:
                s = s + dermix(A[j], i, j, h, mixed)
        jj.append(s - lapA[i])

    # step 4: right-hand sides
    out = np.empty_like(state)
    if upwind:
        # upwinded continuity equation (reading G17): each u_a d_a ln rho uses the
        # upwind-biased derivative
        out[LNRHO] = -(u[0] * der1_upwind(lnrho, 0, h, u[0]) + u[1] * der1_upwind(lnrho, 1, h, u[1])
                       + u[2] * der1_upwind(lnrho, 2, h, u[2])) - divu
    else:
        out[LNRHO] = -(u[0] * g[0] + u[1] * g[1] + u[2] * g[2]) - divu
    rho_inv = np.exp(-lnrho)
    jxb = [jj[1] * B[2] - jj[2] * B[1], jj[2] * B[0] - jj[0] * B[2], jj[0] * B[1] - jj[1] * B[0]]
    uxb = [u[1] * B[2] - u[2] * B[1], u[2] * B[0] - u[0] * B[2], u[0] * B[1] - u[1] * B[0]]
    f = forcing_field(shape, h, forcing)
    for i in range(3):
        adv = u[0] * G[i][0] + u[1] * G[i][1] + u[2] * G[i][2]
        sgl = S[i][0] * g[0] + S[i][1] * g[1] + S[i][2] * g[2]
        out[UX + i] = (-adv - cs * cs * g[i] + jxb[i] * rho_inv
                       + nu * (lapu[i] + graddivu[i] / 3.0 + 2.0 * sgl) + f[i])
        out[AX + i] = uxb[i] + eta * lapA[i]
    return out


def substep(state, w, s, dt, lengths, nu, eta, cs, forcing=None, bext=(0.0, 0.0, 0.0), mixed="bidiagonal",
            upwind=False):
    """One 2N-RK3 substep: w <- alpha_s w + dt RHS(f); f <- f + beta_s w."""
    r = rhs(state, lengths, nu, eta, cs, forcing, bext, mixed, upwind)
    w = RK_ALPHA[s] * w + dt * r
    return state + RK_BETA[s] * w, w


def step(state, dt, lengths, nu, eta, cs, forcing=None, bext=(0.0, 0.0, 0.0), mixed="bidiagonal", upwind=False,
         kick=False):
    """One full RK3 step (three substeps, same forcing parameters in all three: reading G8).  kick=True is the
    alternative reading: no forcing inside the substeps, one impulse u += dt f after the last one."""
    w = np.zeros_like(state)
    for s in range(3):
        state, w = substep(state, w, s, dt, lengths, nu, eta, cs, None if kick else forcing, bext, mixed, upwind)
    if kick and forcing is not None:
        state = state.copy()
        f = forcing_field(state.shape[1:], grid_spacing(state.shape[1:], lengths), forcing)
        for i in range(3):
            state[UX + i] = state[UX + i] + dt * f[i]
    return state


def diagnostics(state, lengths, bext=(0.0, 0.0, 0.0)):
    """rms and max over cells of |u| and |B| (reading G18): rms = sqrt(mean |v|^2)."""
    h = grid_spacing(state.shape[1:], lengths)
    u2 = state[UX] ** 2 + state[UY] ** 2 + state[UZ] ** 2
    B = curl_a(state, h)
    b2 = (B[0] + bext[0]) ** 2 + (B[1] + bext[1]) ** 2 + (B[2] + bext[2]) ** 2
    return {
        "urms": float(np.sqrt(u2.mean())), "umax": float(np.sqrt(u2.max())),
        "brms": float(np.sqrt(b2.mean())), "bmax": float(np.sqrt(b2.max())),
        "lnrho_min": float(state[LNRHO].min()), "lnrho_max": float(state[LNRHO].max()),
        "nonfinite": int(not np.isfinite(state).all()),
    }


def diagnostics_ext(state, lengths, bext=(0.0, 0.0, 0.0), mixed="bidiagonal"):
    """<omega.u>, <j.B> (Eq. 11; mu0 = rho0 = 1) and max |B| / sqrt(rho) (the Alfven term of G15)."""
    h = grid_spacing(state.shape[1:], lengths)
    u = [state[UX], state[UY], state[UZ]]
    a = [state[AX], state[AY], state[AZ]]
    om = [der1(u[2], 1, h) - der1(u[1], 2, h), der1(u[0], 2, h) - der1(u[2], 0, h), der1(u[1], 0, h) - der1(u[0], 1, h)]
    B = curl_a(state, h)
    B = [B[i] + bext[i] for i in range(3)]
    jj = []
    for i in range(3):
        gd = der2(a[i], i, h)
        for j in range(3):
            if j != i:
                gd = gd + dermix(a[j], min(i, j), max(i, j), h, mixed)
        jj.append(gd - (der2(a[i], 0, h) + der2(a[i], 1, h) + der2(a[i], 2, h)))
    hk = sum(om[i] * u[i] for i in range(3)).mean()
    hc = sum(jj[i] * B[i] for i in range(3)).mean()
    va2 = (sum(B[i] ** 2 for i in range(3)) * np.exp(-state[LNRHO])).max()
    return {"kin_hel": float(hk), "cur_hel": float(hc), "va_max": float(np.sqrt(va2))}


def cfl_dt_alfven(umax, va_max, shape, lengths, nu, eta, cs, c_u=0.4, c_nu=0.25):
    """The optional Alfven-speed form of G15: the signal speed c_s becomes sqrt(c_s^2 + max v_A^2)."""
    h = min(grid_spacing(shape, lengths))
    dt_adv = c_u * h / (umax + np.sqrt(cs * cs + va_max * va_max))
    d = max(nu, eta)
    if d <= 0.0:
        return dt_adv
    return min(dt_adv, c_nu * h * h / d)


def cfl_dt(umax, shape, lengths, nu, eta, cs, c_u=0.4, c_nu=0.25):
    """dt = min(C_u h/(max|u| + c_s), C_nu h^2/max(nu, eta)), h = min spacing (reading G15;
    parity unpinned by the paper: the paper's benchmark uses a constant time step)."""
    h = min(grid_spacing(shape, lengths))
    dt_adv = c_u * h / (umax + cs)
    d = max(nu, eta)
    if d <= 0.0:
        return dt_adv
    return min(dt_adv, c_nu * h * h / d)
