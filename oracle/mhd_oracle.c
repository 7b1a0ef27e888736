/*
 * Plain C fp64 oracle: one 2N-RK3 step of isothermal resistive MHD on a triply
 * periodic grid, plus the rms/max diagnostics.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares
 * no code, header, table or constant generator with the CUDA path
 * (paper_2012_08758_b200/csrc).
 *
 * Written from /root/reference/PAPER.md (cited as PAPER.md:<line>):
 *   Eq. 1  D ln rho/Dt = -div u
 *   Eq. 2  Du/Dt = -cs^2 grad ln rho + j x B / rho
 *                  + nu [lap u + 1/3 grad div u + 2 S.grad ln rho] + f
 *   Eq. 3  dA/dt = u x B + eta lap A
 *   B = curl A, j = curl B / mu0, mu0 = 1, S traceless rate of strain
 *   Eq. 4  f(x) = Re{ N f_k exp[i k.x + i phi] }
 *   "6th-order finite difference scheme", stencil radius r = 3
 *   "3rd-order 2N-Runge-Kutta time integration"
 * D/Dt = d/dt + u.grad.  The paper prints no stencil or RK coefficients; the ones
 * below are DESIGN.md readings G1 (maximal-order central stencils), G2 (bidiagonal
 * 12-point mixed stencil; mixed_mode = 1 selects the tensor-product alternative),
 * G3 (diagonal second derivatives use the second-derivative stencil), G4
 * (j = grad div A - lap A), G5 (eta times the component-wise Laplacian), G6, G7
 * (Williamson's alpha, beta), G8 (forcing in all three substeps).
 *
 * Optional (upwind = 1, NEXT-1, reading G17): "In the continuity Equation (1) we have used the
 * high-order upwinding method of Dobler et al. (2006)" (off in the paper's benchmark,
 * PAPER.md:533).  The paper prints no formula.  Reading: the advection term -u.grad ln rho keeps
 * its 6th-order central derivative and gains, per axis a, + |u_a| / (60 h_a) * delta6_a ln rho with
 * delta6 f = f(-3) - 6 f(-2) + 15 f(-1) - 20 f(0) + 15 f(+1) - 6 f(+2) + f(+3): for u_a > 0 the
 * sum is exactly the 5th-order upwind-biased stencil (-2, 15, -60, 20, 30, -3, 0) / (60 h) on points
 * -3 .. +3, mirrored for u_a < 0 (pinned in tests/test_oracle_upwind.py).
 *
 * Every cell is computed by the same straight-line formula; neighbours are found by
 * wrapping each index modulo the grid size.  No blocking, no fusion across cells, no
 * reordering.  The only parallelism is an OpenMP "parallel for" over z planes.
 *
 * Layout: state[7][nz][ny][nx], x fastest; fields lnrho, ux, uy, uz, ax, ay, az.
 *
 * Pins: tests/test_oracle_*.py (P1-P13, P15, P18 of DESIGN.md).  Every pin runs
 * against this C code as well as against the independent numpy restatement
 * (oracle/mhd_numpy.py), and the two are compared with each other (P18).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int nx, ny, nz;
    double lx, ly, lz;
    double nu, eta, cs;
    double bext[3];
    int mixed_mode;      /* 0 = bidiagonal (default reading), 1 = tensor product D_a(D_b f) */
    int has_forcing;
    double fk[3], fphase, fre[3], fim[3];
    int upwind;          /* 0 = off (default, all BASELINE configs), 1 = upwinded continuity equation (G17) */
    int forcing_kick;    /* 0 = f is a term of the RHS in all three substeps (default, reading G8); 1 = the alternative
                            reading: the delta-correlated forcing is an impulse u += dt f added once, after substep 2 */
} orc_params;

static const double C1[3] = {3.0 / 4.0, -3.0 / 20.0, 1.0 / 60.0};
static const double C2_0 = -49.0 / 18.0;
static const double C2[3] = {3.0 / 2.0, -3.0 / 20.0, 1.0 / 90.0};
static const double CM[3] = {270.0 / 720.0, -27.0 / 720.0, 2.0 / 720.0};

static const double RK_ALPHA[3] = {0.0, -5.0 / 9.0, -153.0 / 128.0};
static const double RK_BETA[3] = {1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0};

static long wrap(long i, long n) {
    i %= n;
    if (i < 0) i += n;
    return i;
}

/* value of field f at (x + d[0], y + d[1], z + d[2]), periodic */
static double at(const double* f, const orc_params* p, long x, long y, long z, long dx, long dy, long dz) {
    long xx = wrap(x + dx, p->nx), yy = wrap(y + dy, p->ny), zz = wrap(z + dz, p->nz);
    return f[(size_t)xx + (size_t)p->nx * ((size_t)yy + (size_t)p->ny * (size_t)zz)];
}

static double spacing(const orc_params* p, int a) {
    return a == 0 ? p->lx / p->nx : (a == 1 ? p->ly / p->ny : p->lz / p->nz);
}

static double der1(const double* f, const orc_params* p, long x, long y, long z, int a) {
    double s = 0.0;
    for (int m = 1; m <= 3; m++) {
        long d[3] = {0, 0, 0};
        d[a] = m;
        s += C1[m - 1] * (at(f, p, x, y, z, d[0], d[1], d[2]) - at(f, p, x, y, z, -d[0], -d[1], -d[2]));
    }
    return s / spacing(p, a);
}

static double der2(const double* f, const orc_params* p, long x, long y, long z, int a) {
    double s = C2_0 * at(f, p, x, y, z, 0, 0, 0);
    for (int m = 1; m <= 3; m++) {
        long d[3] = {0, 0, 0};
        d[a] = m;
        s += C2[m - 1] * (at(f, p, x, y, z, d[0], d[1], d[2]) + at(f, p, x, y, z, -d[0], -d[1], -d[2]));
    }
    double h = spacing(p, a);
    return s / (h * h);
}

/* delta6_a f / (60 h_a): the sixth difference that turns the central first derivative into the
 * 5th-order upwind-biased one (G17) */
static const double C6_0 = -20.0;
static const double C6[3] = {15.0, -6.0, 1.0};
static double der6_upwind(const double* f, const orc_params* p, long x, long y, long z, int a) {
    double s = C6_0 * at(f, p, x, y, z, 0, 0, 0);
    for (int m = 1; m <= 3; m++) {
        long d[3] = {0, 0, 0};
        d[a] = m;
        s += C6[m - 1] * (at(f, p, x, y, z, d[0], d[1], d[2]) + at(f, p, x, y, z, -d[0], -d[1], -d[2]));
    }
    return s / (60.0 * spacing(p, a));
}

static double dermix(const double* f, const orc_params* p, long x, long y, long z, int a, int b) {
    double ha = spacing(p, a), hb = spacing(p, b);
    if (p->mixed_mode == 1) {
        /* D_a (D_b f): first-derivative stencil along a applied to first derivatives along b */
        double s = 0.0;
        for (int m = 1; m <= 3; m++) {
            long d[3] = {0, 0, 0};
            d[a] = m;
            s += C1[m - 1] * (der1(f, p, x + d[0], y + d[1], z + d[2], b) - der1(f, p, x - d[0], y - d[1], z - d[2], b));
        }
        return s / ha;
    }
    double s = 0.0;
    for (int m = 1; m <= 3; m++) {
        long da[3] = {0, 0, 0}, db[3] = {0, 0, 0};
        da[a] = m;
        db[b] = m;
        double pp = at(f, p, x, y, z, da[0] + db[0], da[1] + db[1], da[2] + db[2]);
        double mm = at(f, p, x, y, z, -da[0] - db[0], -da[1] - db[1], -da[2] - db[2]);
        double pm = at(f, p, x, y, z, da[0] - db[0], da[1] - db[1], da[2] - db[2]);
        double mp = at(f, p, x, y, z, -da[0] + db[0], -da[1] + db[1], -da[2] + db[2]);
        s += CM[m - 1] * (pp + mm - pm - mp);
    }
    return s / (ha * hb);
}

/* B = curl A (+ uniform external field, reading G16) at one cell */
static void curl_a(const double* const A[3], const orc_params* p, long x, long y, long z, double B[3]) {
    B[0] = der1(A[2], p, x, y, z, 1) - der1(A[1], p, x, y, z, 2) + p->bext[0];
    B[1] = der1(A[0], p, x, y, z, 2) - der1(A[2], p, x, y, z, 0) + p->bext[1];
    B[2] = der1(A[1], p, x, y, z, 0) - der1(A[0], p, x, y, z, 1) + p->bext[2];
}

/* right-hand sides of Eq. 1-3 for every cell: rhs[7][nz][ny][nx] */
void orc_rhs(const double* state, double* rhs, const orc_params* p) {
    const size_t n = (size_t)p->nx * p->ny * p->nz;
    const double* lnrho = state;
    const double* u[3] = {state + n, state + 2 * n, state + 3 * n};
    const double* A[3] = {state + 4 * n, state + 5 * n, state + 6 * n};
    const double hx = spacing(p, 0), hy = spacing(p, 1), hz = spacing(p, 2);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++) {
                const size_t c = (size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z);
                double g[3], G[3][3], lapu[3], graddivu[3], S[3][3];
                double B[3], lapA[3], jj[3], uc[3];
                for (int a = 0; a < 3; a++) g[a] = der1(lnrho, p, x, y, z, a);
                for (int i = 0; i < 3; i++) {
                    uc[i] = u[i][c];
                    for (int j = 0; j < 3; j++) G[i][j] = der1(u[i], p, x, y, z, j);   /* G_ij = d_j u_i */
                }
                double divu = G[0][0] + G[1][1] + G[2][2];
                for (int i = 0; i < 3; i++) {
                    lapu[i] = der2(u[i], p, x, y, z, 0) + der2(u[i], p, x, y, z, 1) + der2(u[i], p, x, y, z, 2);
                    double s = der2(u[i], p, x, y, z, i);
                    for (int j = 0; j < 3; j++)
                        if (j != i) s += dermix(u[j], p, x, y, z, i, j);
                    graddivu[i] = s;
                }
                for (int i = 0; i < 3; i++)
                    for (int j = 0; j < 3; j++)
                        S[i][j] = 0.5 * (G[i][j] + G[j][i]) - (i == j ? divu / 3.0 : 0.0);
                curl_a(A, p, x, y, z, B);
                for (int i = 0; i < 3; i++) {
                    lapA[i] = der2(A[i], p, x, y, z, 0) + der2(A[i], p, x, y, z, 1) + der2(A[i], p, x, y, z, 2);
                    double s = der2(A[i], p, x, y, z, i);
                    for (int j = 0; j < 3; j++)
                        if (j != i) s += dermix(A[j], p, x, y, z, i, j);
                    jj[i] = s - lapA[i];                                                /* j = grad div A - lap A */
                }
                /* Eq. 1 */
                rhs[c] = -(uc[0] * g[0] + uc[1] * g[1] + uc[2] * g[2]) - divu;
                if (p->upwind)
                    for (int a = 0; a < 3; a++) rhs[c] += fabs(uc[a]) * der6_upwind(lnrho, p, x, y, z, a);
                /* forcing, Eq. 4 */
                double f[3] = {0.0, 0.0, 0.0};
                if (p->has_forcing && !p->forcing_kick) {
                    double theta = p->fk[0] * (x * hx) + p->fk[1] * (y * hy) + p->fk[2] * (z * hz) + p->fphase;
                    double ct = cos(theta), st = sin(theta);
                    for (int i = 0; i < 3; i++) f[i] = p->fre[i] * ct - p->fim[i] * st;
                }
                double rho_inv = exp(-lnrho[c]);
                double jxb[3] = {jj[1] * B[2] - jj[2] * B[1], jj[2] * B[0] - jj[0] * B[2], jj[0] * B[1] - jj[1] * B[0]};
                double uxb[3] = {uc[1] * B[2] - uc[2] * B[1], uc[2] * B[0] - uc[0] * B[2], uc[0] * B[1] - uc[1] * B[0]};
                for (int i = 0; i < 3; i++) {
                    double adv = uc[0] * G[i][0] + uc[1] * G[i][1] + uc[2] * G[i][2];
                    double sgl = S[i][0] * g[0] + S[i][1] * g[1] + S[i][2] * g[2];
                    /* Eq. 2 */
                    rhs[(size_t)(1 + i) * n + c] = -adv - p->cs * p->cs * g[i] + jxb[i] * rho_inv
                                                   + p->nu * (lapu[i] + graddivu[i] / 3.0 + 2.0 * sgl) + f[i];
                    /* Eq. 3 */
                    rhs[(size_t)(4 + i) * n + c] = uxb[i] + p->eta * lapA[i];
                }
            }
}

/* one substep s of the 2N scheme: w <- alpha_s w + dt RHS(state); state <- state + beta_s w.
 * scratch holds 7 fields. */
void orc_substep(double* state, double* w, double* scratch, int s, double dt, const orc_params* p) {
    const size_t n7 = (size_t)7 * p->nx * p->ny * p->nz;
    orc_rhs(state, scratch, p);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (long long i = 0; i < (long long)n7; i++) {
        w[i] = RK_ALPHA[s] * w[i] + dt * scratch[i];
        state[i] = state[i] + RK_BETA[s] * w[i];
    }
}

/* one full step: three substeps with the same forcing parameters; w starts at 0 (alpha_0 = 0) */
void orc_step(double* state, double* w, double* scratch, double dt, const orc_params* p) {
    const size_t n7 = (size_t)7 * p->nx * p->ny * p->nz;
    for (size_t i = 0; i < n7; i++) w[i] = 0.0;
    for (int s = 0; s < 3; s++) orc_substep(state, w, scratch, s, dt, p);
    if (p->has_forcing && p->forcing_kick) {
        /* alternative reading of G8: u += dt f(x) once per step, Eq. 4 evaluated as in orc_rhs */
        const size_t n = (size_t)p->nx * p->ny * p->nz;
        const double hx = spacing(p, 0), hy = spacing(p, 1), hz = spacing(p, 2);
        for (long z = 0; z < p->nz; z++)
            for (long y = 0; y < p->ny; y++)
                for (long x = 0; x < p->nx; x++) {
                    const size_t c = (size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z);
                    double theta = p->fk[0] * (x * hx) + p->fk[1] * (y * hy) + p->fk[2] * (z * hz) + p->fphase;
                    double ct = cos(theta), st = sin(theta);
                    for (int i = 0; i < 3; i++) state[(size_t)(1 + i) * n + c] += dt * (p->fre[i] * ct - p->fim[i] * st);
                }
    }
}

/* out: urms, umax, brms, bmax, lnrho_min, lnrho_max, nonfinite (0/1) */
void orc_diag(const double* state, const orc_params* p, double out[7]) {
    const size_t n = (size_t)p->nx * p->ny * p->nz;
    const double* u[3] = {state + n, state + 2 * n, state + 3 * n};
    const double* A[3] = {state + 4 * n, state + 5 * n, state + 6 * n};
    double su = 0.0, sb = 0.0, mu = 0.0, mb = 0.0, lmin = INFINITY, lmax = -INFINITY;
    int bad = 0;
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++) {
                const size_t c = (size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z);
                double u2 = u[0][c] * u[0][c] + u[1][c] * u[1][c] + u[2][c] * u[2][c];
                double B[3];
                curl_a(A, p, x, y, z, B);
                double b2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
                su += u2;
                sb += b2;
                if (u2 > mu) mu = u2;
                if (b2 > mb) mb = b2;
                if (state[c] < lmin) lmin = state[c];
                if (state[c] > lmax) lmax = state[c];
                for (int q = 0; q < 7; q++)
                    if (!isfinite(state[(size_t)q * n + c])) bad = 1;
            }
    out[0] = sqrt(su / (double)n);
    out[1] = sqrt(mu);
    out[2] = sqrt(sb / (double)n);
    out[3] = sqrt(mb);
    out[4] = lmin;
    out[5] = lmax;
    out[6] = (double)bad;
}

/* Extended diagnostics (NEXT-4): volume means of the kinetic helicity omega.u, omega = curl u, and of the current
 * helicity j.B (Eq. 11; mu0 = rho0 = 1; j = grad div A - lap A as in Eq. 2, reading G4;
 * B includes the external field), and the largest Alfven speed |B| / sqrt(rho) (the optional term of the CFL rule,
 * reading G15).  In a periodic box <j> = 0, so the mean of j.B equals that of the fluctuating parts j'.b' of Eq. 11.
 * out: <omega.u>, <j.B>, max |B| rho^(-1/2) */
void orc_diag_ext(const double* state, const orc_params* p, double out[3]) {
    const size_t n = (size_t)p->nx * p->ny * p->nz;
    const double* lnrho = state;
    const double* u[3] = {state + n, state + 2 * n, state + 3 * n};
    const double* A[3] = {state + 4 * n, state + 5 * n, state + 6 * n};
    double hk = 0.0, hc = 0.0, va2 = 0.0;
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++) {
                const size_t c = (size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z);
                double om[3], B[3], jj[3];
                om[0] = der1(u[2], p, x, y, z, 1) - der1(u[1], p, x, y, z, 2);
                om[1] = der1(u[0], p, x, y, z, 2) - der1(u[2], p, x, y, z, 0);
                om[2] = der1(u[1], p, x, y, z, 0) - der1(u[0], p, x, y, z, 1);
                curl_a(A, p, x, y, z, B);
                for (int i = 0; i < 3; i++) {
                    double lap = der2(A[i], p, x, y, z, 0) + der2(A[i], p, x, y, z, 1) + der2(A[i], p, x, y, z, 2);
                    double s = der2(A[i], p, x, y, z, i);
                    for (int j = 0; j < 3; j++)
                        if (j != i) s += dermix(A[j], p, x, y, z, i, j);
                    jj[i] = s - lap;
                }
                hk += om[0] * u[0][c] + om[1] * u[1][c] + om[2] * u[2][c];
                hc += jj[0] * B[0] + jj[1] * B[1] + jj[2] * B[2];
                double v2 = (B[0] * B[0] + B[1] * B[1] + B[2] * B[2]) * exp(-lnrho[c]);
                if (v2 > va2) va2 = v2;
            }
    out[0] = hk / (double)n;
    out[1] = hc / (double)n;
    out[2] = sqrt(va2);
}

/* single derivative operators on a whole scalar field, for the operator pins (P1-P3) */
void orc_der1_field(const double* f, double* out, const orc_params* p, int a) {
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++)
                out[(size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z)] = der1(f, p, x, y, z, a);
}
void orc_der2_field(const double* f, double* out, const orc_params* p, int a) {
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++)
                out[(size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z)] = der2(f, p, x, y, z, a);
}
void orc_der6_upwind_field(const double* f, double* out, const orc_params* p, int a) {
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++)
                out[(size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z)] = der6_upwind(f, p, x, y, z, a);
}
void orc_dermix_field(const double* f, double* out, const orc_params* p, int a, int b) {
    for (long z = 0; z < p->nz; z++)
        for (long y = 0; y < p->ny; y++)
            for (long x = 0; x < p->nx; x++)
                out[(size_t)x + (size_t)p->nx * ((size_t)y + (size_t)p->ny * (size_t)z)] = dermix(f, p, x, y, z, a, b);
}

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
