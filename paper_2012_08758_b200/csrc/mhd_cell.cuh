// Per-cell arithmetic of one 2N-RK3 substep of isothermal resistive MHD (device code).
//
// What it computes (citations: /root/reference/PAPER.md; G<n> = DESIGN.md readings):
//   Eq. 1-3 right-hand sides, forcing Eq. 4, 6th-order
//   radius-3 central differences (G1-G3), j = grad div A - lap A (G4),
//   2N-RK3 update in difference form (G7).
// The function is written against an abstract neighbour fetch so that every kernel variant
// (global-memory loads, shared-memory tiles) evaluates the same expression tree per cell.
#pragma once
#include <cuda_runtime.h>

namespace ac {

enum { LNRHO = 0, UX = 1, UY = 2, UZ = 3, AX = 4, AY = 5, AZ = 6, NFIELDS = 7 };

// Stencil weights with the grid spacing folded in.
//   c1[a][m-1]  = w1_m / h_a          first derivative,  weights of f(+m) - f(-m)
//   c2[a][m-1]  = w2_m / h_a^2        second derivative, weights of f(+m) + f(-m)
//   c20[a]      = w2_0 / h_a^2        second derivative, centre
//   cm[p][m-1]  = wm_m / (h_a h_b)    mixed derivative in plane p (0 = xy, 1 = xz, 2 = yz)
template <typename T>
struct Coeffs {
    T c1[3][3];
    T c2[3][3];
    T c20[3];
    T cm[3][3];
    T c6[3][3];   // upwinding (G17): weights (15, -6, 1) / (60 h_a) of f(+m) + f(-m)
    T c60[3];     //                  centre weight -20 / (60 h_a)
};

template <typename T>
struct Physics {
    T nu, eta, cs2;
    T bext[3];
    T rk_a;  // beta_s * alpha_s / beta_{s-1}   (0 for substep 0)
    T rk_b;  // beta_s * dt
    T fre[3], fim[3];
    int has_forcing;
    int substep;
    int upwind;   // 1: continuity equation with the 5th-order upwind correction (G17)
    int mixed_tensor;   // 1: mixed derivatives as D_a(D_b f) (36 points) instead of the bidiagonal stencil (G2, NEXT-4)
};

template <typename T>
__device__ __forceinline__ T fma_(T a, T b, T c);
template <>
__device__ __forceinline__ double fma_<double>(double a, double b, double c) { return fma(a, b, c); }
template <>
__device__ __forceinline__ float fma_<float>(float a, float b, float c) { return fmaf(a, b, c); }

__device__ __forceinline__ double abs_(double x) { return fabs(x); }
__device__ __forceinline__ float abs_(float x) { return fabsf(x); }
__device__ __forceinline__ double exp_neg(double x) { return exp(-x); }
__device__ __forceinline__ float exp_neg(float x) { return expf(-x); }

// f(+m e_a) and f(-m e_a) of field q through the fetch functor
template <int A, typename F>
__device__ __forceinline__ auto nb(const F& f, int q, int m) {
    if (A == 0) return f(q, m, 0, 0);
    if (A == 1) return f(q, 0, m, 0);
    return f(q, 0, 0, m);
}

// first derivative along axis A
template <typename T, int A, typename F>
__device__ __forceinline__ T d1(const F& f, const Coeffs<T>& c, int q) {
    T r = c.c1[A][0] * (nb<A>(f, q, 1) - nb<A>(f, q, -1));
    r = fma_<T>(c.c1[A][1], nb<A>(f, q, 2) - nb<A>(f, q, -2), r);
    r = fma_<T>(c.c1[A][2], nb<A>(f, q, 3) - nb<A>(f, q, -3), r);
    return r;
}

// second derivative along axis A (centre value passed in)
template <typename T, int A, typename F>
__device__ __forceinline__ T d2(const F& f, const Coeffs<T>& c, int q, T f0) {
    T r = c.c20[A] * f0;
    r = fma_<T>(c.c2[A][0], nb<A>(f, q, 1) + nb<A>(f, q, -1), r);
    r = fma_<T>(c.c2[A][1], nb<A>(f, q, 2) + nb<A>(f, q, -2), r);
    r = fma_<T>(c.c2[A][2], nb<A>(f, q, 3) + nb<A>(f, q, -3), r);
    return r;
}

// upwind correction along axis A: delta6_A f / (60 h_A)
template <typename T, int A, typename F>
__device__ __forceinline__ T d6(const F& f, const Coeffs<T>& c, int q, T f0) {
    T r = c.c60[A] * f0;
    r = fma_<T>(c.c6[A][0], nb<A>(f, q, 1) + nb<A>(f, q, -1), r);
    r = fma_<T>(c.c6[A][1], nb<A>(f, q, 2) + nb<A>(f, q, -2), r);
    r = fma_<T>(c.c6[A][2], nb<A>(f, q, 3) + nb<A>(f, q, -3), r);
    return r;
}

template <int A, int B, typename F>
__device__ __forceinline__ auto corner(const F& f, int q, int sa, int sb) {
    int d[3] = {0, 0, 0};
    d[A] = sa;
    d[B] = sb;
    return f(q, d[0], d[1], d[2]);
}

// mixed derivative in the plane of axes A < B: bidiagonal 12-point stencil (G2, the default reading), or, with
// tensor = true, the alternative reading D_A(D_B f) = first-derivative stencil along A of first derivatives
// along B (36 points, same radius; NEXT-4)
template <typename T, int A, int B, typename F>
__device__ __forceinline__ T dmix(const F& f, const Coeffs<T>& c, int q, bool tensor) {
    constexpr int P = (A == 0 && B == 1) ? 0 : ((A == 0 && B == 2) ? 1 : 2);
    T r = T(0);
    if (tensor) {
#pragma unroll
        for (int m = 1; m <= 3; m++) {
            T dp = T(0), dm = T(0);     // D_B f at +m e_A and at -m e_A
#pragma unroll
            for (int n = 1; n <= 3; n++) {
                dp = fma_<T>(c.c1[B][n - 1], corner<A, B>(f, q, m, n) - corner<A, B>(f, q, m, -n), dp);
                dm = fma_<T>(c.c1[B][n - 1], corner<A, B>(f, q, -m, n) - corner<A, B>(f, q, -m, -n), dm);
            }
            r = fma_<T>(c.c1[A][m - 1], dp - dm, r);
        }
        return r;
    }
#pragma unroll
    for (int m = 1; m <= 3; m++) {
        T s = (corner<A, B>(f, q, m, m) + corner<A, B>(f, q, -m, -m)) -
              (corner<A, B>(f, q, m, -m) + corner<A, B>(f, q, -m, m));
        r = fma_<T>(c.cm[P][m - 1], s, r);
    }
    return r;
}

// Everything a cell needs from its neighbourhood, then the 7 new values.
//   f(q, dx, dy, dz): value of field q at the cell displaced by (dx, dy, dz), |d| <= 3
//   prev[q]: value of field q two substeps back (the "out" buffer; unused for substep 0)
//   fc, fs: cos and sin of (k.x + phase) at this cell (unused without forcing)
template <typename T, typename F>
__device__ __forceinline__ void substep_cell(const F& f, const Coeffs<T>& c, const Physics<T>& p, const T prev[7],
                                             T fc, T fs, T out[7]) {
    const T lnrho = f(LNRHO, 0, 0, 0);
    const T u[3] = {f(UX, 0, 0, 0), f(UY, 0, 0, 0), f(UZ, 0, 0, 0)};
    const T a[3] = {f(AX, 0, 0, 0), f(AY, 0, 0, 0), f(AZ, 0, 0, 0)};

    // grad ln rho
    const T g[3] = {d1<T, 0>(f, c, LNRHO), d1<T, 1>(f, c, LNRHO), d1<T, 2>(f, c, LNRHO)};

    // velocity gradient G[i][j] = d_j u_i
    T G[3][3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        G[i][0] = d1<T, 0>(f, c, UX + i);
        G[i][1] = d1<T, 1>(f, c, UX + i);
        G[i][2] = d1<T, 2>(f, c, UX + i);
    }
    const T divu = G[0][0] + G[1][1] + G[2][2];

    // second derivatives of u: uxx[i][a] = d_aa u_i
    T u2[3][3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        u2[i][0] = d2<T, 0>(f, c, UX + i, u[i]);
        u2[i][1] = d2<T, 1>(f, c, UX + i, u[i]);
        u2[i][2] = d2<T, 2>(f, c, UX + i, u[i]);
    }
    const bool mt = p.mixed_tensor != 0;
    // grad div u: diagonal second derivative + two mixed derivatives (G3)
    T gdu[3];
    gdu[0] = u2[0][0] + dmix<T, 0, 1>(f, c, UY, mt) + dmix<T, 0, 2>(f, c, UZ, mt);
    gdu[1] = u2[1][1] + dmix<T, 0, 1>(f, c, UX, mt) + dmix<T, 1, 2>(f, c, UZ, mt);
    gdu[2] = u2[2][2] + dmix<T, 0, 2>(f, c, UX, mt) + dmix<T, 1, 2>(f, c, UY, mt);

    // magnetic field, Laplacian of A, current density
    T B[3];
    B[0] = d1<T, 1>(f, c, AZ) - d1<T, 2>(f, c, AY) + p.bext[0];
    B[1] = d1<T, 2>(f, c, AX) - d1<T, 0>(f, c, AZ) + p.bext[1];
    B[2] = d1<T, 0>(f, c, AY) - d1<T, 1>(f, c, AX) + p.bext[2];
    T a2[3][3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        a2[i][0] = d2<T, 0>(f, c, AX + i, a[i]);
        a2[i][1] = d2<T, 1>(f, c, AX + i, a[i]);
        a2[i][2] = d2<T, 2>(f, c, AX + i, a[i]);
    }
    T lapA[3], jj[3];
#pragma unroll
    for (int i = 0; i < 3; i++) lapA[i] = a2[i][0] + a2[i][1] + a2[i][2];
    // j_i = d_ii A_i + sum_{j != i} d_ij A_j - lap A_i = mixed terms - the other two second derivatives
    jj[0] = dmix<T, 0, 1>(f, c, AY, mt) + dmix<T, 0, 2>(f, c, AZ, mt) - (a2[0][1] + a2[0][2]);
    jj[1] = dmix<T, 0, 1>(f, c, AX, mt) + dmix<T, 1, 2>(f, c, AZ, mt) - (a2[1][0] + a2[1][2]);
    jj[2] = dmix<T, 0, 2>(f, c, AX, mt) + dmix<T, 1, 2>(f, c, AY, mt) - (a2[2][0] + a2[2][1]);

    // right-hand sides
    T rhs[7];
    rhs[LNRHO] = -(fma_<T>(u[0], g[0], fma_<T>(u[1], g[1], u[2] * g[2]))) - divu;
    if (p.upwind) {
        T up = abs_(u[0]) * d6<T, 0>(f, c, LNRHO, lnrho);
        up = fma_<T>(abs_(u[1]), d6<T, 1>(f, c, LNRHO, lnrho), up);
        up = fma_<T>(abs_(u[2]), d6<T, 2>(f, c, LNRHO, lnrho), up);
        rhs[LNRHO] += up;
    }

    const T rho_inv = exp_neg(lnrho);
    const T jxb[3] = {jj[1] * B[2] - jj[2] * B[1], jj[2] * B[0] - jj[0] * B[2], jj[0] * B[1] - jj[1] * B[0]};
    const T uxb[3] = {u[1] * B[2] - u[2] * B[1], u[2] * B[0] - u[0] * B[2], u[0] * B[1] - u[1] * B[0]};
    const T third = T(1) / T(3);
#pragma unroll
    for (int i = 0; i < 3; i++) {
        const T adv = fma_<T>(u[0], G[i][0], fma_<T>(u[1], G[i][1], u[2] * G[i][2]));
        // 2 S_ij g_j = (G_ij + G_ji) g_j - (2/3) div u g_i
        T sg = (G[i][0] + G[0][i]) * g[0];
        sg = fma_<T>(G[i][1] + G[1][i], g[1], sg);
        sg = fma_<T>(G[i][2] + G[2][i], g[2], sg);
        sg = fma_<T>(T(-2) * third * divu, g[i], sg);
        const T lapu = u2[i][0] + u2[i][1] + u2[i][2];
        const T visc = fma_<T>(third, gdu[i], lapu) + sg;
        T r = fma_<T>(p.nu, visc, fma_<T>(jxb[i], rho_inv, -adv - p.cs2 * g[i]));
        if (p.has_forcing) r += p.fre[i] * fc - p.fim[i] * fs;
        rhs[UX + i] = r;
        rhs[AX + i] = fma_<T>(p.eta, lapA[i], uxb[i]);
    }

    // 2N-RK3 update, difference form: w_{s-1} = (f - prev)/beta_{s-1}
    const T cur[7] = {lnrho, u[0], u[1], u[2], a[0], a[1], a[2]};
#pragma unroll
    for (int q = 0; q < 7; q++) {
        T v = cur[q];
        if (p.substep != 0) v = fma_<T>(p.rk_a, cur[q] - prev[q], v);
        out[q] = fma_<T>(p.rk_b, rhs[q], v);
    }
}

}  // namespace ac
