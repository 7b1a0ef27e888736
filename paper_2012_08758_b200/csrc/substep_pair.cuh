// Fused RK substep, variant "pair-march".
//
// What it computes: exactly the substep of mhd_cell.cuh / the oracle - Eq. 1-3 right-hand sides
// (PAPER.md:166-170), forcing Eq. 4, 6th-order radius-3 central differences
// (readings G1-G3), j = grad div A - lap A (G4), the 2N-RK3 update in difference
// form (G7).
//
// It is the scatter-march of substep_march.cuh (a CTA owns a tile of (x, y) columns and marches along z;
// planes arrive in a shared-memory ring by TMA; the U role carries ln rho and u, the A role carries A and
// hands (j x B)/rho to the U role) with the changes that the ncu profile of that kernel asked for
// (profiles/r01d_march.md: 81 % of the shared-memory data pipe, 12 % of the instructions register moves):
//
// 1. A thread owns a PAIR of cells (x, y), (x, y + 1); the tile is 16 x 16.  The in-plane neighbourhood of
//    the pair is 40 shared-memory loads for a field with an in-plane mixed derivative (25 per single cell
//    before) and 20 for the others (13 before): the y column is shared, and the m = 1 diagonal points of one
//    cell are the x neighbours of the other.  110 instead of 139 stencil loads per cell.
// 2. The pair's z-coupled sums do not fit the register file as 7-level accumulators, so only the sums that
//    involve in-plane differences (the z-mixed derivatives, with d_zz merged in where it is free) stay
//    register accumulators.  Pure z stencils of the centre values (d_z u_x, d_z u_y, d_z / d_zz of A_x, A_y)
//    are GATHERED at finalisation from a 8-plane history of the centre values that the thread keeps in
//    TENSOR MEMORY (tcgen05.st when a plane arrives, tcgen05.ld three planes later): a per-lane scratchpad
//    that costs no shared-memory bandwidth.  The in-plane first derivatives that wait three planes for
//    their z partners are parked there too, and so is the (j x B)/rho mailbox: U warp w and A warp w + 4
//    address the same 32 tensor-memory lanes, so A lane i writes what U lane i reads.  The forcing f of Eq. 4
//    rides on the mailbox ((j x B)/rho + f): the step time follows the longer of the two roles, and the A role
//    had the slack.
// 3. The level shift of the accumulators is folded into the scatter (new[r-1] = old[r] + w v): no
//    register moves in the loop.
//
// Element type E (vec2.cuh): double, or f2 = two fp32 cells (z, z + nz/2) per element.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "layout.cuh"
#include "march_common.cuh"
#include "vec2.cuh"

namespace ac {

constexpr int Q_TX = 16, Q_TY = 16, Q_COLS = Q_TX * Q_TY;
constexpr int Q_PAIRS = Q_COLS / 2;            // column pairs per tile; one U and one A thread per pair
constexpr int Q_WORKERS = 2 * Q_PAIRS;         // 256
constexpr int Q_THREADS = Q_WORKERS + 128;     // + the producer warpgroup (warp 8 lane 0 feeds the ring, warp 9 owns the tensor memory)
constexpr int Q_HX = 4;
constexpr int Q_WX = Q_TX + 2 * Q_HX;          // 24
constexpr int Q_WY = Q_TY + 2 * R;             // 22
constexpr int Q_PLANE = Q_WX * Q_WY;           // 528 elements per field per ring slot
constexpr int Q_NP = 6;                        // ring slots: planes p-3 .. p resident, p+1, p+2 in flight
constexpr int Q_NPP = 3;                       // previous-state ring slots
constexpr int Q_LEAD = 2;
constexpr int Q_ND = 3;                        // (j x B)/rho mailbox depth (the A role runs at most 3 iterations ahead)
constexpr int Q_SLOT_BYTES = M_NF * Q_PLANE * 8;      // 29568
constexpr int Q_PSLOT_BYTES = M_NF * Q_COLS * 8;      // 14336
constexpr int Q_OFF_PREV = Q_NP * Q_SLOT_BYTES;
constexpr int Q_OFF_ZTAB = Q_OFF_PREV + Q_NPP * Q_PSLOT_BYTES;
constexpr int Q_OFF_BARS = Q_OFF_ZTAB + M_CZMAX * 2 * 8;
constexpr int Q_NBARS = 2 * Q_NP + 4 * Q_ND;          // full, done, mailbox [4 warp pairs][depth]
constexpr int Q_OFF_MISC = Q_OFF_BARS + Q_NBARS * 8;  // tensor-memory base address
constexpr int Q_SMEM_BYTES = Q_OFF_MISC + 16;
static_assert(Q_SLOT_BYTES % 128 == 0 && Q_PSLOT_BYTES % 128 == 0, "TMA destinations must stay 128-byte aligned");
static_assert(Q_SMEM_BYTES <= 232448, "exceeds the 227 KB of shared memory a CTA may use");
// MIX build (tensor-product mixed derivatives, NEXT-4): four staged planes of in-plane first derivatives (rows -3 .. 18
// of the 16 tile columns; U: d_x u_y, d_x u_x; A: d_x A_y, d_x A_x) take the place of the z phase table, which that
// build reads from global memory; two more mbarriers per role order the staging.
constexpr int Q_STAGE_FIELD = Q_WY * Q_TX;             // 352 elements
constexpr int QX_OFF_STAGE = Q_OFF_ZTAB;
constexpr int QX_OFF_BARS = QX_OFF_STAGE + 4 * Q_STAGE_FIELD * 8;
constexpr int QX_NBARS = Q_NBARS + 4;                  // + staged / gathered, per role
constexpr int QX_OFF_MISC = QX_OFF_BARS + QX_NBARS * 8;
constexpr int QX_SMEM_BYTES = QX_OFF_MISC + 16;
static_assert(QX_SMEM_BYTES <= 232448, "exceeds the 227 KB of shared memory a CTA may use");

// tensor-memory columns (32-bit) of one lane; an 8-byte element takes two
constexpr int Q_NH = 8;                        // history depth (planes p-6 .. p, one spare)
constexpr int Q_NK = 4;                        // parking depth (written at plane p, read at p + 3)
constexpr int Q_UH_SLOT = 16;                            // U history: [slot][ln rho c0 c1, u_z c0 c1 | u_x c0 c1, u_y c0 c1]
constexpr int Q_TM_UH = 0;
constexpr int Q_TM_UP = Q_TM_UH + Q_NH * Q_UH_SLOT;      // U parking: [slot][cell][gx gy Gxx Gxy Gyx Gyy Gzx Gzy (+ u6x u6y)]
constexpr int Q_UP_CELL = 20;
constexpr int Q_AH_SLOT = 8;                             // A history: [slot][A_x c0 c1, A_y c0 c1]
constexpr int Q_TM_AH = Q_TM_UP + Q_NK * 2 * Q_UP_CELL;
constexpr int Q_TM_AP = Q_TM_AH + Q_NH * Q_AH_SLOT;      // A parking: [slot][cell][Bxip Byip Bz Pxip Pyip]
constexpr int Q_AP_CELL = 12;
constexpr int Q_TM_MB = Q_TM_AP + Q_NK * 2 * Q_AP_CELL;  // mailbox: [depth][cell][3]
constexpr int Q_MB_CELL = 8;
static_assert(Q_TM_MB + Q_ND * 2 * Q_MB_CELL <= 512, "tensor memory has 512 columns");

// wait policy of the pair-march kernel (nanosleep between mbarrier polls; 0 = spin on try_wait)
#ifndef Q_WAIT_MAILBOX
#define Q_WAIT_MAILBOX 20
#endif
#ifndef Q_WAIT_RING_A
#define Q_WAIT_RING_A 20
#endif
#ifndef Q_WAIT_RING_U
#define Q_WAIT_RING_U 0
#endif
#ifndef Q_WAIT_PRODUCER
#define Q_WAIT_PRODUCER 200
#endif

// ---- tensor memory ---------------------------------------------------------------------------------
__device__ __forceinline__ void q_split(double a, uint32_t& lo, uint32_t& hi) {
    lo = (uint32_t)__double2loint(a);
    hi = (uint32_t)__double2hiint(a);
}
__device__ __forceinline__ void q_split(f2 a, uint32_t& lo, uint32_t& hi) {
    lo = (uint32_t)a.v;
    hi = (uint32_t)(a.v >> 32);
}
__device__ __forceinline__ void q_join(double& a, uint32_t lo, uint32_t hi) { a = __hiloint2double((int)hi, (int)lo); }
__device__ __forceinline__ void q_join(f2& a, uint32_t lo, uint32_t hi) { a.v = ((unsigned long long)hi << 32) | lo; }

template <typename E>
__device__ __forceinline__ void q_st1(uint32_t taddr, E a) {
    uint32_t r[2];
    q_split(a, r[0], r[1]);
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(r[0]), "r"(r[1]));
}
// wider stores as single-element stores: a tcgen05.st.x8 wants its 8 source registers consecutive, which cost 8 moves
// per store in the loop; x2 stores take each 8-byte value where it was computed
template <typename E>
__device__ __forceinline__ void q_st2(uint32_t taddr, E a, E b) {
    q_st1<E>(taddr, a);
    q_st1<E>(taddr + 2, b);
}
template <typename E>
__device__ __forceinline__ void q_st4(uint32_t taddr, E a, E b, E c, E d) {
    q_st1<E>(taddr, a);
    q_st1<E>(taddr + 2, b);
    q_st1<E>(taddr + 4, c);
    q_st1<E>(taddr + 6, d);
}
// loads return raw registers; they hold the data only after q_wait_ld + q_tie (the tie takes them as in-out
// operands of an ordered asm so that no use can be scheduled above the wait)
__device__ __forceinline__ void q_ld8(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
}
__device__ __forceinline__ void q_ld4(uint32_t taddr, uint32_t (&r)[4]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(taddr));
}
__device__ __forceinline__ void q_ld2(uint32_t taddr, uint32_t (&r)[2]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(taddr));
}
__device__ __forceinline__ void q_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void q_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void q_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void q_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void q_tie(uint32_t (&r)[N]) {
#pragma unroll
    for (int i = 0; i < N; i++) asm volatile("" : "+r"(r[i]));
}

// ---- the in-plane neighbourhood of a column pair ----------------------------------------------------
// p points at cell 0 of the pair, field q of the plane that has just arrived; cell 1 is one row up.
//   f0[c]        centre values
//   d, s [c][m]  f(x+m) -/+ f(x-m) along x;  e, t [c][m] along y (m = 1..3 -> index m - 1)
//   q[c][m]      f(x+m,y+m) - f(x-m,y+m) - f(x+m,y-m) + f(x-m,y-m): the 4 points of G2's stencil at distance m
// Every quantity of cell 0 and of cell 1 is formed by the same expression, so the result does not
// depend on which cell of a pair a grid point happens to be (P14, translation invariance).
template <typename E, bool SUMS, bool DIAG>
__device__ __forceinline__ void q_load(const E* __restrict__ p, E (&f0)[2], E (&d)[2][3], E (&s)[2][3], E (&e)[2][3],
                                       E (&t)[2][3], E (&q)[2][3]) {
    E col[8];   // rows -3 .. 4 of the pair's column
#pragma unroll
    for (int r = 0; r < 8; r++) col[r] = p[(r - 3) * Q_WX];
    f0[0] = col[3];
    f0[1] = col[4];
#pragma unroll
    for (int m = 1; m <= 3; m++) {
        e[0][m - 1] = vsub(col[3 + m], col[3 - m]);
        e[1][m - 1] = vsub(col[4 + m], col[4 - m]);
        if (SUMS) {
            t[0][m - 1] = vadd(col[3 + m], col[3 - m]);
            t[1][m - 1] = vadd(col[4 + m], col[4 - m]);
        }
    }
#pragma unroll
    for (int c = 0; c < 2; c++)
#pragma unroll
        for (int m = 1; m <= 3; m++) {
            const E a = p[c * Q_WX + m], b = p[c * Q_WX - m];
            d[c][m - 1] = vsub(a, b);
            if (SUMS) s[c][m - 1] = vadd(a, b);
        }
    if (DIAG) {
#define Q_DX(r, m) vsub(p[(r) * Q_WX + (m)], p[(r) * Q_WX - (m)])
        q[0][0] = vsub(d[1][0], Q_DX(-1, 1));
        q[0][1] = vsub(Q_DX(2, 2), Q_DX(-2, 2));
        q[0][2] = vsub(Q_DX(3, 3), Q_DX(-3, 3));
        q[1][0] = vsub(Q_DX(2, 1), d[0][0]);
        q[1][1] = vsub(Q_DX(3, 2), Q_DX(-1, 2));
        q[1][2] = vsub(Q_DX(4, 3), Q_DX(-2, 3));
#undef Q_DX
    }
}

// ---- scatter with the level shift folded in -----------------------------------------------------------
// A[0..5] holds the partial sums of planes p-3 .. p+2 when plane p arrives.  The FIRST contribution of an
// iteration writes level r into slot r - 1 (level 0 leaves the array as `fin`, level 6 starts from the product),
// later contributions of the same iteration update the shifted slots in place.  Level 3 - m takes weight
// dn[m-1], level 3 + m weight up[m-1]; L3 is the new value of level 3 (plane p itself), an expression in A[3]
// for FIRST; after FIRST level 3 sits in A[2].
#define Q_FIRST(A, fin, dn, up, v1, v2, v3, L3) \
    do {                                        \
        fin = vfma(dn[2], v3, A[0]);            \
        A[0] = vfma(dn[1], v2, A[1]);           \
        A[1] = vfma(dn[0], v1, A[2]);           \
        A[2] = (L3);                            \
        A[3] = vfma(up[0], v1, A[4]);           \
        A[4] = vfma(up[1], v2, A[5]);           \
        A[5] = vmul(up[2], v3);                 \
    } while (0)
#define Q_NEXT(A, fin, dn, up, v1, v2, v3)     \
    do {                                        \
        fin = vfma(dn[2], v3, fin);             \
        A[0] = vfma(dn[1], v2, A[0]);           \
        A[1] = vfma(dn[0], v1, A[1]);           \
        A[3] = vfma(up[0], v1, A[3]);           \
        A[4] = vfma(up[1], v2, A[4]);           \
        A[5] = vfma(up[2], v3, A[5]);           \
    } while (0)

template <typename E>
__device__ __forceinline__ void q_zero(E (&A)[2][6]) {
#pragma unroll
    for (int c = 0; c < 2; c++)
#pragma unroll
        for (int r = 0; r < 6; r++) A[c][r] = vzero<E>();
}

// history registers of one load: [f c0, f c1, g c0, g c1]
template <typename E>
__device__ __forceinline__ void q_hist(const uint32_t (&r)[8], E (&f)[2], E (&g)[2]) {
    q_join(f[0], r[0], r[1]);
    q_join(f[1], r[2], r[3]);
    q_join(g[0], r[4], r[5]);
    q_join(g[1], r[6], r[7]);
}

// z derivatives of two fields (f, g) x two cells from the centre history of the last 7 planes: slot (k - 3 + m) % 8
// holds plane p - 3 + m as [f c0, f c1, g c0, g c1].  df, dg = d_z; with ZZ also zf, zg = d_zz; fc, gc = centre values.
template <typename E, bool ZZ, int SLOT>
__device__ __forceinline__ void q_hist_gather(uint32_t base, int k, const E (&c1z)[3], const E (&c2z)[3], E c20z, E (&df)[2],
                                              E (&dg)[2], E (&zf)[2], E (&zg)[2], E (&fc)[2], E (&gc)[2]) {
    uint32_t h0[8], h1[8], h2[8], h3[8], h4[8], h5[8], h6[8];
    const int s0 = k & (Q_NH - 1);
    q_ld8(base + (uint32_t)(s0 * SLOT), h0);
    q_ld8(base + (uint32_t)(((s0 + 2) & (Q_NH - 1)) * SLOT), h6);
    q_ld8(base + (uint32_t)(((s0 + 7) & (Q_NH - 1)) * SLOT), h1);
    q_ld8(base + (uint32_t)(((s0 + 3) & (Q_NH - 1)) * SLOT), h5);
    q_ld8(base + (uint32_t)(((s0 + 6) & (Q_NH - 1)) * SLOT), h2);
    q_ld8(base + (uint32_t)(((s0 + 4) & (Q_NH - 1)) * SLOT), h4);
    q_ld8(base + (uint32_t)(((s0 + 5) & (Q_NH - 1)) * SLOT), h3);
    q_wait_ld();
    q_tie(h0); q_tie(h1); q_tie(h2); q_tie(h3); q_tie(h4); q_tie(h5); q_tie(h6);
    E fa[2], ga[2], fb[2], gb[2];
    q_hist<E>(h3, fc, gc);
    q_hist<E>(h2, fa, ga);
    q_hist<E>(h4, fb, gb);
#pragma unroll
    for (int cc = 0; cc < 2; cc++) {
        df[cc] = vmul(c1z[0], vsub(fa[cc], fb[cc]));
        dg[cc] = vmul(c1z[0], vsub(ga[cc], gb[cc]));
        if (ZZ) {
            zf[cc] = vfma(c2z[0], vadd(fa[cc], fb[cc]), vmul(c20z, fc[cc]));
            zg[cc] = vfma(c2z[0], vadd(ga[cc], gb[cc]), vmul(c20z, gc[cc]));
        }
    }
    q_hist<E>(h1, fa, ga);
    q_hist<E>(h5, fb, gb);
#pragma unroll
    for (int cc = 0; cc < 2; cc++) {
        df[cc] = vfma(c1z[1], vsub(fa[cc], fb[cc]), df[cc]);
        dg[cc] = vfma(c1z[1], vsub(ga[cc], gb[cc]), dg[cc]);
        if (ZZ) {
            zf[cc] = vfma(c2z[1], vadd(fa[cc], fb[cc]), zf[cc]);
            zg[cc] = vfma(c2z[1], vadd(ga[cc], gb[cc]), zg[cc]);
        }
    }
    q_hist<E>(h0, fa, ga);
    q_hist<E>(h6, fb, gb);
#pragma unroll
    for (int cc = 0; cc < 2; cc++) {
        df[cc] = vfma(c1z[2], vsub(fa[cc], fb[cc]), df[cc]);
        dg[cc] = vfma(c1z[2], vsub(ga[cc], gb[cc]), dg[cc]);
        if (ZZ) {
            zf[cc] = vfma(c2z[2], vadd(fa[cc], fb[cc]), zf[cc]);
            zg[cc] = vfma(c2z[2], vadd(ga[cc], gb[cc]), zg[cc]);
        }
    }
}

// ---- tensor-product mixed derivatives in the plane (MIX build; reading G2 alternative, NEXT-4) ------------------
// D_x D_y f is taken as D_y (D_x f): every thread stages D_x f of its two cells, the role's 128 threads add the 2 x 3
// halo rows above and below the tile (96 points per staged field, formed from the ring by the expression the owners
// use, so that a grid point gets the same bits whoever computes it), and after the role's barrier each thread takes
// the y derivative of its pair from the staged plane: 8 loads for two cells and one field, where the bidiagonal
// stencil takes 20.  st points at the role's two staged fields; pa / pb at field a / b of the ring plane, row 0,
// first tile column.
template <typename E>
__device__ __forceinline__ void q_stage(E* __restrict__ st, const E* __restrict__ pa, const E* __restrict__ pb, const E (&c1x)[3],
                                        const E (&own_a)[2], const E (&own_b)[2], int rt, int wp, int lane, int tx, int ty0) {
#pragma unroll
    for (int cc = 0; cc < 2; cc++) {
        st[(ty0 + R + cc) * Q_TX + tx] = own_a[cc];
        st[Q_STAGE_FIELD + (ty0 + R + cc) * Q_TX + tx] = own_b[cc];
    }
    // halo points 0 .. 95 of field a, 96 .. 191 of field b: one each, then lanes 0 .. 15 of every warp a second one
#pragma unroll
    for (int pass = 0; pass < 2; pass++) {
        const int item = pass == 0 ? rt : 128 + wp * 16 + lane;
        if (pass == 0 || lane < 16) {
            const bool second = item >= 96;
            const int r = second ? item - 96 : item;
            const int hrow = r >> 4, hx = r & 15;
            const int row = hrow < R ? hrow : hrow + Q_TY;          // rows 0 1 2 and 19 20 21 of the 22 loaded
            const E* hp = (second ? pb : pa) + row * Q_WX + hx;
            E hd[3];
#pragma unroll
            for (int m = 1; m <= 3; m++) hd[m - 1] = vsub(hp[m], hp[-m]);
            st[(second ? Q_STAGE_FIELD : 0) + row * Q_TX + hx] = m_dot3(c1x, hd);
        }
    }
}
// y differences of the staged field around the two cells of the pair
template <typename E>
__device__ __forceinline__ void q_stage_diff(const E* __restrict__ st, int tx, int ty0, E (&e)[2][3]) {
    E col[8];
#pragma unroll
    for (int r = 0; r < 8; r++) col[r] = st[(ty0 + r) * Q_TX + tx];
#pragma unroll
    for (int m = 1; m <= 3; m++) {
        e[0][m - 1] = vsub(col[3 + m], col[3 - m]);
        e[1][m - 1] = vsub(col[4 + m], col[4 - m]);
    }
}

// UPW: continuity equation with the 5th-order upwind correction (G17); the U role forms
// sum_a |u_a| delta6_a ln rho / (60 h_a) itself (x, y parts parked, the z part scattered).
// MIX: mixed derivatives as tensor products D_a (D_b f) instead of the bidiagonal stencil (ac_set_mixed(1)): the z-mixed
// ones are the z stencil of an in-plane first derivative (scattered like every other z sum), the in-plane ones
// go through q_stage.
// PREV: -1 = the kernel reads MarchArgs::substep to see whether a previous state exists; 0 / 1 = fixed at compile time
// (substep 0 / substeps 1, 2 of the default build: no uniform branches around the 2N-RK3 difference terms)
// FORCE: the same for MarchArgs::has_forcing.
template <typename T, bool UPW, bool MIX = false, int PREV = -1, int FORCE = -1>
__global__ void __launch_bounds__(Q_THREADS, 1)
    substep_pair_kernel(const __grid_constant__ MarchArgs<T> a, const __grid_constant__ CUtensorMap map_in,
                        const __grid_constant__ CUtensorMap map_prev) {
    using E = typename ElemOf<T>::E;
    extern __shared__ __align__(1024) unsigned char smem[];
    E* ztab = (E*)(smem + Q_OFF_ZTAB);
    uint64_t* full = (uint64_t*)(smem + (MIX ? QX_OFF_BARS : Q_OFF_BARS));
    uint64_t* done = full + Q_NP;
    uint64_t* mfull = done + Q_NP;            // [warp pair 0..3][depth]   A -> U mailbox (tensor memory)
    uint64_t* staged = mfull + 4 * Q_ND;      // MIX: [role] the staged plane is complete; gathered = it may be overwritten
    uint64_t* gathered = staged + 2;
    uint32_t* tmem_word = (uint32_t*)(smem + (MIX ? QX_OFF_MISC : Q_OFF_MISC));

    const Layout& L = a.L;
    const MarchCoef<E>& c = a.c;
    const int tid = threadIdx.x;
    // the shuffles tell the compiler that the warp index (and what derives from it: role, tensor-memory addresses)
    // is warp-uniform, so that it lives in uniform registers
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0), lane = tid & 31;
    // warps 0-3 = U  4-7 = A  8 = producer (lane 0)  9 = owns the tensor memory  10, 11 idle
    const int wp = warp & 3;                   // U warp w and A warp w + 4 share tensor-memory lanes and column pairs
    const int tx = lane & 15;
    const int ty0 = 2 * (2 * wp + (lane >> 4));
    const int col0 = ty0 * Q_TX + tx;          // cell c of the pair: col0 + c * Q_TX
    const int x0 = blockIdx.x * Q_TX, y0 = blockIdx.y * Q_TY;
    const int zs = a.z_begin + blockIdx.z * a.cz;
    const int ze = min(zs + a.cz, a.z_end);
    const int niter = ze - zs + 2 * R;      // planes zs-3 .. ze+2
    const int x = x0 + tx, y = y0 + ty0;
    const bool with_prev = PREV < 0 ? a.substep != 0 : PREV != 0;
    const bool has_forcing = FORCE < 0 ? a.has_forcing != 0 : FORCE != 0;

    if (tid == 0) {
        for (int s = 0; s < Q_NP; s++) {
            m_bar_init(&full[s], 1);
            m_bar_init(&done[s], Q_WORKERS / 32);
        }
        for (int s = 0; s < 4 * Q_ND; s++) m_bar_init(&mfull[s], 1);
        if (MIX)
            for (int s = 0; s < 4; s++) m_bar_init(&staged[s], 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 9) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(m_smem_u32(tmem_word)),
                     "n"(512)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    // z phase table of this chunk: (cos, sin)(k_z z + phase) per level, lanes = (z, z + nz/2) for packed pairs
    if (!MIX && has_forcing) {
        const T* tz = a.ftab + 2 * L.nx + 2 * L.ny;
        for (int i = tid; i < ze - zs; i += Q_THREADS) {
            const int z = zs + i;
            const int z2 = (ElemOf<T>::LANES == 2) ? z + L.nz : z;
            ztab[2 * i] = vmake(tz[z], tz[z2]);
            ztab[2 * i + 1] = vmake(tz[a.nz_full + z], tz[a.nz_full + z2]);
        }
    }
    q_fence_before();
    __syncthreads();
    q_fence_after();
    const uint32_t tm = __shfl_sync(0xffffffffu, *tmem_word, 0) + ((uint32_t)(wp * 32) << 16);

    const int cell_off = (ty0 + R) * Q_WX + tx + Q_HX;

    // the kernel is launched with 168 registers per thread (384 threads); the third warpgroup hands its share to
    // the two worker warpgroups.  Worker code must be reachable only through the .inc for ptxas to grant it 232.
    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(M_REGS_PRODUCER));
        if (tid == Q_WORKERS) {
            // ===================================== producer =====================================
            // iteration k processes plane zs - 3 + k and finalises plane zs - 6 + k (which reads the centre values
            // of ring slot k - 3); plane j + 3 reuses the slot of plane j - 3, free once every worker warp has
            // finished iteration j
            auto issue = [&](int k) {
                const int slot = k % Q_NP;
                const bool fin = with_prev && k >= 2 * R;
                m_bar_expect_tx(&full[slot], (uint32_t)(Q_SLOT_BYTES + (fin ? Q_PSLOT_BYTES : 0)));
                m_tma_load_4d(smem + slot * Q_SLOT_BYTES, &map_in, &full[slot], x0 - Q_HX + L.gx, y0, zs + k, 0);
                if (fin)
                    m_tma_load_4d(smem + Q_OFF_PREV + (k % Q_NPP) * Q_PSLOT_BYTES, &map_prev, &full[slot], x0 + L.gx,
                                  y0 + R, zs + k - R, 0);
            };
            for (int k = 0; k <= Q_LEAD && k < niter; k++) issue(k);
            for (int j = 0; j + Q_LEAD + 1 < niter; j++) {
                m_bar_wait<Q_WAIT_PRODUCER>(&done[j % Q_NP], (uint32_t)((j / Q_NP) & 1));
                issue(j + Q_LEAD + 1);
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(M_REGS_WORKER));
        const bool valid_x = x < L.nx;
        // fp64 build: which of the pair's two cells lie inside the grid, kept in a register (the empty asm stops the
        // compiler from rebuilding the two bits from the block and thread ids for every plane)
        uint32_t okm = (valid_x && y < L.ny ? 1u : 0u) | (valid_x && y + 1 < L.ny ? 2u : 0u);
        if (ElemOf<T>::LANES == 1) asm volatile("" : "+r"(okm));
        // element index of the pair's first cell in the plane finalised next: a running 32-bit offset (a padded field has
        // fewer than 2^32 elements, checked by the host) instead of Layout::idx() from scratch for every store
        uint32_t out_idx = (uint32_t)L.idx(x, y, zs);
        if (warp < 4) {
            // =============================== U: ln rho, u ===============================
            E Lx[2][6], Ly[2][6], Lz[2][6], u6z[2][6];
            q_zero(Lx); q_zero(Ly); q_zero(Lz); q_zero(u6z);
            for (int k = 0; k < niter; k++) {
                m_bar_wait<Q_WAIT_RING_U>(&full[k % Q_NP], (uint32_t)((k / Q_NP) & 1));
                const E* pl = (const E*)(smem + (k % Q_NP) * Q_SLOT_BYTES) + cell_off;
                E f0[2], d[2][3], s[2][3], e[2][3], t[2][3], q[2][3];
                E fLx[2], fLy[2], fLz[2], fu6z[2];
                E gx[2], gy[2], Gxx[2], Gxy[2], Gyx[2], Gyy[2], Gzx[2], Gzy[2], lyip[2], ln0[2], ux0[2], u6x[2], u6y[2];
                // ---- ln rho: gradient (and the sixth differences of the upwind term) ----
                q_load<E, UPW, false>(pl, f0, d, s, e, t, q);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    ln0[cc] = f0[cc];
                    gx[cc] = m_dot3(c.c1x, d[cc]);
                    gy[cc] = m_dot3(c.c1y, e[cc]);
                    if (UPW) {
                        u6x[cc] = m_dot3(c.c6x, s[cc], vmul(c.c60x, f0[cc]));
                        u6y[cc] = m_dot3(c.c6y, t[cc], vmul(c.c60y, f0[cc]));
                        Q_FIRST(u6z[cc], fu6z[cc], c.c6z, c.c6z, f0[cc], f0[cc], f0[cc], vfma(c.c60z, f0[cc], u6z[cc][3]));
                    }
                }
                // ---- u_x: d_x, d_y; L_x own; D_xy u_x -> L_y; D_xz u_x -> L_z; d_z u_x from the history ----
                q_load<E, true, !MIX>(pl + 1 * Q_PLANE, f0, d, s, e, t, q);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    ux0[cc] = f0[cc];
                    Gxx[cc] = m_dot3(c.c1x, d[cc]);
                    Gxy[cc] = m_dot3(c.c1y, e[cc]);
                    if (!MIX) lyip[cc] = m_dot3(c.cm3xy, q[cc]);
                    Q_FIRST(Lx[cc], fLx[cc], c.w2z[0], c.w2z[0], f0[cc], f0[cc], f0[cc],
                            m_dot3(c.w2y[0], t[cc], m_dot3(c.w2x[0], s[cc], vfma(c.w20[0], f0[cc], Lx[cc][3]))));
                    if (!MIX) Q_FIRST(Lz[cc], fLz[cc], c.cm3xz, c.ncm3xz, d[cc][0], d[cc][1], d[cc][2], Lz[cc][3]);
                }
                // ---- u_y: d_x, d_y; L_y own; D_xy u_y -> L_x; D_yz u_y -> L_z; d_z u_y from the history ----
                q_load<E, true, !MIX>(pl + 2 * Q_PLANE, f0, d, s, e, t, q);
                q_st4<E>(tm + Q_TM_UH + 8 + (uint32_t)((k & (Q_NH - 1)) * Q_UH_SLOT), ux0[0], ux0[1], f0[0], f0[1]);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    Gyx[cc] = m_dot3(c.c1x, d[cc]);
                    Gyy[cc] = m_dot3(c.c1y, e[cc]);
                    if (!MIX) {
                        Lx[cc][2] = m_dot3(c.cm3xy, q[cc], Lx[cc][2]);
                        Q_FIRST(Ly[cc], fLy[cc], c.w2z[1], c.w2z[1], f0[cc], f0[cc], f0[cc],
                                m_dot3(c.w2y[1], t[cc], m_dot3(c.w2x[1], s[cc], vfma(c.w20[1], f0[cc], vadd(Ly[cc][3], lyip[cc])))));
                        Q_NEXT(Lz[cc], fLz[cc], c.cm3yz, c.ncm3yz, e[cc][0], e[cc][1], e[cc][2]);
                    } else {
                        // 1/3 d_z (d_x u_x + d_y u_y) -> L_z
                        Q_FIRST(Ly[cc], fLy[cc], c.w2z[1], c.w2z[1], f0[cc], f0[cc], f0[cc],
                                m_dot3(c.w2y[1], t[cc], m_dot3(c.w2x[1], s[cc], vfma(c.w20[1], f0[cc], Ly[cc][3]))));
                        const E dxy = vadd(Gxx[cc], Gyy[cc]);
                        Q_FIRST(Lz[cc], fLz[cc], c.c13z, c.nc13z, dxy, dxy, dxy, Lz[cc][3]);
                    }
                }
                if (MIX) {
                    // stage d_x u_y (-> L_x) and d_x u_x (-> L_y) once the role has finished with the previous plane
                    if (k > 0) m_bar_wait<0>(&gathered[0], (uint32_t)((k - 1) & 1));
                    q_stage<E>((E*)(smem + QX_OFF_STAGE), pl - cell_off + 2 * Q_PLANE + Q_HX, pl - cell_off + 1 * Q_PLANE + Q_HX,
                               c.c1x, Gyx, Gxx, tid & 127, wp, lane, tx, ty0);
                    __syncwarp();
                    if (lane == 0) m_bar_arrive(&staged[0]);
                }
                // ---- u_z: d_x, d_y, d_z; L_z own; D_xz u_z -> L_x; D_yz u_z -> L_y ----
                q_load<E, true, false>(pl + 3 * Q_PLANE, f0, d, s, e, t, q);
                q_st4<E>(tm + Q_TM_UH + (uint32_t)((k & (Q_NH - 1)) * Q_UH_SLOT), ln0[0], ln0[1], f0[0], f0[1]);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    Gzx[cc] = m_dot3(c.c1x, d[cc]);
                    Gzy[cc] = m_dot3(c.c1y, e[cc]);
                    Q_NEXT(Lz[cc], fLz[cc], c.w2z[2], c.w2z[2], f0[cc], f0[cc], f0[cc]);
                    Lz[cc][2] = m_dot3(c.w2y[2], t[cc], m_dot3(c.w2x[2], s[cc], vfma(c.w20[2], f0[cc], Lz[cc][2])));
                    if (!MIX) {
                        Q_NEXT(Lx[cc], fLx[cc], c.cm3xz, c.ncm3xz, d[cc][0], d[cc][1], d[cc][2]);
                        Q_NEXT(Ly[cc], fLy[cc], c.cm3yz, c.ncm3yz, e[cc][0], e[cc][1], e[cc][2]);
                    } else {
                        // 1/3 d_z (d_x u_z) -> L_x, 1/3 d_z (d_y u_z) -> L_y
                        Q_NEXT(Lx[cc], fLx[cc], c.c13z, c.nc13z, Gzx[cc], Gzx[cc], Gzx[cc]);
                        Q_NEXT(Ly[cc], fLy[cc], c.c13z, c.nc13z, Gzy[cc], Gzy[cc], Gzy[cc]);
                    }
                }
                if (MIX) {
                    // 1/3 d_y (d_x u_y) -> L_x, 1/3 d_y (d_x u_x) -> L_y of this plane (level 3 sits in slot 2)
                    m_bar_wait<0>(&staged[0], (uint32_t)(k & 1));
                    const E* st = (const E*)(smem + QX_OFF_STAGE);
                    E ey[2][3];
                    q_stage_diff<E>(st, tx, ty0, ey);
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) Lx[cc][2] = m_dot3(c.c13y, ey[cc], Lx[cc][2]);
                    q_stage_diff<E>(st + Q_STAGE_FIELD, tx, ty0, ey);
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) Ly[cc][2] = m_dot3(c.c13y, ey[cc], Ly[cc][2]);
                    __syncwarp();
                    if (lane == 0) m_bar_arrive(&gathered[0]);
                }
                // ---- park the in-plane first derivatives of this plane (needed when it is finalised, 3 iterations on) ----
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    const uint32_t sl = tm + (uint32_t)(Q_TM_UP + ((k % Q_NK) * 2 + cc) * Q_UP_CELL);
                    q_st4<E>(sl, gx[cc], gy[cc], Gxx[cc], Gxy[cc]);
                    q_st4<E>(sl + 8, Gyx[cc], Gyy[cc], Gzx[cc], Gzy[cc]);
                    if (UPW) q_st2<E>(sl + 16, u6x[cc], u6y[cc]);
                }
                // ---- finalise plane zs - 6 + k ----
                if (k >= 2 * R) {
                    const int z = zs + k - 2 * R;
                    const int u = k - 2 * R;
                    const E* pc = (const E*)(smem + ((k - R) % Q_NP) * Q_SLOT_BYTES) + cell_off;
                    q_wait_st();
                    // d_z of ln rho, u from the centre history (plane p - 3 + m sits in slot (k - 3 + m) % 8)
                    E Gxz[2], Gyz[2], uxc[2], uyc[2], gzc[2], Gzzc[2], lnc[2], uzc[2], unused0[2], unused1[2];
                    q_hist_gather<E, false, Q_UH_SLOT>(tm + Q_TM_UH + 8, k, c.c1z, c.c2z, c.c20z, Gxz, Gyz, unused0, unused1, uxc, uyc);
                    q_hist_gather<E, false, Q_UH_SLOT>(tm + Q_TM_UH, k, c.c1z, c.c2z, c.c20z, gzc, Gzzc, unused0, unused1, lnc, uzc);
                    // (j x B) / rho + f from the A role of the same columns
                    m_bar_wait<Q_WAIT_MAILBOX>(&mfull[wp * Q_ND + u % Q_ND], (uint32_t)((u / Q_ND) & 1));
                    q_fence_after();
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) {
                        uint32_t p0[8], p1[8], mb0[4], mb1[2], pu[4];
                        const uint32_t sp = tm + (uint32_t)(Q_TM_UP + (((k - R) % Q_NK) * 2 + cc) * Q_UP_CELL);
                        const uint32_t sm = tm + (uint32_t)(Q_TM_MB + ((u % Q_ND) * 2 + cc) * Q_MB_CELL);
                        q_ld8(sp, p0);
                        q_ld8(sp + 8, p1);
                        q_ld4(sm, mb0);
                        q_ld2(sm + 4, mb1);
                        if (UPW) q_ld4(sp + 16, pu);
                        q_wait_ld();
                        q_tie(p0); q_tie(p1); q_tie(mb0); q_tie(mb1);
                        if (UPW) q_tie(pu);
                        E g0, g1, Gxx0, Gxy0, Gyx0, Gyy0, Gzx0, Gzy0, jxb0, jxb1, jxb2;
                        q_join(g0, p0[0], p0[1]); q_join(g1, p0[2], p0[3]);
                        q_join(Gxx0, p0[4], p0[5]); q_join(Gxy0, p0[6], p0[7]);
                        q_join(Gyx0, p1[0], p1[1]); q_join(Gyy0, p1[2], p1[3]);
                        q_join(Gzx0, p1[4], p1[5]); q_join(Gzy0, p1[6], p1[7]);
                        q_join(jxb0, mb0[0], mb0[1]); q_join(jxb1, mb0[2], mb0[3]); q_join(jxb2, mb1[0], mb1[1]);
                        const E g2 = gzc[cc], Gxz0 = Gxz[cc], Gyz0 = Gyz[cc], Gzz0 = Gzzc[cc];
                        const E lnrho = lnc[cc], ux = uxc[cc], uy = uyc[cc], uz = uzc[cc];
                        const E divu = vadd(vadd(Gxx0, Gyy0), Gzz0);
                        // Eq. 1
                        E rl = vmul(ux, g0);
                        rl = vfma(uy, g1, rl);
                        rl = vfma(uz, g2, rl);
                        rl = vneg(vadd(rl, divu));
                        if (UPW) {
                            E u6x0, u6y0;
                            q_join(u6x0, pu[0], pu[1]);
                            q_join(u6y0, pu[2], pu[3]);
                            E up = vmul(vabs(ux), u6x0);
                            up = vfma(vabs(uy), u6y0, up);
                            rl = vadd(rl, vfma(vabs(uz), fu6z[cc], up));
                        }
                        // 2 S_ij g_j = (G_ij + G_ji) g_j - 2/3 div u g_i
                        const E sxy_ = vadd(Gxy0, Gyx0), sxz_ = vadd(Gxz0, Gzx0), syz_ = vadd(Gyz0, Gzy0);
                        const E dd = vmul(c.n23, divu);
                        E sg0 = vmul(vadd(Gxx0, Gxx0), g0);
                        sg0 = vfma(sxy_, g1, sg0);
                        sg0 = vfma(sxz_, g2, sg0);
                        sg0 = vfma(dd, g0, sg0);
                        E sg1 = vmul(sxy_, g0);
                        sg1 = vfma(vadd(Gyy0, Gyy0), g1, sg1);
                        sg1 = vfma(syz_, g2, sg1);
                        sg1 = vfma(dd, g1, sg1);
                        E sg2 = vmul(sxz_, g0);
                        sg2 = vfma(syz_, g1, sg2);
                        sg2 = vfma(vadd(Gzz0, Gzz0), g2, sg2);
                        sg2 = vfma(dd, g2, sg2);
                        // Eq. 2
                        E adv0 = vmul(ux, Gxx0);
                        adv0 = vfma(uy, Gxy0, adv0);
                        adv0 = vfma(uz, Gxz0, adv0);
                        E adv1 = vmul(ux, Gyx0);
                        adv1 = vfma(uy, Gyy0, adv1);
                        adv1 = vfma(uz, Gyz0, adv1);
                        E adv2 = vmul(ux, Gzx0);
                        adv2 = vfma(uy, Gzy0, adv2);
                        adv2 = vfma(uz, Gzz0, adv2);
                        E r0 = vfma(c.nu, vadd(fLx[cc], sg0), vadd(jxb0, vsub(vmul(c.ncs2, g0), adv0)));
                        E r1 = vfma(c.nu, vadd(fLy[cc], sg1), vadd(jxb1, vsub(vmul(c.ncs2, g1), adv1)));
                        E r2 = vfma(c.nu, vadd(fLz[cc], sg2), vadd(jxb2, vsub(vmul(c.ncs2, g2), adv2)));
                        // 2N-RK3 update, difference form
                        E o0 = lnrho, o1 = ux, o2 = uy, o3 = uz;
                        if (with_prev) {
                            const E* pp = (const E*)(smem + Q_OFF_PREV + (k % Q_NPP) * Q_PSLOT_BYTES) + col0 + cc * Q_TX;
                            o0 = vfma(c.rk_a, vsub(lnrho, pp[0]), o0);
                            o1 = vfma(c.rk_a, vsub(ux, pp[Q_COLS]), o1);
                            o2 = vfma(c.rk_a, vsub(uy, pp[2 * Q_COLS]), o2);
                            o3 = vfma(c.rk_a, vsub(uz, pp[3 * Q_COLS]), o3);
                        }
                        o0 = vfma(c.rk_b, rl, o0);
                        o1 = vfma(c.rk_b, r0, o1);
                        o2 = vfma(c.rk_b, r1, o2);
                        o3 = vfma(c.rk_b, r2, o3);
                        if (ElemOf<T>::LANES == 1 ? (okm & (1u << cc)) != 0 : (valid_x && y + cc < L.ny)) {
                            const uint32_t ci = out_idx + (uint32_t)(cc * L.pitch);
                            a.out[0][ci] = o0;
                            a.out[1][ci] = o1;
                            a.out[2][ci] = o2;
                            a.out[3][ci] = o3;
                        }
                    }
                    q_fence_before();
                    out_idx += (uint32_t)L.plane;
                }
                __syncwarp();
                if (lane == 0) m_bar_arrive(&done[k % Q_NP]);
            }
        } else {
            // =============================== A: vector potential ===============================
            // the forcing of Eq. 4 rides on the mailbox: the A role, which is not on the critical path, adds f_i to
            // (j x B)_i / rho before it hands the sum over
            // cos/sin of k_x x + k_y y, constant along the march
            E cxy[2], sxy[2];
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                cxy[cc] = sxy[cc] = vzero<E>();
                if (has_forcing && valid_x && y + cc < L.ny) {
                    const T cx_ = a.ftab[x], sx_ = a.ftab[L.nx + x];
                    const T cy_ = a.ftab[2 * L.nx + y + cc], sy_ = a.ftab[2 * L.nx + L.ny + y + cc];
                    cxy[cc] = Splat<E>::of((double)(cx_ * cy_ - sx_ * sy_));
                    sxy[cc] = Splat<E>::of((double)(sx_ * cy_ + cx_ * sy_));
                }
            }
            E Pz[2][6], Jx[2][6], Jy[2][6], Jz[2][6];
            q_zero(Pz); q_zero(Jx); q_zero(Jy); q_zero(Jz);
            const E c20xy = vneg(c.nc20xy);     // centre weight of D_xx + D_yy
            for (int k = 0; k < niter; k++) {
                m_bar_wait<Q_WAIT_RING_A>(&full[k % Q_NP], (uint32_t)((k / Q_NP) & 1));
                q_fence_after();   // the mailbox slot written below was read by the U role before the plane was requested
                const E* pl = (const E*)(smem + (k % Q_NP) * Q_SLOT_BYTES) + cell_off;
                E f0[2], d[2][3], s[2][3], e[2][3], t[2][3], q[2][3];
                E fPz[2], fJx[2], fJy[2], fJz[2];
                E Bz[2], Bxip[2], Byip[2], Pxip[2], Pyip[2], jxip[2], jyip[2], ax0[2];
                // ---- A_x: B_z -= d_y A_x; in-plane lap; J_x -= D_yy A_x; D_xy A_x -> J_y; D_xz A_x -> J_z; d_z, d_zz from the history
                E dxax[2], dxay[2];    // MIX only
                q_load<E, true, !MIX>(pl + 4 * Q_PLANE, f0, d, s, e, t, q);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    ax0[cc] = f0[cc];
                    Bz[cc] = vneg(m_dot3(c.c1y, e[cc]));
                    const E px = m_dot3(c.c2x, s[cc]), py = m_dot3(c.c2y, t[cc]);
                    Pxip[cc] = vadd(vfma(c20xy, f0[cc], px), py);
                    jxip[cc] = vneg(vfma(c.c20y, f0[cc], py));
                    if (!MIX) {
                        jyip[cc] = m_dot3(c.cmxy, q[cc]);
                        Q_FIRST(Jz[cc], fJz[cc], c.cmxz, c.ncmxz, d[cc][0], d[cc][1], d[cc][2], Jz[cc][3]);
                    } else {
                        dxax[cc] = m_dot3(c.c1x, d[cc]);
                    }
                }
                // ---- A_y: B_z += d_x A_y; in-plane lap; J_y -= D_xx A_y; D_xy A_y -> J_x; D_yz A_y -> J_z; d_z, d_zz from the history
                q_load<E, true, !MIX>(pl + 5 * Q_PLANE, f0, d, s, e, t, q);
                q_st4<E>(tm + Q_TM_AH + (uint32_t)((k & (Q_NH - 1)) * Q_AH_SLOT), ax0[0], ax0[1], f0[0], f0[1]);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    const E px = m_dot3(c.c2x, s[cc]), py = m_dot3(c.c2y, t[cc]);
                    Pyip[cc] = vadd(vfma(c20xy, f0[cc], px), py);
                    if (!MIX) {
                        Bz[cc] = m_dot3(c.c1x, d[cc], Bz[cc]);
                        jyip[cc] = vsub(jyip[cc], vfma(c.c20x, f0[cc], px));
                        jxip[cc] = m_dot3(c.cmxy, q[cc], jxip[cc]);
                        Q_NEXT(Jz[cc], fJz[cc], c.cmyz, c.ncmyz, e[cc][0], e[cc][1], e[cc][2]);
                    } else {
                        dxay[cc] = m_dot3(c.c1x, d[cc]);
                        Bz[cc] = vadd(Bz[cc], dxay[cc]);
                        jyip[cc] = vneg(vfma(c.c20x, f0[cc], px));
                        // d_z (d_x A_x + d_y A_y) -> J_z
                        const E dxy = vadd(dxax[cc], m_dot3(c.c1y, e[cc]));
                        Q_FIRST(Jz[cc], fJz[cc], c.c1z, c.nc1z, dxy, dxy, dxy, Jz[cc][3]);
                    }
                }
                if (MIX) {
                    // stage d_x A_y (-> J_x) and d_x A_x (-> J_y)
                    if (k > 0) m_bar_wait<0>(&gathered[1], (uint32_t)((k - 1) & 1));
                    q_stage<E>((E*)(smem + QX_OFF_STAGE) + 2 * Q_STAGE_FIELD, pl - cell_off + 5 * Q_PLANE + Q_HX,
                               pl - cell_off + 4 * Q_PLANE + Q_HX, c.c1x, dxay, dxax, tid & 127, wp, lane, tx, ty0);
                    __syncwarp();
                    if (lane == 0) m_bar_arrive(&staged[1]);
                }
                // ---- A_z: B_x += d_y A_z; B_y -= d_x A_z; lap; J_z -= (D_xx + D_yy) A_z; D_xz A_z -> J_x; D_yz A_z -> J_y
                q_load<E, true, false>(pl + 6 * Q_PLANE, f0, d, s, e, t, q);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    Bxip[cc] = m_dot3(c.c1y, e[cc]);
                    Byip[cc] = vneg(m_dot3(c.c1x, d[cc]));
                    const E pxy = vadd(m_dot3(c.c2x, s[cc]), m_dot3(c.c2y, t[cc]));
                    Jz[cc][2] = vsub(vfma(c.nc20xy, f0[cc], Jz[cc][2]), pxy);
                    Q_FIRST(Pz[cc], fPz[cc], c.c2z, c.c2z, f0[cc], f0[cc], f0[cc], vadd(vfma(c.c20all, f0[cc], Pz[cc][3]), pxy));
                    if (!MIX) {
                        Q_FIRST(Jx[cc], fJx[cc], c.cmxz, c.ncmxz, d[cc][0], d[cc][1], d[cc][2], vadd(Jx[cc][3], jxip[cc]));
                        Q_FIRST(Jy[cc], fJy[cc], c.cmyz, c.ncmyz, e[cc][0], e[cc][1], e[cc][2], vadd(Jy[cc][3], jyip[cc]));
                    } else {
                        // d_z (d_x A_z) -> J_x, d_z (d_y A_z) -> J_y
                        const E dxaz = vneg(Byip[cc]), dyaz = Bxip[cc];
                        Q_FIRST(Jx[cc], fJx[cc], c.c1z, c.nc1z, dxaz, dxaz, dxaz, vadd(Jx[cc][3], jxip[cc]));
                        Q_FIRST(Jy[cc], fJy[cc], c.c1z, c.nc1z, dyaz, dyaz, dyaz, vadd(Jy[cc][3], jyip[cc]));
                    }
                }
                if (MIX) {
                    // d_y (d_x A_y) -> J_x, d_y (d_x A_x) -> J_y of this plane (level 3 sits in slot 2)
                    m_bar_wait<0>(&staged[1], (uint32_t)(k & 1));
                    const E* st = (const E*)(smem + QX_OFF_STAGE) + 2 * Q_STAGE_FIELD;
                    E ey[2][3];
                    q_stage_diff<E>(st, tx, ty0, ey);
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) Jx[cc][2] = m_dot3(c.c1y, ey[cc], Jx[cc][2]);
                    q_stage_diff<E>(st + Q_STAGE_FIELD, tx, ty0, ey);
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) Jy[cc][2] = m_dot3(c.c1y, ey[cc], Jy[cc][2]);
                    __syncwarp();
                    if (lane == 0) m_bar_arrive(&gathered[1]);
                }
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    const uint32_t sl = tm + (uint32_t)(Q_TM_AP + ((k % Q_NK) * 2 + cc) * Q_AP_CELL);
                    q_st4<E>(sl, Bxip[cc], Byip[cc], Bz[cc], Pxip[cc]);
                    q_st1<E>(sl + 8, Pyip[cc]);
                }
                // ---- finalise plane zs - 6 + k ----
                if (k >= 2 * R) {
                    const int z = zs + k - 2 * R;
                    const int u = k - 2 * R;
                    const E* pc = (const E*)(smem + ((k - R) % Q_NP) * Q_SLOT_BYTES) + cell_off;
                    q_wait_st();
                    // d_z and d_zz of A_x, A_y from the centre history
                    E dzax[2], dzay[2], zzax[2], zzay[2], axc[2], ayc[2];
                    q_hist_gather<E, true, Q_AH_SLOT>(tm + Q_TM_AH, k, c.c1z, c.c2z, c.c20z, dzax, dzay, zzax, zzay, axc, ayc);
                    E cz_ = vzero<E>(), sz_ = vzero<E>();
                    if (has_forcing) {
                        if (MIX) {
                            const T* tz = a.ftab + 2 * L.nx + 2 * L.ny;
                            const int z2 = (ElemOf<T>::LANES == 2) ? z + L.nz : z;
                            cz_ = vmake(tz[z], tz[z2]);
                            sz_ = vmake(tz[a.nz_full + z], tz[a.nz_full + z2]);
                        } else {
                            cz_ = ztab[2 * (z - zs)];
                            sz_ = ztab[2 * (z - zs) + 1];
                        }
                    }
                    E b0[2], b1[2], b2[2], P0[2], P1[2];
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) {
                        uint32_t p0[8], p1[2];
                        const uint32_t sp = tm + (uint32_t)(Q_TM_AP + (((k - R) % Q_NK) * 2 + cc) * Q_AP_CELL);
                        q_ld8(sp, p0);
                        q_ld2(sp + 8, p1);
                        q_wait_ld();
                        q_tie(p0); q_tie(p1);
                        E Bxip0, Byip0, Bz0, Pxip0, Pyip0;
                        q_join(Bxip0, p0[0], p0[1]); q_join(Byip0, p0[2], p0[3]);
                        q_join(Bz0, p0[4], p0[5]); q_join(Pxip0, p0[6], p0[7]);
                        q_join(Pyip0, p1[0], p1[1]);
                        b0[cc] = vadd(vsub(Bxip0, dzay[cc]), c.bext[0]);
                        b1[cc] = vadd(vadd(dzax[cc], Byip0), c.bext[1]);
                        b2[cc] = vadd(Bz0, c.bext[2]);
                        P0[cc] = vadd(Pxip0, zzax[cc]);
                        P1[cc] = vadd(Pyip0, zzay[cc]);
                        const E j0 = vsub(fJx[cc], zzax[cc]), j1 = vsub(fJy[cc], zzay[cc]), j2 = fJz[cc];
                        const E rho_inv = vexpneg(pc[cc * Q_WX]);
                        E m0 = vmul(rho_inv, vsub(vmul(j1, b2[cc]), vmul(j2, b1[cc])));
                        E m1 = vmul(rho_inv, vsub(vmul(j2, b0[cc]), vmul(j0, b2[cc])));
                        E m2 = vmul(rho_inv, vsub(vmul(j0, b1[cc]), vmul(j1, b0[cc])));
                        if (has_forcing) {
                            // forcing Eq. 4: f_i = re_i cos(theta) - im_i sin(theta)
                            const E fc = vsub(vmul(cxy[cc], cz_), vmul(sxy[cc], sz_));
                            const E fs = vfma(sxy[cc], cz_, vmul(cxy[cc], sz_));
                            m0 = vfma(c.fre[0], fc, vfma(c.nfim[0], fs, m0));
                            m1 = vfma(c.fre[1], fc, vfma(c.nfim[1], fs, m1));
                            m2 = vfma(c.fre[2], fc, vfma(c.nfim[2], fs, m2));
                        }
                        const uint32_t sm = tm + (uint32_t)(Q_TM_MB + ((u % Q_ND) * 2 + cc) * Q_MB_CELL);
                        q_st2<E>(sm, m0, m1);
                        q_st1<E>(sm + 4, m2);
                    }
                    q_wait_st();
                    q_fence_before();
                    __syncwarp();
                    if (lane == 0) m_bar_arrive(&mfull[wp * Q_ND + u % Q_ND]);
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) {
                        const E* pcc = pc + cc * Q_WX;
                        const E ux = pcc[Q_PLANE], uy = pcc[2 * Q_PLANE], uz = pcc[3 * Q_PLANE];
                        const E ax = axc[cc], ay = ayc[cc], az = pcc[6 * Q_PLANE];
                        // Eq. 3: u x B + eta lap A
                        const E r0 = vfma(c.eta, P0[cc], vsub(vmul(uy, b2[cc]), vmul(uz, b1[cc])));
                        const E r1 = vfma(c.eta, P1[cc], vsub(vmul(uz, b0[cc]), vmul(ux, b2[cc])));
                        const E r2 = vfma(c.eta, fPz[cc], vsub(vmul(ux, b1[cc]), vmul(uy, b0[cc])));
                        E o0 = ax, o1 = ay, o2 = az;
                        if (with_prev) {
                            const E* pp = (const E*)(smem + Q_OFF_PREV + (k % Q_NPP) * Q_PSLOT_BYTES) + 4 * Q_COLS + col0 + cc * Q_TX;
                            o0 = vfma(c.rk_a, vsub(ax, pp[0]), o0);
                            o1 = vfma(c.rk_a, vsub(ay, pp[Q_COLS]), o1);
                            o2 = vfma(c.rk_a, vsub(az, pp[2 * Q_COLS]), o2);
                        }
                        o0 = vfma(c.rk_b, r0, o0);
                        o1 = vfma(c.rk_b, r1, o1);
                        o2 = vfma(c.rk_b, r2, o2);
                        if (ElemOf<T>::LANES == 1 ? (okm & (1u << cc)) != 0 : (valid_x && y + cc < L.ny)) {
                            const uint32_t ci = out_idx + (uint32_t)(cc * L.pitch);
                            a.out[4][ci] = o0;
                            a.out[5][ci] = o1;
                            a.out[6][ci] = o2;
                        }
                    }
                    out_idx += (uint32_t)L.plane;
                }
                __syncwarp();
                if (lane == 0) m_bar_arrive(&done[k % Q_NP]);
            }
        }
    }

    // every tensor-memory access has completed (the workers wait for their loads and stores) before the columns go back
    q_fence_before();
    __syncthreads();
    if (warp == 9) {
        q_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_word), "n"(512) : "memory");
    }
}

}  // namespace ac
