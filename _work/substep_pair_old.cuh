// Fused RK substep, variant "pair-march" (the default).
//
// What it computes: exactly the substep of mhd_cell.cuh / the oracle - Eq. 1-3 right-hand sides
// (PAPER.md:166-170), forcing Eq. 4, 6th-order radius-3 central differences
// (readings G1-G3), j = grad div A - lap A (G4), the 2N-RK3 update in difference
// form (G7), and the periodic ghost zones of the buffer it writes (S1, the
// paper's "local boundary transfer") - one launch per substep, nothing else.
//
// It is the scatter-march of substep_march.cuh (a CTA owns a 16 x 8 tile of (x, y) columns and
// marches along z; planes arrive in a shared-memory ring by TMA; everything that couples planes
// is scattered into register accumulators of the pending cells) with three changes that the ncu
// profile of that kernel asked for (profiles/r01d_march.md: 81 % of the shared-memory data pipe,
// 12 % of the instructions register moves, a second launch per substep for the ghost zones):
//
// 1. A thread owns a PAIR of cells (x, y), (x, y + 1).  The in-plane neighbourhood of the pair is
//    40 shared-memory loads for a field with an in-plane mixed derivative (25 per single cell
//    before) and 20 for the others (13 before): the y column is shared, and the m = 1 diagonal
//    points of one cell are the x neighbours of the other.  110 instead of 139 loads per cell.
// 2. The work of a column pair is split over FOUR roles so that the pair's accumulators fit the
//    register file: UH (u_y, u_z) and AH (A_y, A_z) are helpers that only carry linear stencil
//    sums; UF (ln rho, u_x) and AF (A_x) carry their own sums and finalise the cells (non-linear
//    terms, forcing, 2N update, store).  A helper hands its sums to its finaliser through TENSOR
//    MEMORY: warps w and w + 4 of a CTA address the same 32 TMEM lanes, so helper lane i writes
//    (tcgen05.st) what finaliser lane i reads (tcgen05.ld) - a per-lane mailbox that costs no
//    shared-memory bandwidth.  The in-plane first derivatives that wait three planes for their z
//    partners are parked in tensor memory too instead of being carried through registers.
//    AF hands (j x B)/rho to UF through a small shared-memory mailbox as before.
// 3. The level shift of the accumulators is folded into the scatter (new[r-1] = old[r] + w v), so
//    the loop has no register moves except for pure d/dz sums, and warp 9 - idle before - copies
//    the periodic images of every finished plane into the ghost zones, so ghost_fill_kernel and
//    its launch are gone.
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

constexpr int P_PAIRS = M_COLS / 2;        // column pairs per tile; one thread per pair and role
constexpr int P_NSLOT = 8;                 // depth of the helper -> finaliser tensor-memory rings
constexpr int P_NOWN = 4;                  // depth of a finaliser's own parking ring (read 3 planes later)
// tensor-memory columns (32-bit) of one lane; U lanes (warps 0, 1, 4, 5) and A lanes (2, 3, 6, 7) are disjoint
constexpr int P_TM_CELL = 16;              // columns per cell and slot (5 to 8 values)
constexpr int P_TM_CELL_HP = 8;            // columns per cell and slot of the helper's parking ring (4 values)
constexpr int P_TM_HPARK = 0;                                      // helper, written at plane p, read at p + 3
constexpr int P_TM_HCOMP = P_TM_HPARK + P_NSLOT * 2 * P_TM_CELL_HP;   // helper, level-0 sums, read the same iteration
constexpr int P_TM_OWN = P_TM_HCOMP + P_NSLOT * 2 * P_TM_CELL;        // finaliser's own parked in-plane values
static_assert(P_TM_OWN + P_NOWN * 2 * P_TM_CELL <= 512, "tensor memory has 512 columns");

constexpr int P_MBOX_BYTES = 3 * M_COLS * 8;            // (j x B)/rho per depth
constexpr int P_OFF_PREV = M_NP * M_SLOT_BYTES;
constexpr int P_OFF_MBOX = P_OFF_PREV + M_NPP * M_PSLOT_BYTES;
constexpr int P_OFF_ZTAB = P_OFF_MBOX + M_ND * P_MBOX_BYTES;
constexpr int P_OFF_BARS = P_OFF_ZTAB + M_CZMAX * 2 * 8;
constexpr int P_NBARS = 2 * M_NP + 2 * M_ND + 4 * P_NSLOT;    // full, done, mailbox [2 warp pairs], tmem [4 warp pairs]
constexpr int P_OFF_MISC = P_OFF_BARS + P_NBARS * 8;          // tensor-memory base address, ghost-warp progress
constexpr int P_SMEM_BYTES = P_OFF_MISC + 16;
static_assert(P_SMEM_BYTES <= 232448, "exceeds the 227 KB of shared memory a CTA may use");

// ---- tensor memory ---------------------------------------------------------------------------------
__device__ __forceinline__ void p_split(double a, uint32_t& lo, uint32_t& hi) {
    lo = (uint32_t)__double2loint(a);
    hi = (uint32_t)__double2hiint(a);
}
__device__ __forceinline__ void p_split(f2 a, uint32_t& lo, uint32_t& hi) {
    lo = (uint32_t)a.v;
    hi = (uint32_t)(a.v >> 32);
}
__device__ __forceinline__ void p_join(double& a, uint32_t lo, uint32_t hi) { a = __hiloint2double((int)hi, (int)lo); }
__device__ __forceinline__ void p_join(f2& a, uint32_t lo, uint32_t hi) { a.v = ((unsigned long long)hi << 32) | lo; }

template <typename E>
__device__ __forceinline__ void p_tm_st4(uint32_t taddr, E a, E b, E c, E d) {
    uint32_t r[8];
    p_split(a, r[0], r[1]);
    p_split(b, r[2], r[3]);
    p_split(c, r[4], r[5]);
    p_split(d, r[6], r[7]);
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(r[0]),
                 "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
}
template <typename E>
__device__ __forceinline__ void p_tm_st2(uint32_t taddr, E a, E b) {
    uint32_t r[4];
    p_split(a, r[0], r[1]);
    p_split(b, r[2], r[3]);
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3])
                 : "memory");
}
template <typename E>
__device__ __forceinline__ void p_tm_st1(uint32_t taddr, E a) {
    uint32_t r[2];
    p_split(a, r[0], r[1]);
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(r[0]), "r"(r[1]) : "memory");
}
// loads return raw registers; they hold the data only after p_tm_wait_ld, which takes them as in-out operands so
// that no use can be scheduled above it
__device__ __forceinline__ void p_tm_ld8(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void p_tm_ld4(uint32_t taddr, uint32_t (&r)[4]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void p_tm_ld2(uint32_t taddr, uint32_t (&r)[2]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void p_tm_wait_ld(uint32_t (&a)[8], uint32_t (&b)[8], uint32_t (&c)[8], uint32_t (&d)[4]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]), "+r"(a[7]), "+r"(b[0]),
                   "+r"(b[1]), "+r"(b[2]), "+r"(b[3]), "+r"(b[4]), "+r"(b[5]), "+r"(b[6]), "+r"(b[7]), "+r"(c[0]), "+r"(c[1]),
                   "+r"(c[2]), "+r"(c[3]), "+r"(c[4]), "+r"(c[5]), "+r"(c[6]), "+r"(c[7]), "+r"(d[0]), "+r"(d[1]), "+r"(d[2]),
                   "+r"(d[3])
                 :
                 : "memory");
}
__device__ __forceinline__ void p_tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void p_tm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void p_tm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---- the in-plane neighbourhood of a column pair ----------------------------------------------------
// p points at cell 0 of the pair, field q of the plane that has just arrived; cell 1 is one row up.
//   f0[c]        centre values
//   d, s [c][m]  f(x+m) -/+ f(x-m) along x;  e, t [c][m] along y (m = 1..3 -> index m - 1)
//   q[c][m]      f(x+m,y+m) - f(x-m,y+m) - f(x+m,y-m) + f(x-m,y-m): the 4 points of G2's stencil at distance m
// Every quantity of cell 0 and of cell 1 is formed by the same expression, so the result does not
// depend on which cell of a pair a grid point happens to be (P14, translation invariance).
template <typename E, bool SUMS, bool DIAG>
__device__ __forceinline__ void p_load(const E* __restrict__ p, E (&f0)[2], E (&d)[2][3], E (&s)[2][3], E (&e)[2][3],
                                       E (&t)[2][3], E (&q)[2][3]) {
    E col[8];   // rows -3 .. 4 of the pair's column
#pragma unroll
    for (int r = 0; r < 8; r++) col[r] = p[(r - 3) * M_WX];
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
            const E a = p[c * M_WX + m], b = p[c * M_WX - m];
            d[c][m - 1] = vsub(a, b);
            if (SUMS) s[c][m - 1] = vadd(a, b);
        }
    if (DIAG) {
#define P_DX(r, m) vsub(p[(r) * M_WX + (m)], p[(r) * M_WX - (m)])
        q[0][0] = vsub(d[1][0], P_DX(-1, 1));
        q[0][1] = vsub(P_DX(2, 2), P_DX(-2, 2));
        q[0][2] = vsub(P_DX(3, 3), P_DX(-3, 3));
        q[1][0] = vsub(P_DX(2, 1), d[0][0]);
        q[1][1] = vsub(P_DX(3, 2), P_DX(-1, 2));
        q[1][2] = vsub(P_DX(4, 3), P_DX(-2, 3));
#undef P_DX
    }
}

// ---- scatter with the level shift folded in -----------------------------------------------------------
// A[0..5] holds the partial sums of planes p-3 .. p+2 when plane p arrives.  The FIRST contribution of an
// iteration writes level r into slot r - 1 (level 0 leaves the array as `fin`, level 6 starts from the product),
// later contributions of the same iteration update the shifted slots in place.  Level 3 - m takes weight
// dn[m-1], level 3 + m weight up[m-1]; L3 is the new value of level 3 (plane p itself), an expression in A[3]
// for FIRST and in A[2] for a later contribution.
#define P_FIRST(A, fin, dn, up, v1, v2, v3, L3) \
    do {                                        \
        fin = vfma(dn[2], v3, A[0]);            \
        A[0] = vfma(dn[1], v2, A[1]);           \
        A[1] = vfma(dn[0], v1, A[2]);           \
        A[2] = (L3);                            \
        A[3] = vfma(up[0], v1, A[4]);           \
        A[4] = vfma(up[1], v2, A[5]);           \
        A[5] = vmul(up[2], v3);                 \
    } while (0)
#define P_NEXT(A, fin, dn, up, v1, v2, v3)     \
    do {                                        \
        fin = vfma(dn[2], v3, fin);             \
        A[0] = vfma(dn[1], v2, A[0]);           \
        A[1] = vfma(dn[0], v1, A[1]);           \
        A[3] = vfma(up[0], v1, A[3]);           \
        A[4] = vfma(up[1], v2, A[4]);           \
        A[5] = vfma(up[2], v3, A[5]);           \
    } while (0)

template <typename E>
__device__ __forceinline__ void p_zero(E (&A)[2][6]) {
#pragma unroll
    for (int c = 0; c < 2; c++)
#pragma unroll
        for (int r = 0; r < 6; r++) A[c][r] = vzero<E>();
}

// UPW: continuity equation with the 5th-order upwind correction (G17); UF forms
// sum_a |u_a| delta6_a ln rho / (60 h_a) itself (x, y parts parked, the z part scattered).
template <typename T, bool UPW>
__global__ void __launch_bounds__(M_THREADS, 1)
    substep_pair_kernel(const __grid_constant__ MarchArgs<T> a, const __grid_constant__ CUtensorMap map_in,
                        const __grid_constant__ CUtensorMap map_prev) {
    using E = typename ElemOf<T>::E;
    extern __shared__ __align__(1024) unsigned char smem[];
    E* ztab = (E*)(smem + P_OFF_ZTAB);
    uint64_t* full = (uint64_t*)(smem + P_OFF_BARS);
    uint64_t* done = full + M_NP;
    uint64_t* mfull = done + M_NP;            // [warp pair 0..1][depth]   AF -> UF, shared memory mailbox
    uint64_t* tfull = mfull + 2 * M_ND;       // [warp pair 0..3][slot]    helper -> finaliser, tensor memory
    uint32_t* tmem_word = (uint32_t*)(smem + P_OFF_MISC);
    int* prog = (int*)(smem + P_OFF_MISC + 4);   // iterations completed, published by the producer lane

    const Layout& L = a.L;
    const MarchCoef<E>& c = a.c;
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    // warps 0,1 = UH  2,3 = AH  4,5 = UF  6,7 = AF  8 = producer  9-11 = ghost zones (10 also owns the tensor memory)
    const int rw = warp & 1;                   // which half of the tile's pairs this warp serves
    const int wp = warp & 3;                   // helper warp w and finaliser warp w + 4 share tensor-memory lanes
    const int tx = lane & 15;
    const int ty0 = 2 * (2 * rw + (lane >> 4));
    const int col0 = ty0 * M_TX + tx;          // cell c of the pair: col0 + c * M_TX
    const int x0 = blockIdx.x * M_TX, y0 = blockIdx.y * M_TY;
    const int zs = blockIdx.z * a.cz;
    const int ze = min(zs + a.cz, L.nz);
    const int niter = ze - zs + 2 * R;      // planes zs-3 .. ze+2
    const int x = x0 + tx, y = y0 + ty0;
    const bool with_prev = a.substep != 0;
    // which periodic images this tile has to write (S1)
    const bool tile_edge_xy = x0 < R || x0 + M_TX > L.nx - R || y0 < R || y0 + M_TY > L.ny - R;
    const bool chunk_edge_z = a.wrap_z && (zs < R || ze > L.nz - R);
    const bool ghost_active = tile_edge_xy || chunk_edge_z;

    if (tid == 0) {
        for (int s = 0; s < M_NP; s++) {
            m_bar_init(&full[s], 1);
            m_bar_init(&done[s], M_WORKERS / 32);
        }
        for (int s = 0; s < 2 * M_ND; s++) m_bar_init(&mfull[s], 1);
        for (int s = 0; s < 4 * P_NSLOT; s++) m_bar_init(&tfull[s], 1);
        *prog = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 10) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(m_smem_u32(tmem_word)),
                     "n"(512)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    // z phase table of this chunk: (cos, sin)(k_z z + phase) per level, lanes = (z, z + nz/2) for packed pairs
    if (a.has_forcing) {
        const T* tz = a.ftab + 2 * L.nx + 2 * L.ny;
        for (int i = tid; i < ze - zs; i += M_THREADS) {
            const int z = zs + i;
            const int z2 = (ElemOf<T>::LANES == 2) ? z + L.nz : z;
            ztab[2 * i] = vmake(tz[z], tz[z2]);
            ztab[2 * i + 1] = vmake(tz[a.nz_full + z], tz[a.nz_full + z2]);
        }
    }
    p_tm_fence_before();
    __syncthreads();
    p_tm_fence_after();
    const uint32_t tm = *tmem_word + ((uint32_t)(wp * 32) << 16);

    const int cell_off = (ty0 + R) * M_WX + tx + M_HX;

    // the kernel is launched with 168 registers per thread (384 threads); the third warpgroup hands its share to
    // the two worker warpgroups.  Worker code must be reachable only through the .inc for ptxas to grant it 232.
    if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(M_REGS_PRODUCER));
    if (warp == 8) {
        // ===================================== producer =====================================
        // iteration k processes plane zs - 3 + k and finalises plane zs - 6 + k; plane j + 5 reuses the ring
        // slot that every worker warp has released after iteration j.  The lane also publishes how many iterations
        // have completed (prog), which is what the ghost-zone warps wait for.
        if (lane == 0) {
            auto issue = [&](int k) {
                const int slot = k % M_NP;
                const bool fin = with_prev && k >= 2 * R;
                m_bar_expect_tx(&full[slot], (uint32_t)(M_SLOT_BYTES + (fin ? M_PSLOT_BYTES : 0)));
                m_tma_load_4d(smem + slot * M_SLOT_BYTES, &map_in, &full[slot], x0 - M_HX + L.gx, y0, zs + k, 0);
                if (fin)
                    m_tma_load_4d(smem + P_OFF_PREV + (k % M_NPP) * M_PSLOT_BYTES, &map_prev, &full[slot], x0 + L.gx,
                                  y0 + R, zs + k - R, 0);
            };
            for (int k = 0; k < M_LEAD + 2 && k < niter; k++) issue(k);
            const int jend = ghost_active ? niter : niter - (M_LEAD + 2);
            for (int j = 0; j < jend; j++) {
                m_bar_wait<MarchWait<T>::PRODUCER_NS>(&done[j % M_NP], (uint32_t)((j / M_NP) & 1));
                if (ghost_active)
                    asm volatile("st.release.cta.shared.b32 [%0], %1;" ::"r"(m_smem_u32(prog)), "r"(j + 1) : "memory");
                if (j + M_LEAD + 2 < niter) issue(j + M_LEAD + 2);
            }
        }
    } else if (ghost_active) {
        // ===================================== ghost zones (S1), warps 9 - 11 =====================================
        // once iteration k has completed, plane z = zs + k - 6 of the new state is in memory (the workers' stores
        // are ordered before their arrival on done[k], which the producer lane acquires before it releases prog).
        // A lane owns up to two cells of the tile and copies those that lie within R of a face to their periodic
        // images (<= 7 per cell and field).  z images of packed fp32 pairs swap lanes (cell z - nz/2 of the pair
        // below is cell z + nz/2 of the periodic domain).
        const int g = tid - (M_WORKERS + 32);
        int cgx[2], cgy[2];
        bool cval[2], chx[2], chy[2];
#pragma unroll
        for (int j = 0; j < 2; j++) {
            const int cc = g + 96 * j;
            cgx[j] = x0 + (cc & (M_TX - 1));
            cgy[j] = y0 + (cc >> 4);
            cval[j] = cc < M_COLS && cgx[j] < L.nx && cgy[j] < L.ny;
            chx[j] = cgx[j] < R || cgx[j] >= L.nx - R;
            chy[j] = cgy[j] < R || cgy[j] >= L.ny - R;
        }
        for (int k = 2 * R; k < niter; k++) {
            const int z = zs + k - 2 * R;
            // a plane can have two z images when fewer than 2 R planes exist (packed fp32: nz / 2 >= 4)
            const bool hzlo = a.wrap_z && z < R, hzhi = a.wrap_z && z >= L.nz - R;
            const bool hz = hzlo || hzhi;
            const bool need0 = cval[0] && (chx[0] || chy[0] || hz), need1 = cval[1] && (chx[1] || chy[1] || hz);
            if (!__any_sync(0xffffffffu, need0 || need1)) continue;
            for (;;) {
                int have;
                asm volatile("ld.acquire.cta.shared.b32 %0, [%1];" : "=r"(have) : "r"(m_smem_u32(prog)) : "memory");
                if (have > k) break;
                __nanosleep(200);
            }
#pragma unroll
            for (int j = 0; j < 2; j++) {
                if (!(j ? need1 : need0)) continue;
                const int ix = cgx[j] < R ? cgx[j] + L.nx : cgx[j] - L.nx, iy = cgy[j] < R ? cgy[j] + L.ny : cgy[j] - L.ny;
                const size_t src = L.idx(cgx[j], cgy[j], z);
                E v[M_NF];
#pragma unroll
                for (int q = 0; q < M_NF; q++) v[q] = a.out[q][src];
#pragma unroll
                for (int m = 1; m < 12; m++) {   // bit 0: x image, bit 1: y image, bits 2-3: z image (1 = z + nz, 2 = z - nz)
                    const int mz = m >> 2;
                    if (((m & 1) && !chx[j]) || ((m & 2) && !chy[j]) || (mz == 1 && !hzlo) || (mz == 2 && !hzhi)) continue;
                    const size_t dst = L.idx((m & 1) ? ix : cgx[j], (m & 2) ? iy : cgy[j],
                                             mz == 1 ? z + L.nz : (mz == 2 ? z - L.nz : z));
#pragma unroll
                    for (int q = 0; q < M_NF; q++) a.out[q][dst] = mz ? vswap(v[q]) : v[q];
                }
            }
        }
    }
    } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(M_REGS_WORKER));
    if (warp == 0 || warp == 1) {
        // ======================================= UH: u_y, u_z =======================================
        E Gyz[2][6], Gzz[2][6], Ly[2][6], Lzb[2][6], Lxb[2][6];
        p_zero(Gyz); p_zero(Gzz); p_zero(Ly); p_zero(Lzb); p_zero(Lxb);
        for (int k = 0; k < niter; k++) {
            m_bar_wait<MarchWait<T>::RING_A_NS>(&full[k % M_NP], (uint32_t)((k / M_NP) & 1));
            const E* pl = (const E*)(smem + (k % M_NP) * M_SLOT_BYTES) + cell_off;
            E f0[2], d[2][3], s[2][3], e[2][3], t[2][3], q[2][3];
            E fGyz[2], fGzz[2], fLy[2], fLzb[2], fLxb[2], lxip[2], Gyx[2], Gyy[2], Gzx[2], Gzy[2];
            // ---- u_y: d_x, d_y; L_y own; D_xy u_y -> L_x; D_yz u_y -> L_z ----
            p_load<E, true, true>(pl + 2 * M_PLANE, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                Gyx[cc] = m_dot3(c.c1x, d[cc]);
                Gyy[cc] = m_dot3(c.c1y, e[cc]);
                lxip[cc] = m_dot3(c.cm3xy, q[cc]);
                P_FIRST(Gyz[cc], fGyz[cc], c.c1z, c.nc1z, f0[cc], f0[cc], f0[cc], Gyz[cc][3]);
                P_FIRST(Ly[cc], fLy[cc], c.w2z[1], c.w2z[1], f0[cc], f0[cc], f0[cc],
                        m_dot3(c.w2y[1], t[cc], m_dot3(c.w2x[1], s[cc], vfma(c.w20[1], f0[cc], Ly[cc][3]))));
                P_FIRST(Lzb[cc], fLzb[cc], c.cm3yz, c.ncm3yz, e[cc][0], e[cc][1], e[cc][2], Lzb[cc][3]);
            }
            // ---- u_z: d_x, d_y; L_z own; D_xz u_z -> L_x; D_yz u_z -> L_y ----
            p_load<E, true, false>(pl + 3 * M_PLANE, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                Gzx[cc] = m_dot3(c.c1x, d[cc]);
                Gzy[cc] = m_dot3(c.c1y, e[cc]);
                P_FIRST(Gzz[cc], fGzz[cc], c.c1z, c.nc1z, f0[cc], f0[cc], f0[cc], Gzz[cc][3]);
                P_NEXT(Lzb[cc], fLzb[cc], c.w2z[2], c.w2z[2], f0[cc], f0[cc], f0[cc]);
                Lzb[cc][2] = m_dot3(c.w2y[2], t[cc], m_dot3(c.w2x[2], s[cc], vfma(c.w20[2], f0[cc], Lzb[cc][2])));
                P_FIRST(Lxb[cc], fLxb[cc], c.cm3xz, c.ncm3xz, d[cc][0], d[cc][1], d[cc][2], vadd(Lxb[cc][3], lxip[cc]));
                P_NEXT(Ly[cc], fLy[cc], c.cm3yz, c.ncm3yz, e[cc][0], e[cc][1], e[cc][2]);
            }
            // ---- hand over: parked in-plane first derivatives (read 3 planes later), level-0 sums (read now) ----
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                const uint32_t sl = (uint32_t)(((k % P_NSLOT) * 2 + cc) * P_TM_CELL);
                p_tm_st4<E>(tm + P_TM_HPARK + sl / 2, Gyx[cc], Gyy[cc], Gzx[cc], Gzy[cc]);
                p_tm_st4<E>(tm + P_TM_HCOMP + sl, fGyz[cc], fGzz[cc], fLxb[cc], fLy[cc]);
                p_tm_st1<E>(tm + P_TM_HCOMP + sl + 8, fLzb[cc]);
            }
            p_tm_wait_st();
            p_tm_fence_before();
            __syncwarp();
            if (lane == 0) {
                m_bar_arrive(&tfull[wp * P_NSLOT + k % P_NSLOT]);
                m_bar_arrive(&done[k % M_NP]);
            }
        }
    } else if (warp == 2 || warp == 3) {
        // ======================================= AH: A_y, A_z =======================================
        E Bx[2][6], Py[2][6], Jyb[2][6], Jzb[2][6], Jxb[2][6];
        p_zero(Bx); p_zero(Py); p_zero(Jyb); p_zero(Jzb); p_zero(Jxb);
        for (int k = 0; k < niter; k++) {
            m_bar_wait<MarchWait<T>::RING_A_NS>(&full[k % M_NP], (uint32_t)((k / M_NP) & 1));
            const E* pl = (const E*)(smem + (k % M_NP) * M_SLOT_BYTES) + cell_off;
            E f0[2], d[2][3], s[2][3], e[2][3], t[2][3], q[2][3];
            E fBx[2], fPy[2], fJyb[2], fJzb[2], fJxb[2], jxip[2], Bzb[2], Byb[2], Pzip[2];
            // ---- A_y: B_z += d_x A_y; lap; J_y -= (D_xx + D_zz) A_y; D_xy A_y -> J_x; D_yz A_y -> J_z; B_x -= d_z A_y
            p_load<E, true, true>(pl + 5 * M_PLANE, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                Bzb[cc] = m_dot3(c.c1x, d[cc]);
                const E px = m_dot3(c.c2x, s[cc]), py = m_dot3(c.c2y, t[cc]);
                jxip[cc] = m_dot3(c.cmxy, q[cc]);
                P_FIRST(Bx[cc], fBx[cc], c.nc1z, c.c1z, f0[cc], f0[cc], f0[cc], Bx[cc][3]);
                P_FIRST(Py[cc], fPy[cc], c.c2z, c.c2z, f0[cc], f0[cc], f0[cc],
                        vadd(vfma(c.c20all, f0[cc], Py[cc][3]), vadd(px, py)));
                P_FIRST(Jyb[cc], fJyb[cc], c.nc2z, c.nc2z, f0[cc], f0[cc], f0[cc], vsub(vfma(c.nc20xz, f0[cc], Jyb[cc][3]), px));
                P_FIRST(Jzb[cc], fJzb[cc], c.cmyz, c.ncmyz, e[cc][0], e[cc][1], e[cc][2], Jzb[cc][3]);
            }
            // ---- A_z: B_x += d_y A_z; B_y -= d_x A_z; in-plane lap; J_z -= (D_xx + D_yy) A_z; D_xz A_z -> J_x; D_yz A_z -> J_y
            p_load<E, true, false>(pl + 6 * M_PLANE, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                Bx[cc][2] = m_dot3(c.c1y, e[cc], Bx[cc][2]);
                Byb[cc] = vneg(m_dot3(c.c1x, d[cc]));
                const E pxy = vadd(m_dot3(c.c2x, s[cc]), m_dot3(c.c2y, t[cc]));
                Pzip[cc] = vfma(c.c20all, f0[cc], pxy);
                Jzb[cc][2] = vsub(vfma(c.nc20xy, f0[cc], Jzb[cc][2]), pxy);
                P_FIRST(Jxb[cc], fJxb[cc], c.cmxz, c.ncmxz, d[cc][0], d[cc][1], d[cc][2], vadd(Jxb[cc][3], jxip[cc]));
                P_NEXT(Jyb[cc], fJyb[cc], c.cmyz, c.ncmyz, e[cc][0], e[cc][1], e[cc][2]);
            }
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                const uint32_t sl = (uint32_t)(((k % P_NSLOT) * 2 + cc) * P_TM_CELL);
                p_tm_st4<E>(tm + P_TM_HPARK + sl / 2, Bzb[cc], Byb[cc], Pzip[cc], Pzip[cc]);
                p_tm_st4<E>(tm + P_TM_HCOMP + sl, fBx[cc], fPy[cc], fJxb[cc], fJyb[cc]);
                p_tm_st1<E>(tm + P_TM_HCOMP + sl + 8, fJzb[cc]);
            }
            p_tm_wait_st();
            p_tm_fence_before();
            __syncwarp();
            if (lane == 0) {
                m_bar_arrive(&tfull[wp * P_NSLOT + k % P_NSLOT]);
                m_bar_arrive(&done[k % M_NP]);
            }
        }
    } else if (warp == 4 || warp == 5) {
        // =============================== UF: ln rho, u_x; finalises ln rho and u ===============================
        const bool valid_x = x < L.nx;
        // forcing: cos/sin of k_x x + k_y y, constant along the march
        E cxy[2], sxy[2];
#pragma unroll
        for (int cc = 0; cc < 2; cc++) {
            cxy[cc] = sxy[cc] = vzero<E>();
            if (a.has_forcing && valid_x && y + cc < L.ny) {
                const T cx_ = a.ftab[x], sx_ = a.ftab[L.nx + x];
                const T cy_ = a.ftab[2 * L.nx + y + cc], sy_ = a.ftab[2 * L.nx + L.ny + y + cc];
                cxy[cc] = Splat<E>::of((double)(cx_ * cy_ - sx_ * sy_));
                sxy[cc] = Splat<E>::of((double)(sx_ * cy_ + cx_ * sy_));
            }
        }
        E gz[2][6], Gxz[2][6], Lxa[2][6], Lza[2][6], u6z[2][6];
        p_zero(gz); p_zero(Gxz); p_zero(Lxa); p_zero(Lza); p_zero(u6z);
        for (int k = 0; k < niter; k++) {
            m_bar_wait<MarchWait<T>::RING_U_NS>(&full[k % M_NP], (uint32_t)((k / M_NP) & 1));
            const E* pl = (const E*)(smem + (k % M_NP) * M_SLOT_BYTES) + cell_off;
            E f0[2], d[2][3], s[2][3], e[2][3], t[2][3], q[2][3];
            E fgz[2], fGxz[2], fLxa[2], fLza[2], fu6z[2], gx[2], gy[2], Gxx[2], Gxy[2], Lya[2], u6x[2], u6y[2];
            // ---- ln rho: gradient (and the sixth differences of the upwind term) ----
            p_load<E, UPW, false>(pl, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                gx[cc] = m_dot3(c.c1x, d[cc]);
                gy[cc] = m_dot3(c.c1y, e[cc]);
                P_FIRST(gz[cc], fgz[cc], c.c1z, c.nc1z, f0[cc], f0[cc], f0[cc], gz[cc][3]);
                if (UPW) {
                    u6x[cc] = m_dot3(c.c6x, s[cc], vmul(c.c60x, f0[cc]));
                    u6y[cc] = m_dot3(c.c6y, t[cc], vmul(c.c60y, f0[cc]));
                    P_FIRST(u6z[cc], fu6z[cc], c.c6z, c.c6z, f0[cc], f0[cc], f0[cc], vfma(c.c60z, f0[cc], u6z[cc][3]));
                }
            }
            // ---- u_x: d_x, d_y; L_x own; D_xy u_x -> L_y; D_xz u_x -> L_z ----
            p_load<E, true, true>(pl + 1 * M_PLANE, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                Gxx[cc] = m_dot3(c.c1x, d[cc]);
                Gxy[cc] = m_dot3(c.c1y, e[cc]);
                Lya[cc] = m_dot3(c.cm3xy, q[cc]);
                P_FIRST(Gxz[cc], fGxz[cc], c.c1z, c.nc1z, f0[cc], f0[cc], f0[cc], Gxz[cc][3]);
                P_FIRST(Lxa[cc], fLxa[cc], c.w2z[0], c.w2z[0], f0[cc], f0[cc], f0[cc],
                        m_dot3(c.w2y[0], t[cc], m_dot3(c.w2x[0], s[cc], vfma(c.w20[0], f0[cc], Lxa[cc][3]))));
                P_FIRST(Lza[cc], fLza[cc], c.cm3xz, c.ncm3xz, d[cc][0], d[cc][1], d[cc][2], Lza[cc][3]);
            }
            // ---- park the in-plane values of this plane (needed when it is finalised, 3 iterations from now) ----
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                const uint32_t sl = (uint32_t)(P_TM_OWN + ((k % P_NOWN) * 2 + cc) * P_TM_CELL);
                p_tm_st4<E>(tm + sl, gx[cc], gy[cc], Gxx[cc], Gxy[cc]);
                p_tm_st1<E>(tm + sl + 8, Lya[cc]);
                if (UPW) p_tm_st2<E>(tm + sl + 12, u6x[cc], u6y[cc]);
            }
            // ---- finalise plane zs - 6 + k ----
            if (k >= 2 * R) {
                const int z = zs + k - 2 * R;
                const int u = k - 2 * R;
                const E* pc = (const E*)(smem + ((k - R) % M_NP) * M_SLOT_BYTES) + cell_off;
                p_tm_wait_st();
                m_bar_wait<0>(&tfull[wp * P_NSLOT + k % P_NSLOT], (uint32_t)((k / P_NSLOT) & 1));
                p_tm_fence_after();
                // forcing Eq. 4: f_i = re_i cos(theta) - im_i sin(theta)
                E cz_ = vzero<E>(), sz_ = vzero<E>();
                if (a.has_forcing) {
                    cz_ = ztab[2 * (z - zs)];
                    sz_ = ztab[2 * (z - zs) + 1];
                }
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    uint32_t r_own[8], r_hp[8], r_hc[8], r_x[4], r_u[4];
                    const uint32_t so = (uint32_t)(P_TM_OWN + (((k - R) % P_NOWN) * 2 + cc) * P_TM_CELL);
                    const uint32_t sp = (uint32_t)(P_TM_HPARK + (((k - R) % P_NSLOT) * 2 + cc) * P_TM_CELL_HP);
                    const uint32_t sc = (uint32_t)(P_TM_HCOMP + ((k % P_NSLOT) * 2 + cc) * P_TM_CELL);
                    p_tm_ld8(tm + so, r_own);
                    p_tm_ld8(tm + sp, r_hp);
                    p_tm_ld8(tm + sc, r_hc);
                    {
                        uint32_t r2[2], r3[2];
                        p_tm_ld2(tm + so + 8, r2);
                        p_tm_ld2(tm + sc + 8, r3);
                        r_x[0] = r2[0]; r_x[1] = r2[1]; r_x[2] = r3[0]; r_x[3] = r3[1];
                    }
                    if (UPW) {
                        p_tm_ld4(tm + so + 12, r_u);
                        asm volatile("" : "+r"(r_u[0]), "+r"(r_u[1]), "+r"(r_u[2]), "+r"(r_u[3]));
                    }
                    p_tm_wait_ld(r_own, r_hp, r_hc, r_x);
                    if (UPW) asm volatile("" : "+r"(r_u[0]), "+r"(r_u[1]), "+r"(r_u[2]), "+r"(r_u[3])::"memory");
                    E g0, g1, Gxx0, Gxy0, Lya0, Gyx0, Gyy0, Gzx0, Gzy0, Gyz0, Gzz0, Lxb0, Ly0, Lzb0;
                    p_join(g0, r_own[0], r_own[1]); p_join(g1, r_own[2], r_own[3]);
                    p_join(Gxx0, r_own[4], r_own[5]); p_join(Gxy0, r_own[6], r_own[7]);
                    p_join(Lya0, r_x[0], r_x[1]);
                    p_join(Gyx0, r_hp[0], r_hp[1]); p_join(Gyy0, r_hp[2], r_hp[3]);
                    p_join(Gzx0, r_hp[4], r_hp[5]); p_join(Gzy0, r_hp[6], r_hp[7]);
                    p_join(Gyz0, r_hc[0], r_hc[1]); p_join(Gzz0, r_hc[2], r_hc[3]);
                    p_join(Lxb0, r_hc[4], r_hc[5]); p_join(Ly0, r_hc[6], r_hc[7]);
                    p_join(Lzb0, r_x[2], r_x[3]);
                    const E g2 = fgz[cc], Gxz0 = fGxz[cc];
                    const E Lx0 = vadd(fLxa[cc], Lxb0), Ly1 = vadd(Ly0, Lya0), Lz0 = vadd(fLza[cc], Lzb0);
                    const E* pcc = pc + cc * M_WX;
                    const E lnrho = pcc[0], ux = pcc[M_PLANE], uy = pcc[2 * M_PLANE], uz = pcc[3 * M_PLANE];
                    const E divu = vadd(vadd(Gxx0, Gyy0), Gzz0);
                    // (j x B) / rho from the AF role of the same columns
                    if (cc == 0) m_bar_wait<MarchWait<T>::MAILBOX_NS>(&mfull[rw * M_ND + u % M_ND], (uint32_t)((u / M_ND) & 1));
                    const E* mb = (const E*)(smem + P_OFF_MBOX + (u % M_ND) * P_MBOX_BYTES) + col0 + cc * M_TX;
                    const E jxb0 = mb[0], jxb1 = mb[M_COLS], jxb2 = mb[2 * M_COLS];
                    // Eq. 1
                    E rl = vmul(ux, g0);
                    rl = vfma(uy, g1, rl);
                    rl = vfma(uz, g2, rl);
                    rl = vneg(vadd(rl, divu));
                    if (UPW) {
                        E u6x0, u6y0;
                        p_join(u6x0, r_u[0], r_u[1]);
                        p_join(u6y0, r_u[2], r_u[3]);
                        E up = vmul(vabs(ux), u6x0);
                        up = vfma(vabs(uy), u6y0, up);
                        rl = vadd(rl, vfma(vabs(uz), fu6z[cc], up));
                    }
                    E fc = vzero<E>(), fs = vzero<E>();
                    if (a.has_forcing) {
                        fc = vsub(vmul(cxy[cc], cz_), vmul(sxy[cc], sz_));
                        fs = vfma(sxy[cc], cz_, vmul(cxy[cc], sz_));
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
                    E r0 = vfma(c.nu, vadd(Lx0, sg0), vadd(jxb0, vsub(vmul(c.ncs2, g0), adv0)));
                    E r1 = vfma(c.nu, vadd(Ly1, sg1), vadd(jxb1, vsub(vmul(c.ncs2, g1), adv1)));
                    E r2 = vfma(c.nu, vadd(Lz0, sg2), vadd(jxb2, vsub(vmul(c.ncs2, g2), adv2)));
                    if (a.has_forcing) {
                        r0 = vfma(c.fre[0], fc, vfma(c.nfim[0], fs, r0));
                        r1 = vfma(c.fre[1], fc, vfma(c.nfim[1], fs, r1));
                        r2 = vfma(c.fre[2], fc, vfma(c.nfim[2], fs, r2));
                    }
                    // 2N-RK3 update, difference form
                    E o0 = lnrho, o1 = ux, o2 = uy, o3 = uz;
                    if (with_prev) {
                        const E* pp = (const E*)(smem + P_OFF_PREV + (k % M_NPP) * M_PSLOT_BYTES) + col0 + cc * M_TX;
                        o0 = vfma(c.rk_a, vsub(lnrho, pp[0]), o0);
                        o1 = vfma(c.rk_a, vsub(ux, pp[M_COLS]), o1);
                        o2 = vfma(c.rk_a, vsub(uy, pp[2 * M_COLS]), o2);
                        o3 = vfma(c.rk_a, vsub(uz, pp[3 * M_COLS]), o3);
                    }
                    o0 = vfma(c.rk_b, rl, o0);
                    o1 = vfma(c.rk_b, r0, o1);
                    o2 = vfma(c.rk_b, r1, o2);
                    o3 = vfma(c.rk_b, r2, o3);
                    if (valid_x && y + cc < L.ny) {
                        const size_t ci = L.idx(x, y + cc, z);
                        a.out[0][ci] = o0;
                        a.out[1][ci] = o1;
                        a.out[2][ci] = o2;
                        a.out[3][ci] = o3;
                    }
                }
            }
            __syncwarp();
            if (lane == 0) m_bar_arrive(&done[k % M_NP]);
        }
    } else {
        // =============================== AF: A_x (and d_zz A_z); finalises A ===============================
        const bool valid_x = x < L.nx;
        E Bya[2][6], Px[2][6], Jxa[2][6], Jza[2][6], Pzz[2][6];
        p_zero(Bya); p_zero(Px); p_zero(Jxa); p_zero(Jza); p_zero(Pzz);
        for (int k = 0; k < niter; k++) {
            m_bar_wait<MarchWait<T>::RING_A_NS>(&full[k % M_NP], (uint32_t)((k / M_NP) & 1));
            const E* pl = (const E*)(smem + (k % M_NP) * M_SLOT_BYTES) + cell_off;
            E f0[2], d[2][3], s[2][3], e[2][3], t[2][3], q[2][3];
            E fBya[2], fPx[2], fJxa[2], fJza[2], fPzz[2], Bza[2], Jya[2];
            // ---- A_x: B_z -= d_y A_x; lap; J_x -= (D_yy + D_zz) A_x; D_xy A_x -> J_y; D_xz A_x -> J_z; B_y += d_z A_x
            p_load<E, true, true>(pl + 4 * M_PLANE, f0, d, s, e, t, q);
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                Bza[cc] = vneg(m_dot3(c.c1y, e[cc]));
                const E px = m_dot3(c.c2x, s[cc]), py = m_dot3(c.c2y, t[cc]);
                Jya[cc] = m_dot3(c.cmxy, q[cc]);
                P_FIRST(Bya[cc], fBya[cc], c.c1z, c.nc1z, f0[cc], f0[cc], f0[cc], Bya[cc][3]);
                P_FIRST(Px[cc], fPx[cc], c.c2z, c.c2z, f0[cc], f0[cc], f0[cc],
                        vadd(vfma(c.c20all, f0[cc], Px[cc][3]), vadd(px, py)));
                P_FIRST(Jxa[cc], fJxa[cc], c.nc2z, c.nc2z, f0[cc], f0[cc], f0[cc], vsub(vfma(c.nc20yz, f0[cc], Jxa[cc][3]), py));
                P_FIRST(Jza[cc], fJza[cc], c.cmxz, c.ncmxz, d[cc][0], d[cc][1], d[cc][2], Jza[cc][3]);
            }
            // ---- A_z, z part of its Laplacian (the in-plane part comes from AH) ----
#pragma unroll
            for (int cc = 0; cc < 2; cc++) {
                const E fz = pl[6 * M_PLANE + cc * M_WX];
                P_FIRST(Pzz[cc], fPzz[cc], c.c2z, c.c2z, fz, fz, fz, Pzz[cc][3]);
            }
#pragma unroll
            for (int cc = 0; cc < 2; cc++)
                p_tm_st2<E>(tm + (uint32_t)(P_TM_OWN + ((k % P_NOWN) * 2 + cc) * P_TM_CELL), Bza[cc], Jya[cc]);
            // ---- finalise plane zs - 6 + k ----
            if (k >= 2 * R) {
                const int z = zs + k - 2 * R;
                const int u = k - 2 * R;
                const E* pc = (const E*)(smem + ((k - R) % M_NP) * M_SLOT_BYTES) + cell_off;
                p_tm_wait_st();
                m_bar_wait<0>(&tfull[wp * P_NSLOT + k % P_NSLOT], (uint32_t)((k / P_NSLOT) & 1));
                p_tm_fence_after();
                E* mbase = (E*)(smem + P_OFF_MBOX + (u % M_ND) * P_MBOX_BYTES) + col0;
                E b0[2], b1[2], b2[2], P0[2], P1[2], P2[2];
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    uint32_t r_hp[8], r_hc[8], r_own[8], r_x[4];
                    const uint32_t so = (uint32_t)(P_TM_OWN + (((k - R) % P_NOWN) * 2 + cc) * P_TM_CELL);
                    const uint32_t sp = (uint32_t)(P_TM_HPARK + (((k - R) % P_NSLOT) * 2 + cc) * P_TM_CELL_HP);
                    const uint32_t sc = (uint32_t)(P_TM_HCOMP + ((k % P_NSLOT) * 2 + cc) * P_TM_CELL);
                    p_tm_ld8(tm + sp, r_hp);
                    p_tm_ld8(tm + sc, r_hc);
                    {
                        uint32_t r4[4], r2[2];
                        p_tm_ld4(tm + so, r4);
                        p_tm_ld2(tm + sc + 8, r2);
                        r_own[0] = r4[0]; r_own[1] = r4[1]; r_own[2] = r4[2]; r_own[3] = r4[3];
                        r_own[4] = r_own[5] = r_own[6] = r_own[7] = 0u;
                        r_x[0] = r2[0]; r_x[1] = r2[1]; r_x[2] = r_x[3] = 0u;
                    }
                    p_tm_wait_ld(r_own, r_hp, r_hc, r_x);
                    E Bza0, Jya0, Bzb0, Byb0, Pzip0, Bx0, Py0, Jxb0, Jyb0, Jzb0;
                    p_join(Bza0, r_own[0], r_own[1]); p_join(Jya0, r_own[2], r_own[3]);
                    p_join(Bzb0, r_hp[0], r_hp[1]); p_join(Byb0, r_hp[2], r_hp[3]); p_join(Pzip0, r_hp[4], r_hp[5]);
                    p_join(Bx0, r_hc[0], r_hc[1]); p_join(Py0, r_hc[2], r_hc[3]);
                    p_join(Jxb0, r_hc[4], r_hc[5]); p_join(Jyb0, r_hc[6], r_hc[7]);
                    p_join(Jzb0, r_x[0], r_x[1]);
                    b0[cc] = vadd(Bx0, c.bext[0]);
                    b1[cc] = vadd(vadd(fBya[cc], Byb0), c.bext[1]);
                    b2[cc] = vadd(vadd(Bza0, Bzb0), c.bext[2]);
                    const E j0 = vadd(fJxa[cc], Jxb0), j1 = vadd(Jya0, Jyb0), j2 = vadd(fJza[cc], Jzb0);
                    P0[cc] = fPx[cc];
                    P1[cc] = Py0;
                    P2[cc] = vadd(fPzz[cc], Pzip0);
                    const E rho_inv = vexpneg(pc[cc * M_WX]);
                    E* mb = mbase + cc * M_TX;
                    mb[0] = vmul(rho_inv, vsub(vmul(j1, b2[cc]), vmul(j2, b1[cc])));
                    mb[M_COLS] = vmul(rho_inv, vsub(vmul(j2, b0[cc]), vmul(j0, b2[cc])));
                    mb[2 * M_COLS] = vmul(rho_inv, vsub(vmul(j0, b1[cc]), vmul(j1, b0[cc])));
                }
                __syncwarp();
                if (lane == 0) m_bar_arrive(&mfull[rw * M_ND + u % M_ND]);
#pragma unroll
                for (int cc = 0; cc < 2; cc++) {
                    const E* pcc = pc + cc * M_WX;
                    const E ux = pcc[M_PLANE], uy = pcc[2 * M_PLANE], uz = pcc[3 * M_PLANE];
                    const E ax = pcc[4 * M_PLANE], ay = pcc[5 * M_PLANE], az = pcc[6 * M_PLANE];
                    // Eq. 3: u x B + eta lap A
                    const E r0 = vfma(c.eta, P0[cc], vsub(vmul(uy, b2[cc]), vmul(uz, b1[cc])));
                    const E r1 = vfma(c.eta, P1[cc], vsub(vmul(uz, b0[cc]), vmul(ux, b2[cc])));
                    const E r2 = vfma(c.eta, P2[cc], vsub(vmul(ux, b1[cc]), vmul(uy, b0[cc])));
                    E o0 = ax, o1 = ay, o2 = az;
                    if (with_prev) {
                        const E* pp = (const E*)(smem + P_OFF_PREV + (k % M_NPP) * M_PSLOT_BYTES) + 4 * M_COLS + col0 + cc * M_TX;
                        o0 = vfma(c.rk_a, vsub(ax, pp[0]), o0);
                        o1 = vfma(c.rk_a, vsub(ay, pp[M_COLS]), o1);
                        o2 = vfma(c.rk_a, vsub(az, pp[2 * M_COLS]), o2);
                    }
                    o0 = vfma(c.rk_b, r0, o0);
                    o1 = vfma(c.rk_b, r1, o1);
                    o2 = vfma(c.rk_b, r2, o2);
                    if (valid_x && y + cc < L.ny) {
                        const size_t ci = L.idx(x, y + cc, z);
                        a.out[4][ci] = o0;
                        a.out[5][ci] = o1;
                        a.out[6][ci] = o2;
                    }
                }
            }
            __syncwarp();
            if (lane == 0) m_bar_arrive(&done[k % M_NP]);
        }
    }
    }

    // every tensor-memory access has completed (the finalisers wait for their loads) before the columns go back
    p_tm_fence_before();
    __syncthreads();
    if (warp == 10) {
        p_tm_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_word), "n"(512) : "memory");
    }
}

}  // namespace ac
