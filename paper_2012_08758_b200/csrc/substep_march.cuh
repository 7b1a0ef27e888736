// Fused RK substep, variant "scatter-march" (the default).
//
// What it computes: exactly the substep of mhd_cell.cuh / the oracle - Eq. 1-3 right-hand sides
// (PAPER.md:166-170), forcing Eq. 4, 6th-order radius-3 central differences
// (readings G1-G3), j = grad div A - lap A (G4), the 2N-RK3 update in difference
// form (G7) - with the sums re-associated as follows.
//
// A CTA owns a 16 x 8 tile of (x, y) columns and marches along z.  Plane p (all 7 fields, tile +
// halo) is brought into a shared-memory ring by ONE 4-D TMA box load; a second box brings the
// previous-state values (2N register) of the plane that is finalised in the same iteration.
// Each column is served by two threads ("roles"): U carries ln rho and u, A carries A.
//
// When plane p arrives a thread loads only the IN-PLANE neighbourhood of its cell (centre, x row,
// y column, xy diagonals) and forms  dx_m = f(x+m) - f(x-m), dy_m, sx_m = f(x+m) + f(x-m), sy_m.
// These give d_x, d_y, d_xx, d_yy, d_xy of cell p directly.  Everything that couples planes is
// SCATTERED into register accumulators of the pending cells p-3 .. p+3 ("levels" r = 0 .. 6,
// r = 3 being plane p itself):
//     d_z f (z)  = sum_m c1z_m [f(z+m) - f(z-m)]            <- centre value of plane p, weight -/+ c1z_m
//     d_zz f (z) = c20z f(z) + sum_m c2z_m [f(z+m) + f(z-m)]
//     d_xz f (z) = sum_m cm_m [dx_m(z+m) - dx_m(z-m)]       (G2's 12 points, re-associated)
//     d_yz f (z) = sum_m cm_m [dy_m(z+m) - dy_m(z-m)]
// so a cell needs 139 shared-memory loads instead of 277 and a mixed z derivative costs 6 FMAs on
// differences the first derivatives need anyway.  Quantities that enter the equations linearly
// are accumulated already combined: L_i = lap u_i + 1/3 (grad div u)_i, lap A_i,
// J_i = (grad div A - lap A)_i, B_i.  The cell at level 0 (plane p-3) is complete after plane p
// has been scattered; it is then finalised: non-linear terms, forcing, 2N update, store.  The
// periodic ghost zones of the written buffer are refreshed by ghost_fill_kernel after the launch
// (keeping the image stores inside this loop cost 15 % of the U role's issue slots and doubled
// the loop's code size; profiles/r01b_march.md).
//
// Synchronisation: no block-wide barrier in the loop.  full[slot] (TMA transaction bytes) and
// done[iteration] (one arrival per worker warp) mbarriers.  Three warpgroups of 128 threads: U, A and a
// producer whose single working lane refills ring slots 3 planes ahead once every worker warp has
// finished the iteration that last read them.  The CTA is launched with 168 registers per thread;
// setmaxnreg moves the producer's share to the workers (232 each, 40 for the producer).  Giving the
// producer duty to a lane of a worker warp made that warp run every plane twice (the lane diverges
// through the wait loop and does not reconverge), the slowest scheduler then held up the whole CTA.
// The A role hands (j x B)/rho (and the upwind term) to the U role of the same columns through a
// mailbox with one mbarrier per warp pair.
//
// Element type E (vec2.cuh): double, or f2 = two fp32 cells (z, z + nz/2) per element.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "layout.cuh"
#include "vec2.cuh"

#include "march_common.cuh"

namespace ac {

// differences and sums along x (stride 1) or y (stride M_WX) around p
template <typename E, int STRIDE>
__device__ __forceinline__ void m_diff_sum(const E* p, E (&d)[3], E (&s)[3]) {
#pragma unroll
    for (int m = 1; m <= 3; m++) {
        const E a = p[m * STRIDE], b = p[-m * STRIDE];
        d[m - 1] = vsub(a, b);
        s[m - 1] = vadd(a, b);
    }
}
template <typename E, int STRIDE>
__device__ __forceinline__ void m_diff(const E* p, E (&d)[3]) {
#pragma unroll
    for (int m = 1; m <= 3; m++) d[m - 1] = vsub(p[m * STRIDE], p[-m * STRIDE]);
}
template <typename E, int STRIDE>
__device__ __forceinline__ void m_sum(const E* p, E (&s)[3]) {
#pragma unroll
    for (int m = 1; m <= 3; m++) s[m - 1] = vadd(p[m * STRIDE], p[-m * STRIDE]);
}
// in-plane bidiagonal mixed derivative (G2) with weights cm
template <typename E>
__device__ __forceinline__ E m_mixxy(const E* p, const E (&cm)[3]) {
    E r;
#pragma unroll
    for (int m = 1; m <= 3; m++) {
        const E s = vsub(vadd(p[m * M_WX + m], p[-m * M_WX - m]), vadd(p[-m * M_WX + m], p[m * M_WX - m]));
        r = (m == 1) ? vmul(cm[0], s) : vfma(cm[m - 1], s, r);
    }
    return r;
}
// scatter v into the levels m below (r = 3 - m, weight cdn) and m above (r = 3 + m, weight cup) plane p
#define M_SCAT(acc, m, cdn, cup, v)                           \
    do {                                                      \
        acc[3 - (m)] = vfma((cdn), (v), acc[3 - (m)]);        \
        acc[3 + (m)] = vfma((cup), (v), acc[3 + (m)]);        \
    } while (0)

// S1, periodic ghost zones of one state buffer after a substep (the paper's "local boundary
// transfer"; wrap of PAPER.md:111).  Every ghost cell copies its periodic source
// cell, which is always an interior cell, so the order of the copies does not matter.  Tasks
// [0, nb_rows) are the rows that are ghosts in y or z (whole rows, x ghosts included), the remaining
// tasks the x ghosts of M_GHOST_THREADS / (2 gx) interior rows each; blocks take tasks round-robin.  The x ghosts
// are copied as whole 32-byte sectors (gx elements a side: the R ghost cells and the alignment pad next to
// them, which nothing reads), so that no store leaves a partly written sector.  z images of packed fp32
// pairs swap lanes (cell z - nz/2 of the pair below is cell z + nz/2 of the periodic domain).
constexpr int M_GHOST_THREADS = 256;
template <typename E>
__global__ void __launch_bounds__(M_GHOST_THREADS) ghost_fill_kernel(E* __restrict__ base, Layout L, int nb_rows, int na_tasks, int first_row) {
    E* __restrict__ f = base + (size_t)blockIdx.y * L.field;
    const int tid = threadIdx.x;
    const int per_row = 2 * L.gx, rows_per_task = M_GHOST_THREADS / per_row;
    // first_row = 2 R my skips the 6 ghost planes (a slab whose neighbours fill them)
    for (int task = first_row + blockIdx.x; task < nb_rows + na_tasks; task += gridDim.x) {
        if (task < nb_rows) {
            // one ghost row (ghost in y or z), whole: x ghosts included
            const int row = task;
            int y, z;
            if (row < 2 * R * L.my) {            // the 6 ghost planes, all rows
                const int zi = row / L.my;
                z = zi < R ? zi - R : L.nz + zi - R;
                y = row % L.my - R;
            } else {                             // the 6 ghost rows of every interior plane
                const int r2 = row - 2 * R * L.my;
                const int yi = r2 % (2 * R);
                z = r2 / (2 * R);
                y = yi < R ? yi - R : L.ny + yi - R;
            }
            const int ys = y < 0 ? y + L.ny : (y >= L.ny ? y - L.ny : y);
            const int zs = z < 0 ? z + L.nz : (z >= L.nz ? z - L.nz : z);
            const E* __restrict__ src = f + L.idx(0, ys, zs);
            E* __restrict__ dst = f + L.idx(0, y, z);
            for (int x = tid - L.gx; x < L.nx + L.gx; x += M_GHOST_THREADS) {
                const int xs = x < 0 ? x + L.nx : (x >= L.nx ? x - L.nx : x);
                E v = src[xs];
                if (zs != z) v = vswap(v);
                dst[x] = v;
            }
        } else {
            // the 2 x gx x-ghost cells of rows_per_task interior rows
            const long r = (long)(task - nb_rows) * rows_per_task + tid / per_row;
            const int j = tid % per_row;
            if (tid < rows_per_task * per_row && r < (long)L.ny * L.nz) {
                const int y = (int)(r % L.ny), z = (int)(r / L.ny);
                const int x = j < L.gx ? j - L.gx : L.nx + j - L.gx;
                const int xs = j < L.gx ? x + L.nx : x - L.nx;
                f[L.idx(x, y, z)] = f[L.idx(xs, y, z)];
            }
        }
    }
}

// UPW: continuity equation with the 5th-order upwind correction (G17).  The A role, which has
// registers to spare, forms  sum_a |u_a| delta6_a ln rho / (60 h_a)  (x, y parts in plane, z part
// scattered like every other z stencil) and hands it to the U role with (j x B)/rho.
template <typename T, bool UPW>
__global__ void __launch_bounds__(M_THREADS, 1)
    substep_march_kernel(const __grid_constant__ MarchArgs<T> a, const __grid_constant__ CUtensorMap map_in,
                         const __grid_constant__ CUtensorMap map_prev) {
    using E = typename ElemOf<T>::E;
    // declared 1024-byte aligned and used in place: every pointer derived from it keeps the shared
    // address space (LDS/STS); rounding the base through an integer made ptxas fall back to generic LD
    extern __shared__ __align__(1024) unsigned char smem[];
    E* ztab = (E*)(smem + M_OFF_ZTAB);
    uint64_t* full = (uint64_t*)(smem + M_OFF_BARS);
    uint64_t* done = full + M_NP;
    uint64_t* mfull = done + M_NP;     // [pair][depth]

    const Layout& L = a.L;
    const MarchCoef<E>& c = a.c;
    const int tid = threadIdx.x;
    const int role = tid >> 7;              // 0 = U (ln rho, u), 1 = A, 2 = producer (one working lane)
    const int col = tid & (M_COLS - 1);
    const int tx = col & (M_TX - 1), ty = col >> 4;
    const int lane = tid & 31;
    const int pair = (tid >> 5) & 3;        // U warp w and A warp w + 4 serve the same 32 columns
    const int x0 = blockIdx.x * M_TX, y0 = blockIdx.y * M_TY;
    const int zs = a.z_begin + blockIdx.z * a.cz;
    const int ze = min(zs + a.cz, a.z_end);
    const int niter = ze - zs + 2 * R;      // planes zs-3 .. ze+2
    const int x = x0 + tx, y = y0 + ty;
    const bool valid = (x < L.nx) && (y < L.ny);
    const bool with_prev = a.substep != 0;

    if (tid == 0) {
        for (int s = 0; s < M_NP; s++) {
            m_bar_init(&full[s], 1);
            m_bar_init(&done[s], M_WORKERS / 32);
        }
        for (int s = 0; s < 4 * M_ND; s++) m_bar_init(&mfull[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
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
    __syncthreads();

    // iteration k processes plane zs - 3 + k and finalises level zs - 6 + k
    auto issue = [&](int k) {
        const int slot = k % M_NP;
        const bool fin = with_prev && k >= 2 * R;
        m_bar_expect_tx(&full[slot], (uint32_t)(M_SLOT_BYTES + (fin ? M_PSLOT_BYTES : 0)));
        m_tma_load_4d(smem + slot * M_SLOT_BYTES, &map_in, &full[slot], x0 - M_HX + L.gx, y0, zs + k, 0);
        if (fin)
            m_tma_load_4d(smem + M_OFF_PREV + (k % M_NPP) * M_PSLOT_BYTES, &map_prev, &full[slot], x0 + L.gx, y0 + R,
                          zs + k - R, 0);
    };
    // the kernel is launched with 168 registers per thread (384 threads); the producer warpgroup hands its
    // share to the two worker warpgroups
    if (role == 2) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(M_REGS_PRODUCER));
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(M_REGS_WORKER));
    }
    if (role == 2) {
        // ===================================== producer warp =====================================
        // plane k + LEAD reuses the ring slot that every worker warp has released after iteration k - 2
        if (tid == M_WORKERS) {
            for (int k = 0; k < M_LEAD && k < niter; k++) issue(k);
            for (int k = 0; k + M_LEAD < niter; k++) {
                if (k >= 2) m_bar_wait<MarchWait<T>::PRODUCER_NS>(&done[(k - 2) % M_NP], (uint32_t)(((k - 2) / M_NP) & 1));
                issue(k + M_LEAD);
            }
        }
        return;
    }

    const int cell_off = (ty + R) * M_WX + tx + M_HX;

    // forcing: cos/sin of k_x x + k_y y, constant along the march
    E cxy = vzero<E>(), sxy = vzero<E>();
    if (role == 0 && a.has_forcing && valid) {
        const T cx_ = a.ftab[x], sx_ = a.ftab[L.nx + x];
        const T cy_ = a.ftab[2 * L.nx + y], sy_ = a.ftab[2 * L.nx + L.ny + y];
        cxy = Splat<E>::of((double)(cx_ * cy_ - sx_ * sy_));
        sxy = Splat<E>::of((double)(sx_ * cy_ + cx_ * sy_));
    }

    if (role == 0) {
        // ======================================= U role ========================================
        E Gxz[7], Gyz[7], Gzz[7], Lx[7], Ly[7], Lz[7];            // z-coupled accumulators, levels 0..6
        E Gxx[4], Gxy[4], Gyx[4], Gyy[4], Gzx[4], Gzy[4];         // in-plane first derivatives, levels 0..3
        E gz[7], gx[4], gy[4];
#pragma unroll
        for (int r = 0; r < 7; r++) gz[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 4; r++) gx[r] = gy[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 7; r++) Gxz[r] = Gyz[r] = Gzz[r] = Lx[r] = Ly[r] = Lz[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 4; r++) Gxx[r] = Gxy[r] = Gyx[r] = Gyy[r] = Gzx[r] = Gzy[r] = vzero<E>();

        for (int k = 0; k < niter; k++) {
            m_bar_wait<MarchWait<T>::RING_U_NS>(&full[k % M_NP], (uint32_t)((k / M_NP) & 1));
            const E* pl = (const E*)(smem + (k % M_NP) * M_SLOT_BYTES) + cell_off;

            Gxz[6] = Gyz[6] = Gzz[6] = Lx[6] = Ly[6] = Lz[6] = vzero<E>();
            E d[3], s[3], e[3], t[3];
            gz[6] = vzero<E>();
            {
                const E* p = pl;
                const E f0 = p[0];
                m_diff<E, 1>(p, d);
                m_diff<E, M_WX>(p, e);
                gx[3] = m_dot3(c.c1x, d);
                gy[3] = m_dot3(c.c1y, e);
#pragma unroll
                for (int m = 1; m <= 3; m++) M_SCAT(gz, m, c.c1z[m - 1], c.nc1z[m - 1], f0);
            }
            // ---- u_x: d_x, d_y; L_x in-plane; D_xy u_x -> L_y; D_xz u_x -> L_z ----
            {
                const E* p = pl + 1 * M_PLANE;
                const E f0 = p[0];
                m_diff_sum<E, 1>(p, d, s);
                m_diff_sum<E, M_WX>(p, e, t);
                Gxx[3] = m_dot3(c.c1x, d);
                Gxy[3] = m_dot3(c.c1y, e);
                E l = vfma(c.w20[0], f0, Lx[3]);
                l = m_dot3(c.w2x[0], s, l);
                Lx[3] = m_dot3(c.w2y[0], t, l);
                Ly[3] = vadd(Ly[3], m_mixxy(p, c.cm3xy));
#pragma unroll
                for (int m = 1; m <= 3; m++) {
                    M_SCAT(Gxz, m, c.c1z[m - 1], c.nc1z[m - 1], f0);
                    M_SCAT(Lx, m, c.w2z[0][m - 1], c.w2z[0][m - 1], f0);
                    M_SCAT(Lz, m, c.cm3xz[m - 1], c.ncm3xz[m - 1], d[m - 1]);
                }
            }
            // ---- u_y: D_xy u_y -> L_x; D_yz u_y -> L_z ----
            {
                const E* p = pl + 2 * M_PLANE;
                const E f0 = p[0];
                m_diff_sum<E, 1>(p, d, s);
                m_diff_sum<E, M_WX>(p, e, t);
                Gyx[3] = m_dot3(c.c1x, d);
                Gyy[3] = m_dot3(c.c1y, e);
                E l = vfma(c.w20[1], f0, Ly[3]);
                l = m_dot3(c.w2x[1], s, l);
                Ly[3] = m_dot3(c.w2y[1], t, l);
                Lx[3] = vadd(Lx[3], m_mixxy(p, c.cm3xy));
#pragma unroll
                for (int m = 1; m <= 3; m++) {
                    M_SCAT(Gyz, m, c.c1z[m - 1], c.nc1z[m - 1], f0);
                    M_SCAT(Ly, m, c.w2z[1][m - 1], c.w2z[1][m - 1], f0);
                    M_SCAT(Lz, m, c.cm3yz[m - 1], c.ncm3yz[m - 1], e[m - 1]);
                }
            }
            // ---- u_z: D_xz u_z -> L_x; D_yz u_z -> L_y ----
            {
                const E* p = pl + 3 * M_PLANE;
                const E f0 = p[0];
                m_diff_sum<E, 1>(p, d, s);
                m_diff_sum<E, M_WX>(p, e, t);
                Gzx[3] = m_dot3(c.c1x, d);
                Gzy[3] = m_dot3(c.c1y, e);
                E l = vfma(c.w20[2], f0, Lz[3]);
                l = m_dot3(c.w2x[2], s, l);
                Lz[3] = m_dot3(c.w2y[2], t, l);
#pragma unroll
                for (int m = 1; m <= 3; m++) {
                    M_SCAT(Gzz, m, c.c1z[m - 1], c.nc1z[m - 1], f0);
                    M_SCAT(Lz, m, c.w2z[2][m - 1], c.w2z[2][m - 1], f0);
                    M_SCAT(Lx, m, c.cm3xz[m - 1], c.ncm3xz[m - 1], d[m - 1]);
                    M_SCAT(Ly, m, c.cm3yz[m - 1], c.ncm3yz[m - 1], e[m - 1]);
                }
            }

            // ---- finalise level 0 = plane zs - 6 + k ----
            if (k >= 2 * R) {
                const int z = zs + k - 2 * R;
                const E* pc = (const E*)(smem + ((k - R) % M_NP) * M_SLOT_BYTES) + cell_off;
                const E lnrho = pc[0], ux = pc[M_PLANE], uy = pc[2 * M_PLANE], uz = pc[3 * M_PLANE];
                const E divu = vadd(vadd(Gxx[0], Gyy[0]), Gzz[0]);
                // (j x B) / rho (and the upwind term) from the A role of the same columns
                const int u = k - 2 * R;
                m_bar_wait<MarchWait<T>::MAILBOX_NS>(&mfull[pair * M_ND + u % M_ND], (uint32_t)((u / M_ND) & 1));
                const E* mb = (const E*)(smem + M_OFF_MBOX + (u % M_ND) * M_MBOX_BYTES) + col;
                const E jxb0 = mb[0], jxb1 = mb[M_COLS], jxb2 = mb[2 * M_COLS];
                const E g0 = gx[0], g1 = gy[0], g2 = gz[0];
                // Eq. 1
                E rl = vmul(ux, g0);
                rl = vfma(uy, g1, rl);
                rl = vfma(uz, g2, rl);
                rl = vneg(vadd(rl, divu));
                if (UPW) rl = vadd(rl, mb[3 * M_COLS]);
                // forcing Eq. 4: f_i = re_i cos(theta) - im_i sin(theta)
                E fc = vzero<E>(), fs = vzero<E>();
                if (a.has_forcing) {
                    const E cz_ = ztab[2 * (z - zs)], sz_ = ztab[2 * (z - zs) + 1];
                    fc = vsub(vmul(cxy, cz_), vmul(sxy, sz_));
                    fs = vfma(sxy, cz_, vmul(cxy, sz_));
                }
                // 2 S_ij g_j = (G_ij + G_ji) g_j - 2/3 div u g_i
                const E sxy_ = vadd(Gxy[0], Gyx[0]), sxz_ = vadd(Gxz[0], Gzx[0]), syz_ = vadd(Gyz[0], Gzy[0]);
                const E dd = vmul(c.n23, divu);
                E sg0 = vmul(vadd(Gxx[0], Gxx[0]), g0);
                sg0 = vfma(sxy_, g1, sg0);
                sg0 = vfma(sxz_, g2, sg0);
                sg0 = vfma(dd, g0, sg0);
                E sg1 = vmul(sxy_, g0);
                sg1 = vfma(vadd(Gyy[0], Gyy[0]), g1, sg1);
                sg1 = vfma(syz_, g2, sg1);
                sg1 = vfma(dd, g1, sg1);
                E sg2 = vmul(sxz_, g0);
                sg2 = vfma(syz_, g1, sg2);
                sg2 = vfma(vadd(Gzz[0], Gzz[0]), g2, sg2);
                sg2 = vfma(dd, g2, sg2);
                // Eq. 2
                E adv0 = vmul(ux, Gxx[0]);
                adv0 = vfma(uy, Gxy[0], adv0);
                adv0 = vfma(uz, Gxz[0], adv0);
                E adv1 = vmul(ux, Gyx[0]);
                adv1 = vfma(uy, Gyy[0], adv1);
                adv1 = vfma(uz, Gyz[0], adv1);
                E adv2 = vmul(ux, Gzx[0]);
                adv2 = vfma(uy, Gzy[0], adv2);
                adv2 = vfma(uz, Gzz[0], adv2);
                E r0 = vfma(c.nu, vadd(Lx[0], sg0), vadd(jxb0, vsub(vmul(c.ncs2, g0), adv0)));
                E r1 = vfma(c.nu, vadd(Ly[0], sg1), vadd(jxb1, vsub(vmul(c.ncs2, g1), adv1)));
                E r2 = vfma(c.nu, vadd(Lz[0], sg2), vadd(jxb2, vsub(vmul(c.ncs2, g2), adv2)));
                if (a.has_forcing) {
                    r0 = vfma(c.fre[0], fc, vfma(c.nfim[0], fs, r0));
                    r1 = vfma(c.fre[1], fc, vfma(c.nfim[1], fs, r1));
                    r2 = vfma(c.fre[2], fc, vfma(c.nfim[2], fs, r2));
                }
                // 2N-RK3 update, difference form
                E o0 = lnrho, o1 = ux, o2 = uy, o3 = uz;
                if (with_prev) {
                    const E* pp = (const E*)(smem + M_OFF_PREV + (k % M_NPP) * M_PSLOT_BYTES) + col;
                    o0 = vfma(c.rk_a, vsub(lnrho, pp[0]), o0);
                    o1 = vfma(c.rk_a, vsub(ux, pp[M_COLS]), o1);
                    o2 = vfma(c.rk_a, vsub(uy, pp[2 * M_COLS]), o2);
                    o3 = vfma(c.rk_a, vsub(uz, pp[3 * M_COLS]), o3);
                }
                o0 = vfma(c.rk_b, rl, o0);
                o1 = vfma(c.rk_b, r0, o1);
                o2 = vfma(c.rk_b, r1, o2);
                o3 = vfma(c.rk_b, r2, o3);
                const size_t ci = L.idx(x, y, z);
                if (valid) {
                    a.out[0][ci] = o0;
                    a.out[1][ci] = o1;
                    a.out[2][ci] = o2;
                    a.out[3][ci] = o3;
                }
            }
            __syncwarp();
            if (lane == 0) m_bar_arrive(&done[k % M_NP]);
            // next plane: every pending level moves one step closer to completion
#pragma unroll
            for (int r = 0; r < 6; r++) {
                Gxz[r] = Gxz[r + 1]; Gyz[r] = Gyz[r + 1]; Gzz[r] = Gzz[r + 1];
                Lx[r] = Lx[r + 1]; Ly[r] = Ly[r + 1]; Lz[r] = Lz[r + 1];
            }
#pragma unroll
            for (int r = 0; r < 3; r++) {
                Gxx[r] = Gxx[r + 1]; Gxy[r] = Gxy[r + 1];
                Gyx[r] = Gyx[r + 1]; Gyy[r] = Gyy[r + 1]; Gzx[r] = Gzx[r + 1]; Gzy[r] = Gzy[r + 1];
            }
#pragma unroll
            for (int r = 0; r < 6; r++) gz[r] = gz[r + 1];
#pragma unroll
            for (int r = 0; r < 3; r++) { gx[r] = gx[r + 1]; gy[r] = gy[r + 1]; }
        }
    } else {
        // ======================================= A role ========================================
        E Bx[7], By[7], Px[7], Py[7], Pz[7], Jx[7], Jy[7], Jz[7];   // P_i = lap A_i
        E Bz[4];
        E u6z[7], u6x[4], u6y[4];                                    // UPW only: delta6 ln rho / (60 h) per axis
#pragma unroll
        for (int r = 0; r < 7; r++) u6z[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 4; r++) u6x[r] = u6y[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 7; r++) Bx[r] = By[r] = Px[r] = Py[r] = Pz[r] = Jx[r] = Jy[r] = Jz[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 4; r++) Bz[r] = vzero<E>();

        for (int k = 0; k < niter; k++) {
            m_bar_wait<MarchWait<T>::RING_A_NS>(&full[k % M_NP], (uint32_t)((k / M_NP) & 1));
            const E* pl = (const E*)(smem + (k % M_NP) * M_SLOT_BYTES) + cell_off;

            Bx[6] = By[6] = Px[6] = Py[6] = Pz[6] = Jx[6] = Jy[6] = Jz[6] = vzero<E>();
            E d[3], s[3], e[3], t[3];
            if (UPW) {
                // ---- ln rho: sixth differences along x, y (in plane) and z (scattered) ----
                const E* p = pl;
                const E f0 = p[0];
                m_sum<E, 1>(p, s);
                m_sum<E, M_WX>(p, t);
                u6x[3] = m_dot3(c.c6x, s, vmul(c.c60x, f0));
                u6y[3] = m_dot3(c.c6y, t, vmul(c.c60y, f0));
                u6z[6] = vzero<E>();
                u6z[3] = vfma(c.c60z, f0, u6z[3]);
#pragma unroll
                for (int m = 1; m <= 3; m++) M_SCAT(u6z, m, c.c6z[m - 1], c.c6z[m - 1], f0);
            }
            // ---- A_x: B_z -= d_y A_x; lap; J_x -= (D_yy + D_zz) A_x; D_xy A_x -> J_y; D_xz A_x -> J_z; B_y += d_z A_x
            {
                const E* p = pl + 4 * M_PLANE;
                const E f0 = p[0];
                m_diff_sum<E, 1>(p, d, s);
                m_diff_sum<E, M_WX>(p, e, t);
                const E dyax = m_dot3(c.c1y, e);
                const E px = m_dot3(c.c2x, s), py = m_dot3(c.c2y, t);
                Px[3] = vadd(vfma(c.c20all, f0, Px[3]), vadd(px, py));
                Jx[3] = vsub(vfma(c.nc20yz, f0, Jx[3]), py);
                Jy[3] = vadd(Jy[3], m_mixxy(p, c.cmxy));
                Bz[3] = vneg(dyax);
#pragma unroll
                for (int m = 1; m <= 3; m++) {
                    M_SCAT(By, m, c.c1z[m - 1], c.nc1z[m - 1], f0);
                    M_SCAT(Px, m, c.c2z[m - 1], c.c2z[m - 1], f0);
                    M_SCAT(Jx, m, c.nc2z[m - 1], c.nc2z[m - 1], f0);
                    M_SCAT(Jz, m, c.cmxz[m - 1], c.ncmxz[m - 1], d[m - 1]);
                }
            }
            // ---- A_y: B_z += d_x A_y; lap; J_y -= (D_xx + D_zz) A_y; D_xy A_y -> J_x; D_yz A_y -> J_z; B_x -= d_z A_y
            {
                const E* p = pl + 5 * M_PLANE;
                const E f0 = p[0];
                m_diff_sum<E, 1>(p, d, s);
                m_diff_sum<E, M_WX>(p, e, t);
                Bz[3] = m_dot3(c.c1x, d, Bz[3]);
                const E px = m_dot3(c.c2x, s), py = m_dot3(c.c2y, t);
                Py[3] = vadd(vfma(c.c20all, f0, Py[3]), vadd(px, py));
                Jy[3] = vsub(vfma(c.nc20xz, f0, Jy[3]), px);
                Jx[3] = vadd(Jx[3], m_mixxy(p, c.cmxy));
#pragma unroll
                for (int m = 1; m <= 3; m++) {
                    M_SCAT(Bx, m, c.nc1z[m - 1], c.c1z[m - 1], f0);
                    M_SCAT(Py, m, c.c2z[m - 1], c.c2z[m - 1], f0);
                    M_SCAT(Jy, m, c.nc2z[m - 1], c.nc2z[m - 1], f0);
                    M_SCAT(Jz, m, c.cmyz[m - 1], c.ncmyz[m - 1], e[m - 1]);
                }
            }
            // ---- A_z: B_x += d_y A_z; B_y -= d_x A_z; lap; J_z -= (D_xx + D_yy) A_z; D_xz A_z -> J_x; D_yz A_z -> J_y
            {
                const E* p = pl + 6 * M_PLANE;
                const E f0 = p[0];
                m_diff_sum<E, 1>(p, d, s);
                m_diff_sum<E, M_WX>(p, e, t);
                Bx[3] = m_dot3(c.c1y, e, Bx[3]);
                By[3] = vsub(By[3], m_dot3(c.c1x, d));
                const E pxy = vadd(m_dot3(c.c2x, s), m_dot3(c.c2y, t));
                Pz[3] = vadd(vfma(c.c20all, f0, Pz[3]), pxy);
                Jz[3] = vsub(vfma(c.nc20xy, f0, Jz[3]), pxy);
#pragma unroll
                for (int m = 1; m <= 3; m++) {
                    M_SCAT(Pz, m, c.c2z[m - 1], c.c2z[m - 1], f0);
                    M_SCAT(Jx, m, c.cmxz[m - 1], c.ncmxz[m - 1], d[m - 1]);
                    M_SCAT(Jy, m, c.cmyz[m - 1], c.ncmyz[m - 1], e[m - 1]);
                }
            }

            // ---- finalise level 0 ----
            if (k >= 2 * R) {
                const int z = zs + k - 2 * R;
                const E b0 = vadd(Bx[0], c.bext[0]), b1 = vadd(By[0], c.bext[1]), b2 = vadd(Bz[0], c.bext[2]);
                const E j0 = Jx[0], j1 = Jy[0], j2 = Jz[0];
                const int u = k - 2 * R;
                const E* pc = (const E*)(smem + ((k - R) % M_NP) * M_SLOT_BYTES) + cell_off;
                const E rho_inv = vexpneg(pc[0]);
                E* mb = (E*)(smem + M_OFF_MBOX + (u % M_ND) * M_MBOX_BYTES) + col;
                mb[0] = vmul(rho_inv, vsub(vmul(j1, b2), vmul(j2, b1)));
                mb[M_COLS] = vmul(rho_inv, vsub(vmul(j2, b0), vmul(j0, b2)));
                mb[2 * M_COLS] = vmul(rho_inv, vsub(vmul(j0, b1), vmul(j1, b0)));
                if (UPW) {
                    E up = vmul(vabs(pc[M_PLANE]), u6x[0]);
                    up = vfma(vabs(pc[2 * M_PLANE]), u6y[0], up);
                    mb[3 * M_COLS] = vfma(vabs(pc[3 * M_PLANE]), u6z[0], up);
                }
                __syncwarp();
                if (lane == 0) m_bar_arrive(&mfull[pair * M_ND + u % M_ND]);
                const E ux = pc[M_PLANE], uy = pc[2 * M_PLANE], uz = pc[3 * M_PLANE];
                const E ax = pc[4 * M_PLANE], ay = pc[5 * M_PLANE], az = pc[6 * M_PLANE];
                // Eq. 3: u x B + eta lap A
                const E r0 = vfma(c.eta, Px[0], vsub(vmul(uy, b2), vmul(uz, b1)));
                const E r1 = vfma(c.eta, Py[0], vsub(vmul(uz, b0), vmul(ux, b2)));
                const E r2 = vfma(c.eta, Pz[0], vsub(vmul(ux, b1), vmul(uy, b0)));
                E o0 = ax, o1 = ay, o2 = az;
                if (with_prev) {
                    const E* pp = (const E*)(smem + M_OFF_PREV + (k % M_NPP) * M_PSLOT_BYTES) + 4 * M_COLS + col;
                    o0 = vfma(c.rk_a, vsub(ax, pp[0]), o0);
                    o1 = vfma(c.rk_a, vsub(ay, pp[M_COLS]), o1);
                    o2 = vfma(c.rk_a, vsub(az, pp[2 * M_COLS]), o2);
                }
                o0 = vfma(c.rk_b, r0, o0);
                o1 = vfma(c.rk_b, r1, o1);
                o2 = vfma(c.rk_b, r2, o2);
                const size_t ci = L.idx(x, y, z);
                if (valid) {
                    a.out[4][ci] = o0;
                    a.out[5][ci] = o1;
                    a.out[6][ci] = o2;
                }
            }
            __syncwarp();
            if (lane == 0) m_bar_arrive(&done[k % M_NP]);
#pragma unroll
            for (int r = 0; r < 6; r++) {
                Bx[r] = Bx[r + 1]; By[r] = By[r + 1]; Px[r] = Px[r + 1]; Py[r] = Py[r + 1]; Pz[r] = Pz[r + 1];
                Jx[r] = Jx[r + 1]; Jy[r] = Jy[r + 1]; Jz[r] = Jz[r + 1];
            }
#pragma unroll
            for (int r = 0; r < 3; r++) Bz[r] = Bz[r + 1];
            if (UPW) {
#pragma unroll
                for (int r = 0; r < 6; r++) u6z[r] = u6z[r + 1];
#pragma unroll
                for (int r = 0; r < 3; r++) { u6x[r] = u6x[r + 1]; u6y[r] = u6y[r + 1]; }
            }
        }
    }
}

}  // namespace ac
