// S9, stage 1 of the reductions for the 8-byte-element layouts (fp64, packed fp32): rms / max of |u| and
// |B| = |curl A + B_ext|, min / max of ln rho (readings G16, G18).
//
// B needs six first derivatives of A (36 neighbours, radius 3).  The three A fields are streamed plane by
// plane through a shared-memory ring by TMA (one 4-D box of tile + halo x 3 fields per plane, issued by a
// producer warp up to 3 planes ahead), ln rho and u by a second, interior-only box; the loads never wait on
// DRAM.  A worker thread owns one (x, y) column: from the plane that has just landed it takes the pointwise
// fields, the 24 in-plane neighbours (d_x, d_y of A_z, d_x A_y, d_y A_x) and the centre values of A_x, A_y; the z
// derivatives come from a 7-plane register history of those centre values and the in-plane parts of B wait
// 3 planes in registers (31 shared-memory loads per cell; gathering the z neighbours from a longer ring took
// 43 and an 8-slot ring: 1.83 ms against 1.43 ms for this version at 512^3 fp64).  A CTA takes (tile, z chunk) work items round-robin (fixed assignment: deterministic) and leaves one
// partial; reduce_stage2_kernel folds the partials in a fixed order.
#pragma once
#include "kernels.cuh"
#include "substep_march.cuh"

namespace ac {

constexpr int RQ_NP = 4;                                // ring slots: the plane being visited + 3 in flight
constexpr int RQ_CZ = 128;                              // planes per work item
constexpr int RQ_WORKERS = M_COLS;                      // 128 threads, one per column of the 16 x 8 tile
constexpr int RQ_THREADS = RQ_WORKERS + 32;             // + producer warp
constexpr int RQ_SLOT_BYTES = 3 * M_PLANE * 8;          // 8064: A_x, A_y, A_z, tile + halo
constexpr int RQ_PSLOT_BYTES = 4 * M_COLS * 8;          // 4096: ln rho, u, interior tile
constexpr int RQ_OFF_P = RQ_NP * RQ_SLOT_BYTES;
constexpr int RQ_OFF_BARS = RQ_OFF_P + RQ_NP * RQ_PSLOT_BYTES;
constexpr int RQ_SMEM_BYTES = RQ_OFF_BARS + 2 * RQ_NP * 8;
static_assert(RQ_SLOT_BYTES % 128 == 0, "TMA destinations must stay 128-byte aligned");

template <typename T, int LANES>
__device__ __forceinline__ void rq_lds(const unsigned char* p, T (&v)[LANES]) {
    if (LANES == 1) {
        v[0] = *(const T*)p;
    } else {
        const float2 t = *(const float2*)p;
        v[0] = (T)t.x;
        v[LANES - 1] = (T)t.y;
    }
}

template <typename T, int LANES>
__global__ void __launch_bounds__(RQ_THREADS, 3)
    reduce_tma_kernel(const __grid_constant__ ReduceArgs<T> a, const __grid_constant__ CUtensorMap map_a,
                      const __grid_constant__ CUtensorMap map_p, int tiles_x, int tiles_y, int nchunks) {
    extern __shared__ __align__(1024) unsigned char rq_smem[];
    uint64_t* full = (uint64_t*)(rq_smem + RQ_OFF_BARS);
    uint64_t* done = full + RQ_NP;
    const Layout& L = a.L;
    const int tid = threadIdx.x, lane = tid & 31;
    const long nwork = (long)tiles_x * tiles_y * nchunks;
    if (tid == 0) {
        for (int s = 0; s < RQ_NP; s++) {
            m_bar_init(&full[s], 1);
            m_bar_init(&done[s], RQ_WORKERS / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= RQ_WORKERS) {
        // ------------------------------------------ producer ------------------------------------------
        if (tid != RQ_WORKERS) return;
        long issued = 0;                                // running plane counter: ring slot and phase
        for (long w = blockIdx.x; w < nwork; w += gridDim.x) {
            const int x0 = (int)(w % tiles_x) * M_TX, y0 = (int)((w / tiles_x) % tiles_y) * M_TY;
            const int zs = (int)(w / ((long)tiles_x * tiles_y)) * RQ_CZ;
            const int niter = min(zs + RQ_CZ, L.nz) - zs + 2 * R;
            for (int k = 0; k < niter; k++, issued++) {
                // a slot is read only in the iteration its plane arrives in
                const long need = issued - RQ_NP;
                if (need >= 0) m_bar_wait<100>(&done[need % RQ_NP], (uint32_t)((need / RQ_NP) & 1));
                const int slot = (int)(issued % RQ_NP);
                const bool inner = k >= R && k < niter - R;     // plane zs - 3 + k is one of the item's own: bring ln rho, u
                m_bar_expect_tx(&full[slot], (uint32_t)(RQ_SLOT_BYTES + (inner ? RQ_PSLOT_BYTES : 0)));
                m_tma_load_4d(rq_smem + slot * RQ_SLOT_BYTES, &map_a, &full[slot], x0 - M_HX + L.gx, y0, zs + k, 0);
                if (inner)
                    m_tma_load_4d(rq_smem + RQ_OFF_P + slot * RQ_PSLOT_BYTES, &map_p, &full[slot], x0 + L.gx, y0 + R, zs + k,
                                  0);
            }
        }
        return;
    }

    // -------------------------------------------- workers --------------------------------------------
    RedVals acc = red_identity();
    const int tx = tid & (M_TX - 1), ty = tid >> 4;
    const int cell_off = ((ty + R) * M_WX + tx + M_HX) * 8;           // bytes
    long it = 0;
    for (long w = blockIdx.x; w < nwork; w += gridDim.x) {
        const int x = (int)(w % tiles_x) * M_TX + tx, y = (int)((w / tiles_x) % tiles_y) * M_TY + ty;
        const int zs = (int)(w / ((long)tiles_x * tiles_y)) * RQ_CZ;
        const int ze = min(zs + RQ_CZ, L.nz);
        const int niter = ze - zs + 2 * R;
        const bool valid = x < L.nx && y < L.ny;
        T hax[7][LANES], hay[7][LANES];                               // A_x, A_y of planes p-6 .. p (this column)
        T pbx[4][LANES], pby[4][LANES], pbz[4][LANES];                // d_y A_z, d_x A_z, B_z of planes p-3 .. p
#pragma unroll
        for (int r = 0; r < 7; r++)
#pragma unroll
            for (int i = 0; i < LANES; i++) hax[r][i] = hay[r][i] = T(0);
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int i = 0; i < LANES; i++) pbx[r][i] = pby[r][i] = pbz[r][i] = T(0);
#pragma unroll 1
        for (int k = 0; k < niter; k++, it++) {
            const int slot = (int)(it % RQ_NP);
#pragma unroll
            for (int r = 0; r < 6; r++)
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    hax[r][i] = hax[r + 1][i];
                    hay[r][i] = hay[r + 1][i];
                }
#pragma unroll
            for (int r = 0; r < 3; r++)
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    pbx[r][i] = pbx[r + 1][i];
                    pby[r][i] = pby[r + 1][i];
                    pbz[r][i] = pbz[r + 1][i];
                }
            m_bar_wait<0>(&full[slot], (uint32_t)((it / RQ_NP) & 1));
            const unsigned char* p0 = rq_smem + slot * RQ_SLOT_BYTES + cell_off;
            rq_lds<T, LANES>(p0, hax[6]);
            rq_lds<T, LANES>(p0 + M_PLANE * 8, hay[6]);
            if (k >= R && k < niter - R && valid) {
                // the plane is one of the item's own: in-plane parts of B, and the pointwise fields
                auto din = [&](int f, int stride, int axis, T (&r)[LANES]) {
                    const unsigned char* p = p0 + f * (M_PLANE * 8);
                    T r_[LANES];
#pragma unroll
                    for (int m = 1; m <= 3; m++) {
                        T pp[LANES], mm[LANES];
                        rq_lds<T, LANES>(p + m * stride, pp);
                        rq_lds<T, LANES>(p - m * stride, mm);
#pragma unroll
                        for (int i = 0; i < LANES; i++)
                            r_[i] = (m == 1) ? a.c1[axis][0] * (pp[i] - mm[i]) : fma_<T>(a.c1[axis][m - 1], pp[i] - mm[i], r_[i]);
                    }
#pragma unroll
                    for (int i = 0; i < LANES; i++) r[i] = r_[i];
                };
                T azy[LANES], azx[LANES], ayx[LANES], axy[LANES], az[LANES];
                T ux[LANES], uy[LANES], uz[LANES], l[LANES];
                din(2, M_WX * 8, 1, azy);
                din(2, 8, 0, azx);
                din(1, 8, 0, ayx);
                din(0, M_WX * 8, 1, axy);
                rq_lds<T, LANES>(p0 + 2 * M_PLANE * 8, az);
                const unsigned char* pp = rq_smem + RQ_OFF_P + slot * RQ_PSLOT_BYTES + tid * 8;
                rq_lds<T, LANES>(pp, l);
                rq_lds<T, LANES>(pp + M_COLS * 8, ux);
                rq_lds<T, LANES>(pp + 2 * M_COLS * 8, uy);
                rq_lds<T, LANES>(pp + 3 * M_COLS * 8, uz);
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    pbx[3][i] = azy[i];
                    pby[3][i] = azx[i];
                    pbz[3][i] = ayx[i] - axy[i] + a.bext[2];
                    const double u2 = (double)ux[i] * ux[i] + (double)uy[i] * uy[i] + (double)uz[i] * uz[i];
                    acc.su += u2;
                    acc.mu = fmax(acc.mu, u2);
                    acc.lmin = fmin(acc.lmin, (double)l[i]);
                    acc.lmax = fmax(acc.lmax, (double)l[i]);
                    // a non-finite ln rho or A would hide in fmin/fmax: fold it into the sums
                    const double chk = (double)l[i] + (double)hax[6][i] + (double)hay[6][i] + (double)az[i];
                    if (!isfinite(chk)) acc.su += chk;
                }
            }
            if (k >= 2 * R && valid) {                                // plane p - 3 has its 7-plane history: finish B there
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    T ayz = a.c1[2][0] * (hay[4][i] - hay[2][i]);
                    ayz = fma_<T>(a.c1[2][1], hay[5][i] - hay[1][i], ayz);
                    ayz = fma_<T>(a.c1[2][2], hay[6][i] - hay[0][i], ayz);
                    T axz = a.c1[2][0] * (hax[4][i] - hax[2][i]);
                    axz = fma_<T>(a.c1[2][1], hax[5][i] - hax[1][i], axz);
                    axz = fma_<T>(a.c1[2][2], hax[6][i] - hax[0][i], axz);
                    const T bx = pbx[0][i] - ayz + a.bext[0];
                    const T by = axz - pby[0][i] + a.bext[1];
                    const T bz = pbz[0][i];
                    const double b2 = (double)bx * bx + (double)by * by + (double)bz * bz;
                    acc.sb += b2;
                    acc.mb = fmax(acc.mb, b2);
                }
            }
            __syncwarp();
            if (lane == 0) m_bar_arrive(&done[slot]);
        }
    }
    // fold the 4 worker warps (the producer warp has left: no __syncthreads here)
    __shared__ RedVals warp_part[RQ_WORKERS / 32];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc = red_combine(acc, red_shfl_down(acc, d));
    if (lane == 0) warp_part[tid >> 5] = acc;
    asm volatile("bar.sync 1, %0;" ::"n"(RQ_WORKERS) : "memory");
    if (tid == 0) {
        RedVals r = warp_part[0];
        for (int wv = 1; wv < RQ_WORKERS / 32; wv++) r = red_combine(r, warp_part[wv]);
        a.partial[blockIdx.x] = r;
    }
}

}  // namespace ac
