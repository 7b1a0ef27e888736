// S9, stage 1 of the reductions for the 8-byte-element layouts (fp64, packed fp32): rms / max of |u| and
// |B| = |curl A + B_ext|, min / max of ln rho (readings G16, G18).
//
// B needs six first derivatives of A (36 neighbours, radius 3).  The three A fields are streamed plane by
// plane through a shared-memory ring by TMA (one 4-D box of tile + halo x 3 fields per plane, issued by a
// producer warp LEAD planes ahead); a worker thread owns one (x, y) column, and when plane q + 3 has landed it
// gathers the 36 neighbours of cell (x, y, q) from the ring, so no derivative state is carried in registers
// and the loads never wait on DRAM.  ln rho and u of the plane being finished arrive by a second, interior-only
// TMA box in a small ring of their own.  A CTA takes (tile, z chunk) work items round-robin (fixed assignment: deterministic) and leaves one
// partial; reduce_stage2_kernel folds the partials in a fixed order.
#pragma once
#include "kernels.cuh"
#include "substep_march.cuh"

namespace ac {

constexpr int RQ_NP = 8;                                // ring slots: planes q-3 .. q+3 in use + 1 in flight (3 CTAs per SM
                                                        // with a short ring beat 2 CTAs with 11 slots: 1.83 vs 2.13 ms)
constexpr int RQ_CZ = 128;                              // planes per work item
constexpr int RQ_WORKERS = M_COLS;                      // 128 threads, one per column of the 16 x 8 tile
constexpr int RQ_THREADS = RQ_WORKERS + 32;             // + producer warp
constexpr int RQ_SLOT_BYTES = 3 * M_PLANE * 8;          // 8064
constexpr int RQ_PNP = 2;                               // ring of the pointwise fields (ln rho, u): producer lead + 1
constexpr int RQ_PSLOT_BYTES = 4 * M_COLS * 8;          // 4096: interior tile of 4 fields
constexpr int RQ_OFF_P = RQ_NP * RQ_SLOT_BYTES;
constexpr int RQ_OFF_BARS = RQ_OFF_P + RQ_PNP * RQ_PSLOT_BYTES;
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
                // the slot of plane `issued` was last read 7 planes after the plane it held (issued - NP)
                const long need = issued - RQ_NP + 2 * R;
                if (need >= 0) m_bar_wait<100>(&done[need % RQ_NP], (uint32_t)((need / RQ_NP) & 1));
                const int slot = (int)(issued % RQ_NP);
                const bool fin = k >= 2 * R;        // plane zs + k - 6 is finished in this iteration: bring its ln rho, u
                m_bar_expect_tx(&full[slot], (uint32_t)(RQ_SLOT_BYTES + (fin ? RQ_PSLOT_BYTES : 0)));
                m_tma_load_4d(rq_smem + slot * RQ_SLOT_BYTES, &map_a, &full[slot], x0 - M_HX + L.gx, y0, zs + k, 0);
                if (fin)
                    m_tma_load_4d(rq_smem + RQ_OFF_P + (int)(issued % RQ_PNP) * RQ_PSLOT_BYTES, &map_p, &full[slot],
                                  x0 + L.gx, y0 + R, zs + k - R, 0);
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
        for (int k = 0; k < niter; k++, it++) {
            const bool fin = k >= 2 * R;
            m_bar_wait<0>(&full[it % RQ_NP], (uint32_t)((it / RQ_NP) & 1));
            if (fin && valid) {
                T ux[LANES], uy[LANES], uz[LANES], l[LANES];
                const unsigned char* pp = rq_smem + RQ_OFF_P + (int)(it % RQ_PNP) * RQ_PSLOT_BYTES + tid * 8;
                rq_lds<T, LANES>(pp, l);
                rq_lds<T, LANES>(pp + M_COLS * 8, ux);
                rq_lds<T, LANES>(pp + 2 * M_COLS * 8, uy);
                rq_lds<T, LANES>(pp + 3 * M_COLS * 8, uz);
                // plane q + j sits in the slot of running index it - 3 + j
                auto plane = [&](int j) { return rq_smem + (int)((it - R + j) % RQ_NP) * RQ_SLOT_BYTES + cell_off; };
                const unsigned char* p0 = plane(0);
                // first derivative of A field f (0, 1, 2) along x (stride 8 B) or y (stride M_WX * 8 B) in plane q
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
                // and along z: the same column of planes q -+ m
                auto dz = [&](int f, T (&r)[LANES]) {
                    T r_[LANES];
#pragma unroll
                    for (int m = 1; m <= 3; m++) {
                        T pp[LANES], mm[LANES];
                        rq_lds<T, LANES>(plane(m) + f * (M_PLANE * 8), pp);
                        rq_lds<T, LANES>(plane(-m) + f * (M_PLANE * 8), mm);
#pragma unroll
                        for (int i = 0; i < LANES; i++)
                            r_[i] = (m == 1) ? a.c1[2][0] * (pp[i] - mm[i]) : fma_<T>(a.c1[2][m - 1], pp[i] - mm[i], r_[i]);
                    }
#pragma unroll
                    for (int i = 0; i < LANES; i++) r[i] = r_[i];
                };
                T azy[LANES], ayz[LANES], axz[LANES], azx[LANES], ayx[LANES], axy[LANES];
                T ax[LANES], ay[LANES], az[LANES];
                din(2, M_WX * 8, 1, azy);
                dz(1, ayz);
                dz(0, axz);
                din(2, 8, 0, azx);
                din(1, 8, 0, ayx);
                din(0, M_WX * 8, 1, axy);
                rq_lds<T, LANES>(p0, ax);
                rq_lds<T, LANES>(p0 + M_PLANE * 8, ay);
                rq_lds<T, LANES>(p0 + 2 * M_PLANE * 8, az);
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    const T bx = azy[i] - ayz[i] + a.bext[0];
                    const T by = axz[i] - azx[i] + a.bext[1];
                    const T bz = ayx[i] - axy[i] + a.bext[2];
                    const double u2 = (double)ux[i] * ux[i] + (double)uy[i] * uy[i] + (double)uz[i] * uz[i];
                    const double b2 = (double)bx * bx + (double)by * by + (double)bz * bz;
                    acc.su += u2;
                    acc.sb += b2;
                    acc.mu = fmax(acc.mu, u2);
                    acc.mb = fmax(acc.mb, b2);
                    acc.lmin = fmin(acc.lmin, (double)l[i]);
                    acc.lmax = fmax(acc.lmax, (double)l[i]);
                    // a non-finite ln rho or A would hide in fmin/fmax: fold it into the sums
                    const double chk = (double)l[i] + (double)ax[i] + (double)ay[i] + (double)az[i];
                    if (!isfinite(chk)) acc.su += chk;
                }
            }
            __syncwarp();
            if (lane == 0) m_bar_arrive(&done[it % RQ_NP]);
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
