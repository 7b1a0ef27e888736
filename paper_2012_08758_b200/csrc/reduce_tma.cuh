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

// element arithmetic: E = double (one cell) or f2 (the two fp32 cells of a packed pair, add/sub/fma.rn.f32x2)
template <typename E>
__device__ __forceinline__ E rq_lds(const unsigned char* p) {
    return *(const E*)p;
}
template <typename E>
struct RqLanes;
template <>
struct RqLanes<double> {
    static constexpr int N = 1;
    __device__ static void get(double v, double (&o)[2]) { o[0] = v; o[1] = 0.0; }
};
template <>
struct RqLanes<f2> {
    static constexpr int N = 2;
    __device__ static void get(f2 v, double (&o)[2]) {
        float lo, hi;
        vunpack(v, lo, hi);
        o[0] = (double)lo;
        o[1] = (double)hi;
    }
};

// running extrema in the element's own precision: exact, and one FMNMX per lane instead of an fp64 compare-select
template <typename E>
struct RqExt;
template <>
struct RqExt<double> {
    double mu = 0.0, mb = 0.0, lmin = INFINITY, lmax = -INFINITY;
    __device__ void umax(double v) { mu = fmax(mu, v); }
    __device__ void bmax(double v) { mb = fmax(mb, v); }
    __device__ void lminmax(double v) {
        lmin = fmin(lmin, v);
        lmax = fmax(lmax, v);
    }
    __device__ void fold(RedVals& a) const {
        a.mu = fmax(a.mu, mu);
        a.mb = fmax(a.mb, mb);
        a.lmin = fmin(a.lmin, lmin);
        a.lmax = fmax(a.lmax, lmax);
    }
};
template <>
struct RqExt<f2> {
    float mu = 0.f, mb = 0.f, lmin = INFINITY, lmax = -INFINITY;
    __device__ void umax(f2 v) {
        float lo, hi;
        vunpack(v, lo, hi);
        mu = fmaxf(mu, fmaxf(lo, hi));
    }
    __device__ void bmax(f2 v) {
        float lo, hi;
        vunpack(v, lo, hi);
        mb = fmaxf(mb, fmaxf(lo, hi));
    }
    __device__ void lminmax(f2 v) {
        float lo, hi;
        vunpack(v, lo, hi);
        lmin = fminf(lmin, fminf(lo, hi));
        lmax = fmaxf(lmax, fmaxf(lo, hi));
    }
    __device__ void fold(RedVals& a) const {
        a.mu = fmax(a.mu, (double)mu);
        a.mb = fmax(a.mb, (double)mb);
        a.lmin = fmin(a.lmin, (double)lmin);
        a.lmax = fmax(a.lmax, (double)lmax);
    }
};

template <typename T, int LANES>
__global__ void __launch_bounds__(RQ_THREADS, 3)
    reduce_tma_kernel(const __grid_constant__ ReduceArgs<T> a, const __grid_constant__ CUtensorMap map_a,
                      const __grid_constant__ CUtensorMap map_p, int tiles_x, int tiles_y, int nchunks) {
    using E = typename ElemOf<T>::E;
    static_assert(ElemOf<T>::LANES == LANES, "double: 1 lane; float: packed pairs");
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
    RqExt<E> ext;
    const int tx = tid & (M_TX - 1), ty = tid >> 4;
    const int cell_off = ((ty + R) * M_WX + tx + M_HX) * 8;           // bytes
    E c1[3][3], bext[3];
#pragma unroll
    for (int ax = 0; ax < 3; ax++) {
        bext[ax] = Splat<E>::of((double)a.bext[ax]);
#pragma unroll
        for (int m = 0; m < 3; m++) c1[ax][m] = Splat<E>::of((double)a.c1[ax][m]);
    }
    long it = 0;
    for (long w = blockIdx.x; w < nwork; w += gridDim.x) {
        const int x = (int)(w % tiles_x) * M_TX + tx, y = (int)((w / tiles_x) % tiles_y) * M_TY + ty;
        const int zs = (int)(w / ((long)tiles_x * tiles_y)) * RQ_CZ;
        const int ze = min(zs + RQ_CZ, L.nz);
        const int niter = ze - zs + 2 * R;
        const bool valid = x < L.nx && y < L.ny;
        E hax[7], hay[7];                                             // A_x, A_y of planes p-6 .. p (this column)
        E pbx[4], pby[4], pbz[4];                                     // d_y A_z, d_x A_z, B_z of planes p-3 .. p
#pragma unroll
        for (int r = 0; r < 7; r++) hax[r] = hay[r] = vzero<E>();
#pragma unroll
        for (int r = 0; r < 4; r++) pbx[r] = pby[r] = pbz[r] = vzero<E>();
        // the plane loop is unrolled 7 x so that the 7-plane history of A_x, A_y is a rotating register file with
        // compile-time indices (no moves): plane k sits in slot k % 7, H(r) = plane k - 6 + r
#pragma unroll 1
        for (int k0 = 0; k0 < niter; k0 += 7) {
#pragma unroll
            for (int j = 0; j < 7; j++) {
                const int k = k0 + j;
                if (k >= niter) break;
#define RQ_H(arr, r) arr[(j + 1 + (r)) % 7]
                const int slot = (int)(it % RQ_NP);
#pragma unroll
                for (int r = 0; r < 3; r++) {
                    pbx[r] = pbx[r + 1];
                    pby[r] = pby[r + 1];
                    pbz[r] = pbz[r + 1];
                }
                m_bar_wait<0>(&full[slot], (uint32_t)((it / RQ_NP) & 1));
                const unsigned char* p0 = rq_smem + slot * RQ_SLOT_BYTES + cell_off;
                RQ_H(hax, 6) = rq_lds<E>(p0);
                RQ_H(hay, 6) = rq_lds<E>(p0 + M_PLANE * 8);
                if (k >= R && k < niter - R && valid) {
                    // the plane is one of the item's own: in-plane parts of B, and the pointwise fields
                    auto din = [&](int f, int stride, int axis) -> E {
                        const unsigned char* p = p0 + f * (M_PLANE * 8);
                        E r = vmul(c1[axis][0], vsub(rq_lds<E>(p + stride), rq_lds<E>(p - stride)));
                        r = vfma(c1[axis][1], vsub(rq_lds<E>(p + 2 * stride), rq_lds<E>(p - 2 * stride)), r);
                        r = vfma(c1[axis][2], vsub(rq_lds<E>(p + 3 * stride), rq_lds<E>(p - 3 * stride)), r);
                        return r;
                    };
                    pbx[3] = din(2, M_WX * 8, 1);
                    pby[3] = din(2, 8, 0);
                    pbz[3] = vadd(vsub(din(1, 8, 0), din(0, M_WX * 8, 1)), bext[2]);
                    const E az = rq_lds<E>(p0 + 2 * M_PLANE * 8);
                    const unsigned char* pp = rq_smem + RQ_OFF_P + slot * RQ_PSLOT_BYTES + tid * 8;
                    // |u|^2 in the element's own arithmetic (fp64, or packed fp32: the squares are rounded to fp32,
                    // reading G18); sums in fp64; extrema in the element's precision (exact) until the fold
                    const E vx = rq_lds<E>(pp + M_COLS * 8), vy = rq_lds<E>(pp + 2 * M_COLS * 8), vz = rq_lds<E>(pp + 3 * M_COLS * 8);
                    const E lr = rq_lds<E>(pp);
                    const E u2 = vfma(vz, vz, vfma(vy, vy, vmul(vx, vx)));
                    ext.umax(u2);
                    ext.lminmax(lr);
                    double u2d[2], chk[2];
                    RqLanes<E>::get(u2, u2d);
                    // a non-finite ln rho or A would hide in the extrema: fold it into the sums
                    RqLanes<E>::get(vadd(vadd(vadd(RQ_H(hax, 6), RQ_H(hay, 6)), az), lr), chk);
#pragma unroll
                    for (int i = 0; i < LANES; i++) {
                        acc.su += u2d[i];
                        if (!isfinite(chk[i])) acc.su += chk[i];
                    }
                }
                if (k >= 2 * R && valid) {                            // plane p - 3 has its 7-plane history: finish B there
                    E ayz = vmul(c1[2][0], vsub(RQ_H(hay, 4), RQ_H(hay, 2)));
                    ayz = vfma(c1[2][1], vsub(RQ_H(hay, 5), RQ_H(hay, 1)), ayz);
                    ayz = vfma(c1[2][2], vsub(RQ_H(hay, 6), RQ_H(hay, 0)), ayz);
                    E axz = vmul(c1[2][0], vsub(RQ_H(hax, 4), RQ_H(hax, 2)));
                    axz = vfma(c1[2][1], vsub(RQ_H(hax, 5), RQ_H(hax, 1)), axz);
                    axz = vfma(c1[2][2], vsub(RQ_H(hax, 6), RQ_H(hax, 0)), axz);
                    const E bx = vadd(vsub(pbx[0], ayz), bext[0]), by = vadd(vsub(axz, pby[0]), bext[1]), bz = pbz[0];
                    const E b2 = vfma(bz, bz, vfma(by, by, vmul(bx, bx)));
                    ext.bmax(b2);
                    double b2d[2];
                    RqLanes<E>::get(b2, b2d);
#pragma unroll
                    for (int i = 0; i < LANES; i++) acc.sb += b2d[i];
                }
                __syncwarp();
                if (lane == 0) m_bar_arrive(&done[slot]);
                it++;
#undef RQ_H
            }
        }
    }
    ext.fold(acc);
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
