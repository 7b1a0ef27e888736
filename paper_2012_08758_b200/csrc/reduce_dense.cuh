// S9 reductions of a DENSE state, for ac_reduce_dense_noalloc (include/ac_mhd.h): a variant of reduce_stage1_kernel
// (kernels.cuh) that needs no context, no ghost-padded copy of the state and no allocation.
//
// What it computes: sum and max of |u|^2 and of |B|^2 with B = curl A + B_ext (6th-order central first derivatives,
// PAPER.md:85, 119; reading G1), min and max of ln rho: the inputs of the rms / max diagnostics and of the CFL rule
// (reading G15).  Per cell the arithmetic is that of reduce_stage1_kernel, term by term and in its
// order (derivatives in the state's precision T, squares and sums in fp64), so the maxima equal the context path's
// bit for bit and the sums differ by summation order only.
//
// The periodic wrap is taken by index here: the state is the caller's dense [7][nz][ny][nx] array, no
// ghost zones.  A block takes RD_CELLS_PER_BLOCK consecutive cells and writes ONE partial; the partials are the
// kernel's scratch memory (a fixed array of the library, see ac_mhd.cu), folded by reduce_stage2_kernel in a fixed
// order: the result is deterministic.
#pragma once
#include <cuda_runtime.h>

#include "kernels.cuh"

namespace ac {

constexpr int RD_THREADS = 256;
constexpr int RD_CELLS_PER_THREAD = 8;
constexpr int RD_CELLS_PER_BLOCK = RD_THREADS * RD_CELLS_PER_THREAD;          // 2048
constexpr long long RD_MAX_CELLS = 1LL << 27;                                  // 512^3 (BASELINE config 4)
constexpr int RD_MAX_PARTIALS = (int)(RD_MAX_CELLS / RD_CELLS_PER_BLOCK);      // 65536 partials of 48 bytes: 3 MiB

template <typename T>
struct ReduceDenseArgs {
    const T* state;      // dense [7][nz][ny][nx], x fastest (the layout of ac_load_state)
    int nx, ny, nz;
    T c1[3][3];          // first-derivative weights per axis
    T bext[3];
};

// c1[0] (f(+1) - f(-1)) + c1[1] (f(+2) - f(-2)) + c1[2] (f(+3) - f(-3)) along one axis; ip / im = the element offsets
// of the wrapped neighbours at distance m = 1..3
template <typename T>
__device__ __forceinline__ T rd_der1(const T* __restrict__ f, const long long (&ip)[3], const long long (&im)[3],
                                     const T (&c1)[3]) {
    T v = c1[0] * (f[ip[0]] - f[im[0]]);
    v = fma_<T>(c1[1], f[ip[1]] - f[im[1]], v);
    return fma_<T>(c1[2], f[ip[2]] - f[im[2]], v);
}

template <typename T>
__global__ void __launch_bounds__(RD_THREADS) reduce_dense_stage1_kernel(const ReduceDenseArgs<T> a,
                                                                         RedVals* __restrict__ partial) {
    const long long ncell = (long long)a.nx * a.ny * a.nz;
    const long long row = a.nx, plane = (long long)a.nx * a.ny;
    const T* __restrict__ lnrho = a.state + LNRHO * ncell;
    const T* __restrict__ ux = a.state + UX * ncell;
    const T* __restrict__ uy = a.state + UY * ncell;
    const T* __restrict__ uz = a.state + UZ * ncell;
    const T* __restrict__ ax = a.state + AX * ncell;
    const T* __restrict__ ay = a.state + AY * ncell;
    const T* __restrict__ az = a.state + AZ * ncell;
    RedVals acc = red_identity();
#pragma unroll 1
    for (int j = 0; j < RD_CELLS_PER_THREAD; j++) {
        const long long i = (long long)blockIdx.x * RD_CELLS_PER_BLOCK + (long long)j * RD_THREADS + threadIdx.x;
        if (i >= ncell) break;
        const int x = (int)(i % a.nx), y = (int)((i / a.nx) % a.ny), z = (int)(i / plane);
        long long xp[3], xm[3], yp[3], ym[3], zp[3], zm[3];
#pragma unroll
        for (int m = 1; m <= 3; m++) {
            const int xa = x + m < a.nx ? x + m : x + m - a.nx, xb = x - m >= 0 ? x - m : x - m + a.nx;
            const int ya = y + m < a.ny ? y + m : y + m - a.ny, yb = y - m >= 0 ? y - m : y - m + a.ny;
            const int za = z + m < a.nz ? z + m : z + m - a.nz, zb = z - m >= 0 ? z - m : z - m + a.nz;
            xp[m - 1] = i + (xa - x);
            xm[m - 1] = i + (xb - x);
            yp[m - 1] = i + (ya - y) * row;
            ym[m - 1] = i + (yb - y) * row;
            zp[m - 1] = i + (za - z) * plane;
            zm[m - 1] = i + (zb - z) * plane;
        }
        // B = curl A + B_ext, in the order of reduce_stage1_kernel
        const T dyaz = rd_der1<T>(az, yp, ym, a.c1[1]);
        const T dxaz = rd_der1<T>(az, xp, xm, a.c1[0]);
        const T dxay = rd_der1<T>(ay, xp, xm, a.c1[0]);
        const T dyax = rd_der1<T>(ax, yp, ym, a.c1[1]);
        const T dzay = rd_der1<T>(ay, zp, zm, a.c1[2]);
        const T dzax = rd_der1<T>(ax, zp, zm, a.c1[2]);
        const T bx = dyaz - dzay + a.bext[0];
        const T by = dzax - dxaz + a.bext[1];
        const T bz = dxay - dyax + a.bext[2];
        const double b2 = (double)bx * bx + (double)by * by + (double)bz * bz;
        acc.sb += b2;
        acc.mb = fmax(acc.mb, b2);
        const T vx = ux[i], vy = uy[i], vz = uz[i], l = lnrho[i];
        const double u2 = (double)vx * vx + (double)vy * vy + (double)vz * vz;
        acc.su += u2;
        acc.mu = fmax(acc.mu, u2);
        acc.lmin = fmin(acc.lmin, (double)l);
        acc.lmax = fmax(acc.lmax, (double)l);
        // a non-finite ln rho or A would hide in fmin / fmax: fold it into the sums
        const double chk = (double)l + (double)ax[i] + (double)ay[i] + (double)az[i];
        if (!isfinite(chk)) acc.su += chk;
    }
    acc = block_reduce(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}

}  // namespace ac
