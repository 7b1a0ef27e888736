// Extended diagnostics (NEXT-4): volume sums of the kinetic helicity omega.u and the current helicity j.B
// (Eq. 11; mu0 = rho0 = 1) and the largest squared Alfven speed |B|^2 / rho (the
// optional term of the CFL rule, G15), over the current state.  omega = curl u and B = curl A (+ B_ext) from the
// 6th-order first derivatives, j = grad div A - lap A from second and mixed derivatives (G2-G4) - the expressions
// of mhd_cell.cuh.  Called a few times per run, not per step: one thread per cell gathering its 7 x 37 .. 61
// neighbours through the read-only path from the ghost-padded arrays, sums in fp64, per-block partials folded by
// diag_ext_stage2_kernel in a fixed order (deterministic).
#pragma once
#include "kernels.cuh"
#include "mhd_cell.cuh"

namespace ac {

struct ExtVals {
    double hk, hc, va2;
};

template <typename T>
struct DiagExtArgs {
    const void* in[NFIELDS];
    Layout L;            // storage layout: L.nz = planes of storage elements
    Coeffs<T> c;
    T bext[3];
    int mixed_tensor;
    ExtVals* partial;
};

__device__ __forceinline__ ExtVals ext_block_reduce(ExtVals v) {
    __shared__ ExtVals warp_part[32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int lane = tid & 31, wid = tid >> 5;
    const int nwarps = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    auto fold = [](ExtVals& a) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            a.hk += __shfl_down_sync(0xffffffffu, a.hk, d);
            a.hc += __shfl_down_sync(0xffffffffu, a.hc, d);
            a.va2 = fmax(a.va2, __shfl_down_sync(0xffffffffu, a.va2, d));
        }
    };
    fold(v);
    if (lane == 0) warp_part[wid] = v;
    __syncthreads();
    if (wid == 0) {
        v = lane < nwarps ? warp_part[lane] : ExtVals{0.0, 0.0, 0.0};
        fold(v);
    }
    return v;
}

// LANES = 1: one cell per storage element; LANES = 2: packed fp32 pairs (z, z + nz/2), whose z ghost planes hold
// lane-swapped pairs, so that the same lane of the neighbouring element is always the neighbouring cell
template <typename T, int LANES>
__global__ void __launch_bounds__(256) diag_ext_kernel(const __grid_constant__ DiagExtArgs<T> a) {
    const Layout& L = a.L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z * blockDim.z + threadIdx.z;
    ExtVals acc = {0.0, 0.0, 0.0};
    if (x < L.nx && y < L.ny && z < L.nz) {
        const size_t c0 = L.idx(x, y, z);
        const long pitch = L.pitch, plane = (long)L.plane;
#pragma unroll
        for (int lane = 0; lane < LANES; lane++) {
            auto fetch = [&](int q, int dx, int dy, int dz) -> T {
                return __ldg((const T*)a.in[q] + ((c0 + dx + dy * pitch + dz * plane) * LANES + lane));
            };
            const T u[3] = {fetch(UX, 0, 0, 0), fetch(UY, 0, 0, 0), fetch(UZ, 0, 0, 0)};
            const T om0 = d1<T, 1>(fetch, a.c, UZ) - d1<T, 2>(fetch, a.c, UY);
            const T om1 = d1<T, 2>(fetch, a.c, UX) - d1<T, 0>(fetch, a.c, UZ);
            const T om2 = d1<T, 0>(fetch, a.c, UY) - d1<T, 1>(fetch, a.c, UX);
            const T b0 = d1<T, 1>(fetch, a.c, AZ) - d1<T, 2>(fetch, a.c, AY) + a.bext[0];
            const T b1 = d1<T, 2>(fetch, a.c, AX) - d1<T, 0>(fetch, a.c, AZ) + a.bext[1];
            const T b2 = d1<T, 0>(fetch, a.c, AY) - d1<T, 1>(fetch, a.c, AX) + a.bext[2];
            const bool mt = a.mixed_tensor != 0;
            T a2[3][3];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                const T ai = fetch(AX + i, 0, 0, 0);
                a2[i][0] = d2<T, 0>(fetch, a.c, AX + i, ai);
                a2[i][1] = d2<T, 1>(fetch, a.c, AX + i, ai);
                a2[i][2] = d2<T, 2>(fetch, a.c, AX + i, ai);
            }
            // j = grad div A - lap A: the diagonal second derivative cancels
            const T j0 = dmix<T, 0, 1>(fetch, a.c, AY, mt) + dmix<T, 0, 2>(fetch, a.c, AZ, mt) - a2[0][1] - a2[0][2];
            const T j1 = dmix<T, 0, 1>(fetch, a.c, AX, mt) + dmix<T, 1, 2>(fetch, a.c, AZ, mt) - a2[1][0] - a2[1][2];
            const T j2 = dmix<T, 0, 2>(fetch, a.c, AX, mt) + dmix<T, 1, 2>(fetch, a.c, AY, mt) - a2[2][0] - a2[2][1];
            acc.hk += (double)om0 * u[0] + (double)om1 * u[1] + (double)om2 * u[2];
            acc.hc += (double)j0 * b0 + (double)j1 * b1 + (double)j2 * b2;
            const double bb = (double)b0 * b0 + (double)b1 * b1 + (double)b2 * b2;
            const double va2 = bb * exp(-(double)fetch(LNRHO, 0, 0, 0));
            // fmax drops NaNs: a non-finite value shows up in the sums
            acc.va2 = fmax(acc.va2, va2);
            if (!isfinite(va2)) acc.hc += va2;
        }
    }
    acc = ext_block_reduce(acc);
    if (threadIdx.x + threadIdx.y + threadIdx.z == 0)
        a.partial[blockIdx.x + gridDim.x * (blockIdx.y + (size_t)gridDim.y * blockIdx.z)] = acc;
}

// one block folds the per-block partials in a fixed order
__global__ void __launch_bounds__(256) diag_ext_stage2_kernel(const ExtVals* __restrict__ partial, long n,
                                                              ExtVals* __restrict__ result) {
    ExtVals acc = {0.0, 0.0, 0.0};
    for (long i = threadIdx.x; i < n; i += blockDim.x) {
        acc.hk += partial[i].hk;
        acc.hc += partial[i].hc;
        acc.va2 = fmax(acc.va2, partial[i].va2);
    }
    acc = ext_block_reduce(acc);
    if (threadIdx.x == 0) *result = acc;
}

}  // namespace ac
