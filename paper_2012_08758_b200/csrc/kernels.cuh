// CUDA kernels of the hot path: state pack/unpack, forcing tables, the fused RK substep
// (variant "direct": one thread per cell, neighbours through the read-only global path) and the
// two-stage reductions.  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "layout.cuh"
#include "mhd_cell.cuh"

namespace ac {

// ------------------------------------------------------------------------------------------------
// dense <-> padded copies (S1: periodic halo = "local boundary transfer")
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void pack_kernel(const T* __restrict__ dense, T* __restrict__ padded, Layout L) {
    // one thread per padded element that matters: x in [-R, nx+R), y in [-R, ny+R), z in [-R, nz+R)
    const int px = blockIdx.x * blockDim.x + threadIdx.x - R;
    const int py = blockIdx.y * blockDim.y + threadIdx.y - R;
    const int pz = blockIdx.z - R;
    if (px >= L.nx + R || py >= L.ny + R) return;
    int sx = px < 0 ? px + L.nx : (px >= L.nx ? px - L.nx : px);
    int sy = py < 0 ? py + L.ny : (py >= L.ny ? py - L.ny : py);
    int sz = pz < 0 ? pz + L.nz : (pz >= L.nz ? pz - L.nz : pz);
    padded[L.idx(px, py, pz)] = dense[(size_t)sx + (size_t)L.nx * ((size_t)sy + (size_t)L.ny * (size_t)sz)];
}

template <typename T>
__global__ void unpack_kernel(const T* __restrict__ padded, T* __restrict__ dense, Layout L) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    dense[(size_t)x + (size_t)L.nx * ((size_t)y + (size_t)L.ny * (size_t)z)] = padded[L.idx(x, y, z)];
}

// packed fp32 pairs (vec2.cuh): element (x, y, zp) = (cell z = zp, cell z = zp + nz/2); L is the layout in
// 8-byte elements with L.nz = nz/2 planes.  Ghost planes come out lane-swapped by construction.
__global__ void pack_pairs_kernel(const float* __restrict__ dense, float2* __restrict__ padded, Layout L, int nz_full) {
    const int px = blockIdx.x * blockDim.x + threadIdx.x - R;
    const int py = blockIdx.y * blockDim.y + threadIdx.y - R;
    const int pz = blockIdx.z - R;
    if (px >= L.nx + R || py >= L.ny + R) return;
    int sx = px < 0 ? px + L.nx : (px >= L.nx ? px - L.nx : px);
    int sy = py < 0 ? py + L.ny : (py >= L.ny ? py - L.ny : py);
    int z0 = pz, z1 = pz + L.nz;
    z0 = z0 < 0 ? z0 + nz_full : (z0 >= nz_full ? z0 - nz_full : z0);
    z1 = z1 < 0 ? z1 + nz_full : (z1 >= nz_full ? z1 - nz_full : z1);
    const size_t row = (size_t)sx + (size_t)L.nx * (size_t)sy;
    const size_t plane = (size_t)L.nx * L.ny;
    padded[L.idx(px, py, pz)] = make_float2(dense[row + plane * z0], dense[row + plane * z1]);
}

__global__ void unpack_pairs_kernel(const float2* __restrict__ padded, float* __restrict__ dense, Layout L) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const float2 v = padded[L.idx(x, y, z)];
    const size_t row = (size_t)x + (size_t)L.nx * (size_t)y;
    const size_t plane = (size_t)L.nx * L.ny;
    dense[row + plane * z] = v.x;
    dense[row + plane * (z + L.nz)] = v.y;
}

// ------------------------------------------------------------------------------------------------
// z-slab halo (NEXT-3): the 3 bottom and 3 top planes of CELLS of every field (x / y ghost zones
// included) to and from dense buffers [7][3][my * pitch] of T.  LANES = 2: packed fp32 pairs (z, z + nz/2): the
// bottom cells are lane 0 of planes 0..2, the top cells lane 1 of planes nzp-3..nzp-1; of a ghost plane only the
// lane that belongs to the neighbour is written (the other lane is the slab's own cell, kept current by the
// ghost-zone pass).
// ------------------------------------------------------------------------------------------------
template <typename T, int LANES>
__global__ void halo_pack_kernel(const void* __restrict__ state, size_t field_elems, Layout L, T* __restrict__ lo,
                                 T* __restrict__ hi) {
    const size_t per_field = (size_t)R * L.plane;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per_field) return;
    const int q = blockIdx.y;
    const T* f = (const T*)state + (size_t)q * field_elems * LANES;
    // padded plane R + j holds cell plane j
    lo[q * per_field + i] = f[((size_t)R * L.plane + i) * LANES];
    hi[q * per_field + i] = f[((size_t)L.nz * L.plane + i) * LANES + (LANES - 1)];
}
template <typename T, int LANES>
__global__ void halo_unpack_kernel(void* __restrict__ state, size_t field_elems, Layout L, const T* __restrict__ lo,
                                   const T* __restrict__ hi) {
    const size_t per_field = (size_t)R * L.plane;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per_field) return;
    const int q = blockIdx.y;
    T* f = (T*)state + (size_t)q * field_elems * LANES;
    f[i * LANES] = lo[q * per_field + i];                                                   // ghost planes below
    f[((size_t)(L.nz + R) * L.plane + i) * LANES + (LANES - 1)] = hi[q * per_field + i];  // ghost planes above
}

// The same exchange as ONE kernel over peer memory: the ghost planes are pulled straight from the neighbours' state
// arrays (device pointers of the same GPU, or peer-mapped pointers of another GPU: NVLink loads), no staging buffers,
// no library collective.  below / above = the neighbours' buffers that hold THEIR current state, same layout as ours.
template <typename T, int LANES>
__global__ void halo_pull_kernel(void* __restrict__ state, const void* __restrict__ below, const void* __restrict__ above,
                                 size_t field_elems, Layout L) {
    const size_t per_field = (size_t)R * L.plane;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per_field) return;
    const int q = blockIdx.y;
    T* f = (T*)state + (size_t)q * field_elems * LANES;
    const T* fb = (const T*)below + (size_t)q * field_elems * LANES;
    const T* fa = (const T*)above + (size_t)q * field_elems * LANES;
    // ghost planes below <- the top cell planes of the slab below; ghost planes above <- the bottom cell planes of the one above
    f[i * LANES] = fb[((size_t)L.nz * L.plane + i) * LANES + (LANES - 1)];
    f[((size_t)(L.nz + R) * L.plane + i) * LANES + (LANES - 1)] = fa[((size_t)R * L.plane + i) * LANES];
}

// ------------------------------------------------------------------------------------------------
// forcing tables (S7): cos/sin of k_a x_a per axis, phase folded into the z table.
// layout: [cx(nx) sx(nx) cy(ny) sy(ny) cz(nz) sz(nz)]
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void forcing_tables_kernel(T* __restrict__ tab, int nx, int ny, int nz, double kx, double ky, double kz,
                                      double hx, double hy, double hz, double phase) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nx + ny + nz) return;
    double th;
    T *pc, *ps;
    if (i < nx) {
        th = kx * (i * hx);
        pc = tab + i;
        ps = tab + nx + i;
    } else if (i < nx + ny) {
        int j = i - nx;
        th = ky * (j * hy);
        pc = tab + 2 * nx + j;
        ps = tab + 2 * nx + ny + j;
    } else {
        int j = i - nx - ny;
        th = kz * (j * hz) + phase;
        pc = tab + 2 * nx + 2 * ny + j;
        ps = tab + 2 * nx + 2 * ny + nz + j;
    }
    double s, c;
    sincos(th, &s, &c);
    *pc = (T)c;
    *ps = (T)s;
}

template <typename T>
__device__ __forceinline__ void forcing_phase(const T* __restrict__ tab, int nx, int ny, int nz, int x, int y, int z,
                                              T& fc, T& fs) {
    const T cx = __ldg(tab + x), sx = __ldg(tab + nx + x);
    const T cy = __ldg(tab + 2 * nx + y), sy = __ldg(tab + 2 * nx + ny + y);
    const T cz = __ldg(tab + 2 * nx + 2 * ny + z), sz = __ldg(tab + 2 * nx + 2 * ny + nz + z);
    const T cxy = cx * cy - sx * sy, sxy = sx * cy + cx * sy;
    fc = cxy * cz - sxy * sz;
    fs = sxy * cz + cxy * sz;
}

// ------------------------------------------------------------------------------------------------
// fused substep, common argument block
// ------------------------------------------------------------------------------------------------
template <typename T>
struct SubstepArgs {
    const T* in[NFIELDS];
    T* out[NFIELDS];
    const T* ftab;
    Layout L;
    Coeffs<T> c;
    Physics<T> p;
    int z_begin, z_end;   // planes updated by this launch
};

// write a new interior value and its periodic images in the ghost layers (S1 fused into S8)
template <typename T>
__device__ __forceinline__ void store_with_images(T* __restrict__ o, const Layout& L, int x, int y, int z, T v,
                                                  bool edge) {
    o[L.idx(x, y, z)] = v;
    if (!edge) return;
    int xs[2] = {x, x}, ys[2] = {y, y}, zs[2] = {z, z};
    int cx = 1, cy = 1, cz = 1;
    if (x < R) xs[cx++] = x + L.nx; else if (x >= L.nx - R) xs[cx++] = x - L.nx;
    if (y < R) ys[cy++] = y + L.ny; else if (y >= L.ny - R) ys[cy++] = y - L.ny;
    if (z < R) zs[cz++] = z + L.nz; else if (z >= L.nz - R) zs[cz++] = z - L.nz;
    for (int k = 0; k < cz; k++)
        for (int j = 0; j < cy; j++)
            for (int i = 0; i < cx; i++)
                if (i + j + k) o[L.idx(xs[i], ys[j], zs[k])] = v;
}

// Variant "direct": one thread per cell, every stencil point fetched through the read-only
// global/L1 path from the ghost-padded arrays.  Simple and obviously right; kept as the
// debugging / cross-check variant (ac_set_variant(ctx, 1)).
template <typename T>
__global__ void __launch_bounds__(256) substep_direct_kernel(const __grid_constant__ SubstepArgs<T> a) {
    const Layout& L = a.L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = a.z_begin + blockIdx.z * blockDim.z + threadIdx.z;
    if (x >= L.nx || y >= L.ny || z >= a.z_end) return;
    const size_t c0 = L.idx(x, y, z);
    const long pitch = L.pitch;
    const long plane = (long)L.plane;
    auto fetch = [&](int q, int dx, int dy, int dz) -> T {
        return __ldg(a.in[q] + (c0 + dx + dy * pitch + dz * plane));
    };
    T prev[NFIELDS];
#pragma unroll
    for (int q = 0; q < NFIELDS; q++) prev[q] = (a.p.substep != 0) ? a.out[q][c0] : T(0);
    T fc = T(0), fs = T(0);
    if (a.p.has_forcing) forcing_phase<T>(a.ftab, L.nx, L.ny, L.nz, x, y, z, fc, fs);
    T res[NFIELDS];
    substep_cell<T>(fetch, a.c, a.p, prev, fc, fs, res);
    const bool edge = (x < R) | (x >= L.nx - R) | (y < R) | (y >= L.ny - R) | (z < R) | (z >= L.nz - R);
#pragma unroll
    for (int q = 0; q < NFIELDS; q++) store_with_images<T>(a.out[q], L, x, y, z, res[q], edge);
}

// ------------------------------------------------------------------------------------------------
// reductions (S9): sum and max of |u|^2 and |B|^2, min/max of ln rho.  Two stages, fixed order.
// ------------------------------------------------------------------------------------------------
struct RedVals {
    double su, mu, sb, mb, lmin, lmax;
};

__device__ __forceinline__ RedVals red_combine(const RedVals& a, const RedVals& b) {
    RedVals r;
    r.su = a.su + b.su;
    r.sb = a.sb + b.sb;
    r.mu = fmax(a.mu, b.mu);
    r.mb = fmax(a.mb, b.mb);
    r.lmin = fmin(a.lmin, b.lmin);
    r.lmax = fmax(a.lmax, b.lmax);
    return r;
}

__device__ __forceinline__ RedVals red_shfl_down(const RedVals& v, int d) {
    RedVals r;
    r.su = __shfl_down_sync(0xffffffffu, v.su, d);
    r.mu = __shfl_down_sync(0xffffffffu, v.mu, d);
    r.sb = __shfl_down_sync(0xffffffffu, v.sb, d);
    r.mb = __shfl_down_sync(0xffffffffu, v.mb, d);
    r.lmin = __shfl_down_sync(0xffffffffu, v.lmin, d);
    r.lmax = __shfl_down_sync(0xffffffffu, v.lmax, d);
    return r;
}

// NaN-propagating identity: fmax/fmin drop NaNs, so non-finite input is tracked through the sums
__device__ __forceinline__ RedVals red_identity() {
    RedVals r;
    r.su = 0.0;
    r.sb = 0.0;
    r.mu = 0.0;
    r.mb = 0.0;
    r.lmin = INFINITY;
    r.lmax = -INFINITY;
    return r;
}

__device__ __forceinline__ RedVals block_reduce(RedVals v) {
    __shared__ RedVals warp_part[32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int lane = tid & 31, wid = tid >> 5;
    const int nwarps = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = red_combine(v, red_shfl_down(v, d));
    if (lane == 0) warp_part[wid] = v;
    __syncthreads();
    if (wid == 0) {
        v = lane < nwarps ? warp_part[lane] : red_identity();
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v = red_combine(v, red_shfl_down(v, d));
    }
    return v;  // valid in thread 0
}

template <typename T>
struct ReduceArgs {
    const void* in[NFIELDS];   // T elements, or float2 pairs when LANES == 2
    Layout L;                  // layout in storage elements
    T c1[3][3];
    T bext[3];
    RedVals* partial;
};

template <typename T, int LANES>
__device__ __forceinline__ void red_load(const void* base, size_t i, T (&v)[LANES]) {
    if (LANES == 1) {
        v[0] = ((const T*)base)[i];
    } else {
        const float2 t = ((const float2*)base)[i];
        v[0] = (T)t.x;
        v[LANES - 1] = (T)t.y;
    }
}

// stage 1: a block of 32 x 8 threads takes (x, y) tiles of one z chunk at a time (fixed round-robin
// assignment, so the result is deterministic) and marches along z.  Per cell it loads the 7 centre
// values and the 24 in-plane neighbours that curl A needs (d_x, d_y of A_z, d_x A_y, d_y A_x), all
// from the plane it is visiting, so the neighbour loads hit the lines its own block has just
// brought into L1.  The z derivatives of A_x, A_y come from a 7-plane history and the in-plane
// parts of B wait 3 planes; both live in thread-private columns of shared memory (ring-indexed, no
// barrier: a thread only reads what it wrote) so that the registers stay free for the 31 loads in
// flight.  31 loads per cell instead of 43.  One partial per block.
// LANES = 2: packed fp32 pairs (ghost planes hold lane-swapped pairs, so the history needs no care).
constexpr int RED_TX = 32, RED_TY = 8, RED_THREADS = RED_TX * RED_TY, RED_CZ = 32;
template <typename T, int LANES>
constexpr int red_smem_bytes() {
    return (2 * 7 + 3 * 4) * RED_THREADS * LANES * (int)sizeof(T);
}
template <typename T, int LANES>
__global__ void __launch_bounds__(RED_THREADS, 2) reduce_stage1_kernel(const __grid_constant__ ReduceArgs<T> a, int tiles_x,
                                                                       int tiles_y, int nchunks) {
    extern __shared__ __align__(16) unsigned char red_smem[];
    typedef T Col[RED_THREADS][LANES];
    Col* hax = (Col*)red_smem;          // [7]  A_x of planes p-6 .. p, slot = plane mod 7
    Col* hay = hax + 7;                 // [7]
    Col* pbx = hay + 7;                 // [4]  d_y A_z of planes p-3 .. p, slot = plane mod 4
    Col* pby = pbx + 4;                 // [4]  d_x A_z
    Col* pbz = pby + 4;                 // [4]  B_z
    const Layout& L = a.L;
    RedVals acc = red_identity();
    const long pitch = L.pitch, plane = (long)L.plane;
    const long nwork = (long)tiles_x * tiles_y * nchunks;
    const int tid = threadIdx.x;
    const int tx = tid & (RED_TX - 1), ty = tid / RED_TX;
    for (long w = blockIdx.x; w < nwork; w += gridDim.x) {
        const int x = (int)(w % tiles_x) * RED_TX + tx;
        const int y = (int)((w / tiles_x) % tiles_y) * RED_TY + ty;
        const int zs = (int)(w / ((long)tiles_x * tiles_y)) * RED_CZ;
        const int ze = min(zs + RED_CZ, L.nz);
        if (x >= L.nx || y >= L.ny) continue;
        size_t c0 = L.idx(x, y, zs - R);
        int s7 = 0, s4 = 0;                                  // ring slots of the plane being visited
#pragma unroll 1
        for (int p = zs - R; p < ze + R; p++, c0 += plane) {
            T vax[LANES], vay[LANES];
            red_load<T, LANES>(a.in[AX], c0, vax);
            red_load<T, LANES>(a.in[AY], c0, vay);
            if (p >= zs && p < ze) {
                T ux[LANES], uy[LANES], uz[LANES], l[LANES], az[LANES];
                T n[4][6][LANES];                            // the 24 in-plane neighbours
                red_load<T, LANES>(a.in[UX], c0, ux);
                red_load<T, LANES>(a.in[UY], c0, uy);
                red_load<T, LANES>(a.in[UZ], c0, uz);
                red_load<T, LANES>(a.in[LNRHO], c0, l);
                red_load<T, LANES>(a.in[AZ], c0, az);
                const int fq[4] = {AZ, AZ, AY, AX};
                const long fs[4] = {pitch, 1, 1, pitch};
#pragma unroll
                for (int k = 0; k < 4; k++)
#pragma unroll
                    for (int m = 1; m <= 3; m++) {
                        red_load<T, LANES>(a.in[fq[k]], c0 + m * fs[k], n[k][2 * (m - 1)]);
                        red_load<T, LANES>(a.in[fq[k]], c0 - m * fs[k], n[k][2 * (m - 1) + 1]);
                    }
                const int fa[4] = {1, 0, 0, 1};              // axis of the derivative
                T dd[4][LANES];                              // d_y A_z, d_x A_z, d_x A_y, d_y A_x
#pragma unroll
                for (int k = 0; k < 4; k++)
#pragma unroll
                    for (int i = 0; i < LANES; i++) {
                        T v = a.c1[fa[k]][0] * (n[k][0][i] - n[k][1][i]);
                        v = fma_<T>(a.c1[fa[k]][1], n[k][2][i] - n[k][3][i], v);
                        dd[k][i] = fma_<T>(a.c1[fa[k]][2], n[k][4][i] - n[k][5][i], v);
                    }
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    pbx[s4][tid][i] = dd[0][i];
                    pby[s4][tid][i] = dd[1][i];
                    pbz[s4][tid][i] = dd[2][i] - dd[3][i] + a.bext[2];
                    const double u2 = (double)ux[i] * ux[i] + (double)uy[i] * uy[i] + (double)uz[i] * uz[i];
                    acc.su += u2;
                    acc.mu = fmax(acc.mu, u2);
                    acc.lmin = fmin(acc.lmin, (double)l[i]);
                    acc.lmax = fmax(acc.lmax, (double)l[i]);
                    // a non-finite ln rho or A would hide in fmin/fmax: fold it into the sums
                    const double chk = (double)l[i] + (double)vax[i] + (double)vay[i] + (double)az[i];
                    if (!isfinite(chk)) acc.su += chk;
                }
            }
#pragma unroll
            for (int i = 0; i < LANES; i++) {
                hax[s7][tid][i] = vax[i];
                hay[s7][tid][i] = vay[i];
            }
            if (p - R >= zs) {                               // plane p - 3 has its 7-plane history: finish B there
                // slot of plane p - j is (s7 - j) mod 7; plane p - 3 + m  <->  j = 3 - m
                auto slot7 = [&](int j) { const int t = s7 - j; return t < 0 ? t + 7 : t; };
                const int q4 = (s4 + 1) & 3;                 // slot of plane p - 3 in the 4-ring
#pragma unroll
                for (int i = 0; i < LANES; i++) {
                    T ayz = a.c1[2][0] * (hay[slot7(2)][tid][i] - hay[slot7(4)][tid][i]);
                    ayz = fma_<T>(a.c1[2][1], hay[slot7(1)][tid][i] - hay[slot7(5)][tid][i], ayz);
                    ayz = fma_<T>(a.c1[2][2], vay[i] - hay[slot7(6)][tid][i], ayz);
                    T axz = a.c1[2][0] * (hax[slot7(2)][tid][i] - hax[slot7(4)][tid][i]);
                    axz = fma_<T>(a.c1[2][1], hax[slot7(1)][tid][i] - hax[slot7(5)][tid][i], axz);
                    axz = fma_<T>(a.c1[2][2], vax[i] - hax[slot7(6)][tid][i], axz);
                    const T bx = pbx[q4][tid][i] - ayz + a.bext[0];
                    const T by = axz - pby[q4][tid][i] + a.bext[1];
                    const T bz = pbz[q4][tid][i];
                    const double b2 = (double)bx * bx + (double)by * by + (double)bz * bz;
                    acc.sb += b2;
                    acc.mb = fmax(acc.mb, b2);
                }
            }
            s7 = s7 == 6 ? 0 : s7 + 1;
            s4 = (s4 + 1) & 3;
        }
    }
    acc = block_reduce(acc);
    if (threadIdx.x == 0) a.partial[blockIdx.x] = acc;
}

// stage 2: one block folds the per-block partials in a fixed order
__global__ void __launch_bounds__(256) reduce_stage2_kernel(const RedVals* __restrict__ partial, int n,
                                                            RedVals* __restrict__ result) {
    RedVals acc = red_identity();
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc = red_combine(acc, partial[i]);
    acc = block_reduce(acc);
    if (threadIdx.x == 0) *result = acc;
}

}  // namespace ac
