// Host side of the C ABI declared in include/ac_mhd.h.  Argument checks, memory carving, kernel
// launches, the Eq. 4-6 host helpers.  No torch, no exceptions across the boundary.
#include "../../include/ac_mhd.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>
#include <vector>

#include "diag_ext.cuh"
#include "kernels.cuh"
#include "layout.cuh"
#include "mhd_cell.cuh"
#include "reduce_dense.cuh"
#include "reduce_tma.cuh"
#include "substep_march.cuh"
#include "substep_pair.cuh"
#include "vec2.cuh"

namespace {

thread_local char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "CUDA error in %s: %s", what, cudaGetErrorString(e));
    return AC_ECUDA;
}

#define AC_CUDA(call)                                        \
    do {                                                     \
        cudaError_t e__ = (call);                            \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

// stencil weights (G1, G2) and RK coefficients (G7)
const double W1[3] = {3.0 / 4.0, -3.0 / 20.0, 1.0 / 60.0};
const double W2_0 = -49.0 / 18.0;
const double W2[3] = {3.0 / 2.0, -3.0 / 20.0, 1.0 / 90.0};
const double WM[3] = {3.0 / 8.0, -3.0 / 80.0, 1.0 / 360.0};
// upwind correction of the continuity equation (G17): delta6 / 60, weights of f(0) and f(+m) + f(-m)
const double W6_0 = -20.0 / 60.0;
const double W6[3] = {15.0 / 60.0, -6.0 / 60.0, 1.0 / 60.0};
const double RK_ALPHA[3] = {0.0, -5.0 / 9.0, -153.0 / 128.0};
const double RK_BETA[3] = {1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0};

const int RED_BLOCKS = 148 * 8;   // capacity of the partial-result scratch (stage-1 grids are sized from the device's SM count, capped here)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool grid_ok(const ac_grid* g) {
    if (!g) return false;
    if (g->nx < 8 || g->ny < 8 || g->nz < 8) return false;
    if (g->nx % 4 != 0) return false;
    if (!(g->lx > 0.0) || !(g->ly > 0.0) || !(g->lz > 0.0)) return false;
    if (!std::isfinite(g->lx) || !std::isfinite(g->ly) || !std::isfinite(g->lz)) return false;
    return true;
}

size_t elem_size(ac_dtype d) { return d == AC_F64 ? 8 : 4; }

struct Carve {
    size_t field_bytes, ftab_off, partial_off, result_off, total;
};

// es = bytes per storage element (8: fp64 cells or packed fp32 pairs; 4: plain fp32 cells);
// es_tab = bytes per forcing-table entry (the context's dtype)
Carve carve(const ac::Layout& L, size_t es, size_t es_tab, int nz_full) {
    Carve c;
    c.field_bytes = L.field * es;
    size_t off = 2 * AC_NFIELDS * c.field_bytes;
    c.ftab_off = off;
    off += align_up((size_t)2 * (L.nx + L.ny + nz_full) * es_tab, 256);
    c.partial_off = off;
    off += align_up(sizeof(ac::RedVals) * RED_BLOCKS, 256);
    c.result_off = off;
    off += 256;
    c.total = off;
    return c;
}

// The two device layouts a context can use:
//   march  - 8-byte elements: fp64 cells, or fp32 cells packed in (z, z + nz/2) pairs (needs nz even)
//   plain  - fp32 cells, 4-byte elements (direct variant, or odd nz)
bool can_pack(const ac_grid* g) { return g->nz % 2 == 0; }
ac::Layout layout_for(const ac_grid* g, ac_dtype d, bool packed) {
    if (d == AC_F64) return ac::make_layout(g->nx, g->ny, g->nz, 8);
    if (packed) return ac::make_layout(g->nx, g->ny, g->nz / 2, 8);
    return ac::make_layout(g->nx, g->ny, g->nz, 4);
}
size_t store_elem_size(ac_dtype d, bool packed) { return (d == AC_F64 || packed) ? 8 : 4; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// 4-D map (x, y, z, field) over one ghost-padded state buffer of 8-byte elements; box = (wx, wy, 1, 7).
// Boxes must start 16-byte aligned in global memory (an 8-byte-aligned start faults on B200).
int make_state_map(CUtensorMap* map, void* base, const ac::Layout& L, int wx, int wy, int nfields = AC_NFIELDS) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled not available from the driver");
        return AC_ECUDA;
    }
    const size_t es = 8;
    cuuint64_t dims[4] = {(cuuint64_t)L.pitch, (cuuint64_t)L.my, (cuuint64_t)L.mz, (cuuint64_t)nfields};
    cuuint64_t strides[3] = {(cuuint64_t)L.pitch * es, (cuuint64_t)L.plane * es, (cuuint64_t)L.field * es};
    cuuint32_t box[4] = {(cuuint32_t)wx, (cuuint32_t)wy, 1u, (cuuint32_t)nfields};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return AC_ECUDA;
    }
    return AC_OK;
}

}  // namespace

struct ac_ctx {
    ac_grid grid;
    ac_dtype dtype;
    double nu, eta, cs, k_f, helicity;
    double bext[3];
    double c_u, c_nu;
    int upwind;          // 1 = upwinded continuity equation (G17); default 0
    int forcing_kick;    // 1 = alternative reading of G8: one impulse u += dt f per step, applied with substep 2; default 0
    int mixed;           // 0 = bidiagonal mixed stencil (G2, default), 1 = tensor product (pair-march MIX build, direct kernel)
    int variant;         // requested: 0 = pair-march (default), 1 = direct, 2 = scatter-march (one cell per thread)
    bool march;          // the kernel actually used (fp32 with odd nz falls back to direct)
    bool packed;         // fp32 cells stored as (z, z + nz/2) pairs
    ac::Layout L;        // layout in storage elements
    Carve cv;
    char* ws;
    bool owns_ws;
    cudaStream_t stream;
    int cur;  // which of the two state buffers holds the current state
    bool loaded;
    unsigned loaded_mask;  // fields written since the last ac_load_state / configure (ac_load_field)
    long long launches;
    ac::RedVals* host_result;  // pinned
    CUtensorMap map_in[2];     // TMA maps of the two state buffers: tile + halo boxes
    CUtensorMap map_prev[2];   // and interior-tile boxes (previous state of the 2N update)
    CUtensorMap map_a[2];      // tile + halo boxes of the three A fields (reductions)
    CUtensorMap map_p[2];      // interior-tile boxes of ln rho and u (reductions)
    CUtensorMap map_qin[2];    // pair-march kernel: 16 x 16 tile + halo boxes
    CUtensorMap map_qprev[2];  // and interior-tile boxes
    int cz, nchunks;           // z chunking of the march kernel
    int device, sms;           // CUDA device ordinal of the context and its SM count
    bool slab;                 // a z slab of a larger box (ac_set_slab): neighbours own the z ghost planes
    int z0_plane, nz_global;   // index of the slab's first plane in the global grid, planes of the global grid
    int inner_done;            // substep whose inner part has been launched (-1: none)
    int next_substep;          // 0 between full steps; 1, 2 inside a step driven by ac_substep (the idle buffer is live then)

    void* field_ptr(int buf, int q) const { return ws + ((size_t)buf * AC_NFIELDS + q) * cv.field_bytes; }
};

namespace {

// makes the context's device current for the duration of a call (a context may be used while another device is current)
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const ac_ctx* ctx) {
        if (ctx && cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) switched = cudaSetDevice(ctx->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

template <typename T>
void fill_coeffs(const ac_ctx* ctx, ac::Coeffs<T>& c) {
    const double h[3] = {ctx->grid.lx / ctx->grid.nx, ctx->grid.ly / ctx->grid.ny, ctx->grid.lz / ctx->grid.nz};
    for (int a = 0; a < 3; a++) {
        for (int m = 0; m < 3; m++) {
            c.c1[a][m] = (T)(W1[m] / h[a]);
            c.c2[a][m] = (T)(W2[m] / (h[a] * h[a]));
        }
        c.c20[a] = (T)(W2_0 / (h[a] * h[a]));
        c.c60[a] = (T)(W6_0 / h[a]);
        for (int m = 0; m < 3; m++) c.c6[a][m] = (T)(W6[m] / h[a]);
    }
    const int pa[3] = {0, 0, 1}, pb[3] = {1, 2, 2};
    for (int p = 0; p < 3; p++)
        for (int m = 0; m < 3; m++) c.cm[p][m] = (T)(WM[m] / (h[pa[p]] * h[pb[p]]));
}

// one field: dense caller layout -> padded device layout of state buffer `buf` (ghost zones by periodic wrap)
template <typename T>
int load_field_t(ac_ctx* ctx, int buf, int q, const void* field, int src_on_device) {
    const ac::Layout& L = ctx->L;
    const ac_grid& g = ctx->grid;
    const size_t dense_bytes = (size_t)g.nx * g.ny * g.nz * sizeof(T);
    dim3 blk(64, 4, 1);
    dim3 grd((L.nx + 2 * ac::R + blk.x - 1) / blk.x, (L.ny + 2 * ac::R + blk.y - 1) / blk.y, L.nz + 2 * ac::R);
    const T* src;
    if (src_on_device) {
        src = (const T*)field;
    } else {
        // stage the dense field in the other state buffer, whose contents are dead between steps
        T* stage = (T*)ctx->field_ptr(1 - buf, q);
        AC_CUDA(cudaMemcpyAsync(stage, field, dense_bytes, cudaMemcpyHostToDevice, ctx->stream));
        src = stage;
    }
    if (ctx->packed)
        ac::pack_pairs_kernel<<<grd, blk, 0, ctx->stream>>>((const float*)src, (float2*)ctx->field_ptr(buf, q), L, g.nz);
    else
        ac::pack_kernel<T><<<grd, blk, 0, ctx->stream>>>(src, (T*)ctx->field_ptr(buf, q), L);
    ctx->launches++;
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

template <typename T>
int store_field_t(ac_ctx* ctx, int q, void* field, int dst_on_device) {
    const ac::Layout& L = ctx->L;
    const ac_grid& g = ctx->grid;
    const size_t dense_bytes = (size_t)g.nx * g.ny * g.nz * sizeof(T);
    dim3 blk(64, 4, 1);
    dim3 grd((L.nx + blk.x - 1) / blk.x, (L.ny + blk.y - 1) / blk.y, L.nz);
    T* dst = dst_on_device ? (T*)field : (T*)ctx->field_ptr(1 - ctx->cur, q);
    if (ctx->packed)
        ac::unpack_pairs_kernel<<<grd, blk, 0, ctx->stream>>>((const float2*)ctx->field_ptr(ctx->cur, q), (float*)dst, L);
    else
        ac::unpack_kernel<T><<<grd, blk, 0, ctx->stream>>>((const T*)ctx->field_ptr(ctx->cur, q), dst, L);
    ctx->launches++;
    if (!dst_on_device) AC_CUDA(cudaMemcpyAsync(field, dst, dense_bytes, cudaMemcpyDeviceToHost, ctx->stream));
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

// weights of the scatter-march kernel (substep_march.cuh), computed in fp64 and rounded once
template <typename E>
void fill_march_coef(const ac_ctx* ctx, ac::MarchCoef<E>& c, double dt, int s, const ac_forcing* forcing) {
    using S = ac::Splat<E>;
    const double h[3] = {ctx->grid.lx / ctx->grid.nx, ctx->grid.ly / ctx->grid.ny, ctx->grid.lz / ctx->grid.nz};
    double c1[3][3], c2[3][3], c20[3];
    for (int a = 0; a < 3; a++) {
        for (int m = 0; m < 3; m++) {
            c1[a][m] = W1[m] / h[a];
            c2[a][m] = W2[m] / (h[a] * h[a]);
        }
        c20[a] = W2_0 / (h[a] * h[a]);
    }
    for (int m = 0; m < 3; m++) {
        c.c1x[m] = S::of(c1[0][m]);
        c.c1y[m] = S::of(c1[1][m]);
        c.c1z[m] = S::of(c1[2][m]);
        c.nc1z[m] = S::of(-c1[2][m]);
        c.c13y[m] = S::of(c1[1][m] / 3.0);
        c.c13z[m] = S::of(c1[2][m] / 3.0);
        c.nc13z[m] = S::of(-c1[2][m] / 3.0);
        const double mxy = WM[m] / (h[0] * h[1]), mxz = WM[m] / (h[0] * h[2]), myz = WM[m] / (h[1] * h[2]);
        c.cm3xy[m] = S::of(mxy / 3.0);
        c.cm3xz[m] = S::of(mxz / 3.0);
        c.ncm3xz[m] = S::of(-mxz / 3.0);
        c.cm3yz[m] = S::of(myz / 3.0);
        c.ncm3yz[m] = S::of(-myz / 3.0);
        c.cmxy[m] = S::of(mxy);
        c.cmxz[m] = S::of(mxz);
        c.ncmxz[m] = S::of(-mxz);
        c.cmyz[m] = S::of(myz);
        c.ncmyz[m] = S::of(-myz);
        c.c2x[m] = S::of(c2[0][m]);
        c.c2y[m] = S::of(c2[1][m]);
        c.c2z[m] = S::of(c2[2][m]);
        c.nc2x[m] = S::of(-c2[0][m]);
        c.nc2y[m] = S::of(-c2[1][m]);
        c.nc2z[m] = S::of(-c2[2][m]);
    }
    for (int i = 0; i < 3; i++) {
        // L_i = lap u_i + 1/3 (grad div u)_i: the second derivative along axis i carries 4/3
        const double fx = (i == 0) ? 4.0 / 3.0 : 1.0, fy = (i == 1) ? 4.0 / 3.0 : 1.0, fz = (i == 2) ? 4.0 / 3.0 : 1.0;
        for (int m = 0; m < 3; m++) {
            c.w2x[i][m] = S::of(fx * c2[0][m]);
            c.w2y[i][m] = S::of(fy * c2[1][m]);
            c.w2z[i][m] = S::of(fz * c2[2][m]);
        }
        c.w20[i] = S::of(fx * c20[0] + fy * c20[1] + fz * c20[2]);
    }
    for (int m = 0; m < 3; m++) {
        c.c6x[m] = S::of(W6[m] / h[0]);
        c.c6y[m] = S::of(W6[m] / h[1]);
        c.c6z[m] = S::of(W6[m] / h[2]);
    }
    c.c60x = S::of(W6_0 / h[0]);
    c.c60y = S::of(W6_0 / h[1]);
    c.c60z = S::of(W6_0 / h[2]);
    c.c20all = S::of(c20[0] + c20[1] + c20[2]);
    c.nc20yz = S::of(-(c20[1] + c20[2]));
    c.nc20xz = S::of(-(c20[0] + c20[2]));
    c.nc20xy = S::of(-(c20[0] + c20[1]));
    c.c20x = S::of(c20[0]);
    c.c20y = S::of(c20[1]);
    c.c20z = S::of(c20[2]);
    c.nu = S::of(ctx->nu);
    c.eta = S::of(ctx->eta);
    c.ncs2 = S::of(-(ctx->cs * ctx->cs));
    c.n23 = S::of(-2.0 / 3.0);
    for (int i = 0; i < 3; i++) {
        c.bext[i] = S::of(ctx->bext[i]);
        c.fre[i] = S::of(forcing ? forcing->re[i] : 0.0);
        c.nfim[i] = S::of(forcing ? -forcing->im[i] : 0.0);
    }
    c.rk_a = S::of(s == 0 ? 0.0 : RK_BETA[s] * RK_ALPHA[s] / RK_BETA[s - 1]);
    c.rk_b = S::of(RK_BETA[s] * dt);
}

// which planes of the slab a launch updates (AC_PART_* of the header)
enum { PART_ALL = 0, PART_INNER = 1, PART_OUTER = 2 };

// One substep s, or its inner / outer part.  INNER = planes [3, nz - 3): they read no z ghost plane, so they can run
// while the halo exchange is in flight (Fig. 3).  OUTER = the 3 + 3 boundary planes, then the
// ghost zones of the new state and the buffer swap.  ALL = both in one launch.
template <typename T>
int substep_t(ac_ctx* ctx, double dt, const ac_forcing* forcing, int s, int part, bool tables = true) {
    const ac::Layout& L = ctx->L;
    const ac_grid& g = ctx->grid;
    T* ftab = (T*)(ctx->ws + ctx->cv.ftab_off);
    ac_forcing kick;
    if (forcing && ctx->forcing_kick) {
        // alternative reading of G8: nothing in substeps 0 and 1; substep 2 is the last update of the step, and its
        // 2N register is never used again (alpha_0 = 0), so adding f / beta_2 to its right-hand side IS the impulse
        // u += dt f after the step
        if (s < 2) {
            forcing = nullptr;
        } else {
            kick = *forcing;
            for (int i = 0; i < 3; i++) {
                kick.re[i] /= RK_BETA[2];
                kick.im[i] /= RK_BETA[2];
            }
            forcing = &kick;
            tables = true;
        }
    }
    if (forcing && part != PART_OUTER && tables) {
        // a slab sees the global wave with its own origin: phase + k_z z0 (Eq. 4)
        const double hz = g.lz / g.nz;
        const double phase = forcing->phase + forcing->k[2] * (ctx->z0_plane * hz);
        const int n = g.nx + g.ny + g.nz;
        ac::forcing_tables_kernel<T><<<(n + 255) / 256, 256, 0, ctx->stream>>>(
            ftab, g.nx, g.ny, g.nz, forcing->k[0], forcing->k[1], forcing->k[2], g.lx / g.nx, g.ly / g.ny, hz, phase);
        ctx->launches++;
    }
    // plane ranges of this part, in storage planes (packed fp32: the boundary cells sit in the first and last 3 pairs)
    const int nzs = L.nz;
    const bool split = nzs > 2 * ac::R;
    int nr = 0, r0[2], r1[2];
    if (part == PART_ALL || (part == PART_OUTER && !split)) {
        r0[nr] = 0, r1[nr] = nzs, nr++;
    } else if (part == PART_INNER) {
        if (split) r0[nr] = ac::R, r1[nr] = nzs - ac::R, nr++;
    } else {
        r0[nr] = 0, r1[nr] = ac::R, nr++;
        r0[nr] = nzs - ac::R, r1[nr] = nzs, nr++;
    }
    if (ctx->march) {
        using E = typename ac::ElemOf<T>::E;
        ac::MarchArgs<T> a;
        a.ftab = ftab;
        a.L = L;
        a.nz_full = g.nz;
        a.cz = ctx->cz;
        a.has_forcing = forcing ? 1 : 0;
        a.wrap_z = ctx->slab ? 0 : 1;
        a.substep = s;
        fill_march_coef<E>(ctx, a.c, dt, s, forcing);
        for (int q = 0; q < AC_NFIELDS; q++) a.out[q] = (E*)ctx->field_ptr(1 - ctx->cur, q);
        for (int r = 0; r < nr; r++) {
            a.z_begin = r0[r];
            a.z_end = r1[r];
            const int nch = (r1[r] - r0[r] + ctx->cz - 1) / ctx->cz;
            if (ctx->variant == 0) {
                // pair-march: 16 x 16 tiles, a thread owns two cells
                dim3 gq((L.nx + ac::Q_TX - 1) / ac::Q_TX, (L.ny + ac::Q_TY - 1) / ac::Q_TY, nch);
                if (ctx->mixed == 1 && ctx->upwind)
                    ac::substep_pair_kernel<T, true, true><<<gq, ac::Q_THREADS, ac::QX_SMEM_BYTES, ctx->stream>>>(
                        a, ctx->map_qin[ctx->cur], ctx->map_qprev[1 - ctx->cur]);
                else if (ctx->mixed == 1)
                    ac::substep_pair_kernel<T, false, true><<<gq, ac::Q_THREADS, ac::QX_SMEM_BYTES, ctx->stream>>>(
                        a, ctx->map_qin[ctx->cur], ctx->map_qprev[1 - ctx->cur]);
                else if (ctx->upwind)
                    ac::substep_pair_kernel<T, true><<<gq, ac::Q_THREADS, ac::Q_SMEM_BYTES, ctx->stream>>>(
                        a, ctx->map_qin[ctx->cur], ctx->map_qprev[1 - ctx->cur]);
                else {
                    // the default build: previous-state and forcing switches fixed at compile time
                    // (the forcing switch in the fp64 build only: it shortens the A role alone, which the packed
                    // fp32 build cannot afford)
                    constexpr int F1 = std::is_same<T, double>::value ? 1 : -1, F0 = std::is_same<T, double>::value ? 0 : -1;
                    auto kern = s == 0 ? (forcing ? ac::substep_pair_kernel<T, false, false, 0, F1>
                                                  : ac::substep_pair_kernel<T, false, false, 0, F0>)
                                       : (forcing ? ac::substep_pair_kernel<T, false, false, 1, F1>
                                                  : ac::substep_pair_kernel<T, false, false, 1, F0>);
                    kern<<<gq, ac::Q_THREADS, ac::Q_SMEM_BYTES, ctx->stream>>>(a, ctx->map_qin[ctx->cur],
                                                                                ctx->map_qprev[1 - ctx->cur]);
                }
            } else {
                dim3 grd((L.nx + ac::M_TX - 1) / ac::M_TX, (L.ny + ac::M_TY - 1) / ac::M_TY, nch);
                if (ctx->upwind)
                    ac::substep_march_kernel<T, true><<<grd, ac::M_THREADS, ac::M_SMEM_BYTES, ctx->stream>>>(
                        a, ctx->map_in[ctx->cur], ctx->map_prev[1 - ctx->cur]);
                else
                    ac::substep_march_kernel<T, false><<<grd, ac::M_THREADS, ac::M_SMEM_BYTES, ctx->stream>>>(
                        a, ctx->map_in[ctx->cur], ctx->map_prev[1 - ctx->cur]);
            }
            ctx->launches++;
        }
        if (part != PART_INNER) {
            // S1: refresh the ghost zones of the buffer just written.  The z ghost planes of a slab belong to its
            // neighbours (ac_halo_unpack); of packed fp32 pairs one lane is the slab's own cell, so they are kept.
            const int nb_rows = 2 * ac::R * L.my + 2 * ac::R * L.nz;
            const int rows_per_task = ac::M_GHOST_THREADS / (2 * L.gx);
            const int na_tasks = (int)(((long)L.ny * L.nz + rows_per_task - 1) / rows_per_task);
            const int first_row = (ctx->slab && !ctx->packed) ? 2 * ac::R * L.my : 0;
            dim3 gg((unsigned)std::min(nb_rows + na_tasks - first_row, RED_BLOCKS), AC_NFIELDS, 1);
            ac::ghost_fill_kernel<E><<<gg, ac::M_GHOST_THREADS, 0, ctx->stream>>>((E*)ctx->field_ptr(1 - ctx->cur, 0), L,
                                                                              nb_rows, na_tasks, first_row);
            ctx->launches++;
        }
    } else {
        ac::SubstepArgs<T> a;
        a.L = L;
        fill_coeffs<T>(ctx, a.c);
        a.p.nu = (T)ctx->nu;
        a.p.eta = (T)ctx->eta;
        a.p.cs2 = (T)(ctx->cs * ctx->cs);
        for (int i = 0; i < 3; i++) a.p.bext[i] = (T)ctx->bext[i];
        a.p.has_forcing = forcing ? 1 : 0;
        a.p.upwind = ctx->upwind;
        a.p.mixed_tensor = ctx->mixed;
        for (int i = 0; i < 3; i++) {
            a.p.fre[i] = forcing ? (T)forcing->re[i] : T(0);
            a.p.fim[i] = forcing ? (T)forcing->im[i] : T(0);
        }
        a.ftab = ftab;
        a.p.substep = s;
        a.p.rk_a = (s == 0) ? T(0) : (T)(RK_BETA[s] * RK_ALPHA[s] / RK_BETA[s - 1]);
        a.p.rk_b = (T)(RK_BETA[s] * dt);
        for (int q = 0; q < AC_NFIELDS; q++) {
            a.in[q] = (const T*)ctx->field_ptr(ctx->cur, q);
            a.out[q] = (T*)ctx->field_ptr(1 - ctx->cur, q);
        }
        for (int r = 0; r < nr; r++) {
            a.z_begin = r0[r];
            a.z_end = r1[r];
            dim3 blk(32, 4, 2);
            dim3 grd((L.nx + blk.x - 1) / blk.x, (L.ny + blk.y - 1) / blk.y, (r1[r] - r0[r] + blk.z - 1) / blk.z);
            ac::substep_direct_kernel<T><<<grd, blk, 0, ctx->stream>>>(a);
            ctx->launches++;
        }
    }
    if (part != PART_INNER) ctx->cur = 1 - ctx->cur;
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

// substeps [s_begin, s_end) of one RK3 step (ac_step: 0..3; ac_substep: one)
template <typename T>
int step_t(ac_ctx* ctx, double dt, const ac_forcing* forcing, int s_begin = 0, int s_end = 3) {
    for (int s = s_begin; s < s_end; s++) {
        const int rc = substep_t<T>(ctx, dt, forcing, s, PART_ALL, s == s_begin);   // the tables serve all substeps of a step
        if (rc != AC_OK) return rc;
    }
    return AC_OK;
}

template <typename T>
int reduce_t(ac_ctx* ctx, ac_diag* out) {
    const ac::Layout& L = ctx->L;
    const ac_grid& g = ctx->grid;
    ac::ReduceArgs<T> a;
    a.L = L;
    const double h[3] = {g.lx / g.nx, g.ly / g.ny, g.lz / g.nz};
    for (int ax = 0; ax < 3; ax++)
        for (int m = 0; m < 3; m++) a.c1[ax][m] = (T)(W1[m] / h[ax]);
    for (int i = 0; i < 3; i++) a.bext[i] = (T)ctx->bext[i];
    for (int q = 0; q < AC_NFIELDS; q++) a.in[q] = ctx->field_ptr(ctx->cur, q);
    a.partial = (ac::RedVals*)(ctx->ws + ctx->cv.partial_off);
    ac::RedVals* result = (ac::RedVals*)(ctx->ws + ctx->cv.result_off);
    int blocks;
    if (ctx->march) {
        // 8-byte-element layouts (fp64, packed fp32): TMA plane ring (reduce_tma.cuh)
        const int tiles_x = (L.nx + ac::M_TX - 1) / ac::M_TX, tiles_y = (L.ny + ac::M_TY - 1) / ac::M_TY;
        const int nchunks = (L.nz + ac::RQ_CZ - 1) / ac::RQ_CZ;
        blocks = (int)std::min<long>((long)tiles_x * tiles_y * nchunks, std::min(3 * ctx->sms, RED_BLOCKS));
        // fp64 cells, or packed fp32 pairs (a march layout of fp32 is always packed)
        ac::reduce_tma_kernel<T, ac::ElemOf<T>::LANES><<<blocks, ac::RQ_THREADS, ac::RQ_SMEM_BYTES, ctx->stream>>>(
            a, ctx->map_a[ctx->cur], ctx->map_p[ctx->cur], tiles_x, tiles_y, nchunks);
    } else {
        const int tiles_x = (L.nx + ac::RED_TX - 1) / ac::RED_TX, tiles_y = (L.ny + ac::RED_TY - 1) / ac::RED_TY;
        const int nchunks = (L.nz + ac::RED_CZ - 1) / ac::RED_CZ;
        blocks = (int)std::min<long>((long)tiles_x * tiles_y * nchunks, RED_BLOCKS);
        const int sm = ac::red_smem_bytes<T, 1>();
        ac::reduce_stage1_kernel<T, 1><<<blocks, ac::RED_THREADS, sm, ctx->stream>>>(a, tiles_x, tiles_y, nchunks);
    }
    ac::reduce_stage2_kernel<<<1, 256, 0, ctx->stream>>>(a.partial, blocks, result);
    ctx->launches += 2;
    AC_CUDA(cudaGetLastError());
    AC_CUDA(cudaMemcpyAsync(ctx->host_result, result, sizeof(ac::RedVals), cudaMemcpyDeviceToHost, ctx->stream));
    AC_CUDA(cudaStreamSynchronize(ctx->stream));
    const ac::RedVals& r = *ctx->host_result;
    const double ncell = (double)g.nx * g.ny * g.nz;
    out->urms = std::sqrt(r.su / ncell);
    out->umax = std::sqrt(r.mu);
    out->brms = std::sqrt(r.sb / ncell);
    out->bmax = std::sqrt(r.mb);
    out->lnrho_min = r.lmin;
    out->lnrho_max = r.lmax;
    out->nonfinite = !(std::isfinite(r.su) && std::isfinite(r.sb) && std::isfinite(r.lmin) && std::isfinite(r.lmax));
    const double hmin = std::min(h[0], std::min(h[1], h[2]));
    double dt = ctx->c_u * hmin / (out->umax + ctx->cs);
    const double d = std::max(ctx->nu, ctx->eta);
    if (d > 0.0) dt = std::min(dt, ctx->c_nu * hmin * hmin / d);
    out->dt_cfl = dt;
    return AC_OK;
}

// extended diagnostics (diag_ext.cuh); the per-block partials live in the idle state buffer
template <typename T>
int reduce_ext_t(ac_ctx* ctx, double raw[3]) {
    const ac::Layout& L = ctx->L;
    ac::DiagExtArgs<T> a;
    a.L = L;
    fill_coeffs<T>(ctx, a.c);
    for (int i = 0; i < 3; i++) a.bext[i] = (T)ctx->bext[i];
    a.mixed_tensor = ctx->mixed;
    for (int q = 0; q < AC_NFIELDS; q++) a.in[q] = ctx->field_ptr(ctx->cur, q);
    a.partial = (ac::ExtVals*)ctx->field_ptr(1 - ctx->cur, 0);
    ac::ExtVals* result = (ac::ExtVals*)(ctx->ws + ctx->cv.result_off + 128);
    dim3 blk(32, 4, 2);
    dim3 grd((L.nx + blk.x - 1) / blk.x, (L.ny + blk.y - 1) / blk.y, (L.nz + blk.z - 1) / blk.z);
    const long nblocks = (long)grd.x * grd.y * grd.z;
    if ((size_t)nblocks * sizeof(ac::ExtVals) > ctx->cv.field_bytes) return AC_ENOMEM;
    if (ctx->packed)
        ac::diag_ext_kernel<T, 2><<<grd, blk, 0, ctx->stream>>>(a);
    else
        ac::diag_ext_kernel<T, 1><<<grd, blk, 0, ctx->stream>>>(a);
    ac::diag_ext_stage2_kernel<<<1, 256, 0, ctx->stream>>>(a.partial, nblocks, result);
    ctx->launches += 2;
    AC_CUDA(cudaGetLastError());
    ac::ExtVals* host = (ac::ExtVals*)((char*)ctx->host_result + 64);
    AC_CUDA(cudaMemcpyAsync(host, result, sizeof(ac::ExtVals), cudaMemcpyDeviceToHost, ctx->stream));
    AC_CUDA(cudaStreamSynchronize(ctx->stream));
    raw[0] = host->hk;
    raw[1] = host->hc;
    raw[2] = host->va2;
    return AC_OK;
}

// ----- Eq. 4-6 on the host -----------------------------------------------------------------------
void cross(const double a[3], const double b[3], double o[3]) {
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}

bool forcing_ok(const ac_forcing* f) {
    if (!f) return true;
    for (int i = 0; i < 3; i++)
        if (!std::isfinite(f->k[i]) || !std::isfinite(f->re[i]) || !std::isfinite(f->im[i])) return false;
    return std::isfinite(f->phase);
}

uint64_t splitmix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    uint64_t z = x;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

std::vector<std::array<int, 3>>* build_shell(double k_f) {
    auto* v = new (std::nothrow) std::vector<std::array<int, 3>>();
    if (!v) return nullptr;
    const double lo2 = (k_f - 0.5) * (k_f - 0.5), hi2 = (k_f + 0.5) * (k_f + 0.5);
    const int r = (int)std::floor(k_f + 0.5);
    // lexicographic order by construction (kx outermost)
    for (int kx = -r; kx <= r; kx++)
        for (int ky = -r; ky <= r; ky++)
            for (int kz = -r; kz <= r; kz++) {
                const double k2 = (double)kx * kx + (double)ky * ky + (double)kz * kz;
                if (k2 >= lo2 && k2 <= hi2) v->push_back({kx, ky, kz});
            }
    return v;
}

}  // namespace

// =================================================================================================
extern "C" {

size_t ac_workspace_bytes(const ac_grid* grid, ac_dtype dtype) {
    if (!grid_ok(grid) || (dtype != AC_F32 && dtype != AC_F64)) return 0;
    // large enough for either device layout of this dtype (a context may switch variants)
    size_t total = carve(layout_for(grid, dtype, false), store_elem_size(dtype, false), elem_size(dtype), grid->nz).total;
    if (dtype == AC_F32 && can_pack(grid))
        total = std::max(total, carve(layout_for(grid, dtype, true), 8, 4, grid->nz).total);
    return total;
}

}  // extern "C"

namespace {

// choose the kernel and the device layout for the context's variant; builds the TMA maps
int configure(ac_ctx* ctx) {
    const ac_grid* g = &ctx->grid;
    // the tensor-product reading of the mixed derivatives (NEXT-4) exists in the pair-march and in the direct kernel
    ctx->march = ctx->variant != 1 && (ctx->mixed == 0 || ctx->variant == 0) && (ctx->dtype == AC_F64 || can_pack(g));
    ctx->packed = ctx->march && ctx->dtype == AC_F32;
    ctx->L = layout_for(g, ctx->dtype, ctx->packed);
    ctx->cv = carve(ctx->L, store_elem_size(ctx->dtype, ctx->packed), elem_size(ctx->dtype), g->nz);
    // the pair-march kernel addresses its stores with 32-bit element offsets (1024^3 padded: 1.1e9 elements per field)
    if (ctx->march && ctx->variant == 0 && ctx->L.field > 0xffffffffull) return AC_EINVAL;
    ctx->loaded = false;
    ctx->loaded_mask = 0;
    ctx->cur = 0;
    ctx->next_substep = 0;
    {
        // opt-in shared-memory sizes of the reduction kernels, once per configuration
        cudaError_t e = cudaSuccess;
        if (ctx->dtype == AC_F64) {
            e = cudaFuncSetAttribute(ac::reduce_tma_kernel<double, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, ac::RQ_SMEM_BYTES);
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(ac::reduce_stage1_kernel<double, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         ac::red_smem_bytes<double, 1>());
        } else {
            e = cudaFuncSetAttribute(ac::reduce_tma_kernel<float, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, ac::RQ_SMEM_BYTES);
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(ac::reduce_stage1_kernel<float, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         ac::red_smem_bytes<float, 1>());
        }
        if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(reduction smem)");
    }
    if (!ctx->march) return AC_OK;
    for (int b = 0; b < 2; b++) {
        int rc = make_state_map(&ctx->map_in[b], ctx->field_ptr(b, 0), ctx->L, ac::M_WX, ac::M_WY);
        if (rc == AC_OK) rc = make_state_map(&ctx->map_prev[b], ctx->field_ptr(b, 0), ctx->L, ac::M_TX, ac::M_TY);
        if (rc == AC_OK) rc = make_state_map(&ctx->map_a[b], ctx->field_ptr(b, ac::AX), ctx->L, ac::M_WX, ac::M_WY, 3);
        if (rc == AC_OK) rc = make_state_map(&ctx->map_p[b], ctx->field_ptr(b, 0), ctx->L, ac::M_TX, ac::M_TY, 4);
        if (rc == AC_OK) rc = make_state_map(&ctx->map_qin[b], ctx->field_ptr(b, 0), ctx->L, ac::Q_WX, ac::Q_WY);
        if (rc == AC_OK) rc = make_state_map(&ctx->map_qprev[b], ctx->field_ptr(b, 0), ctx->L, ac::Q_TX, ac::Q_TY);
        if (rc != AC_OK) return rc;
    }
    const void* kernels[20] = {(const void*)ac::substep_march_kernel<double, false>,
                              (const void*)ac::substep_march_kernel<double, true>,
                              (const void*)ac::substep_march_kernel<float, false>,
                              (const void*)ac::substep_march_kernel<float, true>,
                              (const void*)ac::substep_pair_kernel<double, false>,
                              (const void*)ac::substep_pair_kernel<double, true>,
                              (const void*)ac::substep_pair_kernel<float, false>,
                              (const void*)ac::substep_pair_kernel<float, true>,
                              (const void*)ac::substep_pair_kernel<double, false, true>,
                              (const void*)ac::substep_pair_kernel<double, true, true>,
                              (const void*)ac::substep_pair_kernel<float, false, true>,
                              (const void*)ac::substep_pair_kernel<float, true, true>,
                              (const void*)ac::substep_pair_kernel<double, false, false, 0, 0>,
                              (const void*)ac::substep_pair_kernel<double, false, false, 1, 0>,
                              (const void*)ac::substep_pair_kernel<float, false, false, 0, -1>,
                              (const void*)ac::substep_pair_kernel<float, false, false, 1, -1>,
                              (const void*)ac::substep_pair_kernel<double, false, false, 0, 1>,
                              (const void*)ac::substep_pair_kernel<double, false, false, 1, 1>,
                              (const void*)ac::substep_pair_kernel<float, false, false, 0, -1>,
                              (const void*)ac::substep_pair_kernel<float, false, false, 1, -1>};
    for (int k = 0; k < 20; k++) {
        if ((ctx->dtype == AC_F64) != (k % 4 < 2)) continue;
        cudaError_t ea = cudaFuncSetAttribute(kernels[k], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              k < 4 ? ac::M_SMEM_BYTES : (k < 8 || k >= 12 ? ac::Q_SMEM_BYTES : ac::QX_SMEM_BYTES));
        if (ea != cudaSuccess) return cuda_fail(ea, "cudaFuncSetAttribute(march kernel smem)");
    }
    // z chunks: every chunk re-reads 6 planes, every wave of CTAs costs (planes + 6) iterations;
    // pick the chunk count that minimises waves x (planes per chunk + 6)
    const int nzp = ctx->L.nz;
    const int tile_x = ctx->variant == 0 ? ac::Q_TX : ac::M_TX, tile_y = ctx->variant == 0 ? ac::Q_TY : ac::M_TY;
    const long tiles = (long)((ctx->L.nx + tile_x - 1) / tile_x) * ((ctx->L.ny + tile_y - 1) / tile_y);
    const int sms = ctx->sms;
    long best_cost = -1;
    int best_n = 1;
    for (int n = 1; n <= 64; n++) {
        const int cz = (nzp + n - 1) / n;
        if (cz > ac::M_CZMAX) continue;
        if (cz < 4 && n > 1) break;
        const int nn = (nzp + cz - 1) / cz;
        const long waves = (tiles * nn + sms - 1) / sms;
        const long cost = waves * (cz + 6);
        if (best_cost < 0 || cost < best_cost) {
            best_cost = cost;
            best_n = nn;
            ctx->cz = cz;
        }
    }
    ctx->nchunks = best_n;
    return AC_OK;
}

}  // namespace

extern "C" {

int ac_init(ac_ctx** out, const ac_grid* grid, ac_dtype dtype, double nu, double eta, double cs, double k_f,
            double helicity, void* workspace_dev, void* cuda_stream) {
    if (!out) return AC_EINVAL;
    *out = nullptr;
    if (!grid_ok(grid) || (dtype != AC_F32 && dtype != AC_F64)) return AC_EINVAL;
    if (!(nu >= 0.0) || !(eta >= 0.0) || !(cs > 0.0) || !std::isfinite(nu) || !std::isfinite(eta) || !std::isfinite(cs))
        return AC_EINVAL;
    if (!(k_f >= 1.0) || !(k_f <= 64.0) || !(helicity >= 0.0) || !(helicity <= 1.0)) return AC_EINVAL;
    if (workspace_dev && ((uintptr_t)workspace_dev % 256) != 0) return AC_EINVAL;

    int dev = 0;
    AC_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    AC_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "device %.160s is sm_%d%d; this library is built for sm_100a only",
                 prop.name, prop.major, prop.minor);
        return AC_ECUDA;
    }

    ac_ctx* ctx = new (std::nothrow) ac_ctx();
    if (!ctx) return AC_ENOMEM;
    ctx->grid = *grid;
    ctx->dtype = dtype;
    ctx->nu = nu;
    ctx->eta = eta;
    ctx->cs = cs;
    ctx->k_f = k_f;
    ctx->helicity = helicity;
    ctx->bext[0] = ctx->bext[1] = ctx->bext[2] = 0.0;
    ctx->c_u = 0.4;
    ctx->c_nu = 0.25;
    ctx->variant = 0;
    ctx->upwind = 0;
    ctx->forcing_kick = 0;
    ctx->mixed = 0;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->launches = 0;
    ctx->host_result = nullptr;
    ctx->cz = 0;
    ctx->nchunks = 1;
    ctx->device = dev;
    ctx->sms = prop.multiProcessorCount;
    ctx->next_substep = 0;
    ctx->slab = false;
    ctx->z0_plane = 0;
    ctx->nz_global = grid->nz;
    ctx->inner_done = -1;
    if (workspace_dev) {
        ctx->ws = (char*)workspace_dev;
        ctx->owns_ws = false;
    } else {
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, ac_workspace_bytes(grid, dtype));
        if (e != cudaSuccess) {
            cudaGetLastError();
            delete ctx;
            return e == cudaErrorMemoryAllocation ? AC_ENOMEM : cuda_fail(e, "cudaMalloc(workspace)");
        }
        ctx->ws = (char*)p;
        ctx->owns_ws = true;
    }
    int rc = configure(ctx);
    if (rc == AC_OK) {
        cudaError_t e = cudaMallocHost((void**)&ctx->host_result, 128);   // RedVals at 0, ExtVals at 64
        if (e != cudaSuccess) rc = cuda_fail(e, "cudaMallocHost");
    }
    if (rc != AC_OK) {
        if (ctx->owns_ws) cudaFree(ctx->ws);
        delete ctx;
        return rc;
    }
    *out = ctx;
    return AC_OK;
}

int ac_load_state(ac_ctx* ctx, const void* const fields[AC_NFIELDS], int src_on_device) {
    DeviceGuard guard(ctx);
    if (!ctx || !fields) return AC_EINVAL;
    for (int q = 0; q < AC_NFIELDS; q++)
        if (!fields[q]) return AC_EINVAL;
    ctx->cur = 0;
    ctx->loaded = false;
    ctx->loaded_mask = 0;
    ctx->next_substep = 0;          // a whole new state starts a new step
    ctx->inner_done = -1;
    for (int q = 0; q < AC_NFIELDS; q++) {
        const int rc = ac_load_field(ctx, q, fields[q], src_on_device);
        if (rc != AC_OK) return rc;
    }
    return AC_OK;
}

int ac_load_field(ac_ctx* ctx, int q, const void* field, int src_on_device) {
    DeviceGuard guard(ctx);
    if (!ctx || !field || q < 0 || q >= AC_NFIELDS) return AC_EINVAL;
    // inside a step the idle buffer holds the previous state (2N register): nothing may be staged there, and
    // replacing a field of the current state would corrupt the register as well
    if (ctx->next_substep != 0) return AC_ESTATE;
    const int rc = ctx->dtype == AC_F64 ? load_field_t<double>(ctx, ctx->cur, q, field, src_on_device)
                                        : load_field_t<float>(ctx, ctx->cur, q, field, src_on_device);
    if (rc != AC_OK) return rc;
    ctx->loaded_mask |= 1u << q;
    if (ctx->loaded_mask == (1u << AC_NFIELDS) - 1u) ctx->loaded = true;
    return AC_OK;
}

int ac_store_state(ac_ctx* ctx, void* const fields[AC_NFIELDS], int dst_on_device) {
    DeviceGuard guard(ctx);
    if (!ctx || !fields) return AC_EINVAL;
    for (int q = 0; q < AC_NFIELDS; q++)
        if (!fields[q]) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    if (!dst_on_device && ctx->next_substep != 0) return AC_ESTATE;   // the host path stages in the idle buffer
    for (int q = 0; q < AC_NFIELDS; q++) {
        const int rc = ctx->dtype == AC_F64 ? store_field_t<double>(ctx, q, fields[q], dst_on_device)
                                            : store_field_t<float>(ctx, q, fields[q], dst_on_device);
        if (rc != AC_OK) return rc;
    }
    if (!dst_on_device) AC_CUDA(cudaStreamSynchronize(ctx->stream));
    return AC_OK;
}

int ac_store_field(ac_ctx* ctx, int q, void* field, int dst_on_device) {
    DeviceGuard guard(ctx);
    if (!ctx || !field || q < 0 || q >= AC_NFIELDS) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    if (!dst_on_device && ctx->next_substep != 0) return AC_ESTATE;
    const int rc = ctx->dtype == AC_F64 ? store_field_t<double>(ctx, q, field, dst_on_device)
                                        : store_field_t<float>(ctx, q, field, dst_on_device);
    if (rc != AC_OK) return rc;
    if (!dst_on_device) AC_CUDA(cudaStreamSynchronize(ctx->stream));
    return AC_OK;
}

int ac_step(ac_ctx* ctx, double dt, const ac_forcing* forcing) {
    DeviceGuard guard(ctx);
    if (!ctx) return AC_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return AC_EINVAL;
    if (!forcing_ok(forcing)) return AC_EINVAL;
    if (!ctx->loaded || ctx->next_substep != 0 || ctx->inner_done != -1) return AC_ESTATE;
    return ctx->dtype == AC_F64 ? step_t<double>(ctx, dt, forcing) : step_t<float>(ctx, dt, forcing);
}

int ac_substep(ac_ctx* ctx, int s, double dt, const ac_forcing* forcing) {
    DeviceGuard guard(ctx);
    if (!ctx || s < 0 || s > 2) return AC_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return AC_EINVAL;
    if (!forcing_ok(forcing)) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    if (s != ctx->next_substep || ctx->inner_done != -1) return AC_ESTATE;   // substeps run in order 0, 1, 2: the 2N register is the buffers' difference
    const int rc = ctx->dtype == AC_F64 ? step_t<double>(ctx, dt, forcing, s, s + 1) : step_t<float>(ctx, dt, forcing, s, s + 1);
    if (rc == AC_OK) ctx->next_substep = (s + 1) % 3;
    return rc;
}

int ac_substep_part(ac_ctx* ctx, int s, double dt, const ac_forcing* forcing, int part) {
    DeviceGuard guard(ctx);
    if (!ctx || s < 0 || s > 2 || (part != AC_PART_INNER && part != AC_PART_OUTER)) return AC_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return AC_EINVAL;
    if (!forcing_ok(forcing)) return AC_EINVAL;
    if (!ctx->loaded || s != ctx->next_substep) return AC_ESTATE;
    if (part == AC_PART_INNER ? ctx->inner_done != -1 : ctx->inner_done != s) return AC_ESTATE;   // inner first, once
    const int rc = ctx->dtype == AC_F64 ? substep_t<double>(ctx, dt, forcing, s, part == AC_PART_INNER ? PART_INNER : PART_OUTER)
                                        : substep_t<float>(ctx, dt, forcing, s, part == AC_PART_INNER ? PART_INNER : PART_OUTER);
    if (rc != AC_OK) return rc;
    if (part == AC_PART_INNER) {
        ctx->inner_done = s;
    } else {
        ctx->inner_done = -1;
        ctx->next_substep = (s + 1) % 3;
    }
    return AC_OK;
}

int ac_set_slab(ac_ctx* ctx, int z0_plane, int nz_global) {
    if (!ctx) return AC_EINVAL;
    if (nz_global < ctx->grid.nz || z0_plane < 0 || z0_plane + ctx->grid.nz > nz_global) return AC_EINVAL;
    if (ctx->next_substep != 0 || ctx->inner_done != -1) return AC_ESTATE;
    ctx->slab = nz_global != ctx->grid.nz;
    ctx->z0_plane = z0_plane;
    ctx->nz_global = nz_global;
    return AC_OK;
}

size_t ac_halo_bytes(const ac_ctx* ctx) {
    if (!ctx) return 0;
    return (size_t)AC_NFIELDS * ac::R * ctx->L.plane * elem_size(ctx->dtype);
}

int ac_halo_pack(ac_ctx* ctx, void* send_lo_dev, void* send_hi_dev, void* cuda_stream) {
    DeviceGuard guard(ctx);
    if (!ctx || !send_lo_dev || !send_hi_dev) return AC_EINVAL;
    if (!ctx->loaded || ctx->inner_done != -1) return AC_ESTATE;
    cudaStream_t st = cuda_stream ? (cudaStream_t)cuda_stream : ctx->stream;
    const ac::Layout& L = ctx->L;
    const size_t per_field = (size_t)ac::R * L.plane;
    dim3 grd((unsigned)((per_field + 255) / 256), AC_NFIELDS, 1);
    void* state = ctx->field_ptr(ctx->cur, 0);
    if (ctx->dtype == AC_F64)
        ac::halo_pack_kernel<double, 1><<<grd, 256, 0, st>>>(state, L.field, L, (double*)send_lo_dev, (double*)send_hi_dev);
    else if (ctx->packed)
        ac::halo_pack_kernel<float, 2><<<grd, 256, 0, st>>>(state, L.field, L, (float*)send_lo_dev, (float*)send_hi_dev);
    else
        ac::halo_pack_kernel<float, 1><<<grd, 256, 0, st>>>(state, L.field, L, (float*)send_lo_dev, (float*)send_hi_dev);
    ctx->launches++;
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

int ac_halo_unpack(ac_ctx* ctx, const void* recv_lo_dev, const void* recv_hi_dev, void* cuda_stream) {
    DeviceGuard guard(ctx);
    if (!ctx || !recv_lo_dev || !recv_hi_dev) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    cudaStream_t st = cuda_stream ? (cudaStream_t)cuda_stream : ctx->stream;
    const ac::Layout& L = ctx->L;
    const size_t per_field = (size_t)ac::R * L.plane;
    dim3 grd((unsigned)((per_field + 255) / 256), AC_NFIELDS, 1);
    void* state = ctx->field_ptr(ctx->cur, 0);
    if (ctx->dtype == AC_F64)
        ac::halo_unpack_kernel<double, 1><<<grd, 256, 0, st>>>(state, L.field, L, (const double*)recv_lo_dev, (const double*)recv_hi_dev);
    else if (ctx->packed)
        ac::halo_unpack_kernel<float, 2><<<grd, 256, 0, st>>>(state, L.field, L, (const float*)recv_lo_dev, (const float*)recv_hi_dev);
    else
        ac::halo_unpack_kernel<float, 1><<<grd, 256, 0, st>>>(state, L.field, L, (const float*)recv_lo_dev, (const float*)recv_hi_dev);
    ctx->launches++;
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

int ac_halo_pull(ac_ctx* ctx, const void* below_workspace, const void* above_workspace, void* cuda_stream) {
    DeviceGuard guard(ctx);
    if (!ctx || !below_workspace || !above_workspace) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    cudaStream_t st = cuda_stream ? (cudaStream_t)cuda_stream : ctx->stream;
    const ac::Layout& L = ctx->L;
    const size_t per_field = (size_t)ac::R * L.plane;
    dim3 grd((unsigned)((per_field + 255) / 256), AC_NFIELDS, 1);
    // every rank of a run makes the same calls in the same order, so the neighbours' current state sits at the same
    // offset of their workspace as ours does in ours
    const size_t off = (size_t)((char*)ctx->field_ptr(ctx->cur, 0) - ctx->ws);
    void* state = ctx->field_ptr(ctx->cur, 0);
    const void* below = (const char*)below_workspace + off;
    const void* above = (const char*)above_workspace + off;
    if (ctx->dtype == AC_F64)
        ac::halo_pull_kernel<double, 1><<<grd, 256, 0, st>>>(state, below, above, L.field, L);
    else if (ctx->packed)
        ac::halo_pull_kernel<float, 2><<<grd, 256, 0, st>>>(state, below, above, L.field, L);
    else
        ac::halo_pull_kernel<float, 1><<<grd, 256, 0, st>>>(state, below, above, L.field, L);
    ctx->launches++;
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

void* ac_workspace_ptr(ac_ctx* ctx) { return ctx ? (void*)ctx->ws : nullptr; }

int ac_ipc_export(ac_ctx* ctx, void* handle64) {
    DeviceGuard guard(ctx);
    if (!ctx || !handle64) return AC_EINVAL;
    if (!ctx->owns_ws) return AC_ESTATE;       // only a workspace the library allocated starts at a cudaMalloc base
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "the header promises a 64-byte handle");
    cudaIpcMemHandle_t h;
    AC_CUDA(cudaIpcGetMemHandle(&h, ctx->ws));
    memcpy(handle64, &h, 64);
    return AC_OK;
}

int ac_ipc_open(const void* handle64, void** workspace_out) {
    if (!handle64 || !workspace_out) return AC_EINVAL;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle64, 64);
    AC_CUDA(cudaIpcOpenMemHandle(workspace_out, h, cudaIpcMemLazyEnablePeerAccess));
    return AC_OK;
}

int ac_ipc_close(void* workspace) {
    if (!workspace) return AC_EINVAL;
    AC_CUDA(cudaIpcCloseMemHandle(workspace));
    return AC_OK;
}

int ac_diag_combine(const ac_ctx* ctx, const double* raws, int nranks, ac_diag* out) {
    if (!ctx || !raws || !out || nranks < 1) return AC_EINVAL;
    double su = 0.0, sb = 0.0, mu = 0.0, mb = 0.0, lmin = INFINITY, lmax = -INFINITY;
    for (int r = 0; r < nranks; r++) {       // rank order: deterministic
        const double* v = raws + 6 * r;
        su += v[0];
        sb += v[2];
        mu = std::max(mu, v[1]);
        mb = std::max(mb, v[3]);
        lmin = std::min(lmin, v[4]);
        lmax = std::max(lmax, v[5]);
    }
    const ac_grid& g = ctx->grid;
    const double ncell = (double)g.nx * g.ny * (double)ctx->nz_global;
    out->urms = std::sqrt(su / ncell);
    out->umax = std::sqrt(mu);
    out->brms = std::sqrt(sb / ncell);
    out->bmax = std::sqrt(mb);
    out->lnrho_min = lmin;
    out->lnrho_max = lmax;
    out->nonfinite = !(std::isfinite(su) && std::isfinite(sb) && std::isfinite(lmin) && std::isfinite(lmax));
    const double hmin = std::min(g.lx / g.nx, std::min(g.ly / g.ny, g.lz / g.nz));
    double dt = ctx->c_u * hmin / (out->umax + ctx->cs);
    const double d = std::max(ctx->nu, ctx->eta);
    if (d > 0.0) dt = std::min(dt, ctx->c_nu * hmin * hmin / d);
    out->dt_cfl = dt;
    return AC_OK;
}

int ac_state_layout(const ac_ctx* ctx, ac_layout_info* out) {
    if (!ctx || !out) return AC_EINVAL;
    const ac::Layout& L = ctx->L;
    out->elem_bytes = (int)store_elem_size(ctx->dtype, ctx->packed);
    out->packed_pairs = ctx->packed ? 1 : 0;
    out->gx = L.gx;
    out->pitch = L.pitch;
    out->my = L.my;
    out->mz = L.mz;
    out->plane_elems = L.plane;
    out->field_elems = L.field;
    return AC_OK;
}

void* ac_field_device_ptr(ac_ctx* ctx, int q) {
    if (!ctx || q < 0 || q >= AC_NFIELDS) return nullptr;
    return ctx->field_ptr(ctx->cur, q);
}

int ac_reduce(ac_ctx* ctx, ac_diag* out) {
    DeviceGuard guard(ctx);
    if (!ctx || !out) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    return ctx->dtype == AC_F64 ? reduce_t<double>(ctx, out) : reduce_t<float>(ctx, out);
}

int ac_reduce_raw(ac_ctx* ctx, double out[6]) {
    DeviceGuard guard(ctx);
    if (!ctx || !out) return AC_EINVAL;
    if (!ctx->loaded) return AC_ESTATE;
    ac_diag d;
    const int rc = ctx->dtype == AC_F64 ? reduce_t<double>(ctx, &d) : reduce_t<float>(ctx, &d);
    if (rc != AC_OK) return rc;
    const ac::RedVals& r = *ctx->host_result;
    out[0] = r.su;
    out[1] = r.mu;
    out[2] = r.sb;
    out[3] = r.mb;
    out[4] = r.lmin;
    out[5] = r.lmax;
    return AC_OK;
}

int ac_reduce_ext_raw(ac_ctx* ctx, double out[3]) {
    DeviceGuard guard(ctx);
    if (!ctx || !out) return AC_EINVAL;
    if (!ctx->loaded || ctx->next_substep != 0) return AC_ESTATE;    // the partials are staged in the idle buffer
    return ctx->dtype == AC_F64 ? reduce_ext_t<double>(ctx, out) : reduce_ext_t<float>(ctx, out);
}

int ac_reduce_ext(ac_ctx* ctx, ac_diag_ext* out) {
    if (!ctx || !out) return AC_EINVAL;
    if (!ctx->loaded || ctx->next_substep != 0) return AC_ESTATE;
    ac_diag d;
    int rc = ac_reduce(ctx, &d);
    if (rc != AC_OK) return rc;
    double raw[3];
    rc = ac_reduce_ext_raw(ctx, raw);
    if (rc != AC_OK) return rc;
    const ac_grid& g = ctx->grid;
    const double ncell = (double)g.nx * g.ny * g.nz;
    out->kin_hel = raw[0] / ncell;
    out->cur_hel = raw[1] / ncell;
    out->va_max = std::sqrt(raw[2]);
    out->nonfinite = d.nonfinite || !(std::isfinite(raw[0]) && std::isfinite(raw[1]) && std::isfinite(raw[2]));
    // G15 with the Alfven term: the signal speed c_s becomes sqrt(c_s^2 + max v_A^2)
    const double hmin = std::min(g.lx / g.nx, std::min(g.ly / g.ny, g.lz / g.nz));
    double dt = ctx->c_u * hmin / (d.umax + std::sqrt(ctx->cs * ctx->cs + raw[2]));
    const double dd = std::max(ctx->nu, ctx->eta);
    if (dd > 0.0) dt = std::min(dt, ctx->c_nu * hmin * hmin / dd);
    out->dt_cfl_alfven = dt;
    return AC_OK;
}

int ac_forcing_params(double k_f, double helicity, double cs, const ac_grid* grid, double u1, double u2, double u3,
                      double dt, double f0, ac_forcing* out) {
    if (!out || !grid_ok(grid)) return AC_EINVAL;
    if (!(k_f >= 1.0) || !(k_f <= 64.0) || !(helicity >= 0.0) || !(helicity <= 1.0) || !(cs > 0.0)) return AC_EINVAL;
    if (!(u1 >= 0.0 && u1 < 1.0 && u2 >= 0.0 && u2 < 1.0 && u3 >= 0.0 && u3 < 1.0)) return AC_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt) || !std::isfinite(f0)) return AC_EINVAL;
    std::vector<std::array<int, 3>>* shp = build_shell(k_f);
    if (!shp) return AC_ENOMEM;
    if (shp->empty()) {
        delete shp;
        return AC_EINVAL;
    }
    const auto& sh = *shp;
    size_t idx = (size_t)std::floor(u1 * (double)sh.size());
    if (idx >= sh.size()) idx = sh.size() - 1;
    const double k[3] = {(double)sh[idx][0], (double)sh[idx][1], (double)sh[idx][2]};
    delete shp;
    const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
    const double kabs = std::sqrt(k2);
    const double pi = 3.14159265358979323846;
    // e-hat = cos(psi) e1 + sin(psi) e2, e1 = normalise(k x a), a = axis of smallest |k_a|, e2 = k^ x e1 (G9)
    int ai = 0;
    for (int i = 1; i < 3; i++)
        if (std::fabs(k[i]) < std::fabs(k[ai])) ai = i;
    double a[3] = {0, 0, 0};
    a[ai] = 1.0;
    double e1[3], e2[3], khat[3] = {k[0] / kabs, k[1] / kabs, k[2] / kabs};
    cross(k, a, e1);
    const double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    for (int i = 0; i < 3; i++) e1[i] /= n1;
    cross(khat, e1, e2);
    const double psi = 2.0 * pi * u3;
    double eh[3];
    for (int i = 0; i < 3; i++) eh[i] = std::cos(psi) * e1[i] + std::sin(psi) * e2[i];
    // Eq. 6: f_k = [k x (k x e) - i sigma |k| (k x e)] / [sqrt(1 + sigma^2) k^2 sqrt(1 - (k.e)^2/k^2)]
    double kxe[3], kxkxe[3];
    cross(k, eh, kxe);
    cross(k, kxe, kxkxe);
    const double sigma = helicity;
    const double kde = k[0] * eh[0] + k[1] * eh[1] + k[2] * eh[2];
    const double den = std::sqrt(1.0 + sigma * sigma) * k2 * std::sqrt(1.0 - kde * kde / k2);
    // Eq. 5: N = f0 cs sqrt(|k| cs / dt)
    const double N = f0 * cs * std::sqrt(kabs * cs / dt);
    // the integer shell vector counts periods per box side: k_a 2 pi / l_a
    out->k[0] = k[0] * (2.0 * pi / grid->lx);
    out->k[1] = k[1] * (2.0 * pi / grid->ly);
    out->k[2] = k[2] * (2.0 * pi / grid->lz);
    out->phase = -pi + 2.0 * pi * u2;
    for (int i = 0; i < 3; i++) {
        out->re[i] = N * kxkxe[i] / den;
        out->im[i] = N * (-sigma * kabs * kxe[i]) / den;
    }
    return AC_OK;
}

int ac_forcing_from_draws(const ac_ctx* ctx, double u1, double u2, double u3, double dt, double f0, ac_forcing* out) {
    if (!ctx) return AC_EINVAL;
    // the wave vectors count periods of the GLOBAL box: a slab knows its share of it (ac_set_slab)
    ac_grid g = ctx->grid;
    g.lz = ctx->grid.lz / ctx->grid.nz * ctx->nz_global;
    g.nz = ctx->nz_global;
    return ac_forcing_params(ctx->k_f, ctx->helicity, ctx->cs, &g, u1, u2, u3, dt, f0, out);
}

int ac_make_forcing(const ac_ctx* ctx, uint64_t seed, uint64_t step, double dt, double f0, ac_forcing* out) {
    if (!ctx || !out) return AC_EINVAL;
    const uint64_t key = splitmix64(seed);
    double u[3];
    for (uint64_t i = 0; i < 3; i++) u[i] = (double)(splitmix64(key ^ (3 * step + i)) >> 11) * (1.0 / 9007199254740992.0);
    return ac_forcing_from_draws(ctx, u[0], u[1], u[2], dt, f0, out);
}

int ac_set_bext(ac_ctx* ctx, const double b[3]) {
    if (!ctx || !b) return AC_EINVAL;
    for (int i = 0; i < 3; i++) {
        if (!std::isfinite(b[i])) return AC_EINVAL;
        ctx->bext[i] = b[i];
    }
    return AC_OK;
}

int ac_set_cfl(ac_ctx* ctx, double c_u, double c_nu) {
    if (!ctx || !(c_u > 0.0) || !(c_nu > 0.0)) return AC_EINVAL;
    ctx->c_u = c_u;
    ctx->c_nu = c_nu;
    return AC_OK;
}

int ac_set_upwind(ac_ctx* ctx, int on) {
    if (!ctx || (on != 0 && on != 1)) return AC_EINVAL;
    ctx->upwind = on;
    return AC_OK;
}

int ac_set_forcing_mode(ac_ctx* ctx, int mode) {
    if (!ctx || (mode != 0 && mode != 1)) return AC_EINVAL;
    if (ctx->next_substep != 0 || ctx->inner_done != -1) return AC_ESTATE;
    ctx->forcing_kick = mode;
    return AC_OK;
}

int ac_set_mixed(ac_ctx* ctx, int mode) {
    DeviceGuard guard(ctx);
    if (!ctx || (mode != 0 && mode != 1)) return AC_EINVAL;
    if (mode == ctx->mixed) return AC_OK;
    // variants 1 and 2 run the tensor-product reading in the direct kernel, whose fp32 device layout differs
    cudaStreamSynchronize(ctx->stream);
    ctx->mixed = mode;
    return configure(ctx);
}

int ac_set_variant(ac_ctx* ctx, int variant) {
    DeviceGuard guard(ctx);
    if (!ctx) return AC_EINVAL;
    if (variant < 0 || variant > 2) return AC_EINVAL;
    if (variant == ctx->variant) return AC_OK;
    // the variants use different device layouts in fp32: a loaded state would have to be re-packed
    cudaStreamSynchronize(ctx->stream);
    ctx->variant = variant;
    return configure(ctx);
}

long long ac_launch_count(const ac_ctx* ctx) { return ctx ? ctx->launches : 0; }

void ac_free(ac_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard guard(ctx);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->owns_ws) cudaFree(ctx->ws);
    if (ctx->host_result) cudaFreeHost(ctx->host_result);
    delete ctx;
}

// ---- ac_reduce_dense_noalloc: the one entry point that allocates nothing ---------------------------------------
// Its scratch memory (the per-block partials of reduce_dense_stage1_kernel) is this fixed array: every GPU that loads
// the library holds its 3 MiB until the process exits.  In HOST code the name below is a host-side stand-in, not a
// device address; the kernels get the address cudaGetSymbolAddress returns for the current device, looked up once per
// device (noalloc_scratch) in this same file.
}  // extern "C"

static __device__ __align__(256) unsigned char g_noalloc_scratch[(size_t)ac::RD_MAX_PARTIALS * sizeof(ac::RedVals)];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
void* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

// device address of g_noalloc_scratch on the CURRENT device; set-up once per device, no allocation
int noalloc_scratch(int dev, void** out) {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        AC_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return AC_ECUDA;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return AC_OK;
}

template <typename T>
int reduce_dense_t(const void* state_dev, const ac_grid* g, const double bext[3], ac::RedVals* partial, double* raw_dev,
                   cudaStream_t stream) {
    ac::ReduceDenseArgs<T> a;
    a.state = (const T*)state_dev;
    a.nx = g->nx, a.ny = g->ny, a.nz = g->nz;
    const double h[3] = {g->lx / g->nx, g->ly / g->ny, g->lz / g->nz};
    for (int ax = 0; ax < 3; ax++)
        for (int m = 0; m < 3; m++) a.c1[ax][m] = (T)(W1[m] / h[ax]);
    for (int i = 0; i < 3; i++) a.bext[i] = (T)(bext ? bext[i] : 0.0);
    const long long ncell = (long long)g->nx * g->ny * g->nz;
    const int blocks = (int)((ncell + ac::RD_CELLS_PER_BLOCK - 1) / ac::RD_CELLS_PER_BLOCK);   // <= RD_MAX_PARTIALS
    // every partial that stage 2 reads is written by stage 1 of this call: nothing in the scratch array has to start
    // at zero, whatever the previous call left there
    ac::reduce_dense_stage1_kernel<T><<<blocks, ac::RD_THREADS, 0, stream>>>(a, partial);
    ac::reduce_stage2_kernel<<<1, 256, 0, stream>>>(partial, blocks, (ac::RedVals*)raw_dev);
    AC_CUDA(cudaGetLastError());
    return AC_OK;
}

}  // namespace

extern "C" {

int ac_reduce_dense_noalloc(const void* state_dev, ac_dtype dtype, const ac_grid* grid, const double bext[3],
                            double* raw_dev, void* cuda_stream) {
    if (!state_dev || !raw_dev || ((uintptr_t)raw_dev % 8) != 0) return AC_EINVAL;
    if (!grid_ok(grid) || (dtype != AC_F32 && dtype != AC_F64)) return AC_EINVAL;
    if (bext && !(std::isfinite(bext[0]) && std::isfinite(bext[1]) && std::isfinite(bext[2]))) return AC_EINVAL;
    if ((long long)grid->nx * grid->ny * grid->nz > ac::RD_MAX_CELLS) return AC_ELIMIT;
    int dev = 0;
    AC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return AC_EINVAL;
    // both pointers must be memory the current device owns (a host pointer would fault in the kernel, or silently
    // read host memory where the GPU can reach it)
    const void* ptrs[2] = {state_dev, raw_dev};
    for (const void* p : ptrs) {
        cudaPointerAttributes at;
        AC_CUDA(cudaPointerGetAttributes(&at, p));
        if (!(at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) ||
            (at.type == cudaMemoryTypeDevice && at.device != dev))
            return AC_EINVAL;
    }
    void* scratch = nullptr;
    const int rc = noalloc_scratch(dev, &scratch);
    if (rc != AC_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    return dtype == AC_F64 ? reduce_dense_t<double>(state_dev, grid, bext, (ac::RedVals*)scratch, raw_dev, stream)
                           : reduce_dense_t<float>(state_dev, grid, bext, (ac::RedVals*)scratch, raw_dev, stream);
}

long long ac_noalloc_max_cells(void) { return ac::RD_MAX_CELLS; }

const char* ac_strerror(int status) {
    switch (status) {
        case AC_OK: return "ok";
        case AC_EINVAL: return "invalid argument";
        case AC_ENOMEM: return "out of memory or workspace too small";
        case AC_ECUDA: return g_cuda_err;
        case AC_ESTATE: return "no state loaded (call ac_load_state first)";
        case AC_ELIMIT: return "grid larger than the fixed scratch array of ac_reduce_dense_noalloc (2^27 cells = 512^3)";
        default: return "unknown status";
    }
}

const char* ac_version(void) { return "ac_mhd 0.1 sm_100a"; }

}  // extern "C"
