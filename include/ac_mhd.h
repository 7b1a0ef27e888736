/*
 * ac_mhd.h - C ABI of the B200-native MHD time-stepping library (libac_mhd.so).
 *
 * The library advances the state (ln rho, u, A) of compressible isothermal resistive MHD on a
 * triply periodic grid by full 2N-RK3 time steps and reduces rms/max diagnostics.  Everything on
 * the path runs in hand-written sm_100a CUDA kernels; there is no CPU fallback: every entry point
 * that needs the device returns AC_ECUDA if there is none.
 *
 * What is computed (citations: /root/reference/PAPER.md line numbers; "G<n>" = reading listed
 * in DESIGN.md where the paper is silent):
 *   Eq. 1  D ln rho/Dt = -div u
 *   Eq. 2  Du/Dt = -cs^2 grad ln rho + j x B / rho
 *                  + nu [lap u + 1/3 grad div u + 2 S.grad ln rho] + f
 *   Eq. 3  dA/dt = u x B + eta lap A     (B = curl A, j = curl B, mu0 = 1)
 *   Eq. 4  f(x) = Re{N f_k exp[i k.x + i phi]}, Eq. 5 N, Eq. 6 f_k
 *   6th-order central finite differences, stencil radius 3 (G1-G3)
 *   3rd-order 2N-storage Runge-Kutta, two state buffers swapped per substep (G7)
 *   runtime reductions ("global averages")
 *
 * Conventions
 *   - Fields, in this order everywhere: lnrho, ux, uy, uz, ax, ay, az  (AC_NFIELDS = 7).
 *   - A caller-visible field is a dense array of nz*ny*nx elements, x fastest:
 *       index = x + nx*(y + ny*z),  element type = the context's dtype (float or double).
 *   - Cell (x, y, z) sits at position (x*lx/nx, y*ly/ny, z*lz/nz).
 *   - All functions return 0 (AC_OK) or a negative ac_status; no exceptions cross the ABI.
 *   - Device work is enqueued on the CUDA stream given to ac_init and is asynchronous unless
 *     stated otherwise.  A context must be used from one host thread at a time.
 *   - Ownership: the library owns everything it allocates; the caller owns every pointer it
 *     passes in, and may free or reuse it as soon as the call returns, except the workspace
 *     given to ac_init, which must outlive the context.
 */
#ifndef AC_MHD_H
#define AC_MHD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AC_NFIELDS 7

typedef struct ac_ctx ac_ctx; /* opaque */

typedef enum { AC_F32 = 0, AC_F64 = 1 } ac_dtype;

typedef enum {
    AC_OK = 0,
    AC_EINVAL = -1, /* NULL pointer, bad grid (n < 8, nx % 4 != 0), non-positive L or cs, negative nu/eta, bad dt */
    AC_ENOMEM = -2, /* device or host allocation failed / workspace too small */
    AC_ECUDA = -3,  /* CUDA error (sticky); text from ac_strerror(AC_ECUDA) on the same thread */
    AC_ESTATE = -4, /* ac_step / ac_reduce / ac_store_state before ac_load_state; a call that is not allowed between substeps */
    AC_ELIMIT = -5  /* ac_reduce_dense_noalloc: more than AC_NOALLOC_MAX_CELLS cells */
} ac_status;

/* Periodic box: n cells and side length per axis; spacing h_a = l_a / n_a (l = 2 pi). */
typedef struct {
    int nx, ny, nz;
    double lx, ly, lz;
} ac_grid;

/* Forcing of one time step (Eq. 4), N of Eq. 5 folded into re, im:
 *   f(x) = re * cos(k.x + phase) - im * sin(k.x + phase).
 * k is in radians per unit length (integer components for l = 2 pi). */
typedef struct {
    double k[3];
    double phase;
    double re[3];
    double im[3];
} ac_forcing;

/* Diagnostics (G18): rms = sqrt(mean over cells of |v|^2), max of |v|.
 * B = curl A (+ external field).  dt_cfl per G15.  nonfinite != 0 if any reduced value is NaN/Inf. */
typedef struct {
    double urms, umax, brms, bmax;
    double lnrho_min, lnrho_max;
    double dt_cfl;
    int nonfinite;
} ac_diag;

/* Bytes of device memory a context needs for this grid and dtype: 2 x 7 ghost-padded field
 * arrays (the two state buffers of PAPER.md:143; the 2N register lives implicitly in their
 * difference) plus forcing tables and reduction scratch.  Returns 0 for an invalid grid. */
size_t ac_workspace_bytes(const ac_grid* grid, ac_dtype dtype);

/* Create a context.
 *   nu, eta, cs        viscosity, magnetic diffusivity, isothermal sound speed
 *   k_f, helicity      forcing shell centre and sigma in [0, 1]; used only by
 *                      ac_make_forcing / ac_forcing_from_draws
 *   workspace_dev      device pointer to at least ac_workspace_bytes() bytes, 256-byte aligned,
 *                      or NULL to let the library cudaMalloc (and free in ac_free)
 *   cuda_stream        a cudaStream_t (as void*), or NULL for the legacy default stream
 * Errors: AC_EINVAL, AC_ENOMEM, AC_ECUDA (no device / not sm_100). */
int ac_init(ac_ctx** out, const ac_grid* grid, ac_dtype dtype, double nu, double eta, double cs,
            double k_f, double helicity, void* workspace_dev, void* cuda_stream);

/* Copy the 7 fields in (dense caller layout -> padded device layout, ghost zones filled by
 * periodic wrap: the "local boundary transfer" of PAPER.md:153).  src_on_device: 0 = host
 * pointers (pinned memory makes the copy asynchronous), 1 = device pointers.  The caller may
 * reuse its buffers when the call returns only if they are pageable host memory or after
 * synchronising the stream. */
int ac_load_state(ac_ctx* ctx, const void* const fields[AC_NFIELDS], int src_on_device);

/* Copy the current state out into 7 dense arrays.  Host destinations: the call synchronises the
 * stream before returning.  Device destinations: asynchronous on the stream. */
int ac_store_state(ac_ctx* ctx, void* const fields[AC_NFIELDS], int dst_on_device);

/* The same for ONE field (q = AC_LNRHO .. AC_AZ order: ln rho, ux, uy, uz, ax, ay, az), so that a
 * caller can stream a state that is too large to hold twice (1024^3 fp64: 8.6 GB per field next
 * to the 122.6 GB workspace).  ac_load_field writes field q of the current state; the context
 * counts as loaded once all 7 fields have been written since ac_init / the last ac_load_state.
 * A host source is staged in the idle state buffer.  Errors: AC_EINVAL, AC_ESTATE (store), AC_ECUDA. */
int ac_load_field(ac_ctx* ctx, int q, const void* field, int src_on_device);
int ac_store_field(ac_ctx* ctx, int q, void* field, int dst_on_device);

/* One full RK3 time step = 3 fused substep kernels (S1-S8 of DESIGN.md), each followed by the
 * ghost-zone kernel (S1) in the default variant, asynchronous.
 * forcing == NULL: no forcing.  The same forcing parameters are used in all 3 substeps (G8).
 * Errors: AC_EINVAL (dt <= 0 or non-finite), AC_ESTATE, AC_ECUDA. */
int ac_step(ac_ctx* ctx, double dt, const ac_forcing* forcing);

/* ---- building blocks of a z-slab decomposition over several GPUs --------------------
 * A rank owns nz_local planes of the global grid (its ac_grid carries nz = nz_local and lz = its share of the box)
 * and the usual 3 ghost planes per side.  Between substeps the ghost planes must hold the neighbour ranks' boundary
 * planes instead of the rank's own periodic images: the caller runs ONE substep with ac_substep (which also refreshes
 * the x / y ghost zones and, harmlessly, writes the local periodic images into the z ghost planes), then overwrites
 * the z ghost planes of every field of the current state with the neighbours' planes.  In the padded layout
 * (ac_state_layout; element (x, y, z) of field q at ac_field_device_ptr(ctx, q) + (x + gx) + pitch * (y + 3) +
 * plane_elems * (z + 3) elements) the planes to send, [nz_local, nz_local + 3) upwards and [3, 6) downwards, and the
 * planes to receive, [0, 3) and [nz_local + 3, nz_local + 6), are contiguous blocks of 3 * plane_elems elements per
 * field, so the exchange can be 2 x 7 plain copies (layouts with packed_pairs == 0 only); ac_halo_pack /
 * ac_halo_unpack below do the same through two dense buffers for every layout, packed fp32 pairs included.
 * ac_substep: substep s = 0, 1, 2 of the 2N-RK3 step; three calls with the same dt and forcing equal ac_step.
 *   The substeps must come in order (AC_ESTATE otherwise; ac_load_state restarts at 0): between substeps the idle
 *   state buffer holds the previous state, from which the 2N register is rebuilt.  Therefore, after substep 0 or 1,
 *   ac_step, ac_load_field, ac_reduce_ext and the HOST-destination forms of ac_store_state / ac_store_field (which
 *   stage in that buffer) return AC_ESTATE; device-destination stores and ac_reduce stay available.
 * ac_reduce_raw: the unnormalised reductions of this rank's cells, out = {sum |u|^2, max |u|^2, sum |B|^2, max |B|^2,
 * min ln rho, max ln rho}, to be combined across ranks (sum, max, sum, max, min, max).  Synchronises the stream. */
typedef struct {
    int elem_bytes;          /* 8: double or packed fp32 pair; 4: plain float */
    int packed_pairs;        /* 1: an element holds cells z and z + nz/2 (fp32 default variant) */
    int gx, pitch, my, mz;   /* x ghost offset, row pitch, padded rows and planes, in elements */
    size_t plane_elems, field_elems;
} ac_layout_info;
int ac_substep(ac_ctx* ctx, int s, double dt, const ac_forcing* forcing);

/* ---- the slab as the paper runs it ("it is critical to carry out computations in parallel with
 * communication", the six functions of a substep PAPER.md:153-158, Fig. 3) -------------------------------------
 * ac_set_slab: declares the context a slab of a global grid of nz_global planes whose first plane is z0_plane
 *   (nz_global == nz: an ordinary periodic box again).  From then on: the forcing of ac_step / ac_substep* is the
 *   GLOBAL wave (the slab adds k_z z0 to the phase itself) and ac_make_forcing / ac_forcing_from_draws take the
 *   global box length for k; the substep kernels leave the z ghost planes to ac_halo_unpack.
 * ac_substep_part: substep s in two launches.  AC_PART_INNER updates the planes [3, nz - 3), which read no z ghost
 *   plane and can therefore run while the halo of the current state is still in flight; AC_PART_OUTER updates the
 *   3 + 3 boundary planes (after ac_halo_unpack), refreshes the x / y ghost zones and swaps the buffers.  INNER
 *   then OUTER equal ac_substep bit for bit.  Errors as ac_substep; AC_ESTATE for OUTER without INNER or twice.
 * ac_halo_bytes: size of ONE halo buffer, 7 fields x 3 planes x (my * pitch) cells of the context's dtype.
 * ac_halo_pack: the 3 bottom planes of cells of the CURRENT state (all fields, x / y ghost zones included) into
 *   send_lo (for the rank below: its upper ghost planes) and the 3 top planes into send_hi (for the rank above),
 *   dense [7][3][my * pitch]; works for packed fp32 pairs too (it picks the lanes).  ac_halo_unpack: recv_lo (the
 *   top planes of the rank below) into the ghost planes below, recv_hi into those above.  Both run on cuda_stream
 *   (NULL: the context's stream) so that a caller can keep the exchange on a second stream; the caller orders them
 *   against the substeps with events: pack after the previous OUTER / ac_substep, unpack before the next OUTER.
 * ac_diag_combine: the diagnostics of the whole box from nranks ac_reduce_raw results (raws[6 * nranks], folded in
 *   rank order: sum, max, sum, max, min, max) with the context's CFL constants; pure host arithmetic. */
#define AC_PART_INNER 1
#define AC_PART_OUTER 2
int ac_set_slab(ac_ctx* ctx, int z0_plane, int nz_global);
int ac_substep_part(ac_ctx* ctx, int s, double dt, const ac_forcing* forcing, int part);
size_t ac_halo_bytes(const ac_ctx* ctx);
int ac_halo_pack(ac_ctx* ctx, void* send_lo_dev, void* send_hi_dev, void* cuda_stream);
int ac_halo_unpack(ac_ctx* ctx, const void* recv_lo_dev, const void* recv_hi_dev, void* cuda_stream);
int ac_diag_combine(const ac_ctx* ctx, const double* raws, int nranks, ac_diag* out);

/* The exchange as one kernel over peer memory (no staging buffers, no library collective on the data path):
 * ac_halo_pull copies the top 3 cell planes of the slab below and the bottom 3 of the slab above straight from THEIR
 * state arrays into this context's z ghost planes (all fields, x / y ghost zones included, packed fp32 lanes picked),
 * on cuda_stream (NULL: the context's).  below_workspace / above_workspace = the base of the neighbours' workspaces as
 * THIS process can address them: ac_workspace_ptr of a context of the same process, or the pointer ac_ipc_open
 * returns for a handle another process exported with ac_ipc_export (CUDA IPC: the same GPU, or a peer GPU over
 * NVLink).  All ranks must have the same local grid, dtype and variant and make the same calls in the same order
 * (the neighbours' current state is then at the same workspace offset as ours).  The caller orders the pull after the
 * neighbours' previous substep has finished (events; cudaIpcEventHandle between processes) and before its own
 * AC_PART_OUTER.  ac_ipc_export needs a workspace the library allocated itself (ac_init with workspace_dev = NULL);
 * the handle is 64 bytes (cudaIpcMemHandle_t).  Errors: AC_EINVAL, AC_ESTATE, AC_ECUDA. */
int ac_halo_pull(ac_ctx* ctx, const void* below_workspace, const void* above_workspace, void* cuda_stream);
void* ac_workspace_ptr(ac_ctx* ctx);
int ac_ipc_export(ac_ctx* ctx, void* handle64);
int ac_ipc_open(const void* handle64, void** workspace_out);
int ac_ipc_close(void* workspace);
int ac_state_layout(const ac_ctx* ctx, ac_layout_info* out);
void* ac_field_device_ptr(ac_ctx* ctx, int q);
int ac_reduce_raw(ac_ctx* ctx, double out[6]);

/* rms/max reductions of |u| and |B| and min/max of ln rho over the current state, and the CFL
 * time step dt = min(C_u h/(umax + cs), C_nu h^2/max(nu, eta)) (G15).  Deterministic (fixed
 * two-stage tree, no floating-point atomics).  Synchronises the stream. */
int ac_reduce(ac_ctx* ctx, ac_diag* out);

/* Extended diagnostics: volume means of the kinetic helicity omega.u (omega = curl u) and of the
 * current helicity j.B (Eq. 11, with mu0 = rho0 = 1; j = grad div A - lap A as in
 * Eq. 2, B = curl A + external field; in a periodic box <j> = 0, so <j.B> is also the mean of the fluctuating parts
 * j'.b' of Eq. 11), the largest Alfven speed |B| / sqrt(rho), and the CFL step with the Alfven term of reading G15,
 * dt = min(C_u h / (umax + sqrt(cs^2 + va_max^2)), C_nu h^2 / max(nu, eta)).  Runs ac_reduce plus one gather
 * kernel; deterministic; synchronises the stream.  Scratch lives in the idle state buffer, so inside a step driven
 * by ac_substep (after substep 0 or 1) the call returns AC_ESTATE.
 * ac_reduce_ext_raw: this rank's {sum omega.u, sum j.B, max |B|^2 / rho} for a slab decomposition (sum, sum, max). */
typedef struct {
    double kin_hel, cur_hel, va_max;
    double dt_cfl_alfven;
    int nonfinite;
} ac_diag_ext;
int ac_reduce_ext(ac_ctx* ctx, ac_diag_ext* out);
int ac_reduce_ext_raw(ac_ctx* ctx, double out[3]);

/* ac_reduce_dense_noalloc: the reductions of ac_reduce_raw WITHOUT a context and without any allocation, for callers
 * that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses that forbid it).  It calls no
 * cudaMalloc / cudaFree / cudaMallocHost and no allocating library routine, does no host <-> device copy and does not
 * synchronise: two kernel launches on cuda_stream (NULL: the default stream) of the CURRENT device.
 *   state_dev  DEVICE pointer, dense [7][nz][ny][nx] elements of dtype (float / double), x fastest, field order
 *              ln rho, u_x, u_y, u_z, A_x, A_y, A_z: the array ac_load_state takes.  No ghost zones: the periodic
 *              wrap is taken by index.  Read only; owned by the caller.
 *   grid       as for ac_init (n >= 8 per axis, nx % 4 == 0); bext: uniform imposed field added to curl A, or NULL.
 *   raw_dev    DEVICE pointer to 6 doubles (8-byte aligned), written by the second launch: {sum |u|^2, max |u|^2,
 *              sum |B|^2, max |B|^2, min ln rho, max ln rho} with B = curl A + B_ext (6th-order first derivatives,
 *              PAPER.md:85, 119; G1), i.e. ac_reduce_raw's six numbers; ac_diag_combine (nranks = 1) turns a host copy
 *              of them into rms / max values and the CFL step (G15).  Per cell the arithmetic is that of ac_reduce,
 *              so the maxima equal ac_reduce_raw's bit for bit, the sums to summation order (deterministic: fixed
 *              two-stage tree); a non-finite ln rho or A makes sum |u|^2 non-finite.
 * Scratch: the per-block partials live in a fixed array inside the library (static __device__, 3 MiB, held by every GPU
 * that loads the library until the process exits), so the size is LIMITED: at most AC_NOALLOC_MAX_CELLS = 2^27 cells
 * (512^3, BASELINE config 4; ac_noalloc_max_cells() returns it); more returns AC_ELIMIT and launches nothing.  Every
 * call on a device shares that array and finds the previous call's partials in it; a call writes every partial it reads,
 * so nothing has to be cleared - but two calls that overlap on the GPU (different streams of one device, or different
 * host threads without ordering) RACE on it: order them on one stream or with events.  The first call on each device
 * looks the array's device address up (cudaGetSymbolAddress; no allocation): under graph capture make one call on the
 * device before the capture begins.
 * Errors: AC_EINVAL (NULL / misaligned / non-device pointers, pointers of another device, bad grid or dtype, non-finite
 * bext), AC_ELIMIT, AC_ECUDA. */
#define AC_NOALLOC_MAX_CELLS (1LL << 27)
int ac_reduce_dense_noalloc(const void* state_dev, ac_dtype dtype, const ac_grid* grid, const double bext[3],
                            double* raw_dev, void* cuda_stream);
long long ac_noalloc_max_cells(void);

/* Host helpers for Eq. 4-6 (no device work).
 * ac_forcing_from_draws: u1, u2, u3 in [0, 1) choose the shell vector (index floor(u1*len) into
 *   the lexicographically sorted shell k_f - 1/2 <= |k| <= k_f + 1/2, G11), the phase
 *   (-pi + 2 pi u2) and the angle of e-hat around k (2 pi u3, G9); amplitude N = f0 cs sqrt(|k| cs/dt).
 * ac_make_forcing: the same with u_i = (splitmix64(splitmix64(seed) ^ (3*step + i)) >> 11) * 2^-53. */
int ac_forcing_from_draws(const ac_ctx* ctx, double u1, double u2, double u3, double dt, double f0,
                          ac_forcing* out);
/* The same without a context (pure host arithmetic, usable on a machine without a GPU):
 * k_f, helicity (sigma), cs and the box as given to ac_init.  Errors: AC_EINVAL. */
int ac_forcing_params(double k_f, double helicity, double cs, const ac_grid* grid, double u1, double u2, double u3,
                      double dt, double f0, ac_forcing* out);
int ac_make_forcing(const ac_ctx* ctx, uint64_t seed, uint64_t step, double dt, double f0, ac_forcing* out);

/* Optional knobs.  ac_set_bext: uniform external field added to curl A in j x B, u x B and the
 * |B| diagnostics (test hook for the Alfven-wave check, G16; default 0).  ac_set_cfl: C_u, C_nu
 * (defaults 0.4, 0.25).  ac_set_variant: substep kernel variant (0 = default/fastest,
 * others documented in DESIGN.md; AC_EINVAL if unknown). */
int ac_set_bext(ac_ctx* ctx, const double b[3]);
/* ac_set_upwind: 1 = the continuity equation uses the high-order upwinding the paper's production
 * runs used (Dobler et al. 2006; off in its benchmark, and in every
 * BASELINE config).  Reading G17: -u.grad ln rho keeps the 6th-order central derivative and gains
 * + sum_a |u_a| / (60 h_a) [f(-3) - 6 f(-2) + 15 f(-1) - 20 f(0) + 15 f(+1) - 6 f(+2) + f(+3)],
 * which makes each u_a d_a ln rho the 5th-order upwind-biased derivative.  Default 0. */
int ac_set_upwind(ac_ctx* ctx, int on);
/* ac_set_forcing_mode: how the forcing of Eq. 4 enters the three substeps, which the paper does not say (G8).
 * 0 (default, every reported number) = f is a term of the right-hand side in all three substeps; 1 = the forcing is
 * delta-correlated and acts as ONE impulse u += dt f per time step, after the last substep (the
 * Pencil-Code convention behind Eq. 5's dt^-1/2).  The net impulse is the same, the O(dt^2) coupling terms differ.
 * Not between the substeps of a step (AC_ESTATE). */
int ac_set_forcing_mode(ac_ctx* ctx, int mode);
/* ac_set_mixed: reading of the mixed-derivative scheme, which the paper does not print (G2).  0 (default, all
 * reported parity and every BASELINE config) = bidiagonal 12-point stencil; 1 = tensor product D_a(D_b f), 36
 * points, also radius 3 and 6th order, taken as D_z (D_x f), D_z (D_y f), D_y (D_x f).  With the default kernel
 * (variant 0) mode 1 is a build of the same fused substep kernel in which the z-mixed terms are z stencils of the
 * in-plane first derivatives and the in-plane ones are y stencils of d_x f staged in shared memory (SURVEY.md 8(f)
 * NEXT-4, "staged intermediates"); variants 1 and 2 run the direct kernel.  Like ac_set_variant it must be called
 * before ac_load_state (a loaded state is dropped: AC_ESTATE until the next load). */
int ac_set_mixed(ac_ctx* ctx, int mode);
int ac_set_cfl(ac_ctx* ctx, double c_u, double c_nu);
int ac_set_variant(ac_ctx* ctx, int variant);

/* Number of kernels this context has launched so far (for the bench's gpu_launches). */
long long ac_launch_count(const ac_ctx* ctx);

/* Destroy the context (ac_free(NULL) is a no-op).  Synchronises the stream first. */
void ac_free(ac_ctx* ctx);

/* Static text for a status; for AC_ECUDA the last CUDA error text seen on this thread. */
const char* ac_strerror(int status);

/* Library version string, e.g. "ac_mhd 0.1 sm_100a". */
const char* ac_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AC_MHD_H */
