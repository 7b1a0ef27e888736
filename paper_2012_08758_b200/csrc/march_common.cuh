// Definitions shared by the z-march substep kernels (substep_pair.cuh, substep_march.cuh) and the reductions:
// tile geometry, shared-memory ring layout, the weight block, mbarrier / TMA primitives.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "layout.cuh"
#include "vec2.cuh"

namespace ac {

constexpr int M_TX = 16, M_TY = 8, M_COLS = M_TX * M_TY;
constexpr int M_WORKERS = 2 * M_COLS;          // U and A roles
constexpr int M_THREADS = M_WORKERS + 128;    // + the producer warpgroup (one working lane) that feeds the ring
constexpr int M_REGS_WORKER = 240, M_REGS_PRODUCER = 24;   // setmaxnreg: 128 x (240 + 240 + 24) = 384 x 168, the registers the CTA is launched with
constexpr int M_HX = 4;                  // x halo of the tile in shared memory (>= R; 32 bytes keeps TMA boxes aligned)
constexpr int M_WX = M_TX + 2 * M_HX;    // 24
constexpr int M_WY = M_TY + 2 * R;       // 14
constexpr int M_PLANE = M_WX * M_WY;     // elements per field per plane slot
constexpr int M_NP = 8;                  // ring slots: planes p-3 .. p resident, p+1 .. p+3 in flight
constexpr int M_NPP = 5;                 // previous-state ring slots
constexpr int M_ND = 5;                  // mailbox depth: the A role runs at most 5 iterations ahead of the U role
constexpr int M_LEAD = 3;                // planes issued ahead of the one being processed
constexpr int M_CZMAX = 512;             // longest z chunk (bounds the z phase table in shared memory)
constexpr int M_NF = 7;

constexpr int M_SLOT_BYTES = M_NF * M_PLANE * 8;        // 18816 (multiple of 128)
constexpr int M_PSLOT_BYTES = M_NF * M_COLS * 8;        // 7168
constexpr int M_MBOX_BYTES = 4 * M_COLS * 8;            // 4096 per depth: (j x B)/rho and the upwind term
constexpr int M_OFF_PREV = M_NP * M_SLOT_BYTES;
constexpr int M_OFF_MBOX = M_OFF_PREV + M_NPP * M_PSLOT_BYTES;
constexpr int M_OFF_ZTAB = M_OFF_MBOX + M_ND * M_MBOX_BYTES;
constexpr int M_OFF_BARS = M_OFF_ZTAB + M_CZMAX * 2 * 8;
constexpr int M_NBARS = 2 * M_NP + 4 * M_ND;
constexpr int M_SMEM_BYTES = M_OFF_BARS + M_NBARS * 8;
static_assert(M_SLOT_BYTES % 128 == 0 && M_PSLOT_BYTES % 128 == 0, "TMA destinations must stay 128-byte aligned");
static_assert(M_SMEM_BYTES <= 232448, "exceeds the 227 KB of shared memory a CTA may use");

// Weights with the grid spacing (and, for the U role, the 1/3 of grad div and the 4/3 of the
// diagonal second derivative) folded in; n* = negated copies (packed fp32 has no negate modifier in PTX).
template <typename E>
struct MarchCoef {
    E c1x[3], c1y[3], c1z[3], nc1z[3];
    // U role: L_i = lap u_i + 1/3 (grad div u)_i
    E w2x[3][3], w2y[3][3], w2z[3][3], w20[3];      // [component][m-1]; w20 = centre weight summed over the axes
    E cm3xy[3], cm3xz[3], ncm3xz[3], cm3yz[3], ncm3yz[3];
    // A role
    E c2x[3], c2y[3], c2z[3], nc2x[3], nc2y[3], nc2z[3];
    E c20all, nc20yz, nc20xz, nc20xy, c20x, c20y, c20z;
    E cmxy[3], cmxz[3], ncmxz[3], cmyz[3], ncmyz[3];
    // upwind correction of the continuity equation (G17; UPW kernels only): delta6 / (60 h)
    E c6x[3], c6y[3], c6z[3], c60x, c60y, c60z;
    // physics and time stepping
    E nu, eta, ncs2, bext[3], rk_a, rk_b, fre[3], nfim[3], n23;
    // tensor-product mixed derivatives (pair-march MIX build): 1/3 of the first-derivative weights
    E c13y[3], c13z[3], nc13z[3];
};

template <typename T>
struct MarchArgs {
    using E = typename ElemOf<T>::E;
    E* out[M_NF];        // buffer 1-cur: previous state on entry (read through map_prev), new state on exit
    const T* ftab;       // forcing tables [cx(nx) sx(nx) cy(ny) sy(ny) cz(nzfull) sz(nzfull)]
    Layout L;            // layout in 8-byte elements; L.nz = number of (packed) planes
    int nz_full;         // planes of the caller's grid (= L.nz, or 2 L.nz for packed fp32)
    int cz;              // planes per z chunk (<= M_CZMAX)
    int z_begin, z_end;  // planes [z_begin, z_end) are updated by this launch (the whole grid, or the inner / outer part of a slab)
    int substep;
    int has_forcing;
    int wrap_z;          // 1: write the periodic z images too (single box); 0: a slab neighbour fills the z ghost planes
    MarchCoef<E> c;
};

// ---- mbarrier / TMA primitives -------------------------------------------------------------------
__device__ __forceinline__ uint32_t m_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void m_bar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(m_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void m_bar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(m_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void m_bar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(m_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool m_bar_try(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(m_smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// try_wait suspends the warp for a hardware-limited time by itself; SLEEP_NS > 0 adds a nanosleep between polls
template <int SLEEP_NS>
__device__ __forceinline__ void m_bar_wait(uint64_t* bar, uint32_t parity) {
    while (!m_bar_try(bar, parity)) {
        if (SLEEP_NS > 0) __nanosleep(SLEEP_NS);
    }
}
// Measured at 512^3 on B200 (16 combinations of 0 / 20 ns at the four wait sites): the fp64 kernel is fastest
// (21.7 ms per step against 22.7 without any sleep and 28.5 with the U role sleeping alone) when the U role
// sleeps at the mailbox and the A role at the ring; the packed fp32 kernel is fastest without any sleep
// (10.85 against 11.3-11.9 ms).  Swapping which role gets the higher warp ids made no difference.  Over 40
// steps both kernels run into the 1000 W power cap (SM clock 1725 MHz fp64 / 1845 MHz fp32: 22.5 / 11.4 ms);
// the ranking of the policies stays the same there and longer sleeps change nothing.
template <typename T>
struct MarchWait {
    static constexpr int MAILBOX_NS = ElemOf<T>::LANES == 1 ? 20 : 0;   // U role waiting for (j x B)/rho
    static constexpr int RING_A_NS = ElemOf<T>::LANES == 1 ? 20 : 0;    // A role waiting for its next plane
    static constexpr int RING_U_NS = 0;
    static constexpr int PRODUCER_NS = 200;   // once per plane (~1 us); 20 ns polled 54 times per plane for nothing
};
__device__ __forceinline__ void m_tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2,
                                              int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::
            "r"(m_smem_u32(dst)),
        "l"(map), "r"(m_smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

// ---- small stencil helpers -----------------------------------------------------------------------
template <typename E>
__device__ __forceinline__ E m_dot3(const E (&c)[3], const E (&d)[3]) {
    E r = vmul(c[0], d[0]);
    r = vfma(c[1], d[1], r);
    r = vfma(c[2], d[2], r);
    return r;
}
template <typename E>
__device__ __forceinline__ E m_dot3(const E (&c)[3], const E (&d)[3], E r) {
    r = vfma(c[0], d[0], r);
    r = vfma(c[1], d[1], r);
    r = vfma(c[2], d[2], r);
    return r;
}
}  // namespace ac
