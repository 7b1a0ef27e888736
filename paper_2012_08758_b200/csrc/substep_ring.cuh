// Fused RK substep, variant "ring" (the default): 2.5-D streaming with TMA.
//
// A CTA owns an xy tile of TX x TY cells and marches along z over a chunk of planes.  For every z
// plane ONE 4-D TMA box load (x, y, 1 plane, 7 fields) brings the tile plus its r = 3 xy halo of
// all seven fields from the ghost-padded arrays into a ring of NP plane slots in shared memory,
// completion signalled on an mbarrier per slot.  Planes z-3..z+3 are resident while plane z is
// computed, the remaining slots are prefetched ahead.  Each thread owns one (x, y) column and
// evaluates the whole right-hand side and the 2N-RK3 update for its cell from shared memory
// (S1-S8 of DESIGN.md); results go straight to global memory (coalesced rows) together with the
// periodic ghost images of boundary cells.  xy-halo re-reads hit L2; every input plane is read
// from HBM once per tile row/column neighbourhood.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"
#include "layout.cuh"
#include "mhd_cell.cuh"

namespace ac {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2,
                                            int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::
            "r"(smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

template <typename T, int TX_, int TY_, int NP_, int HXS_>
struct RingCfg {
    static constexpr int TX = TX_, TY = TY_, NP = NP_, HXS = HXS_;
    static constexpr int WX = TX + 2 * HXS;           // smem row length (elements)
    static constexpr int WY = TY + 2 * R;             // smem rows per plane
    static constexpr int PLANE = WX * WY;             // elements per field per plane
    static constexpr int BOX_BYTES = NFIELDS * PLANE * (int)sizeof(T);
    static constexpr int SLOT_BYTES = (BOX_BYTES + 127) / 128 * 128;
    static constexpr int SMEM_BYTES = NP * SLOT_BYTES + NP * 8 + 128;
    static constexpr int THREADS = TX * TY;
    static_assert(NP >= 2 * R + 2, "ring needs the 7 resident planes plus at least one prefetch slot");
    static_assert((WX * sizeof(T)) % 16 == 0, "TMA box rows must be a multiple of 16 bytes");
};

template <typename T, typename Cfg>
__global__ void __launch_bounds__(Cfg::THREADS, 1)
    substep_ring_kernel(const __grid_constant__ SubstepArgs<T> a, const __grid_constant__ CUtensorMap map_in, int cz) {
    constexpr int TX = Cfg::TX, TY = Cfg::TY, NP = Cfg::NP, HXS = Cfg::HXS, WX = Cfg::WX, PLANE = Cfg::PLANE;
    extern __shared__ unsigned char smem_raw[];
    // 128-byte aligned base for the TMA destinations
    unsigned char* smem = (unsigned char*)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
    uint64_t* bars = (uint64_t*)(smem + NP * Cfg::SLOT_BYTES);

    const Layout& L = a.L;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int tid = ty * TX + tx;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int zs = blockIdx.z * cz;
    const int ze = min(zs + cz, L.nz);
    const int x = x0 + tx, y = y0 + ty;
    const bool valid = (x < L.nx) && (y < L.ny);

    if (tid == 0) {
        for (int s = 0; s < NP; s++) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // plane p (interior z coordinate, may be in the ghosts) -> ring slot (p - (zs - R)) % NP
    const int pfirst = zs - R, plast = ze - 1 + R;
    auto issue = [&](int p) {
        const int k = p - pfirst;
        const int slot = k % NP;
        mbar_expect_tx(&bars[slot], (uint32_t)Cfg::BOX_BYTES);
        tma_load_4d(smem + slot * Cfg::SLOT_BYTES, &map_in, &bars[slot], x0 - HXS + L.gx, y0, p + R, 0);
    };
    if (tid == 0) {
        for (int p = pfirst; p < pfirst + NP && p <= plast; p++) issue(p);
    }

    const int cell_off = (ty + R) * WX + tx + HXS;
    const bool edge_xy = (x < R) | (x >= L.nx - R) | (y < R) | (y >= L.ny - R);

    // wait for the first 6 planes once; inside the loop only the newest plane (z + 3) is waited for
    for (int p = pfirst; p < pfirst + 2 * R; p++) mbar_wait(&bars[(p - pfirst) % NP], (uint32_t)(((p - pfirst) / NP) & 1));

    for (int z = zs; z < ze; z++) {
        {
            const int k = z + R - pfirst;
            mbar_wait(&bars[k % NP], (uint32_t)((k / NP) & 1));
        }
        const T* sp[2 * R + 1];
#pragma unroll
        for (int d = 0; d < 2 * R + 1; d++) {
            const int k = z - R + d - pfirst;
            sp[d] = (const T*)(smem + (k % NP) * Cfg::SLOT_BYTES) + cell_off;
        }
        if (valid) {
            const size_t c0 = L.idx(x, y, z);
            T prev[NFIELDS];
#pragma unroll
            for (int q = 0; q < NFIELDS; q++) prev[q] = (a.p.substep != 0) ? a.out[q][c0] : T(0);
            T fc = T(0), fs = T(0);
            if (a.p.has_forcing) forcing_phase<T>(a.ftab, L.nx, L.ny, L.nz, x, y, z, fc, fs);
            auto fetch = [&](int q, int dx, int dy, int dz) -> T { return sp[dz + R][q * PLANE + dy * WX + dx]; };
            T res[NFIELDS];
            substep_cell<T>(fetch, a.c, a.p, prev, fc, fs, res);
            const bool edge = edge_xy | (z < R) | (z >= L.nz - R);
#pragma unroll
            for (int q = 0; q < NFIELDS; q++) store_with_images<T>(a.out[q], L, x, y, z, res[q], edge);
        }
        __syncthreads();  // every thread is done with plane z - 3: its slot may be refilled
        if (tid == 0) {
            const int p = z - R + NP;
            if (p <= plast) issue(p);
        }
    }
}

}  // namespace ac
