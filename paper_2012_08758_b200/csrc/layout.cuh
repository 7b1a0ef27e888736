// Ghost-padded device layout of one field (the paper's m = n + 2r grid).
//
// A field is stored as mz x my x pitch elements, x fastest.  Cell (x, y, z) of the periodic
// domain lives at padded index (x + gx, y + 3, z + 3); the r = 3 ghost layers on every side hold
// periodic images of the opposite side ("wrapping ghost zones around").  gx is 32
// bytes' worth of elements so that interior rows start on a 32-byte sector boundary and TMA boxes
// (16-byte granular) can start at x - gx' for any tile; the pitch is a multiple of 32 bytes.
#pragma once
#include <cstddef>

namespace ac {

constexpr int R = 3;  // stencil radius

struct Layout {
    int nx, ny, nz;      // interior cells
    int gx;              // ghost offset in x (>= R)
    int pitch, my, mz;   // padded extents
    size_t plane;        // pitch * my
    size_t field;        // pitch * my * mz  (elements per padded field)

    __host__ __device__ size_t idx(int x, int y, int z) const {  // interior coordinates, may run into the ghosts
        return (size_t)(x + gx) + (size_t)pitch * (size_t)(y + R) + plane * (size_t)(z + R);
    }
};

inline Layout make_layout(int nx, int ny, int nz, size_t elem_size) {
    Layout L;
    L.nx = nx;
    L.ny = ny;
    L.nz = nz;
    L.gx = (int)(32 / elem_size);
    int per32 = (int)(32 / elem_size);
    L.pitch = ((nx + 2 * L.gx + per32 - 1) / per32) * per32;
    L.my = ny + 2 * R;
    L.mz = nz + 2 * R;
    L.plane = (size_t)L.pitch * L.my;
    L.field = L.plane * L.mz;
    // keep every field 256-byte aligned inside the workspace
    size_t per256 = 256 / elem_size;
    L.field = ((L.field + per256 - 1) / per256) * per256;
    return L;
}

}  // namespace ac
