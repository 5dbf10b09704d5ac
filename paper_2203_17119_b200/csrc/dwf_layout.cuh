// Device-side helpers for the tiled native layout (see dwf_internal.h / DESIGN.md §4).
#pragma once
#include "dwf_internal.h"

namespace dwf {

struct Coord {
    int x[4];
};

// tile index <-> tile coordinates (the ONE place that fixes the order in which tiles are laid out in
// memory and scheduled; x fastest)
__host__ __device__ inline void tile_coords(const Geom& g, int tile, int c[4]) {
    c[0] = tile % g.NT[0];
    int r = tile / g.NT[0];
    c[1] = r % g.NT[1];
    r /= g.NT[1];
    c[2] = r % g.NT[2];
    c[3] = r / g.NT[2];
}
__host__ __device__ inline int tile_index(const Geom& g, const int c[4]) {
    return ((c[3] * g.NT[2] + c[2]) * g.NT[1] + c[1]) * g.NT[0] + c[0];
}

// (tile, lane, parity) -> global coordinates
__host__ __device__ inline Coord site_coords(const Geom& g, int tile, int lane, int parity) {
    const int txh_n = g.T[0] >> 1;
    int txh = lane % txh_n;
    int r = lane / txh_n;
    int ty = r % g.T[1];
    r /= g.T[1];
    int tz = r % g.T[2];
    int tt = r / g.T[2];
    int tc[4];
    tile_coords(g, tile, tc);
    Coord c;
    c.x[1] = tc[1] * g.T[1] + ty;
    c.x[2] = tc[2] * g.T[2] + tz;
    c.x[3] = tc[3] * g.T[3] + tt;
    int xpar = (parity + c.x[1] + c.x[2] + c.x[3]) & 1;
    c.x[0] = tc[0] * g.T[0] + 2 * txh + xpar;
    return c;
}

// global coordinates -> native site index tile*TS + lane (parity is implied by the coordinates)
__host__ __device__ inline void native_site(const Geom& g, const int x[4], int& tile, int& lane) {
    int ix = x[0] / g.T[0], tx = x[0] - ix * g.T[0];
    int iy = x[1] / g.T[1], ty = x[1] - iy * g.T[1];
    int iz = x[2] / g.T[2], tz = x[2] - iz * g.T[2];
    int it = x[3] / g.T[3], tt = x[3] - it * g.T[3];
    const int tc[4] = {ix, iy, iz, it};
    tile = tile_index(g, tc);
    lane = ((tt * g.T[2] + tz) * g.T[1] + ty) * (g.T[0] >> 1) + (tx >> 1);
}

__host__ __device__ inline long long lex_index(const Geom& g, const int x[4]) {
    return (((long long)x[3] * g.L[2] + x[2]) * g.L[1] + x[1]) * g.L[0] + x[0];
}

}  // namespace dwf
