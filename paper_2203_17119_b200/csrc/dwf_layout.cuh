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

// ---- lane order inside a tile (the ONE place that fixes it) -------------------------------------------------------
// lane = ((tt*T2 + tz)*T1 + py)*(T0/2) + tx/2  with  py = ty ^ tz  when the tile is 4 wide in y and z (g.swz), else
// py = ty.  The XOR rotates the y rows of every (tz, tt) plane differently, so that in the Dhop kernels' shared-memory
// slices the lanes of a quarter warp and their +-y / +-x face neighbours fall into 8 distinct 16-byte bank groups
// (DESIGN.md section 5.1); it leaves every t-slab, z-face and y-row a contiguous run, as the TMA boxes need.
__host__ __device__ inline int lane_from_local(const Geom& g, const int y[4]) {
    const int py = g.swz ? (y[1] ^ y[2]) : y[1];
    return ((y[3] * g.T[2] + y[2]) * g.T[1] + py) * (g.T[0] >> 1) + (y[0] >> 1);
}
// lane -> tile-local coordinates of the site of parity `tile_parity_offset + ...`: x[0] needs the parity of the site
__host__ __device__ inline void local_from_lane(const Geom& g, int lane, int xpar_base, int x[4]) {
    const int txh_n = g.T[0] >> 1;
    const int txh = lane % txh_n;
    int r = lane / txh_n;
    const int py = r % g.T[1];
    r /= g.T[1];
    x[2] = r % g.T[2];
    x[3] = r / g.T[2];
    x[1] = g.swz ? (py ^ x[2]) : py;
    x[0] = 2 * txh + ((xpar_base + x[1] + x[2] + x[3]) & 1);
}

// (tile, lane, parity) -> global coordinates
__host__ __device__ inline Coord site_coords(const Geom& g, int tile, int lane, int parity) {
    int tc[4];
    tile_coords(g, tile, tc);
    // tile origins are even in every direction or the tile extent is even: the local parity offset is the parity of the origin
    const int opar = (tc[1] * g.T[1] + tc[2] * g.T[2] + tc[3] * g.T[3] + tc[0] * g.T[0]) & 1;
    int x[4];
    local_from_lane(g, lane, parity + opar, x);
    Coord c;
    for (int mu = 0; mu < 4; ++mu) c.x[mu] = tc[mu] * g.T[mu] + x[mu];
    return c;
}

// global coordinates -> native site index tile*TS + lane (parity is implied by the coordinates)
__host__ __device__ inline void native_site(const Geom& g, const int x[4], int& tile, int& lane) {
    int tc[4], y[4];
    for (int mu = 0; mu < 4; ++mu) { tc[mu] = x[mu] / g.T[mu]; y[mu] = x[mu] - tc[mu] * g.T[mu]; }
    tile = tile_index(g, tc);
    lane = lane_from_local(g, y);
}

__host__ __device__ inline long long lex_index(const Geom& g, const int x[4]) {
    return (((long long)x[3] * g.L[2] + x[2]) * g.L[1] + x[1]) * g.L[0] + x[0];
}

}  // namespace dwf
