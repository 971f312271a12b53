// k_stage_common.cuh -- tiling shared by the fused stage kernels (k_hydro.cu, k_rad.cu).
//
// 2.5-D marching tiles: a CTA owns a TX x TY patch of columns and marches along z over a chunk of
// planes.  At step k it holds
//   * a ring of five planes k-1..k+3 of the cell-centred reconstruction variables of its own
//     columns in shared memory (the z stencil of PPM for cell k+1),
//   * plane k with a star-shaped halo of 3 cells in x and y (the x/y stencils of the tile cells
//     and of the one cell beyond each tile edge whose face state a tile-edge flux needs).
// Fluxes live in registers / shared memory only; HBM sees one read of the conserved state (plus
// halo re-reads that L2 absorbs) and one write of the updated state per stage.
#pragma once

#include "qk_internal.h"

namespace qk {

constexpr int TX = 32;            // tile width  (x, one warp per row: coalesced 256-byte rows)
constexpr int TY = 8;             // tile height (y)
constexpr int NT = TX * TY;       // threads per CTA
constexpr int RING = 5;           // planes k-1..k+3
constexpr int HALO = 3;           // in-plane star halo
constexpr int N_HALO_X = 2 * HALO * TY;          // halo cells left/right of the tile rows
constexpr int N_HALO = N_HALO_X + 2 * HALO * TX; // + below/above the tile columns
constexpr int N_EDGE_X = 2 * TY;                 // cells -1 and TX of every row
constexpr int N_EDGE = N_EDGE_X + 2 * TX;        // + cells -1 and TY of every column

static_assert(N_HALO <= NT, "one halo cell per thread");
static_assert(N_EDGE <= NT && TX + TY <= NT, "one edge item per thread");

__device__ __forceinline__ int ring_slot(int plane) { return (plane + 2 * RING) % RING; }

// tile-local coordinates of halo cell h (0 <= h < N_HALO)
__device__ __forceinline__ void halo_cell(int h, int &lx, int &ly)
{
    if (h < N_HALO_X) {
        ly = h / (2 * HALO);
        const int q = h - ly * (2 * HALO);
        lx = q < HALO ? q - HALO : TX + (q - HALO);
    } else {
        const int u = h - N_HALO_X;
        const int r = u / TX;
        lx = u - r * TX;
        ly = r < HALO ? r - HALO : TY + (r - HALO);
    }
}

// tile-local coordinates of edge cell e (0 <= e < N_EDGE): the cells one beyond the tile along x
// (e < N_EDGE_X) or along y; `high` tells which side
__device__ __forceinline__ void edge_cell(int e, int &lx, int &ly, bool &along_x, bool &high)
{
    if (e < N_EDGE_X) {
        along_x = true;
        ly = e >> 1;
        high = (e & 1) != 0;
        lx = high ? TX : -1;
    } else {
        along_x = false;
        const int u = e - N_EDGE_X;
        high = u >= TX;
        lx = high ? u - TX : u;
        ly = high ? TY : -1;
    }
}

__device__ __forceinline__ bool in_array(const Geom &g, int i, int j)
{
    return i >= -NG && i < g.nx + NG && j >= -NG && j < g.ny + NG;
}

}  // namespace qk
