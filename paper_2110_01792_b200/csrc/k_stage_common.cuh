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
#include "qk_math.cuh"

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

// ---- per-cell / per-face building blocks shared by the tile kernels and the sweep kernels ------

// The select-only PPM limiter of qk_math.cuh (ppm_face_states_t<true>) for NV variables of one cell in
// lockstep: every elementary step is issued for all variables before the next step starts, so that the
// fp64 pipe (8-cycle latency, one warp instruction per 2 cycles per scheduler) always has NV independent
// operations in flight.  Same operations in the same order per variable, hence the same bits.
template <int NV, typename Q>
__device__ __forceinline__ void ppm_lockstep(Q q, double lo[NV], double hi[NV])
{
    const double w7 = 7.0 / 12.0, w1 = 1.0 / 12.0;
    double a[NV], b[NV], c[NV], d[NV], e[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { a[v] = q(v, 0); b[v] = q(v, 1); c[v] = q(v, 2); d[v] = q(v, 3); e[v] = q(v, 4); }
    double lf[NV], hf[NV], fl[NV], ce[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) lf[v] = w7 * (b[v] + c[v]) - w1 * (d[v] + a[v]);
#pragma unroll
    for (int v = 0; v < NV; ++v) hf[v] = w7 * (c[v] + d[v]) - w1 * (e[v] + b[v]);
#pragma unroll
    for (int v = 0; v < NV; ++v) fl[v] = lesser(b[v], lesser(c[v], d[v]));
#pragma unroll
    for (int v = 0; v < NV; ++v) ce[v] = greater(b[v], greater(c[v], d[v]));
#pragma unroll
    for (int v = 0; v < NV; ++v) lf[v] = lesser(greater(lf[v], fl[v]), ce[v]);
#pragma unroll
    for (int v = 0; v < NV; ++v) hf[v] = lesser(greater(hf[v], fl[v]), ce[v]);
    double below[NV], above[NV], s[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { below[v] = c[v] - lf[v]; above[v] = hf[v] - c[v]; }
    // monotonized-central slope (mc_slope) of (b, c, d)
    double dW[NV], dE[NV], dC[NV], bound[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { dW[v] = c[v] - b[v]; dE[v] = d[v] - c[v]; }
#pragma unroll
    for (int v = 0; v < NV; ++v) dC[v] = 0.5 * (d[v] - b[v]);
#pragma unroll
    for (int v = 0; v < NV; ++v) bound[v] = lesser(fabs(dC[v]), lesser(2.0 * fabs(dW[v]), 2.0 * fabs(dE[v])));
#pragma unroll
    for (int v = 0; v < NV; ++v) s[v] = (dW[v] * dE[v] <= 0.0) ? 0.0 : (dC[v] > 0.0 ? bound[v] : -bound[v]);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const bool extremum = below[v] * above[v] <= 0.0;
        const double ab = fabs(below[v]), aa = fabs(above[v]);
        const bool fix_lo = ab >= 2.0 * aa;
        const bool fix_hi = !fix_lo && (aa >= 2.0 * ab);
        const double lo_fix = c[v] - 2.0 * above[v], hi_fix = c[v] + 2.0 * below[v];
        const double lo_ext = c[v] - 0.5 * s[v], hi_ext = c[v] + 0.5 * s[v];
        lo[v] = extremum ? lo_ext : (fix_lo ? lo_fix : lf[v]);
        hi[v] = extremum ? hi_ext : (fix_hi ? hi_fix : hf[v]);
    }
}

// PLM: face states q -+ s/2 with the monotonized-central slope of the three cell averages
template <int NV, typename Q>
__device__ __forceinline__ void plm_states(Q q, double lo[NV], double hi[NV])
{
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const double c = q(v, 2);
        const double s = mc_slope(q(v, 1), c, q(v, 3));
        lo[v] = c - 0.5 * s;
        hi[v] = c + 0.5 * s;
    }
}

// Marching sweeps: the raw interface value at the high face of one cell is the raw interface value at the low
// face of the next (the same expression of eq 22 on the same four cells), so it is carried in `ifc` instead of
// being evaluated twice; q(v, 0) is then never read.  Same values as ppm_cell / rad_ppm_cell.
template <int BL, int NV, typename Q>
__device__ __forceinline__ void ppm_states_carry(Q q, double ifc[NV], double lo[NV], double hi[NV])
{
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const double b = q(v, 1), c = q(v, 2), d = q(v, 3), e = q(v, 4);
        const double hi_raw = ppm_interface(b, c, d, e);
        ppm_limit_t<BL != 0>(ifc[v], hi_raw, b, c, d, lo[v], hi[v]);
        ifc[v] = hi_raw;
    }
}

// flattened PPM face states of all five primitives of one cell; q(v, m) = value of variable v at
// stencil offset m-2
template <int BL = 0, typename Q>
__device__ __forceinline__ void ppm_cell(Q q, double chi, double lo[5], double hi[5])
{
    if (BL == 2) {
        double l[5], h[5];
        ppm_lockstep<5>(q, l, h);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double c = q(v, 2);
            lo[v] = c + chi * (l[v] - c);
            hi[v] = c + chi * (h[v] - c);
        }
        return;
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double c = q(v, 2);
        double l, h;
        ppm_face_states_t<BL != 0>(q(v, 0), q(v, 1), c, q(v, 3), q(v, 4), l, h);
        lo[v] = c + chi * (l - c);          // flatten toward the cell average
        hi[v] = c + chi * (h - c);
    }
}

// HLLC flux through a face with normal DIR; L, R = (rho, vx, vy, vz, P); F in conserved order
template <int DIR>
__device__ __forceinline__ void face_flux(double gamma, const double L[5], const double R[5], double F[5])
{
    constexpr int n = 1 + DIR, t1 = 1 + (DIR + 1) % 3, t2 = 1 + (DIR + 2) % 3;
    const Flux5 f = hllc_flux(gamma, L[0], L[n], L[t1], L[t2], L[4], R[0], R[n], R[t1], R[t2], R[4]);
    F[0] = f.m; F[n] = f.pn; F[t1] = f.pt1; F[t2] = f.pt2; F[4] = f.e;
}

// PPM face states of (E, fx, fy, fz) of one cell, q(v, m) = variable v at stencil offset m-2; a face
// state with |f|^2 > 1 or E <= 0 reverts to the cell average.  Returns the number of
// reverted states.
template <int BL = 0, typename Q>
__device__ __forceinline__ int rad_ppm_cell(Q q, double lo[4], double hi[4])
{
    double ctr[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) ctr[v] = q(v, 2);
    if (BL == 2) {
        ppm_lockstep<4>(q, lo, hi);
    } else {
#pragma unroll
        for (int v = 0; v < 4; ++v)
            ppm_face_states_t<BL != 0>(q(v, 0), q(v, 1), ctr[v], q(v, 3), q(v, 4), lo[v], hi[v]);
    }
    int nfall = 0;
    double f2 = (lo[1] * lo[1] + lo[2] * lo[2]) + lo[3] * lo[3];
    if (f2 > 1.0 || !(lo[0] > 0.0)) {
#pragma unroll
        for (int v = 0; v < 4; ++v) lo[v] = ctr[v];
        ++nfall;
    }
    f2 = (hi[1] * hi[1] + hi[2] * hi[2]) + hi[3] * hi[3];
    if (f2 > 1.0 || !(hi[0] > 0.0)) {
#pragma unroll
        for (int v = 0; v < 4; ++v) hi[v] = ctr[v];
        ++nfall;
    }
    return nfall;
}

template <int DIR>
__device__ __forceinline__ int rad_face_flux(double c, double c_hat, bool tau_corr, double tau, const double L[4],
                                             const double R[4], double G[4])
{
    int guard;
    const Rad4 g = rad_hll_flux(c, c_hat, L[0], L[1], L[2], L[3], R[0], R[1], R[2], R[3], DIR, tau, tau_corr, guard);
    G[0] = g.e; G[1] = g.x; G[2] = g.y; G[3] = g.z;
    return guard;
}

}  // namespace qk
