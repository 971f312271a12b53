// k_recon.cuh -- per-cell reconstruction building blocks of the sweep kernels (k_sweep.cuh): PPM / PLM face
// states of all variables of one cell and the first-order fallback of the radiation
// states.  Device inline functions only; every formula in the evaluation order DESIGN.md section 3 fixes.
#pragma once

#include "qk_internal.h"
#include "qk_math.cuh"

namespace qk {

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

// First-order fallback per face state (R3): a state with |f|^2 > 1 or E <= 0 reverts, all four
// variables, to the cell average q(v, 2).  Returns the number of reverted states.
template <typename Q>
__device__ __forceinline__ int rad_fallback(Q q, double lo[4], double hi[4])
{
    int nfall = 0;
    double f2 = (lo[1] * lo[1] + lo[2] * lo[2]) + lo[3] * lo[3];
    if (f2 > 1.0 || !(lo[0] > 0.0)) {
#pragma unroll
        for (int v = 0; v < 4; ++v) lo[v] = q(v, 2);
        ++nfall;
    }
    f2 = (hi[1] * hi[1] + hi[2] * hi[2]) + hi[3] * hi[3];
    if (f2 > 1.0 || !(hi[0] > 0.0)) {
#pragma unroll
        for (int v = 0; v < 4; ++v) hi[v] = q(v, 2);
        ++nfall;
    }
    return nfall;
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
    return rad_fallback(q, lo, hi);
}

}  // namespace qk
