// k_sweep.cuh -- direction-split, barrier-free sweep kernels shared by the hydro and radiation stages.
//
// The stage kernels are bound by the latency of the fp64 pipe rather than by HBM (a stage
// moves ~530 B/cell, 1.4 ms of HBM time, against 2.7 ms measured).  The sweeps trade a few hundred bytes per
// cell of extra traffic for instruction streams that never wait on another warp:
//
//   sweep_x_kernel     : one thread per cell, one warp per 30-cell x segment walking 8 rows, row segments
//                        staged global -> shared by cp.async one row ahead.  Lane l owns cell
//                        30 b - 1 + l; the high face state of the left neighbour and the flux of the
//                        right neighbour arrive by warp shuffle, so lanes 1..30 produce a flux
//                        difference and lanes 0, 31 are halo lanes.  Writes D = dF_x.
//   sweep_march_kernel : one thread per (x, other) column, marching along y or z over a chunk of
//                        cells.  The five-cell reconstruction window of the column lives in a
//                        thread-private shared-memory ring (no __syncthreads anywhere); the high face
//                        state and the low-face flux of the previous cell stay in registers.
//                        MODE 1 (y): D = D + dF_y.   MODE 2 (z): out = RK stage update with
//                        (D + dF_z), i.e. the paper's sum order ((dFx + dFy) + dFz), plus
//                        the policy's `finish` epilogue: the reconstruction variables of the updated
//                        cell for the next stage and, after the last stage, its CFL speed.
//
// `PH` is the physics policy (k_sweep.cu): NV reconstructed variables, SW_NR window variables per
// cell (the last one may be a face auxiliary such as kappa_R rho), `states` = limited face states of
// one cell, `flux<DIR>` = Riemann flux through a face.  Each face state / face of the grid is counted
// by exactly one thread for the integer diagnostics (same convention as the oracle: states of the
// cells -1..n and faces 0..n of the sweep direction, other two indices interior).
#pragma once

#include "k_stage_common.cuh"

namespace qk {

#ifndef QK_SW_NT
#define QK_SW_NT 128
#endif
#ifndef QK_SW_MINB1
#define QK_SW_MINB1 4
#endif
#ifndef QK_SW_MINB2
#define QK_SW_MINB2 3
#endif
#ifndef QK_SW_XROWS
#define QK_SW_XROWS 4
#endif
#ifndef QK_SW_XMINB
#define QK_SW_XMINB 5
#endif
constexpr int SW_NT = QK_SW_NT;       // threads per CTA of the marching kernels (lanes along x)
constexpr int SW_NR = 5;              // variables per cell kept in the marching window
constexpr int SW_XW = 30;             // cells updated per warp in the x sweep
constexpr int SW_XROWS = QK_SW_XROWS; // rows (warps) per CTA in the x sweep

template <int NV> struct FieldsRW { double *f[NV]; };
template <int NV> struct FieldsRO { const double *f[NV]; };

// dtdx_dev != nullptr: dt/dx is read from device memory (qk_hydro_step_cfl: the timestep never visits the host)
struct RkArgs { double dtdx; int stage; const double *dtdx_dev; };

__device__ __forceinline__ void sweep_count(Counters *ctr, int nfall, int nguard)
{
    for (int off = 16; off > 0; off >>= 1) {
        nfall += __shfl_xor_sync(0xffffffffu, nfall, off);
        nguard += __shfl_xor_sync(0xffffffffu, nguard, off);
    }
    if ((threadIdx.x & 31) == 0) {
        if (nfall) atomicAdd((unsigned long long *)&ctr->fallback, (unsigned long long)nfall);
        if (nguard) atomicAdd((unsigned long long *)&ctr->guard, (unsigned long long)nguard);
    }
}

// ---- x sweep -------------------------------------------------------------------------------------------
// Each warp owns one 30-cell x segment and walks SW_XNROW consecutive rows of it.  The 36-cell row
// segment of every source array the stencils of its 32 lanes touch is copied global -> shared with
// cp.async (no register staging), one row ahead of the arithmetic, into a warp-private double buffer:
// the copy of row r+1 overlaps the PPM / Riemann work of row r and the only synchronisation is
// __syncwarp.  (Loading the stencils straight from global memory exposed one full memory latency per
// variable: 45 % of the stall samples, profiles/r1_hydro_ncu.md.)
#ifndef QK_SW_XNROW
#define QK_SW_XNROW 8
#endif
constexpr int SW_XNROW = QK_SW_XNROW;   // rows walked by one warp
constexpr int SW_XSEG = SW_XW + 6;      // staged cells per row: lanes' cells -1..30 plus the +-2 stencil halo
constexpr int SW_NSRC = 6;              // source arrays per policy (window variables are built from them)

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <class PH>
__global__ void __launch_bounds__(32 * SW_XROWS, QK_SW_XMINB) sweep_x_kernel(PH ph, Geom g, FieldsRW<PH::NV> D, Counters *ctr)
{
    constexpr int NV = PH::NV;
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ double stage[SW_XROWS][2][SW_NSRC][SW_XSEG];
    const int lane = threadIdx.x, wy = threadIdx.y;
    const int k = blockIdx.z;
    const int j0 = ((int)blockIdx.y * SW_XROWS + wy) * SW_XNROW;
    const int i0 = (int)blockIdx.x * SW_XW;
    const int i = i0 - 1 + lane;                              // this lane's cell
    int nfall = 0, nguard = 0;
    const int nrow = min(SW_XNROW, g.ny - j0);                // warp-uniform; <= 0 for warps past the last row

    // cells staged by this lane: i0-3+lane, and for lanes 0..3 also i0+29+lane (clamped into the array)
    const int ia = min(i0 - 3 + lane, g.nx + NG - 1), ib = min(i0 + 29 + lane, g.nx + NG - 1);
    auto issue = [&](int r) {
        const int rowbase = g.at(0, j0 + r, k);
        double(*buf)[SW_XSEG] = stage[wy][r & 1];
#pragma unroll
        for (int sidx = 0; sidx < SW_NSRC; ++sidx) {
            const double *src = ph.src(sidx) + rowbase;
            cp_async8(&buf[sidx][lane], src + ia);
            if (lane < SW_XSEG - 32) cp_async8(&buf[sidx][32 + lane], src + ib);
        }
        cp_async_commit();
    };
    if (nrow > 0) issue(0);
    for (int r = 0; r < nrow; ++r) {
        if (r + 1 < nrow) { issue(r + 1); cp_async_wait<1>(); }
        else              { cp_async_wait<0>(); }
        __syncwarp();
        const double(*buf)[SW_XSEG] = stage[wy][r & 1];
        const int cidx = g.at(min(i, g.nx), j0 + r, k);      // lanes beyond cell n are not stored, not counted
        double lo[NV], hi[NV], L[NV], F[NV];
        const int nf = ph.template states<PH::BL_X>([&](int v, int m) { return ph.win(v, buf, lane + m); },
                                                     ph.win_aux(buf, lane + 2), lo, hi);
#pragma unroll
        for (int v = 0; v < NV; ++v) L[v] = __shfl_up_sync(FULL, hi[v], 1);
        const int gd = ph.template flux<0>(L, lo, ph.win(SW_NR - 1, buf, lane + 1), ph.win(SW_NR - 1, buf, lane + 2), F);   // face i-1/2
        const bool interior = lane >= 1 && lane <= SW_XW && i < g.nx;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const double Fh = __shfl_down_sync(FULL, F[v], 1);
            if (interior) D.f[v][cidx] = Fh - F[v];
        }
        if (PH::COUNTS) {
            const bool last = lane >= 1 && i == g.nx;
            if (interior || i == -1 || last) nfall += nf;
            if (interior || last) nguard += gd;
        }
        __syncwarp();                                         // all lanes done with buf before it is refilled
    }
    if (PH::COUNTS) sweep_count(ctr, nfall, nguard);
}

// DIR = 1 (march along y; blockIdx.y = k) or 2 (march along z; blockIdx.y = j)
template <class PH, int DIR, int MODE>
__global__ void __launch_bounds__(SW_NT, MODE == 2 ? QK_SW_MINB2 : QK_SW_MINB1) sweep_march_kernel(PH ph, Geom g, int len, FieldsRW<PH::NV> D, RkArgs rk,
                                                            FieldsRO<PH::NV> U, FieldsRO<PH::NV> U0,
                                                            FieldsRW<PH::NV> out, FieldsRW<PH::NV> pout, Counters *ctr,
                                                            StateCache *cache)
{
    constexpr int NV = PH::NV;
    const double dtdx = (MODE == 2 && rk.dtdx_dev) ? __ldg(rk.dtdx_dev) : rk.dtdx;
    typename PH::Tail tail;                             // per-thread reduction state of the MODE 2 epilogue
    __shared__ double ring[5 * SW_NR * SW_NT];          // [slot][var][thread], thread-private columns
    const int tid = threadIdx.x;
    const int i = blockIdx.x * SW_NT + tid;
    const bool active = i < g.nx;
    const int o = blockIdx.y;
    const int n_m = DIR == 1 ? g.ny : g.nz;
    const int m0 = (int)blockIdx.z * len;
    const int m1 = min(m0 + len, n_m);
    const int s = DIR == 1 ? g.sy : g.sz;
    const int ic = min(i, g.nx - 1);
    const int base = DIR == 1 ? g.at(ic, 0, o) : g.at(ic, o, 0);     // cell m = 0 of the column

    // rotating ring offsets of the cells m-1, m, m+1, m+2, m+3
    int r0 = 0 * SW_NR * SW_NT + tid, r1 = 1 * SW_NR * SW_NT + tid, r2 = 2 * SW_NR * SW_NT + tid,
        r3 = 3 * SW_NR * SW_NT + tid, r4 = 4 * SW_NR * SW_NT + tid;
    // prologue: cells m0-3..m0 -> r0..r3 (they are cells m-1..m+2 of the first step m = m0-2)
    {
        const int rr[4] = {r0, r1, r2, r3};
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int cidx = base + (m0 - 3 + p) * s;
#pragma unroll
            for (int v = 0; v < SW_NR; ++v) ring[rr[p] + v * SW_NT] = ph.ld(v, cidx);
        }
    }
    double pend[SW_NR];
#pragma unroll
    for (int v = 0; v < SW_NR; ++v) pend[v] = ph.ld(v, base + (m0 + 1) * s);
    double aux_next = ph.aux(base + (m0 - 1) * s);
    double hiP[NV], Flo[NV], ifc[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        hiP[v] = 0.0; Flo[v] = 0.0;
        // raw eq 22 interface at the low face of the first cell reconstructed (cells m0-3..m0 are in r0..r3)
        ifc[v] = ppm_interface(ring[r0 + v * SW_NT], ring[r1 + v * SW_NT], ring[r2 + v * SW_NT], ring[r3 + v * SW_NT]);
    }
    int nfall = 0, nguard = 0;

    for (int m = m0 - 2; m < m1; ++m) {
#pragma unroll
        for (int v = 0; v < SW_NR; ++v) ring[r4 + v * SW_NT] = pend[v];
        const double aux = aux_next;
        if (m + 1 < m1) {
            const int cn = base + (m + 4) * s;
#pragma unroll
            for (int v = 0; v < SW_NR; ++v) pend[v] = ph.ld(v, cn);
            aux_next = ph.aux(base + (m + 2) * s);
        }
        const int cidx = base + m * s;
        // own-cell inputs of the update, consumed at the end of the step
        double din[NV], u[NV], u0[NV];
        if (m >= m0) {
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                din[v] = D.f[v][cidx];
                if (MODE == 2) {
                    u[v] = U.f[v][cidx];
                    u0[v] = rk.stage == 1 ? U0.f[v][cidx] : 0.0;
                }
            }
        }
        // limited face states of cell m+1
        double lo[NV], hi[NV], Fhi[NV];
        {
            const int rr[5] = {r0, r1, r2, r3, r4};
            const auto win = [&](int v, int q) { return ring[rr[q] + v * SW_NT]; };
            const int nf = PH::CARRY ? ph.template states_carry<PH::BL_MARCH>(win, aux, ifc, lo, hi)
                                     : ph.template states<PH::BL_MARCH>(win, aux, lo, hi);
            const int mm = m + 1;
            if (PH::COUNTS && active && ((mm >= m0 && mm < m1) || mm == -1 || mm == n_m)) nfall += nf;
        }
        if (m >= m0 - 1) {      // face m+1/2 = low face of cell m+1
            const int gd = ph.template flux<DIR>(hiP, lo, ring[r1 + (SW_NR - 1) * SW_NT], ring[r2 + (SW_NR - 1) * SW_NT], Fhi);
            const int mm = m + 1;
            if (PH::COUNTS && active && ((mm >= m0 && mm < m1) || mm == n_m)) nguard += gd;
        }
        if (m >= m0 && active) {
            double fresh[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const double div = din[v] + (Fhi[v] - Flo[v]);
                if (MODE == 1) {
                    D.f[v][cidx] = div;
                } else {
                    const double us = u[v] - dtdx * div;
                    fresh[v] = rk.stage == 0 ? us : 0.5 * u0[v] + 0.5 * us;
                    out.f[v][cidx] = fresh[v];
                }
            }
            // the reconstruction variables of the updated cell, for the next stage (and its CFL speed)
            if (MODE == 2) ph.finish(cidx, fresh, pout, rk.stage == 1, tail);
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) { hiP[v] = hi[v]; Flo[v] = Fhi[v]; }
        const int t = r0; r0 = r1; r1 = r2; r2 = r3; r3 = r4; r4 = t;
    }
    if (PH::COUNTS) sweep_count(ctr, nfall, nguard);
    if (MODE == 2) ph.finish_block(tail, rk.stage == 1, ctr, cache);
}

}  // namespace qk
