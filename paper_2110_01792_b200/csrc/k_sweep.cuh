// k_sweep.cuh -- the two stencil kernels of an RK stage, shared by the hydro and the radiation policy (k_sweep.cu).
//
// The sweeps read the RECONSTRUCTION variables of the stage's state -- primitives W = (rho, v, P), or
// S = (E_r, f = F_r/(c E_r)), PAPER.md:178 -- which the kernel that produced the state wrote next to it (z sweep,
// exchange); no face flux ever exists in HBM, only the running flux difference D:
//
//   sweep_x_kernel     : one warp per 30-cell x segment walking 8 rows; row segments staged global -> shared by
//                        16-byte cp.async one row ahead, converted by the staging lanes; both face states of the
//                        lane's cell, left neighbour's high state and right neighbour's flux by warp shuffle.
//                        Writes D = dF_x.
//   sweep_march_kernel : one thread per (x, other) column marching along y or z over a chunk of cells; the
//                        five-cell window of the column lives in a thread-private shared-memory ring (no barrier
//                        anywhere), the high face state, the low-face flux and the raw eq 22 interface value of
//                        the previous cell stay in registers; the own-cell inputs of the update are copied global ->
//                        shared by cp.async at the top of a step and read at its end (they never occupy registers
//                        during the Riemann solve: that is what lets the z sweep run at 4 CTAs per SM).  y: D += dF_y.  z: RK stage update
//                        with (dF_x + dF_y) + dF_z (the paper's sum order) and, after the last hydro
//                        stage, the CFL signal speed of the new state (eq 21).
//
// HBM traffic per cell and stage (hydro): x reads W + chi (48 B), writes D (40); y reads W + chi + D (88), writes D
// (40); z reads W + chi + D + U (120: the density of W is U's own array) + U^n in stage 2 (40), writes the new state
// and its primitives v, P (72): 408-448 B with the flattening kernel's 40.  Two leaner layouts were built and measured slower: reading
// the conserved state and converting every loaded cell (no W arrays, 80 B less, +20 % time: the division chains of
// cons -> prim run 4 x per cell instead of once), and one fused x+y kernel that writes D once (128 B less, +50 % time
// at 168 registers / 3 warps per scheduler).
//
// `PH` is the physics policy: NV reconstructed variables, SW_NR window variables per cell (the last one may be a
// face auxiliary such as kappa_R rho), `states` = limited face states of one cell, `flux<DIR>` = Riemann flux through a face.  Each face state / face of the grid is counted by exactly
// one thread for the integer diagnostics (same convention as the oracle: states of the cells -1..n and faces
// 0..n of the sweep direction, other two indices interior).
#pragma once

#include "k_recon.cuh"

namespace qk {

constexpr int SW_NT = 128;            // threads per CTA: z march = 128 columns along x; xy kernel = 4 warps
constexpr int SW_NR = 5;              // window variables per cell
constexpr int SW_XW = 30;             // cells updated per warp row in the xy kernel (lanes 1..30; 0 and 31 are halo lanes)
constexpr int SW_XCOLS = 38;          // staged columns per warp row: cells i0-4 .. i0+33 (16-byte aligned start)
constexpr int SW_XYWARPS = SW_NT / 32;

template <int NV> struct FieldsRW { double *f[NV]; };
template <int NV> struct FieldsRO { const double *f[NV]; };

// dtdx_dev != nullptr: dt/dx is read from device memory (qk_hydro_step_cfl: the timestep never visits the host)
struct RkArgs { double dtdx; int stage; const double *dtdx_dev; };

__device__ __forceinline__ void sweep_count(Counters *ctr, int nfall, int nguard, int nbad)
{
    for (int off = 16; off > 0; off >>= 1) {
        nfall += __shfl_xor_sync(0xffffffffu, nfall, off);
        nguard += __shfl_xor_sync(0xffffffffu, nguard, off);
        nbad += __shfl_xor_sync(0xffffffffu, nbad, off);
    }
    if ((threadIdx.x & 31) == 0) {
        if (nfall) atomicAdd((unsigned long long *)&ctr->fallback, (unsigned long long)nfall);
        if (nguard) atomicAdd((unsigned long long *)&ctr->guard, (unsigned long long)nguard);
        if (nbad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)nbad);
    }
}

// ---- x sweep ---------------------------------------------------------------------------------------------
// One warp per 30-cell x segment, walking SW_XNROW consecutive rows.  Lane l owns cell i = i0 - 1 + l (lanes 0
// and 31 are halo lanes); the 38 cells i0-4 .. i0+33 of a row are staged as 19 pairs: lane l < 19 copies the
// pair (i0 - 4 + 2l, +1) of every source array global -> shared with one 16-byte cp.async (every row of every
// field starts 32-byte aligned and i0 is even, so with an even row pitch no pair straddles a 16-byte boundary;
// odd pitches fall back to two 8-byte copies), one row ahead of the arithmetic, into a warp-private double
// buffer: no register staging, the copy of row r+1 overlaps the PPM / Riemann work of row r.  Every lane
// reconstructs both face states of its cell, the left neighbour's high state and the right neighbour's flux
// arrive by shuffle, and lanes 1..30 write D = dF_x.  Only __syncwarp.
constexpr int SW_XNROW = 8;             // rows walked by one warp

__device__ __forceinline__ void cp_async16(double *smem_dst, const double *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <class PH>
__global__ void __launch_bounds__(SW_NT, PH::X_MINB) sweep_x_kernel(PH ph, Geom g, int k0, FieldsRW<PH::NV> D, Counters *ctr)
{
    constexpr int NV = PH::NV, NSRC = PH::NSRC;
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ __align__(16) double stage_all[SW_XYWARPS][2][NSRC][SW_XCOLS];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int k = (int)blockIdx.z + k0;                       // the launch covers the planes k0 .. k0 + gridDim.z - 1
    const int j0 = ((int)blockIdx.y * SW_XYWARPS + wid) * SW_XNROW;
    const int i0 = (int)blockIdx.x * SW_XW;
    const int nrow = min(SW_XNROW, g.ny - j0);                // warp-uniform; <= 0 for warps past the last row
    if (nrow <= 0) return;                                    // there is no CTA-wide barrier
    double(*stage)[NSRC][SW_XCOLS] = stage_all[wid];
    const int i = i0 - 1 + lane;                              // own cell
    const int col = lane + 3;                                 // its staged column
    const bool owner = lane >= 1 && lane <= SW_XW && i < g.nx;      // lanes that store and count
    const int xi = min(i, g.nx);
    const bool stager = lane < SW_XCOLS / 2;
    // the last pairs of the last warp of a row may lie beyond the array: clamp (those columns feed no stored result)
    const int xs = min(i0 - NG + 2 * lane, g.nx + NG - 2);
    const bool vec = (g.sy & 1) == 0;
    int nfall = 0, nguard = 0;

    auto issue = [&](int r) {
        if (stager) {
            const int src = g.at(xs, j0 + r, k);
#pragma unroll
            for (int q = 0; q < NSRC; ++q) {
                const double *p = ph.src(q) + src;
                double *d = &stage[r & 1][q][2 * lane];
                if (vec) cp_async16(d, p);
                else { cp_async8(d, p); cp_async8(d + 1, p + 1); }
            }
        }
        cp_async_commit();
    };
    issue(0);
    for (int r = 0; r < nrow; ++r) {
        if (r + 1 < nrow) { issue(r + 1); cp_async_wait<1>(); }
        else              { cp_async_wait<0>(); }
        __syncwarp();
        const double(*buf)[SW_XCOLS] = stage[r & 1];
        const int cidx = g.at(xi, j0 + r, k);
        double lo[NV], hi[NV], L[NV], F[NV];
        const int nf = ph.template states<PH::BL_X>([&](int v, int q) { return ph.win(v, buf, col - 2 + q); },
                                                     ph.win_aux(buf, col), lo, hi);
#pragma unroll
        for (int v = 0; v < NV; ++v) L[v] = __shfl_up_sync(FULL, hi[v], 1);
        const int gd = ph.template flux<0>(L, lo, ph.win(SW_NR - 1, buf, col - 1), ph.win(SW_NR - 1, buf, col), F);   // face i-1/2
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const double Fh = __shfl_down_sync(FULL, F[v], 1);
            if (owner) D.f[v][cidx] = Fh - F[v];
        }
        if (PH::COUNTS) {
            const bool last = lane >= 1 && i == g.nx;
            if (owner || i == -1 || last) nfall += nf;
            if (owner || last) nguard += gd;
        }
        __syncwarp();                                         // all lanes done with the buffer before it is refilled
    }
    if (PH::COUNTS) sweep_count(ctr, nfall, nguard, 0);
}

// ---- y and z sweeps: marching columns ----------------------------------------------------------------------
// DIR = 1: march along y (blockIdx.y = k), D += dF_y.  DIR = 2: march along z (blockIdx.y = j), RK stage update
// from (dF_x + dF_y) + dF_z (the paper's sum order).
// NT = threads per CTA = columns along x per CTA (128, 64 or 32: the launcher takes the width that wastes the fewest
// lanes on the row length; the CTAs per SM scale with 128 / NT, so the resident warps stay the same)
template <class PH, int DIR, int NT>
__global__ void __launch_bounds__(NT, (DIR == 2 ? PH::Z_MINB : PH::Y_MINB) * (SW_NT / NT)) sweep_march_kernel(PH ph, Geom g, int len, int o0, FieldsRW<PH::NV> D, RkArgs rk,
                                                                   FieldsRO<PH::NV> U, FieldsRO<PH::NV> U0, FieldsRW<PH::NV> out,
                                                                   FieldsRW<PH::NV> pout, Counters *ctr, StateCache *cache)
{
    constexpr int NV = PH::NV;
    const double dtdx = (DIR == 2 && rk.dtdx_dev) ? __ldg(rk.dtdx_dev) : rk.dtdx;
    typename PH::Tail tail;                             // per-thread reduction state of the z epilogue
    __shared__ double ring[5 * SW_NR * NT];          // [slot][var][thread], thread-private columns
    // own-cell inputs of the update (D; for z also U and U^n), staged global -> shared by cp.async: [array][var][thread]
    __shared__ double own[(DIR == 2 ? 3 : 1) * PH::NV * NT];   // z: D, U, U^n of the cell being updated, staged by cp.async
    const int tid = threadIdx.x;
    const int i = blockIdx.x * NT + tid;
    const bool active = i < g.nx;
    const int o = (int)blockIdx.y + o0;                 // y sweep: the launch covers the planes o0 .. o0 + gridDim.y - 1
    const int n_m = DIR == 1 ? g.ny : g.nz;
    const int m0 = (int)blockIdx.z * len;
    const int m1 = min(m0 + len, n_m);
    const int s = DIR == 1 ? g.sy : g.sz;
    const int ic = min(i, g.nx - 1);
    const int base = DIR == 1 ? g.at(ic, 0, o) : g.at(ic, o, 0);     // cell m = 0 of the column

    // rotating ring offsets of the cells m-1, m, m+1, m+2, m+3
    int r0 = 0 * SW_NR * NT + tid, r1 = 1 * SW_NR * NT + tid, r2 = 2 * SW_NR * NT + tid,
        r3 = 3 * SW_NR * NT + tid, r4 = 4 * SW_NR * NT + tid;
    // prologue: cells m0-3..m0 -> r0..r3 (they are cells m-1..m+2 of the first step m = m0-2)
    {
        const int rr[4] = {r0, r1, r2, r3};
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int cidx = base + (m0 - 3 + p) * s;
#pragma unroll
            for (int v = 0; v < SW_NR; ++v) ring[rr[p] + v * NT] = ph.ld(v, cidx);
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
        ifc[v] = ppm_interface(ring[r0 + v * NT], ring[r1 + v * NT], ring[r2 + v * NT], ring[r3 + v * NT]);
    }
    int nfall = 0, nguard = 0;

    for (int m = m0 - 2; m < m1; ++m) {
#pragma unroll
        for (int v = 0; v < SW_NR; ++v) ring[r4 + v * NT] = pend[v];
        const double aux = aux_next;
        if (m + 1 < m1) {
            const int cn = base + (m + 4) * s;
#pragma unroll
            for (int v = 0; v < SW_NR; ++v) pend[v] = ph.ld(v, cn);
            aux_next = ph.aux(base + (m + 2) * s);
        }
        const int cidx = base + m * s;
        // own-cell inputs of the update, consumed at the end of the step
        if (m >= m0) {
            {     // global -> shared without passing through registers: they land while the Riemann solve runs
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    cp_async8(&own[(0 * NV + v) * NT + tid], D.f[v] + cidx);
                    if (DIR == 2) {
                        cp_async8(&own[(1 * NV + v) * NT + tid], U.f[v] + cidx);
                        if (rk.stage == 1) cp_async8(&own[(2 * NV + v) * NT + tid], U0.f[v] + cidx);
                    }
                }
                cp_async_commit();
            }
        }
        // limited face states of cell m+1
        double lo[NV], hi[NV], Fhi[NV];
        {
            const int rr[5] = {r0, r1, r2, r3, r4};
            const auto win = [&](int v, int q) { return ring[rr[q] + v * NT]; };
            const int nf = PH::CARRY ? ph.template states_carry<PH::BL_MARCH>(win, aux, ifc, lo, hi)
                                     : ph.template states<PH::BL_MARCH>(win, aux, lo, hi);
            const int mm = m + 1;
            if (PH::COUNTS && active && ((mm >= m0 && mm < m1) || mm == -1 || mm == n_m)) nfall += nf;
        }
        if (m >= m0 - 1) {      // face m+1/2 = low face of cell m+1
            const int gd = ph.template flux<DIR>(hiP, lo, ring[r1 + (SW_NR - 1) * NT], ring[r2 + (SW_NR - 1) * NT], Fhi);
            const int mm = m + 1;
            if (PH::COUNTS && active && ((mm >= m0 && mm < m1) || mm == n_m)) nguard += gd;
        }
        if (m >= m0) cp_async_wait<0>();
        if (m >= m0 && active) {
            double fresh[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const double dv = own[(0 * NV + v) * NT + tid];
                const double div = dv + (Fhi[v] - Flo[v]);                  // dF_x + dF_y, then (dF_x + dF_y) + dF_z
                if (DIR == 1) {
                    D.f[v][cidx] = div;
                } else {
                    const double us = own[(1 * NV + v) * NT + tid] - dtdx * div;
                    fresh[v] = rk.stage == 0 ? us : 0.5 * own[(2 * NV + v) * NT + tid] + 0.5 * us;
                    out.f[v][cidx] = fresh[v];
                }
            }
            // the reconstruction variables of the updated cell, for the next stage (and its CFL speed)
            if (DIR == 2) ph.finish(cidx, fresh, pout, rk.stage == 1, tail);
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) { hiP[v] = hi[v]; Flo[v] = Fhi[v]; }
        const int t = r0; r0 = r1; r1 = r2; r2 = r3; r3 = r4; r4 = t;
    }
    if (PH::COUNTS) sweep_count(ctr, nfall, nguard, 0);
    if (DIR == 2) ph.finish_block(tail, rk.stage == 1, ctr, cache);
}

}  // namespace qk
