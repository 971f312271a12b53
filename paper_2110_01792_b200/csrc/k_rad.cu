// k_rad.cu -- fused radiation-transport stage: one kernel per SSP-RK2 stage.
//
//   rad_stage_kernel : (E_r, F_r), rho, kappa_R -> reduced flux f = F_r/(c E_r),
//                      PPM face states of (E_r, f) in x, y, z with the paper's limiters and no
//                      flattening, first-order fallback per face state (R3), closure
//                      (eq 23-25) + HLL flux with the guarded optical-depth correction
//                      (R5/R6), unsplit divergence ((dGx+dGy)+dGz) and the RK
//                      stage combination, in one pass.
//
// Same 2.5-D z-marching tiles as the hydro stage (k_stage_common.cuh).  The fifth slot of the
// shared-memory planes holds kappa_R rho, whose two-cell average gives tau_face.  Face states and
// fluxes never leave the SM.  The integer diagnostics (fallback states, guarded faces) are counted
// so that every face state / face of the grid is counted by exactly one thread (see `counts`).
#include "k_stage_common.cuh"
#include "qk_math.cuh"

namespace qk {

struct RadCell { double E, fx, fy, fz, kr; };   // reconstruction variables + kappa_R rho

__device__ __forceinline__ RadCell load_rad_cell(double c, const CRad4p &R, const double *__restrict__ rho,
                                                 const double *__restrict__ kR, int cidx)
{
    RadCell s;
    const double E = R.E[cidx], cE = c * E;
    s.E = E;
    s.fx = R.Fx[cidx] / cE;
    s.fy = R.Fy[cidx] / cE;
    s.fz = R.Fz[cidx] / cE;
    s.kr = kR[cidx] * rho[cidx];
    return s;
}

__device__ __forceinline__ RadCell benign_rad() { return RadCell{1.0, 0.0, 0.0, 0.0, 0.0}; }

struct RadSmem {
    double ring[RING][5][TY][TX];                   // (E, fx, fy, fz, kappa_R rho), planes k-1..k+3
    union {
        double W[5][TY + 2 * HALO][TX + 2 * HALO];  // plane k with star halo (phase P)
        struct {
            double gx[4][TY][TX];                   // x flux at faces 1..TX   (phases F, U)
            double gy[4][TY][TX];                   // y flux at faces 1..TY
        } fl;
    };
    double hiX[4][TY][TX + 1];                      // high-x face state of cells -1..TX-1
    double hiY[4][TY + 1][TX];                      // high-y face state of cells -1..TY-1
    double loXe[4][TY];                             // low-x face state of cell TX
    double loYe[4][TX];                             // low-y face state of cell TY
};

__global__ void __launch_bounds__(NT, 2) rad_stage_kernel(Geom g, double c, double c_hat, double dx, int tau_corr_i,
                                                          double dtdx, int stage, CRad4p R, CRad4p R0,
                                                          const double *__restrict__ rho, const double *__restrict__ kR,
                                                          Rad4p out, int lz, Counters *ctr)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RadSmem &s = *reinterpret_cast<RadSmem *>(smem_raw);
    const bool tau_corr = tau_corr_i != 0;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = (int)blockIdx.x * TX, j0 = (int)blockIdx.y * TY;
    const int k0 = (int)blockIdx.z * lz;
    const int k1 = min(k0 + lz, g.nz);
    const int gi = i0 + tx, gj = j0 + ty;
    const bool own_ok = in_array(g, gi, gj);
    const bool active = gi < g.nx && gj < g.ny;

    int hx = 0, hy = 0;
    const bool is_halo = t < N_HALO;
    if (is_halo) halo_cell(t, hx, hy);
    const bool halo_ok = is_halo && in_array(g, i0 + hx, j0 + hy);

    int ex = 0, ey = 0; bool e_along_x = false, e_high = false;
    const bool is_edge = t < N_EDGE;
    if (is_edge) edge_cell(t, ex, ey, e_along_x, e_high);

    // `counts`: who counts which face states / faces (each exactly once over the grid; the oracle
    // counts the states of cells -1..n of the direction and the faces 0..n, other two indices interior)
    const bool cnt_own_x = gi <= g.nx && gj < g.ny;            // own cell's x states and its low x face
    const bool cnt_own_y = gj <= g.ny && gi < g.nx;
    const bool cnt_edge = is_edge && (e_along_x ? (j0 + ey < g.ny && (i0 + ex == -1 || i0 + ex == g.nx))
                                                : (i0 + ex < g.nx && (j0 + ey == -1 || j0 + ey == g.ny)));
    const bool cnt_hiface = t < TX + TY && (t < TY ? (i0 + TX == g.nx && j0 + t < g.ny)
                                                   : (j0 + TY == g.ny && i0 + (t - TY) < g.nx));

    int bad = 0, nfall = 0, nguard = 0;
    // prologue: planes k0-3..k0 of the own columns
    for (int p = k0 - 3; p <= k0; ++p) {
        const RadCell u = own_ok ? load_rad_cell(c, R, rho, kR, g.at(gi, gj, p)) : benign_rad();
        const int sl = ring_slot(p);
        s.ring[sl][0][ty][tx] = u.E; s.ring[sl][1][ty][tx] = u.fx; s.ring[sl][2][ty][tx] = u.fy;
        s.ring[sl][3][ty][tx] = u.fz; s.ring[sl][4][ty][tx] = u.kr;
        if (p == k0 && active && !(u.E > 0.0)) ++bad;
    }
    RadCell pend_own = own_ok ? load_rad_cell(c, R, rho, kR, g.at(gi, gj, k0 + 1)) : benign_rad();
    RadCell pend_halo = benign_rad();
    double hiZ[4], GzLo[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) { hiZ[v] = 0.0; GzLo[v] = 0.0; }

    for (int k = k0 - 2; k < k1; ++k) {
        // ---- commit the loads issued during the previous step --------------------------------
        {
            const int sl = ring_slot(k + 3);
            s.ring[sl][0][ty][tx] = pend_own.E; s.ring[sl][1][ty][tx] = pend_own.fx;
            s.ring[sl][2][ty][tx] = pend_own.fy; s.ring[sl][3][ty][tx] = pend_own.fz;
            s.ring[sl][4][ty][tx] = pend_own.kr;
            if (active && k + 3 > k0 && k + 3 < k1 && !(pend_own.E > 0.0)) ++bad;
        }
        if (k >= k0) {
            if (is_halo) {
                s.W[0][hy + HALO][hx + HALO] = pend_halo.E; s.W[1][hy + HALO][hx + HALO] = pend_halo.fx;
                s.W[2][hy + HALO][hx + HALO] = pend_halo.fy; s.W[3][hy + HALO][hx + HALO] = pend_halo.fz;
                s.W[4][hy + HALO][hx + HALO] = pend_halo.kr;
            }
            const int sl = ring_slot(k);
#pragma unroll
            for (int v = 0; v < 5; ++v) s.W[v][ty + HALO][tx + HALO] = s.ring[sl][v][ty][tx];
        }
        __syncthreads();   // S1
        // ---- issue the loads of the next step -------------------------------------------------
        if (k + 1 < k1) {
            pend_own = own_ok ? load_rad_cell(c, R, rho, kR, g.at(gi, gj, k + 4)) : benign_rad();
            if (k + 1 >= k0)
                pend_halo = halo_ok ? load_rad_cell(c, R, rho, kR, g.at(i0 + hx, j0 + hy, k + 1)) : benign_rad();
        }
        // ---- phase P: PPM face states, fallback, optical depths of the faces -------------------
        double loZn[4], hiZn[4];
        const bool in_chunk = k >= k0;
        {
            const int s0 = ring_slot(k - 1), s1 = ring_slot(k), s2 = ring_slot(k + 1), s3 = ring_slot(k + 2),
                      s4 = ring_slot(k + 3);
            const int sl[5] = {s0, s1, s2, s3, s4};
            const int nf = rad_ppm_cell([&](int v, int m) { return s.ring[sl[m]][v][ty][tx]; }, loZn, hiZn);
            const int kk = k + 1;       // the cell these z states belong to
            if (active && ((kk >= k0 && kk < k1) || kk == -1 || kk == g.nz)) nfall += nf;
        }
        const double tauZ = (0.5 * (s.ring[ring_slot(k)][4][ty][tx] + s.ring[ring_slot(k + 1)][4][ty][tx])) * dx;
        double loX[4], loY[4];
        double tauX = 0.0, tauY = 0.0, tauHi = 0.0;
        if (in_chunk) {
            double hi[4];
            const int y = ty + HALO, x = tx + HALO;
            int nf = rad_ppm_cell([&](int v, int m) { return s.W[v][y][x + m - 2]; }, loX, hi);
            if (cnt_own_x) nfall += nf;
#pragma unroll
            for (int v = 0; v < 4; ++v) s.hiX[v][ty][tx + 1] = hi[v];
            nf = rad_ppm_cell([&](int v, int m) { return s.W[v][y + m - 2][x]; }, loY, hi);
            if (cnt_own_y) nfall += nf;
#pragma unroll
            for (int v = 0; v < 4; ++v) s.hiY[v][ty + 1][tx] = hi[v];
            tauX = (0.5 * (s.W[4][y][x - 1] + s.W[4][y][x])) * dx;
            tauY = (0.5 * (s.W[4][y - 1][x] + s.W[4][y][x])) * dx;
            if (t < TY)           tauHi = (0.5 * (s.W[4][t + HALO][TX - 1 + HALO] + s.W[4][t + HALO][TX + HALO])) * dx;
            else if (t < TX + TY) tauHi = (0.5 * (s.W[4][TY - 1 + HALO][t - TY + HALO] + s.W[4][TY + HALO][t - TY + HALO])) * dx;
            if (is_edge) {
                double lo[4];
                const int yy = ey + HALO, xx = ex + HALO;
                if (e_along_x) {
                    nf = rad_ppm_cell([&](int v, int m) { return s.W[v][yy][xx + m - 2]; }, lo, hi);
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        if (e_high) s.loXe[v][ey] = lo[v];
                        else        s.hiX[v][ey][0] = hi[v];
                    }
                } else {
                    nf = rad_ppm_cell([&](int v, int m) { return s.W[v][yy + m - 2][xx]; }, lo, hi);
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        if (e_high) s.loYe[v][ex] = lo[v];
                        else        s.hiY[v][0][ex] = hi[v];
                    }
                }
                if (cnt_edge) nfall += nf;
            }
        }
        __syncthreads();   // S2: face states visible; plane W no longer read
        // ---- phase F: HLL fluxes ----------------------------------------------------------------
        double GzHi[4], GxLo[4], GyLo[4];
        double uc[4] = {1.0, 0.0, 0.0, 0.0}, u0[4] = {1.0, 0.0, 0.0, 0.0};
        if (k >= k0 - 1) {                                             // face k+1/2 = low face of cell k+1
            const int gd = rad_face_flux<2>(c, c_hat, tau_corr, tauZ, hiZ, loZn, GzHi);
            const int m = k + 1;
            if (active && ((m >= k0 && m < k1) || m == g.nz)) nguard += gd;
        }
        if (in_chunk) {
            if (active) {
                const int cidx = g.at(gi, gj, k);
                uc[0] = R.E[cidx]; uc[1] = R.Fx[cidx]; uc[2] = R.Fy[cidx]; uc[3] = R.Fz[cidx];
                if (stage == 1) { u0[0] = R0.E[cidx]; u0[1] = R0.Fx[cidx]; u0[2] = R0.Fy[cidx]; u0[3] = R0.Fz[cidx]; }
            }
            double L[4];
#pragma unroll
            for (int v = 0; v < 4; ++v) L[v] = s.hiX[v][ty][tx];
            int gd = rad_face_flux<0>(c, c_hat, tau_corr, tauX, L, loX, GxLo);   // low x face of the own cell
            if (cnt_own_x) nguard += gd;
#pragma unroll
            for (int v = 0; v < 4; ++v) L[v] = s.hiY[v][ty][tx];
            gd = rad_face_flux<1>(c, c_hat, tau_corr, tauY, L, loY, GyLo);
            if (cnt_own_y) nguard += gd;
            if (tx >= 1) {
#pragma unroll
                for (int v = 0; v < 4; ++v) s.fl.gx[v][ty][tx - 1] = GxLo[v];
            }
            if (ty >= 1) {
#pragma unroll
                for (int v = 0; v < 4; ++v) s.fl.gy[v][ty - 1][tx] = GyLo[v];
            }
            if (t < TX + TY) {      // the faces at the high end of the tile
                double Rr[4], G[4];
                if (t < TY) {
#pragma unroll
                    for (int v = 0; v < 4; ++v) { L[v] = s.hiX[v][t][TX]; Rr[v] = s.loXe[v][t]; }
                    gd = rad_face_flux<0>(c, c_hat, tau_corr, tauHi, L, Rr, G);
#pragma unroll
                    for (int v = 0; v < 4; ++v) s.fl.gx[v][t][TX - 1] = G[v];
                } else {
                    const int cx = t - TY;
#pragma unroll
                    for (int v = 0; v < 4; ++v) { L[v] = s.hiY[v][TY][cx]; Rr[v] = s.loYe[v][cx]; }
                    gd = rad_face_flux<1>(c, c_hat, tau_corr, tauHi, L, Rr, G);
#pragma unroll
                    for (int v = 0; v < 4; ++v) s.fl.gy[v][TY - 1][cx] = G[v];
                }
                if (cnt_hiface) nguard += gd;
            }
        }
        __syncthreads();   // S3: fluxes visible
        // ---- phase U: divergence and stage update ----------------------------------------------
        if (in_chunk && active) {
            double res[4];
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                const double div = ((s.fl.gx[v][ty][tx] - GxLo[v]) + (s.fl.gy[v][ty][tx] - GyLo[v])) + (GzHi[v] - GzLo[v]);
                const double us = uc[v] - dtdx * div;
                res[v] = stage == 0 ? us : 0.5 * u0[v] + 0.5 * us;
            }
            const int cidx = g.at(gi, gj, k);
            out.E[cidx] = res[0]; out.Fx[cidx] = res[1]; out.Fy[cidx] = res[2]; out.Fz[cidx] = res[3];
        }
#pragma unroll
        for (int v = 0; v < 4; ++v) { GzLo[v] = GzHi[v]; hiZ[v] = hiZn[v]; }
        __syncthreads();   // S4: flux buffers (aliasing plane W) and ring slot k-1 free
    }
    // x/y states and faces were counted for every plane of the chunk only (in_chunk), as the oracle
    // counts interior planes only; reduce the integer diagnostics over the warp before the atomics
    for (int off = 16; off > 0; off >>= 1) {
        nfall += __shfl_xor_sync(0xffffffffu, nfall, off);
        nguard += __shfl_xor_sync(0xffffffffu, nguard, off);
        bad += __shfl_xor_sync(0xffffffffu, bad, off);
    }
    if (tx == 0) {
        if (nfall) atomicAdd((unsigned long long *)&ctr->fallback, (unsigned long long)nfall);
        if (nguard) atomicAdd((unsigned long long *)&ctr->guard, (unsigned long long)nguard);
        if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
    }
}

static int rad_chunk_length(int nz_planes, int tiles_xy)
{
    int lz = 32;
    while (lz > 16 && (long long)tiles_xy * ((nz_planes + lz - 1) / lz) < 148 * 2 * 4) lz -= 8;
    if (lz > nz_planes) lz = nz_planes;
    return lz < 1 ? 1 : lz;
}

int launch_rad_stage(const Geom &g, const PhysConsts &pc, double dtdx, int stage, CRad4p R, CRad4p R0, const double *rho,
                     const double *kappaR, Rad4p out, Counters *ctr, cudaStream_t st)
{
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(rad_stage_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RadSmem));
        configured = true;
    }
    const int bx = (g.nx + TX - 1) / TX, by = (g.ny + TY - 1) / TY;
    const int lz = rad_chunk_length(g.nz, bx * by);
    dim3 grid(bx, by, (g.nz + lz - 1) / lz), block(TX, TY);
    rad_stage_kernel<<<grid, block, sizeof(RadSmem), st>>>(g, pc.c, pc.c_hat, pc.dx, (pc.flags & QK_FLAG_TAU_CORR) ? 1 : 0,
                                                           dtdx, stage, R, R0, rho, kappaR, out, lz, ctr);
    return 1;
}

}  // namespace qk
