// k_rad_ref.cu -- unfused radiation-transport kernels, intermediates in HBM.
// Same role as k_hydro_ref.cu: first GPU statement of the stage and on-device cross-check of the
// fused kernel in k_rad.cu.
//
//   rad_prim : S = (E_r, f = F_r/(c E_r)) for every cell, ghosts included
//   flux<d>  : PPM states (no flattening), first-order fallback per face state when |f|>1 or
//              E_r<=0 (R3), closure + HLL with tau correction
//   update   : SSP-RK2 stage combination as for hydro
#include "qk_internal.h"
#include "qk_math.cuh"

namespace qk {

__global__ void __launch_bounds__(256) rad_prim_kernel(Geom g, double c, CRad4p R, Rad4p S, Counters *ctr)
{
    int bad = 0;
    for (int cidx = blockIdx.x * blockDim.x + threadIdx.x; cidx < g.ntot; cidx += gridDim.x * blockDim.x) {
        const double E = R.E[cidx], cE = c * E;
        S.E[cidx] = E;
        S.Fx[cidx] = R.Fx[cidx] / cE;
        S.Fy[cidx] = R.Fy[cidx] / cE;
        S.Fz[cidx] = R.Fz[cidx] / cE;
        if (!(E > 0.0)) {   // only interior cells count (their ghost images would double count)
            const int kk = cidx / g.sz, rem = cidx - kk * g.sz, jj = rem / g.sy, ii = rem - jj * g.sy;
            if (ii >= NG && ii < NG + g.nx && jj >= NG && jj < NG + g.ny && kk >= NG && kk < NG + g.nz) ++bad;
        }
    }
    if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
}

struct RadState { double E, fx, fy, fz; };

// both PPM face states of cell c along stride s, each reverted to the cell average when
// non-causal; nfall counts the reverted states
__device__ __forceinline__ void rad_cell_states(CRad4p S, int cidx, int s, RadState &lo, RadState &hi, int &nfall)
{
    ppm_face_states(S.E[cidx - 2 * s], S.E[cidx - s], S.E[cidx], S.E[cidx + s], S.E[cidx + 2 * s], lo.E, hi.E);
    ppm_face_states(S.Fx[cidx - 2 * s], S.Fx[cidx - s], S.Fx[cidx], S.Fx[cidx + s], S.Fx[cidx + 2 * s], lo.fx, hi.fx);
    ppm_face_states(S.Fy[cidx - 2 * s], S.Fy[cidx - s], S.Fy[cidx], S.Fy[cidx + s], S.Fy[cidx + 2 * s], lo.fy, hi.fy);
    ppm_face_states(S.Fz[cidx - 2 * s], S.Fz[cidx - s], S.Fz[cidx], S.Fz[cidx + s], S.Fz[cidx + 2 * s], lo.fz, hi.fz);
    nfall = 0;
    double f2 = (lo.fx * lo.fx + lo.fy * lo.fy) + lo.fz * lo.fz;
    if (f2 > 1.0 || !(lo.E > 0.0)) {
        lo.E = S.E[cidx]; lo.fx = S.Fx[cidx]; lo.fy = S.Fy[cidx]; lo.fz = S.Fz[cidx];
        nfall += 1;
    }
    f2 = (hi.fx * hi.fx + hi.fy * hi.fy) + hi.fz * hi.fz;
    if (f2 > 1.0 || !(hi.E > 0.0)) {
        hi.E = S.E[cidx]; hi.fx = S.Fx[cidx]; hi.fy = S.Fy[cidx]; hi.fz = S.Fz[cidx];
        nfall += 2;
    }
}

template <int DIR>
__global__ void __launch_bounds__(128) rad_flux_kernel(Geom g, double c, double c_hat, double dx, bool tau_corr, CRad4p S,
                                                       const double *__restrict__ rho, const double *__restrict__ kR,
                                                       Rad4p flux, Counters *ctr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    const int ex = g.nx + (DIR == 0), ey = g.ny + (DIR == 1), ez = g.nz + (DIR == 2);
    int nfall = 0, guard = 0;
    if (i < ex && j < ey && k < ez) {
        const int s = DIR == 0 ? 1 : (DIR == 1 ? g.sy : g.sz);
        const int cidx = g.at(i, j, k);
        const int pos = DIR == 0 ? i : (DIR == 1 ? j : k);
        const int npos = DIR == 0 ? g.nx : (DIR == 1 ? g.ny : g.nz);
        RadState loL, hiL, loR, hiR;
        int fallL, fallR;
        rad_cell_states(S, cidx - s, s, loL, hiL, fallL);
        rad_cell_states(S, cidx, s, loR, hiR, fallR);
        // Each face state is counted once over the grid: the face owns the high state of its
        // left cell and the low state of its right cell; the two states no flux uses (low
        // state of cell -1, high state of cell n) are counted at the first and last face.
        nfall = ((fallL >> 1) & 1) + (fallR & 1);
        if (pos == 0) nfall += fallL & 1;
        if (pos == npos) nfall += (fallR >> 1) & 1;
        const double tau = (0.5 * (kR[cidx - s] * rho[cidx - s] + kR[cidx] * rho[cidx])) * dx;
        const Rad4 G = rad_hll_flux(c, c_hat, hiL.E, hiL.fx, hiL.fy, hiL.fz, loR.E, loR.fx, loR.fy, loR.fz, DIR, tau,
                                    tau_corr, guard);
        flux.E[cidx] = G.e; flux.Fx[cidx] = G.x; flux.Fy[cidx] = G.y; flux.Fz[cidx] = G.z;
    }
    for (int off = 16; off > 0; off >>= 1) {
        nfall += __shfl_xor_sync(0xffffffffu, nfall, off);
        guard += __shfl_xor_sync(0xffffffffu, guard, off);
    }
    if ((threadIdx.x & 31) == 0) {
        if (nfall) atomicAdd((unsigned long long *)&ctr->fallback, (unsigned long long)nfall);
        if (guard) atomicAdd((unsigned long long *)&ctr->guard, (unsigned long long)guard);
    }
}

__device__ __forceinline__ double rk_update4(double u, double u0, double dtdx, const double *__restrict__ gx,
                                             const double *__restrict__ gy, const double *__restrict__ gz, int cidx,
                                             int sy, int sz, int stage)
{
    const double div = ((gx[cidx + 1] - gx[cidx]) + (gy[cidx + sy] - gy[cidx])) + (gz[cidx + sz] - gz[cidx]);
    const double us = u - dtdx * div;
    return stage == 0 ? us : 0.5 * u0 + 0.5 * us;
}

__global__ void __launch_bounds__(128) rad_update_kernel(Geom g, double dtdx, int stage, CRad4p R, CRad4p R0, CRad4p gx,
                                                         CRad4p gy, CRad4p gz, Rad4p out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.nx) return;
    const int cidx = g.at(i, blockIdx.y, blockIdx.z);
    out.E[cidx] = rk_update4(R.E[cidx], R0.E[cidx], dtdx, gx.E, gy.E, gz.E, cidx, g.sy, g.sz, stage);
    out.Fx[cidx] = rk_update4(R.Fx[cidx], R0.Fx[cidx], dtdx, gx.Fx, gy.Fx, gz.Fx, cidx, g.sy, g.sz, stage);
    out.Fy[cidx] = rk_update4(R.Fy[cidx], R0.Fy[cidx], dtdx, gx.Fy, gy.Fy, gz.Fy, cidx, g.sy, g.sz, stage);
    out.Fz[cidx] = rk_update4(R.Fz[cidx], R0.Fz[cidx], dtdx, gx.Fz, gy.Fz, gz.Fz, cidx, g.sy, g.sz, stage);
}

int launch_rad_prim(const Geom &g, double c, CRad4p R, Rad4p S, Counters *ctr, cudaStream_t st)
{
    int blocks = (g.ntot + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    rad_prim_kernel<<<blocks, 256, 0, st>>>(g, c, R, S, ctr);
    return 1;
}

int launch_rad_flux(const Geom &g, const PhysConsts &pc, int dir, CRad4p S, const double *rho, const double *kappaR,
                    Rad4p flux, Counters *ctr, cudaStream_t st)
{
    dim3 grid((g.nx + (dir == 0) + 127) / 128, g.ny + (dir == 1), g.nz + (dir == 2));
    const bool tc = (pc.flags & QK_FLAG_TAU_CORR) != 0;
    if (dir == 0) rad_flux_kernel<0><<<grid, 128, 0, st>>>(g, pc.c, pc.c_hat, pc.dx, tc, S, rho, kappaR, flux, ctr);
    else if (dir == 1) rad_flux_kernel<1><<<grid, 128, 0, st>>>(g, pc.c, pc.c_hat, pc.dx, tc, S, rho, kappaR, flux, ctr);
    else rad_flux_kernel<2><<<grid, 128, 0, st>>>(g, pc.c, pc.c_hat, pc.dx, tc, S, rho, kappaR, flux, ctr);
    return 1;
}

int launch_rad_update(const Geom &g, double dtdx, int stage, CRad4p R, CRad4p R0, CRad4p gx, CRad4p gy, CRad4p gz,
                      Rad4p out, cudaStream_t st)
{
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    rad_update_kernel<<<grid, 128, 0, st>>>(g, dtdx, stage, R, R0, gx, gy, gz, out);
    return 1;
}

}  // namespace qk
