// k_hydro_ref.cu -- unfused hydro kernels (one kernel per sub-step of PAPER.md:120-172, all
// intermediates in HBM).  This is the first, simplest GPU statement of the hydro stage; the
// fused stage kernel of k_hydro.cu replaces it on the hot path.  It stays selectable
// (QK_PATH_UNFUSED) as an on-device cross-check of the fused kernel: both are hand-written
// CUDA, neither is a CPU fallback.
//
//   prim     : W = (rho, v, P) for every cell, ghosts included
//   flatten  : chi = min over directions and +-1 neighbours of chi~_d    (H6)
//   flux<d>  : PPM states of the two cells next to a face, flattened; HLLC
//   update   : U - (dt/dx)((dFx+dFy)+dFz), SSP-RK2 stage combination
#include "qk_internal.h"
#include "qk_math.cuh"

namespace qk {

__global__ void __launch_bounds__(256) prim_kernel(int ntot, double gamma, CHydro5 U, Hydro5 W, Counters *ctr)
{
    int bad = 0;
    for (int cidx = blockIdx.x * blockDim.x + threadIdx.x; cidx < ntot; cidx += gridDim.x * blockDim.x) {
        const Prim w = cons_to_prim(gamma, U.rho[cidx], U.mx[cidx], U.my[cidx], U.mz[cidx], U.E[cidx]);
        W.rho[cidx] = w.rho; W.mx[cidx] = w.vx; W.my[cidx] = w.vy; W.mz[cidx] = w.vz; W.E[cidx] = w.P;
        if (!(w.rho > 0.0) || !(w.P > 0.0)) ++bad;
    }
    if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
}

// chi~_d at cell c (stride s along d) from the primitive fields
__device__ __forceinline__ double chi_dir(double gamma, const double *__restrict__ P, const double *__restrict__ vn,
                                          int cidx, int s)
{
    return flatten_coeff_1d(gamma, P[cidx - 2 * s], P[cidx - s], P[cidx], P[cidx + s], P[cidx + 2 * s],
                            vn[cidx - s], vn[cidx + s]);
}

// chi for the cells -1..n in every direction (the cells whose face states a flux needs)
__global__ void __launch_bounds__(128) flatten_kernel(Geom g, double gamma, CHydro5 W, double *__restrict__ chi)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x - 1;
    const int j = (int)blockIdx.y - 1, k = (int)blockIdx.z - 1;
    if (i > g.nx) return;
    const int cidx = g.at(i, j, k);
    double x = 1.0;
    x = lesser(x, lesser(chi_dir(gamma, W.E, W.mx, cidx - 1, 1),
                         lesser(chi_dir(gamma, W.E, W.mx, cidx, 1), chi_dir(gamma, W.E, W.mx, cidx + 1, 1))));
    x = lesser(x, lesser(chi_dir(gamma, W.E, W.my, cidx - g.sy, g.sy),
                         lesser(chi_dir(gamma, W.E, W.my, cidx, g.sy), chi_dir(gamma, W.E, W.my, cidx + g.sy, g.sy))));
    x = lesser(x, lesser(chi_dir(gamma, W.E, W.mz, cidx - g.sz, g.sz),
                         lesser(chi_dir(gamma, W.E, W.mz, cidx, g.sz), chi_dir(gamma, W.E, W.mz, cidx + g.sz, g.sz))));
    chi[cidx] = x;
}

// flattened PPM state of `q` at the high face of cell c-s and at the low face of cell c
__device__ __forceinline__ void face_pair(const double *__restrict__ q, int cidx, int s, double chiL, double chiR,
                                          double &left, double &right)
{
    const double qm3 = q[cidx - 3 * s], qm2 = q[cidx - 2 * s], qm1 = q[cidx - s];
    const double q0 = q[cidx], qp1 = q[cidx + s], qp2 = q[cidx + 2 * s];
    double lo, hi;
    ppm_face_states(qm3, qm2, qm1, q0, qp1, lo, hi);      // cell c-s: use its high face
    left = qm1 + chiL * (hi - qm1);
    ppm_face_states(qm2, qm1, q0, qp1, qp2, lo, hi);      // cell c: use its low face
    right = q0 + chiR * (lo - q0);
}

template <int DIR>
__global__ void __launch_bounds__(128) hydro_flux_kernel(Geom g, double gamma, CHydro5 W, const double *__restrict__ chi,
                                                         Hydro5 flux)
{
    // faces 0..n along DIR (the low face of cells 0..n), interior range in the other two
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    const int ex = g.nx + (DIR == 0), ey = g.ny + (DIR == 1), ez = g.nz + (DIR == 2);
    if (i >= ex || j >= ey || k >= ez) return;
    const int s = DIR == 0 ? 1 : (DIR == 1 ? g.sy : g.sz);
    const int cidx = g.at(i, j, k);
    const double *vn = DIR == 0 ? W.mx : (DIR == 1 ? W.my : W.mz);
    const double *vt1 = DIR == 0 ? W.my : (DIR == 1 ? W.mz : W.mx);
    const double *vt2 = DIR == 0 ? W.mz : (DIR == 1 ? W.mx : W.my);
    const double chiL = chi[cidx - s], chiR = chi[cidx];
    double rL, rR, uL, uR, vL, vR, wL, wR, pL, pR;
    face_pair(W.rho, cidx, s, chiL, chiR, rL, rR);
    face_pair(vn, cidx, s, chiL, chiR, uL, uR);
    face_pair(vt1, cidx, s, chiL, chiR, vL, vR);
    face_pair(vt2, cidx, s, chiL, chiR, wL, wR);
    face_pair(W.E, cidx, s, chiL, chiR, pL, pR);
    const Flux5 F = hllc_flux(gamma, rL, uL, vL, wL, pL, rR, uR, vR, wR, pR);
    double *fn = DIR == 0 ? flux.mx : (DIR == 1 ? flux.my : flux.mz);
    double *ft1 = DIR == 0 ? flux.my : (DIR == 1 ? flux.mz : flux.mx);
    double *ft2 = DIR == 0 ? flux.mz : (DIR == 1 ? flux.mx : flux.my);
    flux.rho[cidx] = F.m; fn[cidx] = F.pn; ft1[cidx] = F.pt1; ft2[cidx] = F.pt2; flux.E[cidx] = F.e;
}

__device__ __forceinline__ double rk_update(double u, double u0, double dtdx, const double *__restrict__ fx,
                                            const double *__restrict__ fy, const double *__restrict__ fz, int cidx,
                                            int sy, int sz, int stage)
{
    const double div = ((fx[cidx + 1] - fx[cidx]) + (fy[cidx + sy] - fy[cidx])) + (fz[cidx + sz] - fz[cidx]);
    const double us = u - dtdx * div;
    return stage == 0 ? us : 0.5 * u0 + 0.5 * us;
}

__global__ void __launch_bounds__(128) hydro_update_kernel(Geom g, double dtdx, int stage, CHydro5 U, CHydro5 U0,
                                                           CHydro5 fx, CHydro5 fy, CHydro5 fz, Hydro5 out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.nx) return;
    const int cidx = g.at(i, blockIdx.y, blockIdx.z);
    out.rho[cidx] = rk_update(U.rho[cidx], U0.rho[cidx], dtdx, fx.rho, fy.rho, fz.rho, cidx, g.sy, g.sz, stage);
    out.mx[cidx] = rk_update(U.mx[cidx], U0.mx[cidx], dtdx, fx.mx, fy.mx, fz.mx, cidx, g.sy, g.sz, stage);
    out.my[cidx] = rk_update(U.my[cidx], U0.my[cidx], dtdx, fx.my, fy.my, fz.my, cidx, g.sy, g.sz, stage);
    out.mz[cidx] = rk_update(U.mz[cidx], U0.mz[cidx], dtdx, fx.mz, fy.mz, fz.mz, cidx, g.sy, g.sz, stage);
    out.E[cidx] = rk_update(U.E[cidx], U0.E[cidx], dtdx, fx.E, fy.E, fz.E, cidx, g.sy, g.sz, stage);
}

int launch_prim(const Geom &g, double gamma, CHydro5 U, Hydro5 W, Counters *ctr, cudaStream_t st)
{
    int blocks = (g.ntot + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    prim_kernel<<<blocks, 256, 0, st>>>(g.ntot, gamma, U, W, ctr);
    return 1;
}

int launch_flatten(const Geom &g, double gamma, CHydro5 W, double *chi, cudaStream_t st)
{
    dim3 grid((g.nx + 2 + 127) / 128, g.ny + 2, g.nz + 2);
    flatten_kernel<<<grid, 128, 0, st>>>(g, gamma, W, chi);
    return 1;
}

int launch_hydro_flux(const Geom &g, double gamma, int dir, CHydro5 W, const double *chi, Hydro5 flux, cudaStream_t st)
{
    dim3 grid((g.nx + (dir == 0) + 127) / 128, g.ny + (dir == 1), g.nz + (dir == 2));
    if (dir == 0) hydro_flux_kernel<0><<<grid, 128, 0, st>>>(g, gamma, W, chi, flux);
    else if (dir == 1) hydro_flux_kernel<1><<<grid, 128, 0, st>>>(g, gamma, W, chi, flux);
    else hydro_flux_kernel<2><<<grid, 128, 0, st>>>(g, gamma, W, chi, flux);
    return 1;
}

int launch_hydro_update(const Geom &g, double dtdx, int stage, CHydro5 U, CHydro5 U0, CHydro5 fx, CHydro5 fy,
                        CHydro5 fz, Hydro5 out, cudaStream_t st)
{
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    hydro_update_kernel<<<grid, 128, 0, st>>>(g, dtdx, stage, U, U0, fx, fy, fz, out);
    return 1;
}

}  // namespace qk
