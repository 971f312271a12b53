// k_exchange.cu -- per-cell implicit matter-radiation exchange, eq 26-43.
//
// One thread per interior cell, x fastest so that every field access of a warp is one
// coalesced 256-byte row segment.  No spatial coupling: the kernel is a pointwise map that
// reads 11 doubles and writes 8 (152 B/cell) around a Newton loop of a few iterations
// (HBM-bound).  Counters are reduced per warp before the atomics.
#include "qk_internal.h"
#include "qk_math.cuh"
#include "qk_fastmath.cuh"

namespace qk {

#ifndef QK_EX_MINB
#define QK_EX_MINB 7     // <= 73 registers: 1.09 -> 1.02 ms at 256^3 (6: 1.04, 5: 1.10); 8 spills into the Newton loop (1.45 ms)
#endif
__global__ void __launch_bounds__(128, QK_EX_MINB) exchange_kernel(Geom g, ExchangeConsts kc, double dt, const double *__restrict__ rho,
                                                       double *__restrict__ mx, double *__restrict__ my,
                                                       double *__restrict__ mz, double *__restrict__ E,
                                                       double *__restrict__ Er, double *__restrict__ Fx,
                                                       double *__restrict__ Fy, double *__restrict__ Fz,
                                                       const double *__restrict__ kP, const double *__restrict__ kR,
                                                       const double *__restrict__ src, Hydro5 Wout, Rad4p Sout, Counters *ctr, StateCache *cache)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    int iters = 0, fail = 0, bad = 0, bad_hydro = 0;
    double smax = 0.0;
    if (i < g.nx) {
        const int cidx = g.at(i, j, k);
        double m0 = mx[cidx], m1 = my[cidx], m2 = mz[cidx];
        double e = E[cidx], er = Er[cidx];
        double f0 = Fx[cidx], f1 = Fy[cidx], f2 = Fz[cidx];
        const double S = src ? dt * src[cidx] : 0.0;              // eq 27: energy added during the substep (X13)
        const int rc = exchange_cell(kc, dt, rho[cidx], m0, m1, m2, e, er, f0, f1, f2, kP[cidx], kR[cidx], S, iters);
        fail = (rc == 4);
        bad = (rc == 5);
        if (!kc.static_matter) { mx[cidx] = m0; my[cidx] = m1; mz[cidx] = m2; }
        E[cidx] = e; Er[cidx] = er;
        Fx[cidx] = f0; Fy[cidx] = f1; Fz[cidx] = f2;
        if (Wout.rho) {
            // reconstruction variables of the updated cell for the next hydro / radiation stage and its CFL
            // speed (same operations as prim_kernel, rad_prim_kernel and cfl_max_speed_kernel)
            Prim p;
            double sp;
            cell_prim_speed(kc.gamma, rho[cidx], m0, m1, m2, e, true, p, sp);
            Wout.rho[cidx] = p.rho; Wout.mx[cidx] = p.vx; Wout.my[cidx] = p.vy; Wout.mz[cidx] = p.vz; Wout.E[cidx] = p.P;
            if (!(p.rho > 0.0) || !(p.P > 0.0)) bad_hydro = 1;
            else smax = sp;
            const double cE = kc.c * er;
            Sout.E[cidx] = er; Sout.Fx[cidx] = f0 / cE; Sout.Fy[cidx] = f1 / cE; Sout.Fz[cidx] = f2 / cE;
        }
    }
    int tot = iters, mxit = iters;
    for (int off = 16; off > 0; off >>= 1) {
        tot += __shfl_xor_sync(0xffffffffu, tot, off);
        mxit = max(mxit, __shfl_xor_sync(0xffffffffu, mxit, off));
        fail += __shfl_xor_sync(0xffffffffu, fail, off);
        bad += __shfl_xor_sync(0xffffffffu, bad, off);
        bad_hydro += __shfl_xor_sync(0xffffffffu, bad_hydro, off);
        const double o = __shfl_xor_sync(0xffffffffu, smax, off);
        if (o > smax) smax = o;
    }
    if ((threadIdx.x & 31) == 0) {
        if (tot) atomicAdd((unsigned long long *)&ctr->newton_total, (unsigned long long)tot);
        if (mxit > 0) atomicMax(&ctr->newton_max, mxit);
        if (fail) atomicAdd((unsigned long long *)&ctr->newton_fail, (unsigned long long)fail);
        if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
        if (Wout.rho) {
            const unsigned long long bits = (unsigned long long)__double_as_longlong(smax);
            if (bits > *(volatile unsigned long long *)&cache->smax_bits) atomicMax(&cache->smax_bits, bits);
            if (bad_hydro) atomicAdd((unsigned long long *)&cache->cfl_bad, (unsigned long long)bad_hydro);
        }
    }
}

// kappa = kappa0 q^|e|, q = rho/rho0 (e > 0) or rho0/rho (e < 0), by repeated multiplication (X14): the density
// power laws of the paper's tests, interior cells, evaluated before a radiation subcycle
__global__ void __launch_bounds__(128) opacity_law_kernel(Geom g, const double *__restrict__ rho, double *__restrict__ kP,
                                                          double *__restrict__ kR, double kP0, double kR0, double rho0, int e)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.nx) return;
    const int cidx = g.at(i, blockIdx.y, blockIdx.z);
    const double r = rho[cidx];
    const double q = e < 0 ? rho0 / r : r / rho0;
    const int n = e < 0 ? -e : e;
    double kp = kP0, kr = kR0;
    for (int m = 0; m < n; ++m) { kp = kp * q; kr = kr * q; }
    kP[cidx] = kp; kR[cidx] = kr;
}

int launch_opacity_law(const Geom &g, const double *rho, double *kP, double *kR, double kP0, double kR0, double rho0,
                       int e, cudaStream_t st)
{
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    opacity_law_kernel<<<grid, 128, 0, st>>>(g, rho, kP, kR, kP0, kR0, rho0, e);
    return 1;
}

int launch_exchange(const Geom &g, const PhysConsts &pc, double dt, const double *rho, double *mx, double *my,
                    double *mz, double *E, double *Er, double *Fx, double *Fy, double *Fz, const double *kP,
                    const double *kR, const double *src, Hydro5 Wout, Rad4p Sout, Counters *ctr, StateCache *cache,
                    cudaStream_t st)
{
    ExchangeConsts kc;
    kc.c = pc.c; kc.c_hat = pc.c_hat; kc.a_rad = pc.a_rad; kc.kB_mu = pc.kB_mu; kc.gamma = pc.gamma;
    kc.tol = pc.newton_tol; kc.maxit = pc.newton_maxit;
    kc.alpha = pc.eos_alpha; kc.eos_alpha_t3 = pc.eos_alpha > 0.0;
    kc.literal_stop = (pc.flags & QK_FLAG_NEWTON_LITERAL) != 0;
    kc.static_matter = (pc.flags & QK_FLAG_STATIC_MATTER) != 0;
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    exchange_kernel<<<grid, 128, 0, st>>>(g, kc, dt, rho, mx, my, mz, E, Er, Fx, Fy, Fz, kP, kR, src, Wout, Sout, ctr, cache);
    return 1;
}

}  // namespace qk
