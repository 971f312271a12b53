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

constexpr int QK_EX_MINB = 7;    // 72 registers, 40 B of spills: 1.04 -> 1.00 ms at 256^3 (6 CTAs / 80 registers 1.04, 8 / 64 1.00, 9 / 56 1.23, 5 / 96 1.16)
template <bool KT>
__global__ void __launch_bounds__(128, KT ? 5 : QK_EX_MINB) exchange_kernel(Geom g, ExchangeConsts kc, double dt_host, const double *__restrict__ dt_dev, const double *__restrict__ rho,
                                                       double *__restrict__ mx, double *__restrict__ my,
                                                       double *__restrict__ mz, double *__restrict__ E,
                                                       double *__restrict__ Er, double *__restrict__ Fx,
                                                       double *__restrict__ Fy, double *__restrict__ Fz,
                                                       const double *__restrict__ kP, const double *__restrict__ kR,
                                                       const double *__restrict__ src, Hydro5 Wout, Rad4p Sout, Counters *ctr, StateCache *cache)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    const double dt = dt_dev ? __ldg(dt_dev) : dt_host;
    int iters = 0, fail = 0, bad = 0, bad_hydro = 0;
    double smax = 0.0;
    if (i < g.nx) {
        const int cidx = g.at(i, j, k);
        double m0 = mx[cidx], m1 = my[cidx], m2 = mz[cidx];
        double e = E[cidx], er = Er[cidx];
        double f0 = Fx[cidx], f1 = Fy[cidx], f2 = Fz[cidx];
        const double S = src ? dt * src[cidx] : 0.0;              // eq 27: energy added during the substep (X13)
        double kp = kP[cidx], kr = kR[cidx];
        if (KT) opacity_density_part(rho[cidx], kc.kP0, kc.kR0, kc.rho0, kc.opac_exp, kp, kr);
        const int rc = exchange_cell<KT>(kc, dt, rho[cidx], m0, m1, m2, e, er, f0, f1, f2, kp, kr, S, iters);
        fail = (rc == 4);
        bad = (rc == 5);
        if (!kc.static_matter) { mx[cidx] = m0; my[cidx] = m1; mz[cidx] = m2; }
        E[cidx] = e; Er[cidx] = er;
        Fx[cidx] = f0; Fy[cidx] = f1; Fz[cidx] = f2;
        {
            // CFL signal speed of the updated cell (eq 21) and, when asked, its reconstruction variables for the next
            // hydro / radiation stage (same operations as cfl_max_speed_kernel, prim_kernel and rad_prim_kernel)
            Prim p;
            double sp;
            cell_prim_speed(kc.gamma, rho[cidx], m0, m1, m2, e, true, p, sp);
            if (!(p.rho > 0.0) || !(p.P > 0.0)) bad_hydro = 1;
            else smax = sp;
            if (Wout.mx) {        // rho and E_r are read from the state by the next stage: not stored again
                Wout.mx[cidx] = p.vx; Wout.my[cidx] = p.vy; Wout.mz[cidx] = p.vz; Wout.E[cidx] = p.P;
                const double cE = kc.c * er;
                Sout.Fx[cidx] = f0 / cE; Sout.Fy[cidx] = f1 / cE; Sout.Fz[cidx] = f2 / cE;
            }
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
        {
            const unsigned long long bits = (unsigned long long)__double_as_longlong(smax);
            if (bits > *(volatile unsigned long long *)&cache->smax_bits) atomicMax(&cache->smax_bits, bits);
            if (bad_hydro) atomicAdd((unsigned long long *)&cache->cfl_bad, (unsigned long long)bad_hydro);
        }
    }
}

// kappa = kappa0 (rho/rho0)^e (T/T0)^(texp2/2) for the interior cells (X14; the laws of the paper's tests,
// PAPER.md:464, 528, and Kramers-like temperature laws), from the density and gas temperature of the current
// state, evaluated before the transport part of a radiation subcycle
__global__ void __launch_bounds__(128) opacity_law_kernel(Geom g, ExchangeConsts kc, CHydro5 U, double *__restrict__ kP,
                                                          double *__restrict__ kR)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.nx) return;
    const int cidx = g.at(i, blockIdx.y, blockIdx.z);
    const double r = U.rho[cidx];
    double kp, kr;
    opacity_density_part(r, kc.kP0, kc.kR0, kc.rho0, kc.opac_exp, kp, kr);
    if (kc.texp2 != 0) {
        const double mx = U.mx[cidx], my = U.my[cidx], mz = U.mz[cidx];
        const double msq = (mx * mx + my * my) + mz * mz;
        const double Eg = U.E[cidx] - 0.5 * msq / r;
        const double T = kc.eos_alpha_t3 ? sqrt(sqrt(4.0 * Eg / kc.alpha)) : Eg / (r * kc.kB_mu / (kc.gamma - 1.0));
        const double tp = temperature_power(T, kc.T0, kc.texp2);
        kp = kp * tp; kr = kr * tp;
    }
    kP[cidx] = kp; kR[cidx] = kr;
}

static ExchangeConsts exchange_consts(const PhysConsts &pc)
{
    ExchangeConsts kc;
    kc.c = pc.c; kc.c_hat = pc.c_hat; kc.a_rad = pc.a_rad; kc.kB_mu = pc.kB_mu; kc.gamma = pc.gamma;
    kc.tol = pc.newton_tol; kc.maxit = pc.newton_maxit;
    kc.alpha = pc.eos_alpha; kc.eos_alpha_t3 = pc.eos_alpha > 0.0;
    kc.literal_stop = (pc.flags & QK_FLAG_NEWTON_LITERAL) != 0;
    kc.static_matter = (pc.flags & QK_FLAG_STATIC_MATTER) != 0;
    kc.kappa_T = pc.opac_rho0 > 0.0 && pc.opac_texp2 != 0;
    kc.texp2 = pc.opac_texp2; kc.opac_exp = pc.opac_exp;
    kc.T0 = pc.opac_T0; kc.kP0 = pc.opac_kP0; kc.kR0 = pc.opac_kR0; kc.rho0 = pc.opac_rho0;
    return kc;
}

int launch_opacity_law(const Geom &g, const PhysConsts &pc, CHydro5 U, double *kP, double *kR, cudaStream_t st)
{
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    opacity_law_kernel<<<grid, 128, 0, st>>>(g, exchange_consts(pc), U, kP, kR);
    return 1;
}

int launch_exchange(const Geom &g, const PhysConsts &pc, double dt, const double *dt_dev, const double *rho, double *mx, double *my,
                    double *mz, double *E, double *Er, double *Fx, double *Fy, double *Fz, const double *kP,
                    const double *kR, const double *src, Hydro5 Wout, Rad4p Sout, Counters *ctr, StateCache *cache,
                    cudaStream_t st)
{
    const ExchangeConsts kc = exchange_consts(pc);
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    if (kc.kappa_T)
        exchange_kernel<true><<<grid, 128, 0, st>>>(g, kc, dt, dt_dev, rho, mx, my, mz, E, Er, Fx, Fy, Fz, kP, kR, src, Wout, Sout, ctr, cache);
    else
        exchange_kernel<false><<<grid, 128, 0, st>>>(g, kc, dt, dt_dev, rho, mx, my, mz, E, Er, Fx, Fy, Fz, kP, kR, src, Wout, Sout, ctr, cache);
    return 1;
}

}  // namespace qk
