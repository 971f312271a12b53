// k_sweep.cu -- physics policies and launchers of the direction-split sweep path (k_sweep.cuh).
//
// Hydro stage:  prim (cons -> rho, v, P, all cells)  ->  chi (flattening, H6)
//   -> x sweep (D = dFx) -> y sweep (D += dFy) -> z sweep (U' = RK(U, (dFx+dFy)+dFz)).
// Radiation stage:  rad prim (E_r, f = F_r/(c E_r))  -> x, y, z sweeps the same way.
#include <stdlib.h>

#include "k_sweep.cuh"
#include "qk_fastmath.cuh"

#ifndef QK_BLX_H
#define QK_BLX_H 1
#endif
#ifndef QK_BLM_H
#define QK_BLM_H 0
#endif
#ifndef QK_BLX_R
#define QK_BLX_R 1
#endif
#ifndef QK_BLM_R
#define QK_BLM_R 1
#endif

namespace qk {

// Out-of-line plain-operator versions of the face fluxes: taken only by the faces whose operands left
// the range in which the branch-free division / square root of qk_fastmath.cuh are exact.
__device__ __noinline__ Flux5 hllc_flux_slow(double gamma, double rL, double uL, double vL, double wL, double pL,
                                             double rR, double uR, double vR, double wR, double pR)
{
    return hllc_flux(gamma, rL, uL, vL, wL, pL, rR, uR, vR, wR, pR);
}

template <int CL>
__device__ __noinline__ Rad4 rad_hll_flux_slow(double c, double c_hat, double EL, double fxL, double fyL, double fzL,
                                               double ER, double fxR, double fyR, double fzR, int n, double tau,
                                               bool tau_corr, int *guard)
{
    int gd;
    const Rad4 G = rad_hll_flux<CL>(c, c_hat, EL, fxL, fyL, fzL, ER, fxR, fyR, fzR, n, tau, tau_corr, gd);
    *guard = gd;
    return G;
}

// ---- hydro ------------------------------------------------------------------------------------------
// RECON: 0 = PPM, 1 = PLM with the MC limiter
template <int RECON>
struct HydroPhT {
    static constexpr int NV = 5;
    static constexpr bool COUNTS = false;
    // select-only PPM limiter (same values): measured faster in the x sweep, slower in the marching sweeps
    static constexpr int BL_X = QK_BLX_H, BL_MARCH = QK_BLM_H;
    static constexpr bool CARRY = true;    // marching sweeps carry the raw interface value (measured: -1.5 %)   // 0 branches, 1 selects, 2 selects in lockstep
    const double *w[5];        // rho, vx, vy, vz, P (ghost cells included)
    const double *chi;         // flattening coefficient of the cells -1..n
    double gamma;
    __device__ __forceinline__ double ld(int v, int cidx) const { return __ldg(w[v] + cidx); }
    __device__ __forceinline__ double aux(int cidx) const { return __ldg(chi + cidx); }
    // x sweep: staged sources 0..4 = W, 5 = chi
    __device__ __forceinline__ const double *src(int s) const { return s < 5 ? w[s] : chi; }
    __device__ __forceinline__ double win(int v, const double (*buf)[SW_XSEG], int p) const { return buf[v][p]; }
    __device__ __forceinline__ double win_aux(const double (*buf)[SW_XSEG], int p) const { return buf[5][p]; }
    template <int BL, class Q>
    __device__ __forceinline__ int states(Q q, double x, double lo[5], double hi[5]) const
    {
        if (RECON == 1) {
            double l[5], h[5];
            plm_states<5>(q, l, h);
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                const double c = q(v, 2);
                lo[v] = c + x * (l[v] - c);         // flatten toward the cell average
                hi[v] = c + x * (h[v] - c);
            }
        } else {
            ppm_cell<BL>(q, x, lo, hi);
        }
        return 0;
    }
    template <int BL, class Q>
    __device__ __forceinline__ int states_carry(Q q, double x, double ifc[5], double lo[5], double hi[5]) const
    {
        if (RECON == 1) return states<BL>(q, x, lo, hi);
        double l[5], h[5];
        ppm_states_carry<BL, 5>(q, ifc, l, h);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double c = q(v, 2);
            lo[v] = c + x * (l[v] - c);         // flatten toward the cell average
            hi[v] = c + x * (h[v] - c);
        }
        return 0;
    }
    // MODE 2 epilogue: primitives of the updated cell for the next stage's sweeps and,
    // after the last stage, the cell's CFL signal speed |v| + c_s (eq 21), same operations as
    // prim_kernel / cfl_max_speed_kernel.
    struct Tail { double smax = 0.0; int bad = 0; };
    __device__ __forceinline__ void finish(int cidx, const double u[5], const FieldsRW<5> &wout, bool last, Tail &t) const
    {
        Prim p;
        double sp;
        cell_prim_speed(gamma, u[0], u[1], u[2], u[3], u[4], last, p, sp);
        wout.f[0][cidx] = p.rho; wout.f[1][cidx] = p.vx; wout.f[2][cidx] = p.vy; wout.f[3][cidx] = p.vz;
        wout.f[4][cidx] = p.P;
        if (!(p.rho > 0.0) || !(p.P > 0.0)) { ++t.bad; return; }
        if (last && sp > t.smax) t.smax = sp;
    }
    __device__ __forceinline__ void finish_block(Tail &t, bool last, Counters *ctr, StateCache *cache) const
    {
        double smax = t.smax;
        int bad = t.bad;
        for (int off = 16; off > 0; off >>= 1) {
            const double o = __shfl_xor_sync(0xffffffffu, smax, off);
            if (o > smax) smax = o;
            bad += __shfl_xor_sync(0xffffffffu, bad, off);
        }
        if ((threadIdx.x & 31) == 0) {
            if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
            if (last) {
                const unsigned long long bits = (unsigned long long)__double_as_longlong(smax);
                // most warps lose against the running maximum: look before paying for the atomic
                if (bits > *(volatile unsigned long long *)&cache->smax_bits) atomicMax(&cache->smax_bits, bits);
                if (bad) atomicAdd((unsigned long long *)&cache->cfl_bad, (unsigned long long)bad);
            }
        }
    }
    template <int DIR>
    __device__ __forceinline__ int flux(const double L[5], const double R[5], double, double, double F[5]) const
    {
#ifdef QK_PLAIN_DIVSQRT
        face_flux<DIR>(gamma, L, R, F);
#else
        constexpr int n = 1 + DIR, t1 = 1 + (DIR + 1) % 3, t2 = 1 + (DIR + 2) % 3;
        unsigned risk = 0;
        Flux5 f = hllc_flux_fast(gamma, L[0], L[n], L[t1], L[t2], L[4], R[0], R[n], R[t1], R[t2], R[4], risk);
        if (risk) f = hllc_flux_slow(gamma, L[0], L[n], L[t1], L[t2], L[4], R[0], R[n], R[t1], R[t2], R[4]);
        F[0] = f.m; F[n] = f.pn; F[t1] = f.pt1; F[t2] = f.pt2; F[4] = f.e;
#endif
        return 0;
    }
};

// ---- radiation --------------------------------------------------------------------------------------
// RECON as for hydro; CL: 0 = Levermore closure (eq 23-25), 1 = Eddington approximation
template <int RECON, int CL>
struct RadPhT {
    static constexpr int NV = 4;
    static constexpr bool COUNTS = true;
    static constexpr int BL_X = QK_BLX_R, BL_MARCH = QK_BLM_R;
    static constexpr bool CARRY = false;   // measured slower with the select-only limiter (+1.5 %)
    const double *s[4];        // E_r, fx, fy, fz
    const double *rho, *kR;
    double c, c_hat, dx;
    int tau_corr;
    __device__ __forceinline__ double ld(int v, int cidx) const
    {
        if (v < 4) return __ldg(s[v] + cidx);
        return __ldg(kR + cidx) * __ldg(rho + cidx);      // kappa_R rho of the cell
    }
    __device__ __forceinline__ double aux(int) const { return 0.0; }
    // x sweep: staged sources 0..3 = S, 4 = kappa_R, 5 = rho
    __device__ __forceinline__ const double *src(int i) const { return i < 4 ? s[i] : (i == 4 ? kR : rho); }
    __device__ __forceinline__ double win(int v, const double (*buf)[SW_XSEG], int p) const
    {
        return v < 4 ? buf[v][p] : buf[4][p] * buf[5][p];
    }
    __device__ __forceinline__ double win_aux(const double (*)[SW_XSEG], int) const { return 0.0; }
    template <int BL, class Q>
    __device__ __forceinline__ int states(Q q, double, double lo[4], double hi[4]) const
    {
        if (RECON == 0) return rad_ppm_cell<BL>(q, lo, hi);
        plm_states<4>(q, lo, hi);
        int nfall = 0;      // first-order fallback per face state, as in rad_ppm_cell
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
    template <int BL, class Q>
    __device__ __forceinline__ int states_carry(Q q, double x, double ifc[4], double lo[4], double hi[4]) const
    {
        if (RECON == 1) return states<BL>(q, x, lo, hi);
        ppm_states_carry<BL, 4>(q, ifc, lo, hi);
        int nfall = 0;      // first-order fallback per face state, as in rad_ppm_cell
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
    // MODE 2 epilogue: (E_r, f = F_r / (c E_r)) of the updated cell, as rad_prim_kernel
    struct Tail { int bad = 0; };
    __device__ __forceinline__ void finish(int cidx, const double r[4], const FieldsRW<4> &sout, bool, Tail &t) const
    {
        const double cE = c * r[0];
        sout.f[0][cidx] = r[0];
        sout.f[1][cidx] = r[1] / cE;
        sout.f[2][cidx] = r[2] / cE;
        sout.f[3][cidx] = r[3] / cE;
        if (!(r[0] > 0.0)) ++t.bad;
    }
    __device__ __forceinline__ void finish_block(Tail &t, bool, Counters *ctr, StateCache *) const
    {
        int bad = t.bad;
        for (int off = 16; off > 0; off >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, off);
        if ((threadIdx.x & 31) == 0 && bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
    }
    template <int DIR>
    __device__ __forceinline__ int flux(const double L[4], const double R[4], double krL, double krR, double G[4]) const
    {
        const double tau = (0.5 * (krL + krR)) * dx;
#ifdef QK_PLAIN_DIVSQRT
        return rad_face_flux<DIR>(c, c_hat, tau_corr != 0, tau, L, R, G);
#else
        unsigned risk = 0;
        int guard;
        Rad4 g = rad_hll_flux_fast<CL>(c, c_hat, L[0], L[1], L[2], L[3], R[0], R[1], R[2], R[3], DIR, tau, tau_corr != 0,
                                   guard, risk);
        if (risk) g = rad_hll_flux_slow<CL>(c, c_hat, L[0], L[1], L[2], L[3], R[0], R[1], R[2], R[3], DIR, tau,
                                        tau_corr != 0, &guard);
        G[0] = g.e; G[1] = g.x; G[2] = g.y; G[3] = g.z;
        return guard;
#endif
    }
};

// ---- flattening coefficient in two pointwise passes (H6) -------------------------------
// pass 1: chi~_x, chi~_y, chi~_z of every cell of [-2, n+1]^3 (one evaluation per cell and direction);
// pass 2: chi = min over the three directions and the -1, 0, +1 neighbours along each, cells [-1, n]^3.
__global__ void __launch_bounds__(128) chi_dir_kernel(Geom g, double gamma, const double *__restrict__ P,
                                                      const double *__restrict__ vx, const double *__restrict__ vy,
                                                      const double *__restrict__ vz, double *__restrict__ cx,
                                                      double *__restrict__ cy, double *__restrict__ cz)
{
    // threads are dealt out over the (nx+4) x (ny+4) cells of a plane in row-major order: no idle tail per row
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int w = g.nx + 4;
    if (t >= w * (g.ny + 4)) return;
    const int jj = t / w;
    const int i = t - jj * w - 2, j = jj - 2, k = (int)blockIdx.y - 2;
    const int c = g.at(i, j, k), sy = g.sy, sz = g.sz;
    const double P0 = P[c];
    cx[c] = flatten_coeff_1d(gamma, P[c - 2], P[c - 1], P0, P[c + 1], P[c + 2], vx[c - 1], vx[c + 1]);
    cy[c] = flatten_coeff_1d(gamma, P[c - 2 * sy], P[c - sy], P0, P[c + sy], P[c + 2 * sy], vy[c - sy], vy[c + sy]);
    cz[c] = flatten_coeff_1d(gamma, P[c - 2 * sz], P[c - sz], P0, P[c + sz], P[c + 2 * sz], vz[c - sz], vz[c + sz]);
}

__global__ void __launch_bounds__(128) chi_min_kernel(Geom g, const double *__restrict__ cx, const double *__restrict__ cy,
                                                      const double *__restrict__ cz, double *__restrict__ chi)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int w = g.nx + 2;
    if (t >= w * (g.ny + 2)) return;
    const int jj = t / w;
    const int i = t - jj * w - 1, j = jj - 1, k = (int)blockIdx.y - 1;
    const int c = g.at(i, j, k), sy = g.sy, sz = g.sz;
    double x = 1.0;      // same nesting as the oracle: min(1, min(lo, min(mid, hi))) per direction
    x = lesser(x, lesser(cx[c - 1], lesser(cx[c], cx[c + 1])));
    x = lesser(x, lesser(cy[c - sy], lesser(cy[c], cy[c + sy])));
    x = lesser(x, lesser(cz[c - sz], lesser(cz[c], cz[c + sz])));
    chi[c] = x;
}

int launch_chi_two_pass(const Geom &g, double gamma, CHydro5 W, double *cx, double *cy, double *cz, double *chi,
                        cudaStream_t st)
{
    dim3 g1(((g.nx + 4) * (g.ny + 4) + 127) / 128, g.nz + 4), g2(((g.nx + 2) * (g.ny + 2) + 127) / 128, g.nz + 2);
    chi_dir_kernel<<<g1, 128, 0, st>>>(g, gamma, W.E, W.mx, W.my, W.mz, cx, cy, cz);
    chi_min_kernel<<<g2, 128, 0, st>>>(g, cx, cy, cz, chi);
    return 2;
}

static int sweep_len(int n_m, long long columns)
{
    static int forced = -1;
    if (forced < 0) {
        const char *e = getenv("QK_SWEEP_LEN");
        forced = e ? atoi(e) : 0;
    }
    int len = forced > 0 ? forced : 32;
    // keep at least ~8 waves of warps on 148 SMs x 16 warps
    while (forced <= 0 && len > 8 && columns / 32 * ((n_m + len - 1) / len) < 148LL * 16 * 8) len /= 2;
    if (len > n_m) len = n_m;
    return len < 1 ? 1 : len;
}

template <class PH>
static int launch_sweeps(const PH &ph, const Geom &g, double dtdx, int stage, FieldsRW<PH::NV> D, FieldsRO<PH::NV> U,
                         FieldsRO<PH::NV> U0, FieldsRW<PH::NV> out, FieldsRW<PH::NV> pout, Counters *ctr,
                         StateCache *cache, cudaStream_t st, int which, const double *dtdx_dev = nullptr)
{
    const RkArgs rk{dtdx, stage, dtdx_dev};
    int n = 0;
    if (which & 1) {
        constexpr int rows = SW_XROWS * SW_XNROW;
        dim3 grid((g.nx + SW_XW - 1) / SW_XW, (g.ny + rows - 1) / rows, g.nz), block(32, SW_XROWS);
        sweep_x_kernel<PH><<<grid, block, 0, st>>>(ph, g, D, ctr);
        ++n;
    }
    const int bx = (g.nx + SW_NT - 1) / SW_NT;
    if (which & 2) {
        const int len = sweep_len(g.ny, (long long)g.nx * g.nz);
        dim3 grid(bx, g.nz, (g.ny + len - 1) / len);
        sweep_march_kernel<PH, 1, 1><<<grid, SW_NT, 0, st>>>(ph, g, len, D, rk, U, U0, out, pout, ctr, cache);
        ++n;
    }
    if (which & 4) {
        const int len = sweep_len(g.nz, (long long)g.nx * g.ny);
        dim3 grid(bx, g.ny, (g.nz + len - 1) / len);
        sweep_march_kernel<PH, 2, 2><<<grid, SW_NT, 0, st>>>(ph, g, len, D, rk, U, U0, out, pout, ctr, cache);
        ++n;
    }
    return n;
}

int launch_hydro_sweeps(const Geom &g, double gamma, unsigned scheme, double dtdx, int stage, CHydro5 W,
                        const double *chi, Hydro5 D, CHydro5 U, CHydro5 U0, Hydro5 out, Hydro5 Wout, Counters *ctr,
                        StateCache *cache, cudaStream_t st, int which, const double *dtdx_dev)
{
    FieldsRW<5> d{{D.rho, D.mx, D.my, D.mz, D.E}}, o{{out.rho, out.mx, out.my, out.mz, out.E}};
    FieldsRO<5> u{{U.rho, U.mx, U.my, U.mz, U.E}}, u0{{U0.rho, U0.mx, U0.my, U0.mz, U0.E}};
    FieldsRW<5> wo{{Wout.rho, Wout.mx, Wout.my, Wout.mz, Wout.E}};
    auto go = [&](auto ph) {
        ph.w[0] = W.rho; ph.w[1] = W.mx; ph.w[2] = W.my; ph.w[3] = W.mz; ph.w[4] = W.E;
        ph.chi = chi; ph.gamma = gamma;
        return launch_sweeps(ph, g, dtdx, stage, d, u, u0, o, wo, ctr, cache, st, which, dtdx_dev);
    };
    return (scheme & QK_FLAG_PLM) ? go(HydroPhT<1>()) : go(HydroPhT<0>());
}

int launch_rad_sweeps(const Geom &g, const PhysConsts &pc, double dtdx, int stage, CRad4p S, const double *rho,
                      const double *kappaR, Rad4p D, CRad4p R, CRad4p R0, Rad4p out, Rad4p Sout, Counters *ctr,
                      cudaStream_t st, int which)
{
    FieldsRW<4> d{{D.E, D.Fx, D.Fy, D.Fz}}, o{{out.E, out.Fx, out.Fy, out.Fz}};
    FieldsRO<4> u{{R.E, R.Fx, R.Fy, R.Fz}}, u0{{R0.E, R0.Fx, R0.Fy, R0.Fz}};
    FieldsRW<4> so{{Sout.E, Sout.Fx, Sout.Fy, Sout.Fz}};
    auto go = [&](auto ph) {
        ph.s[0] = S.E; ph.s[1] = S.Fx; ph.s[2] = S.Fy; ph.s[3] = S.Fz;
        ph.rho = rho; ph.kR = kappaR;
        ph.c = pc.c; ph.c_hat = pc.c_hat; ph.dx = pc.dx; ph.tau_corr = (pc.flags & QK_FLAG_TAU_CORR) ? 1 : 0;
        return launch_sweeps(ph, g, dtdx, stage, d, u, u0, o, so, ctr, nullptr, st, which);
    };
    const bool plm = (pc.flags & QK_FLAG_PLM) != 0;
    const int cl = (pc.flags & QK_FLAG_EDDINGTON) ? 1 : ((pc.flags & QK_FLAG_MINERBO) ? 2 : 0);
    if (plm) return cl == 1 ? go(RadPhT<1, 1>()) : (cl == 2 ? go(RadPhT<1, 2>()) : go(RadPhT<1, 0>()));
    return cl == 1 ? go(RadPhT<0, 1>()) : (cl == 2 ? go(RadPhT<0, 2>()) : go(RadPhT<0, 0>()));
}

}  // namespace qk
