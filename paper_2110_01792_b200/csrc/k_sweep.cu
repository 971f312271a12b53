// k_sweep.cu -- physics policies and launchers of the stencil kernels of an RK stage (k_sweep.cuh) and the
// flattening-coefficient kernel.
//
// Hydro stage:  chi (flattening, H6) -> x sweep (D = dFx) -> y sweep (D += dFy) -> z sweep
// (U' = RK(U, D + dFz)).  Radiation stage:  x, y, z sweeps, same code with the radiation policy.
#include "k_sweep.cuh"
#include "qk_fastmath.cuh"
#include <type_traits>

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
    static constexpr int NV = 5, NSRC = 6;
    static constexpr bool COUNTS = false;
    // PPM limiter with branches in every sweep.  The select-only form (same values) was faster in the x sweep while its
    // division chains still branched; since the operand-window Riemann solver and the 16-byte row staging the x sweep is
    // bound by instruction issue and the fp64 pipe, and the branches skip the MC slope of every cell that is no
    // extremum: 0.712 -> 0.637 ms at 256^3 (lock-step form: 0.69 ms)
    static constexpr int BL_X = 0, BL_MARCH = 0;
    static constexpr bool CARRY = true;    // marching sweeps carry the raw interface value (measured: -1.5 %)
    // CTAs per SM.  z runs at 4 (126 registers, no spill) only because its update inputs are staged by cp.async and
    // never sit in registers during the Riemann solve: 0.81 -> 0.77 ms; with register loads 4 CTAs spill (1.10 ms).
    // y at 5 (96 registers) spills: 0.62 -> 0.78 ms.  x at 6 (78 registers, no spill): 0.637 -> 0.627 ms.
    static constexpr int X_MINB = 6, Y_MINB = 4, Z_MINB = 4;
    const double *w[5];        // rho, vx, vy, vz, P (ghost cells included)
    const double *chi;         // flattening coefficient of the cells -1..n
    double gamma;
    __device__ __forceinline__ double ld(int v, int cidx) const { return __ldg(w[v] + cidx); }
    __device__ __forceinline__ double aux(int cidx) const { return __ldg(chi + cidx); }
    // x sweep: staged sources 0..4 = W, 5 = chi
    __device__ __forceinline__ const double *src(int q) const { return q < 5 ? w[q] : chi; }
    __device__ __forceinline__ double win(int v, const double (*buf)[SW_XCOLS], int p) const { return buf[v][p]; }
    __device__ __forceinline__ double win_aux(const double (*buf)[SW_XCOLS], int p) const { return buf[5][p]; }
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
    // z epilogue: primitives of the updated cell for the next stage's sweeps and, after the last
    // stage, the cell's CFL signal speed |v| + c_s (eq 21), same operations as prim_kernel / cfl_max_speed_kernel
    struct Tail { double smax = 0.0; int bad = 0; };
    __device__ __forceinline__ void finish(int cidx, const double u[5], const FieldsRW<5> &wout, bool last, Tail &t) const
    {
        Prim p;
        double sp;
        cell_prim_speed(gamma, u[0], u[1], u[2], u[3], u[4], last, p, sp);
        // rho is its own primitive: the next stage reads it from the state this kernel has just written (8 B/cell less)
        wout.f[1][cidx] = p.vx; wout.f[2][cidx] = p.vy; wout.f[3][cidx] = p.vz;
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
        constexpr int n = 1 + DIR, t1 = 1 + (DIR + 1) % 3, t2 = 1 + (DIR + 2) % 3;
        unsigned risk = 0;
        Flux5 f = hllc_flux_fast(gamma, L[0], L[n], L[t1], L[t2], L[4], R[0], R[n], R[t1], R[t2], R[4], risk);
        if (risk) f = hllc_flux_slow(gamma, L[0], L[n], L[t1], L[t2], L[4], R[0], R[n], R[t1], R[t2], R[4]);
        F[0] = f.m; F[n] = f.pn; F[t1] = f.pt1; F[t2] = f.pt2; F[4] = f.e;
        return 0;
    }
};

// ---- radiation --------------------------------------------------------------------------------------
// RECON as for hydro; CL: 0 = Levermore closure (eq 23-25), 1 = Eddington approximation, 2 = Minerbo
template <int RECON, int CL>
struct RadPhT {
    static constexpr int NV = 4, NSRC = 6;
    static constexpr bool COUNTS = true;
    static constexpr int BL_X = 1, BL_MARCH = 1;
    static constexpr bool CARRY = false;   // measured slower with the select-only limiter (+1.5 %)
    static constexpr int X_MINB = 5, Y_MINB = 4, Z_MINB = 4;
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
    __device__ __forceinline__ const double *src(int q) const { return q < 4 ? s[q] : (q == 4 ? kR : rho); }
    __device__ __forceinline__ double win(int v, const double (*buf)[SW_XCOLS], int p) const
    {
        return v < 4 ? buf[v][p] : buf[4][p] * buf[5][p];
    }
    __device__ __forceinline__ double win_aux(const double (*)[SW_XCOLS], int) const { return 0.0; }
    template <int BL, class Q>
    __device__ __forceinline__ int states(Q q, double, double lo[4], double hi[4]) const
    {
        if (RECON == 0) return rad_ppm_cell<BL>(q, lo, hi);
        plm_states<4>(q, lo, hi);
        return rad_fallback(q, lo, hi);
    }
    template <int BL, class Q>
    __device__ __forceinline__ int states_carry(Q q, double x, double ifc[4], double lo[4], double hi[4]) const
    {
        if (RECON == 1) return states<BL>(q, x, lo, hi);
        ppm_states_carry<BL, 4>(q, ifc, lo, hi);
        return rad_fallback(q, lo, hi);
    }
    // z epilogue: (E_r, f = F_r / (c E_r)) of the updated cell, as rad_prim_kernel
    struct Tail { int bad = 0; };
    __device__ __forceinline__ void finish(int cidx, const double r[4], const FieldsRW<4> &sout, bool, Tail &t) const
    {
        const double cE = c * r[0];           // E_r is its own reconstruction variable: read from the state next stage
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
        unsigned risk = 0;
        int guard;
        Rad4 g = rad_hll_flux_fast<CL>(c, c_hat, L[0], L[1], L[2], L[3], R[0], R[1], R[2], R[3], DIR, tau, tau_corr != 0,
                                   guard, risk);
        if (risk) g = rad_hll_flux_slow<CL>(c, c_hat, L[0], L[1], L[2], L[3], R[0], R[1], R[2], R[3], DIR, tau,
                                        tau_corr != 0, &guard);
        G[0] = g.e; G[1] = g.x; G[2] = g.y; G[3] = g.z;
        return guard;
    }
};

// ---- flattening coefficient in two pointwise passes (H6) -------------------------------
// (A single kernel marching along z -- P, v of a 32 x 8 tile and its halo in a shared plane, chi~_z from a register
// window, 40 B/cell instead of 89 -- was built and measured slower: 0.42 ms against 0.31 ms at 256^3, one barrier
// per plane at 16 resident warps.)
// pass 1: chi~_x, chi~_y, chi~_z of every cell of [-2, n+1]^3 (one evaluation per cell and direction);
// pass 2: chi = min over the three directions and the -1, 0, +1 neighbours along each, cells [-1, n]^3.
__global__ void __launch_bounds__(128) chi_dir_kernel(Geom g, int k0, double gamma, const double *__restrict__ P,
                                                      const double *__restrict__ vx, const double *__restrict__ vy,
                                                      const double *__restrict__ vz, double *__restrict__ cx,
                                                      double *__restrict__ cy, double *__restrict__ cz)
{
    // threads are dealt out over the (nx+4) x (ny+4) cells of a plane in row-major order: no idle tail per row
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int w = g.nx + 4;
    if (t >= w * (g.ny + 4)) return;
    const int jj = t / w;
    const int i = t - jj * w - 2, j = jj - 2, k = (int)blockIdx.y + k0;
    const int c = g.at(i, j, k), sy = g.sy, sz = g.sz;
    const double P0 = P[c];
    cx[c] = flatten_coeff_1d(gamma, P[c - 2], P[c - 1], P0, P[c + 1], P[c + 2], vx[c - 1], vx[c + 1]);
    cy[c] = flatten_coeff_1d(gamma, P[c - 2 * sy], P[c - sy], P0, P[c + sy], P[c + 2 * sy], vy[c - sy], vy[c + sy]);
    cz[c] = flatten_coeff_1d(gamma, P[c - 2 * sz], P[c - sz], P0, P[c + sz], P[c + 2 * sz], vz[c - sz], vz[c + sz]);
}

__global__ void __launch_bounds__(128) chi_min_kernel(Geom g, int k0, const double *__restrict__ cx, const double *__restrict__ cy,
                                                      const double *__restrict__ cz, double *__restrict__ chi)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int w = g.nx + 2;
    if (t >= w * (g.ny + 2)) return;
    const int jj = t / w;
    const int i = t - jj * w - 1, j = jj - 1, k = (int)blockIdx.y + k0;
    const int c = g.at(i, j, k), sy = g.sy, sz = g.sz;
    double x = 1.0;      // same nesting as the oracle: min(1, min(lo, min(mid, hi))) per direction
    x = lesser(x, lesser(cx[c - 1], lesser(cx[c], cx[c + 1])));
    x = lesser(x, lesser(cy[c - sy], lesser(cy[c], cy[c + sy])));
    x = lesser(x, lesser(cz[c - sz], lesser(cz[c], cz[c + sz])));
    chi[c] = x;
}

// The same two passes with two x-adjacent cells per thread and 16-byte accesses, for even nx (every row of every
// field then starts 16-byte aligned at even x indices): half the load / store instructions, twice the bytes in
// flight per thread -- these kernels wait on memory latency, not on arithmetic.  Pairs start at i = -2.
__device__ __forceinline__ double2 ld2(const double *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }

__global__ void __launch_bounds__(128) chi_dir2_kernel(Geom g, int k0, double gamma, const double *__restrict__ P,
                                                       const double *__restrict__ vx, const double *__restrict__ vy,
                                                       const double *__restrict__ vz, double *__restrict__ cx,
                                                       double *__restrict__ cy, double *__restrict__ cz)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int w2 = (g.nx + 4) / 2;
    if (t >= w2 * (g.ny + 4)) return;
    const int jj = t / w2;
    const int i = 2 * (t - jj * w2) - 2, j = jj - 2, k = (int)blockIdx.y + k0;
    const int c = g.at(i, j, k), sy = g.sy, sz = g.sz;
    const double2 p0 = ld2(P + c);
    double2 r;
    {
        const double2 pa = ld2(P + c - 2), pc = ld2(P + c + 2), va = ld2(vx + c - 2), vb = ld2(vx + c), vc = ld2(vx + c + 2);
        r.x = flatten_coeff_1d(gamma, pa.x, pa.y, p0.x, p0.y, pc.x, va.y, vb.y);
        r.y = flatten_coeff_1d(gamma, pa.y, p0.x, p0.y, pc.x, pc.y, vb.x, vc.x);
        *reinterpret_cast<double2 *>(cx + c) = r;
    }
    {
        const double2 a = ld2(P + c - 2 * sy), b = ld2(P + c - sy), d = ld2(P + c + sy), e = ld2(P + c + 2 * sy);
        const double2 vm = ld2(vy + c - sy), vp = ld2(vy + c + sy);
        r.x = flatten_coeff_1d(gamma, a.x, b.x, p0.x, d.x, e.x, vm.x, vp.x);
        r.y = flatten_coeff_1d(gamma, a.y, b.y, p0.y, d.y, e.y, vm.y, vp.y);
        *reinterpret_cast<double2 *>(cy + c) = r;
    }
    {
        const double2 a = ld2(P + c - 2 * sz), b = ld2(P + c - sz), d = ld2(P + c + sz), e = ld2(P + c + 2 * sz);
        const double2 vm = ld2(vz + c - sz), vp = ld2(vz + c + sz);
        r.x = flatten_coeff_1d(gamma, a.x, b.x, p0.x, d.x, e.x, vm.x, vp.x);
        r.y = flatten_coeff_1d(gamma, a.y, b.y, p0.y, d.y, e.y, vm.y, vp.y);
        *reinterpret_cast<double2 *>(cz + c) = r;
    }
}

__global__ void __launch_bounds__(128) chi_min2_kernel(Geom g, int k0, const double *__restrict__ cx, const double *__restrict__ cy,
                                                       const double *__restrict__ cz, double *__restrict__ chi)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int w2 = (g.nx + 4) / 2;
    if (t >= w2 * (g.ny + 2)) return;
    const int jj = t / w2;
    const int i = 2 * (t - jj * w2) - 2, j = jj - 1, k = (int)blockIdx.y + k0;
    const int c = g.at(i, j, k), sy = g.sy, sz = g.sz;
    const double2 xm = ld2(cx + c);
    const double xl = __ldg(cx + c - 1), xr = __ldg(cx + c + 2);
    const double2 ya = ld2(cy + c - sy), yb = ld2(cy + c), yc = ld2(cy + c + sy);
    const double2 za = ld2(cz + c - sz), zb = ld2(cz + c), zc = ld2(cz + c + sz);
    double2 r;       // same nesting as the oracle: min(1, min(lo, min(mid, hi))) per direction
    r.x = lesser(1.0, lesser(xl, lesser(xm.x, xm.y)));
    r.x = lesser(r.x, lesser(ya.x, lesser(yb.x, yc.x)));
    r.x = lesser(r.x, lesser(za.x, lesser(zb.x, zc.x)));
    r.y = lesser(1.0, lesser(xm.x, lesser(xm.y, xr)));
    r.y = lesser(r.y, lesser(ya.y, lesser(yb.y, yc.y)));
    r.y = lesser(r.y, lesser(za.y, lesser(zb.y, zc.y)));
    if (i >= 0 && i + 1 < g.nx) *reinterpret_cast<double2 *>(chi + c) = r;      // chi lives on [-1, nx]: the two end pairs
    else if (i < 0) chi[c + 1] = r.y;                                             // (-2, -1) and (nx, nx+1) store one cell
    else chi[c] = r.x;
}

// ---- flattening coefficient in ONE pass, no chi~ arrays ------------------------------------------------------
// One thread per (i, j) column of [-1, nx] x [-1, ny] marching along z over a chunk of planes.  chi~_z of the three
// planes k-1, k, k+1 comes from a register window of the column's own P and v_z (each evaluated once); chi~_x and
// chi~_y of the three neighbours along x and y are evaluated in place from P and v_x / v_y of the cell's row and
// of the rows j +- 1..3 -- those loads are L1 / L2 hits on lines the neighbouring lanes and warps fetch anyway.
// No shared memory, no barrier (the rejected one-kernel variant of round 2, paid one barrier
// per plane).  HBM traffic: P, v once and chi once, 44 B/cell measured instead of the two passes' 89.
// The value is the two-pass result bit for bit: the same flatten_coeff_1d on the same operands, and the same
// nesting of the minimum.
// 32 x 4 tiles at 5 CTAs per SM (96 registers, no spill): 0.250 ms at 256^3; 32 x 8 at 3 (80 registers, 76 B of
// spills) 0.275 ms, 32 x 2 at 10: 0.253 ms; grouping the loads by direction instead of issuing all 24 first: 0.35 ms.
constexpr int CHI_TX = 32, CHI_TY = 4, CHI_MINB = 5;

__device__ __forceinline__ void prefetch_l2(const double *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__global__ void __launch_bounds__(CHI_TX * CHI_TY, CHI_MINB) chi_march_kernel(Geom g, int m0, int m1, int len, double gamma,
                                                                    const double *__restrict__ P, const double *__restrict__ vx,
                                                                    const double *__restrict__ vy, const double *__restrict__ vz,
                                                                    double *__restrict__ chi)
{
    const int i = (int)blockIdx.x * CHI_TX + (int)threadIdx.x - 1;
    const int j = (int)blockIdx.y * CHI_TY + (int)threadIdx.y - 1;
    if (i > g.nx || j > g.ny) return;
    const int ka = m0 + (int)blockIdx.z * len, kb = min(ka + len, m1);
    const int sy = g.sy, sz = g.sz;
    int c = g.at(i, j, ka);
    // z window of the column: P(k-1..k+2), v_z(k), v_z(k+1); chi~_z(k-1), chi~_z(k)
    double pa, pb, pc, pd, wa, wb, czm, cz0;
    {
        const double q3 = __ldg(P + c - 3 * sz), q2 = __ldg(P + c - 2 * sz);
        pa = __ldg(P + c - sz); pb = __ldg(P + c); pc = __ldg(P + c + sz); pd = __ldg(P + c + 2 * sz);
        const double u2 = __ldg(vz + c - 2 * sz), u1 = __ldg(vz + c - sz);
        wa = __ldg(vz + c); wb = __ldg(vz + c + sz);
        czm = flatten_coeff_1d(gamma, q3, q2, pa, pb, pc, u2, wa);
        cz0 = flatten_coeff_1d(gamma, q2, pa, pb, pc, pd, u1, wb);
    }
    for (int k = ka; k < kb; ++k, c += sz) {
        // all 24 loads of the step are issued before the first evaluation: the kernel lives on memory-level parallelism
        const double pe = __ldg(P + c + 3 * sz), wc = __ldg(vz + c + 2 * sz);
        // the four lines of this column's data that the step two planes on touches for the first time, asked into the
        // L2 now (no register, no dependency): its loads then miss the L1 only as far as the L2 (0.254 -> 0.235 ms)
        if (k + 2 < kb) {
            const int cp = c + 2 * sz;
            prefetch_l2(P + cp + 3 * sz); prefetch_l2(vz + cp + 2 * sz); prefetch_l2(vx + cp); prefetch_l2(vy + cp);
        }
        const double xm3 = __ldg(P + c - 3), xm2 = __ldg(P + c - 2), xm1 = __ldg(P + c - 1);
        const double xp1 = __ldg(P + c + 1), xp2 = __ldg(P + c + 2), xp3 = __ldg(P + c + 3);
        const double um2 = __ldg(vx + c - 2), um1 = __ldg(vx + c - 1), u0 = __ldg(vx + c), up1 = __ldg(vx + c + 1), up2 = __ldg(vx + c + 2);
        const double ym3 = __ldg(P + c - 3 * sy), ym2 = __ldg(P + c - 2 * sy), ym1 = __ldg(P + c - sy);
        const double yp1 = __ldg(P + c + sy), yp2 = __ldg(P + c + 2 * sy), yp3 = __ldg(P + c + 3 * sy);
        const double vm2 = __ldg(vy + c - 2 * sy), vm1 = __ldg(vy + c - sy), v0 = __ldg(vy + c), vp1 = __ldg(vy + c + sy), vp2 = __ldg(vy + c + 2 * sy);
        const double czp = flatten_coeff_1d(gamma, pa, pb, pc, pd, pe, wa, wc);       // chi~_z(k+1)
        const double cxm = flatten_coeff_1d(gamma, xm3, xm2, xm1, pb, xp1, um2, u0);
        const double cx0 = flatten_coeff_1d(gamma, xm2, xm1, pb, xp1, xp2, um1, up1);
        const double cxp = flatten_coeff_1d(gamma, xm1, pb, xp1, xp2, xp3, u0, up2);
        const double cym = flatten_coeff_1d(gamma, ym3, ym2, ym1, pb, yp1, vm2, v0);
        const double cy0 = flatten_coeff_1d(gamma, ym2, ym1, pb, yp1, yp2, vm1, vp1);
        const double cyp = flatten_coeff_1d(gamma, ym1, pb, yp1, yp2, yp3, v0, vp2);
        double x = 1.0;      // same nesting as the oracle: min(1, min(lo, min(mid, hi))) per direction
        x = lesser(x, lesser(cxm, lesser(cx0, cxp)));
        x = lesser(x, lesser(cym, lesser(cy0, cyp)));
        x = lesser(x, lesser(czm, lesser(cz0, czp)));
        chi[c] = x;
        pa = pb; pb = pc; pc = pd; pd = pe; wa = wb; wb = wc; czm = cz0; cz0 = czp;
    }
}

// chunk length of the flattening march: whole waves of CTAs, long chunks (a chunk's prologue costs about half a step)
static int chi_len(int nplanes, int ctas_xy, int per_sm)
{
    const double per_wave = 148.0 * per_sm;
    int best = nplanes < 1 ? 1 : nplanes;
    double best_cost = 1e30;
    for (int len = 4; len <= 96; ++len) {
        if (len > nplanes) break;
        const int chunks = (nplanes + len - 1) / len;
        const double waves = (double)ctas_xy * chunks / per_wave;
        const double waves_up = (double)(long long)(waves + 0.999999);
        const double cost = (1.0 + 0.5 / len) * (waves_up / waves) * ((double)chunks * len / nplanes);
        if (cost < best_cost - 1e-12) { best_cost = cost; best = len; }
    }
    return best;
}

// chi~_d for the planes [d0, d1) (within [-2, nz+2)), then chi for the planes [m0, m1) (within [-1, nz+1)); an empty
// range launches nothing.  The whole box is (-2, nz+2, -1, nz+1); a decomposed box does the planes that need no
// neighbour data first.
int launch_chi(const Geom &g, double gamma, CHydro5 W, double *cx, double *cy, double *cz, double *chi, int d0, int d1,
               int m0, int m1, int path, cudaStream_t st)
{
    int n = 0;
    // path 0: by box size.  Boxes whose three chi~ arrays stay in the 126 MB L2 between the two passes (up to ~160^3)
    // are faster with the two passes (128^3: 0.054 against 0.071 ms); beyond that the single pass wins (192^3: 0.118
    // against 0.134 ms, 256^3: 0.250 against 0.290 ms, 320^3: 0.467 against 0.543 ms) and moves half the bytes.
    if (path == 2 || (path == 0 && 3.0 * 8.0 * (double)g.ntot > 100.0e6)) {
        if (m1 > m0) {
            const int bx = (g.nx + 2 + CHI_TX - 1) / CHI_TX, by = (g.ny + 2 + CHI_TY - 1) / CHI_TY;
            const int len = chi_len(m1 - m0, bx * by, CHI_MINB);
            dim3 grid(bx, by, (m1 - m0 + len - 1) / len);
            chi_march_kernel<<<grid, dim3(CHI_TX, CHI_TY), 0, st>>>(g, m0, m1, len, gamma, W.E, W.mx, W.my, W.mz, chi);
            ++n;
        }
        return n;
    }
    const bool vec = (g.nx & 1) == 0;
    if (d1 > d0) {
        if (vec) {
            dim3 g1(((g.nx + 4) / 2 * (g.ny + 4) + 127) / 128, d1 - d0);
            chi_dir2_kernel<<<g1, 128, 0, st>>>(g, d0, gamma, W.E, W.mx, W.my, W.mz, cx, cy, cz);
        } else {
            dim3 g1(((g.nx + 4) * (g.ny + 4) + 127) / 128, d1 - d0);
            chi_dir_kernel<<<g1, 128, 0, st>>>(g, d0, gamma, W.E, W.mx, W.my, W.mz, cx, cy, cz);
        }
        ++n;
    }
    if (m1 > m0) {
        if (vec) {
            dim3 g2(((g.nx + 4) / 2 * (g.ny + 2) + 127) / 128, m1 - m0);
            chi_min2_kernel<<<g2, 128, 0, st>>>(g, m0, cx, cy, cz, chi);
        } else {
            dim3 g2(((g.nx + 2) * (g.ny + 2) + 127) / 128, m1 - m0);
            chi_min_kernel<<<g2, 128, 0, st>>>(g, m0, cx, cy, cz, chi);
        }
        ++n;
    }
    return n;
}

// Marching chunk length.  A chunk of `len` cells costs len + ~3 cells of work (window prologue, two extra
// reconstructions), so long chunks are cheaper per cell; but the launch must still fill the GPU with whole waves of
// CTAs: with `ctas_per_sm` resident CTAs a grid of 9.2 waves runs for 10.  Among the lengths 16..64 take the one with
// the least (work per cell) x (rounded-up waves / waves); boxes too small for ~8 waves of warps use short chunks.
static int sweep_len(int n_m, int ctas_xy, int ctas_per_sm)
{
    const double per_wave = 148.0 * ctas_per_sm;
    if ((double)ctas_xy * ((n_m + 31) / 32) < 2.0 * per_wave) {      // small box: more, shorter chunks
        int len = 32;
        while (len > 8 && (double)ctas_xy * ((n_m + len - 1) / len) < 2.0 * per_wave) len /= 2;
        return len > n_m ? (n_m < 1 ? 1 : n_m) : len;
    }
    int best = 32;
    double best_cost = 1e30;
    for (int len = 16; len <= 64 && len <= n_m; ++len) {
        const int chunks = (n_m + len - 1) / len;
        const double waves = (double)ctas_xy * chunks / per_wave;
        const double waves_up = (double)(long long)(waves + 0.999999);
        // the last chunk of a column may be short: the longest chunk sets a CTA's time
        const double cost = (1.0 + 3.0 / len) * (waves_up / waves) * ((double)chunks * len / n_m);
        if (cost < best_cost - 1e-12) { best_cost = cost; best = len; }
    }
    return best;
}

template <class PH>
static int launch_sweeps(const PH &ph, const Geom &g, double dtdx, int stage, FieldsRW<PH::NV> D, FieldsRO<PH::NV> U,
                         FieldsRO<PH::NV> U0, FieldsRW<PH::NV> out, FieldsRW<PH::NV> pout, Counters *ctr,
                         StateCache *cache, cudaStream_t st, int which, const double *dtdx_dev, int k0, int k1)
{
    const RkArgs rk{dtdx, stage, dtdx_dev};
    int n = 0;
    if ((which & 1) && k1 > k0) {        // x sweep of the planes [k0, k1)
        constexpr int rows = SW_XYWARPS * SW_XNROW;
        dim3 grid((g.nx + SW_XW - 1) / SW_XW, (g.ny + rows - 1) / rows, k1 - k0);
        sweep_x_kernel<PH><<<grid, SW_NT, 0, st>>>(ph, g, k0, D, ctr);
        ++n;
    }
    // marching sweeps: CTA width 128, 64 or 32 columns -- the one that pads the row length least, the wider on ties
    // (192 cells: three CTAs of 64 instead of a full and a half-empty CTA of 128: hydro step at 192^3 2.73 -> 3.26 G/s;
    // 64^3: 1.03 -> 1.26 G/s; 256^3 unchanged)
    int nt = SW_NT;
    for (int cand = SW_NT / 2; cand >= 32; cand /= 2)
        if ((g.nx + cand - 1) / cand * cand < (g.nx + nt - 1) / nt * nt) nt = cand;
    const int bx = (g.nx + nt - 1) / nt;
    auto march = [&](auto dir, auto width) {
        constexpr int DIR = decltype(dir)::value, NT = decltype(width)::value;
        constexpr int per_sm = (DIR == 2 ? PH::Z_MINB : PH::Y_MINB) * (SW_NT / NT);
        if (DIR == 1) {                  // y sweep of the planes [k0, k1)
            const int len = sweep_len(g.ny, bx * (k1 - k0), per_sm);
            dim3 grid(bx, k1 - k0, (g.ny + len - 1) / len);
            sweep_march_kernel<PH, DIR, NT><<<grid, NT, 0, st>>>(ph, g, len, k0, D, rk, U, U0, out, pout, ctr, cache);
        } else {                         // z sweep: always the whole box
            const int len = sweep_len(g.nz, bx * g.ny, per_sm);
            dim3 grid(bx, g.ny, (g.nz + len - 1) / len);
            sweep_march_kernel<PH, DIR, NT><<<grid, NT, 0, st>>>(ph, g, len, 0, D, rk, U, U0, out, pout, ctr, cache);
        }
    };
    auto march_nt = [&](auto dir) {
        if (nt == 128) march(dir, std::integral_constant<int, 128>());
        else if (nt == 64) march(dir, std::integral_constant<int, 64>());
        else march(dir, std::integral_constant<int, 32>());
    };
    if ((which & 2) && k1 > k0) { march_nt(std::integral_constant<int, 1>()); ++n; }
    if (which & 4) { march_nt(std::integral_constant<int, 2>()); ++n; }
    return n;
}

// `which`: bit 0 = x sweep (D = dF_x), bit 1 = y sweep (D += dF_y), bit 2 = z sweep (RK stage update); x and y
// sweeps cover the planes [k0, k1)
int launch_hydro_sweeps(const Geom &g, double gamma, unsigned scheme, double dtdx, int stage, CHydro5 W,
                        const double *chi, Hydro5 D, CHydro5 U, CHydro5 U0, Hydro5 out, Hydro5 Wout, Counters *ctr,
                        StateCache *cache, cudaStream_t st, int which, const double *dtdx_dev, int k0, int k1)
{
    FieldsRW<5> d{{D.rho, D.mx, D.my, D.mz, D.E}}, o{{out.rho, out.mx, out.my, out.mz, out.E}};
    FieldsRO<5> u{{U.rho, U.mx, U.my, U.mz, U.E}}, u0{{U0.rho, U0.mx, U0.my, U0.mz, U0.E}};
    FieldsRW<5> wo{{Wout.rho, Wout.mx, Wout.my, Wout.mz, Wout.E}};
    auto go = [&](auto ph) {
        ph.w[0] = W.rho; ph.w[1] = W.mx; ph.w[2] = W.my; ph.w[3] = W.mz; ph.w[4] = W.E;
        ph.chi = chi; ph.gamma = gamma;
        return launch_sweeps(ph, g, dtdx, stage, d, u, u0, o, wo, ctr, cache, st, which, dtdx_dev, k0, k1);
    };
    return (scheme & QK_FLAG_PLM) ? go(HydroPhT<1>()) : go(HydroPhT<0>());
}

int launch_rad_sweeps(const Geom &g, const PhysConsts &pc, double dtdx, int stage, CRad4p S, const double *rho,
                      const double *kappaR, Rad4p D, CRad4p R, CRad4p R0, Rad4p out, Rad4p Sout, Counters *ctr,
                      cudaStream_t st, int which, const double *dtdx_dev, int k0, int k1)
{
    FieldsRW<4> d{{D.E, D.Fx, D.Fy, D.Fz}}, o{{out.E, out.Fx, out.Fy, out.Fz}};
    FieldsRO<4> u{{R.E, R.Fx, R.Fy, R.Fz}}, u0{{R0.E, R0.Fx, R0.Fy, R0.Fz}};
    FieldsRW<4> so{{Sout.E, Sout.Fx, Sout.Fy, Sout.Fz}};
    auto go = [&](auto ph) {
        ph.s[0] = S.E; ph.s[1] = S.Fx; ph.s[2] = S.Fy; ph.s[3] = S.Fz;
        ph.rho = rho; ph.kR = kappaR;
        ph.c = pc.c; ph.c_hat = pc.c_hat; ph.dx = pc.dx; ph.tau_corr = (pc.flags & QK_FLAG_TAU_CORR) ? 1 : 0;
        return launch_sweeps(ph, g, dtdx, stage, d, u, u0, o, so, ctr, nullptr, st, which, dtdx_dev, k0, k1);
    };
    const bool plm = (pc.flags & QK_FLAG_PLM) != 0;
    const int cl = (pc.flags & QK_FLAG_EDDINGTON) ? 1 : ((pc.flags & QK_FLAG_MINERBO) ? 2 : 0);
    if (plm) return cl == 1 ? go(RadPhT<1, 1>()) : (cl == 2 ? go(RadPhT<1, 2>()) : go(RadPhT<1, 0>()));
    return cl == 1 ? go(RadPhT<0, 1>()) : (cl == 2 ? go(RadPhT<0, 2>()) : go(RadPhT<0, 0>()));
}

// ---- reconstruction variables of a whole field set (all cells, ghosts included): only when no kernel has left
// them next to the state -- after qk_set_state / qk_set_raw, and every stage with Dirichlet faces, whose ghost
// cells hold caller-supplied conserved values ---------------------------------------------------------------
__global__ void __launch_bounds__(256) prim_kernel(Geom g, double gamma, CHydro5 U, Hydro5 W, Counters *ctr)
{
    int bad = 0;
    for (int cidx = blockIdx.x * blockDim.x + threadIdx.x; cidx < g.ntot; cidx += gridDim.x * blockDim.x) {
        const Prim w = cons_to_prim(gamma, U.rho[cidx], U.mx[cidx], U.my[cidx], U.mz[cidx], U.E[cidx]);
        W.rho[cidx] = w.rho; W.mx[cidx] = w.vx; W.my[cidx] = w.vy; W.mz[cidx] = w.vz; W.E[cidx] = w.P;
        if (!(w.rho > 0.0) || !(w.P > 0.0)) {   // only interior cells count (their ghost images would double count)
            const int kk = cidx / g.sz, rem = cidx - kk * g.sz, jj = rem / g.sy, ii = rem - jj * g.sy;
            if (ii >= NG && ii < NG + g.nx && jj >= NG && jj < NG + g.ny && kk >= NG && kk < NG + g.nz) ++bad;
        }
    }
    if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
}

__global__ void __launch_bounds__(256) rad_prim_kernel(Geom g, double c, CRad4p R, Rad4p S, Counters *ctr)
{
    int bad = 0;
    for (int cidx = blockIdx.x * blockDim.x + threadIdx.x; cidx < g.ntot; cidx += gridDim.x * blockDim.x) {
        const double E = R.E[cidx], cE = c * E;
        S.E[cidx] = E;
        S.Fx[cidx] = R.Fx[cidx] / cE;
        S.Fy[cidx] = R.Fy[cidx] / cE;
        S.Fz[cidx] = R.Fz[cidx] / cE;
        if (!(E > 0.0)) {
            const int kk = cidx / g.sz, rem = cidx - kk * g.sz, jj = rem / g.sy, ii = rem - jj * g.sy;
            if (ii >= NG && ii < NG + g.nx && jj >= NG && jj < NG + g.ny && kk >= NG && kk < NG + g.nz) ++bad;
        }
    }
    if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
}

int launch_prim(const Geom &g, double gamma, CHydro5 U, Hydro5 W, Counters *ctr, cudaStream_t st)
{
    int blocks = (g.ntot + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    prim_kernel<<<blocks, 256, 0, st>>>(g, gamma, U, W, ctr);
    return 1;
}

int launch_rad_prim(const Geom &g, double c, CRad4p R, Rad4p S, Counters *ctr, cudaStream_t st)
{
    int blocks = (g.ntot + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    rad_prim_kernel<<<blocks, 256, 0, st>>>(g, c, R, S, ctr);
    return 1;
}

}  // namespace qk
