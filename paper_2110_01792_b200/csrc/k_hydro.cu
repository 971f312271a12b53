// k_hydro.cu -- fused hydro stage: two kernels per SSP-RK2 stage.
//
//   flatten_march_kernel : conserved state -> multidimensional shock-flattening coefficient chi
//                          (H6) for the cells -1..n of every direction.  8 B/cell out.
//   hydro_stage_kernel   : conserved state + chi -> primitives, PPM face states in
//                          x, y, z with the paper's limiters (eq 22), flattening,
//                          HLLC fluxes, unsplit divergence ((dFx+dFy)+dFz,
//                          PAPER.md:408) and the RK stage combination, in one pass.
//
// Both march TX x TY tiles along z (k_stage_common.cuh).  Primitives are recomputed from the
// conserved state where needed (3 divisions per cell) instead of being stored: the stage is
// bound by the fp64 pipe, not by HBM, and face states / fluxes never
// leave the SM.  The chi pre-pass exists because chi of the one cell beyond a tile edge depends
// on a radius-4 neighbourhood across the edge; computing it once per cell costs 48 B/cell of
// traffic and saves recomputing those neighbourhoods in every tile.
#include "k_stage_common.cuh"
#include "qk_math.cuh"

namespace qk {

struct Cons5 { double r, mx, my, mz, e; };

__device__ __forceinline__ Cons5 load_cons(const CHydro5 &U, int cidx)
{
    Cons5 u;
    u.r = U.rho[cidx]; u.mx = U.mx[cidx]; u.my = U.my[cidx]; u.mz = U.mz[cidx]; u.e = U.E[cidx];
    return u;
}

__device__ __forceinline__ Cons5 benign_cons() { return Cons5{1.0, 0.0, 0.0, 0.0, 1.0}; }

// ---------------------------------------------------------------------------------------------
// chi pre-pass
// ---------------------------------------------------------------------------------------------
struct FlattenSmem {
    double ringP[RING][TY][TX];             // pressure, planes k-1..k+3 of the own columns
    double ringV[RING][TY][TX];             // v_z
    double P[TY + 2 * HALO][TX + 2 * HALO];  // plane k with star halo
    double vx[TY + 2 * HALO][TX + 2 * HALO];
    double vy[TY + 2 * HALO][TX + 2 * HALO];
    double cx[TY][TX + 2];                  // chi~_x of cells -1..TX of every row
    double cy[TY + 2][TX];                  // chi~_y of cells -1..TY of every column
};

// Tiles cover the cells -1..n in x and y; the march covers planes -1..nz.
__global__ void __launch_bounds__(NT) flatten_march_kernel(Geom g, double gamma, CHydro5 U, double *__restrict__ chi,
                                                           int lz)
{
    __shared__ FlattenSmem s;
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = -1 + (int)blockIdx.x * TX, j0 = -1 + (int)blockIdx.y * TY;
    const int k0 = -1 + (int)blockIdx.z * lz;
    const int k1 = min(k0 + lz, g.nz + 1);
    const int gi = i0 + tx, gj = j0 + ty;
    const bool own_ok = in_array(g, gi, gj);
    const bool writes = gi <= g.nx && gj <= g.ny;

    int hx = 0, hy = 0;
    const bool is_halo = t < N_HALO;
    if (is_halo) halo_cell(t, hx, hy);
    const bool halo_ok = is_halo && in_array(g, i0 + hx, j0 + hy);

    // prologue: planes k0-3..k0 of the own columns
    for (int p = k0 - 3; p <= k0; ++p) {
        const Cons5 u = own_ok ? load_cons(U, g.at(gi, gj, p)) : benign_cons();
        const Prim w = cons_to_prim(gamma, u.r, u.mx, u.my, u.mz, u.e);
        s.ringP[ring_slot(p)][ty][tx] = w.P;
        s.ringV[ring_slot(p)][ty][tx] = w.vz;
    }
    Cons5 pend_own = own_ok ? load_cons(U, g.at(gi, gj, k0 + 1)) : benign_cons();
    Cons5 pend_halo = benign_cons();
    double cz_prev = 1.0, cz_cur = 1.0;    // chi~_z of cells k-1 and k

    for (int k = k0 - 2; k < k1; ++k) {
        // ---- commit the loads issued during the previous step --------------------------------
        {
            const Prim w = cons_to_prim(gamma, pend_own.r, pend_own.mx, pend_own.my, pend_own.mz, pend_own.e);
            s.ringP[ring_slot(k + 3)][ty][tx] = w.P;
            s.ringV[ring_slot(k + 3)][ty][tx] = w.vz;
        }
        if (k >= k0) {
            if (is_halo) {
                const Prim w = cons_to_prim(gamma, pend_halo.r, pend_halo.mx, pend_halo.my, pend_halo.mz, pend_halo.e);
                s.P[hy + HALO][hx + HALO] = w.P;
                s.vx[hy + HALO][hx + HALO] = w.vx;
                s.vy[hy + HALO][hx + HALO] = w.vy;
            }
        }
        // the centre of plane k needs v_x, v_y too: recompute from the conserved state (prefetched
        // below as pend_ctr) -- see the load block
        __syncthreads();   // S1: ring + halo visible
        // ---- issue the loads of the next step -------------------------------------------------
        if (k + 1 < k1) {
            pend_own = own_ok ? load_cons(U, g.at(gi, gj, k + 4)) : benign_cons();
            if (k + 1 >= k0) pend_halo = halo_ok ? load_cons(U, g.at(i0 + hx, j0 + hy, k + 1)) : benign_cons();
        }
        // chi~_z of cell k+1 from the ring (planes k-1..k+3)
        const double cz_next = flatten_coeff_1d(gamma, s.ringP[ring_slot(k - 1)][ty][tx], s.ringP[ring_slot(k)][ty][tx],
                                                s.ringP[ring_slot(k + 1)][ty][tx], s.ringP[ring_slot(k + 2)][ty][tx],
                                                s.ringP[ring_slot(k + 3)][ty][tx], s.ringV[ring_slot(k)][ty][tx],
                                                s.ringV[ring_slot(k + 2)][ty][tx]);
        if (k >= k0) {
            // centre of plane k: P from the ring, v_x and v_y from the conserved state
            {
                const Cons5 u = own_ok ? load_cons(U, g.at(gi, gj, k)) : benign_cons();
                s.P[ty + HALO][tx + HALO] = s.ringP[ring_slot(k)][ty][tx];
                s.vx[ty + HALO][tx + HALO] = u.mx / u.r;
                s.vy[ty + HALO][tx + HALO] = u.my / u.r;
            }
            __syncthreads();   // S1b: plane k complete
            // chi~_x, chi~_y of the own cell and of the edge cells
            {
                const int y = ty + HALO, x = tx + HALO;
                s.cx[ty][tx + 1] = flatten_coeff_1d(gamma, s.P[y][x - 2], s.P[y][x - 1], s.P[y][x], s.P[y][x + 1],
                                                    s.P[y][x + 2], s.vx[y][x - 1], s.vx[y][x + 1]);
                s.cy[ty + 1][tx] = flatten_coeff_1d(gamma, s.P[y - 2][x], s.P[y - 1][x], s.P[y][x], s.P[y + 1][x],
                                                    s.P[y + 2][x], s.vy[y - 1][x], s.vy[y + 1][x]);
            }
            if (t < N_EDGE) {
                int lx, ly; bool along_x, high;
                edge_cell(t, lx, ly, along_x, high);
                const int y = ly + HALO, x = lx + HALO;
                if (along_x)
                    s.cx[ly][high ? TX + 1 : 0] = flatten_coeff_1d(gamma, s.P[y][x - 2], s.P[y][x - 1], s.P[y][x],
                                                                   s.P[y][x + 1], s.P[y][x + 2], s.vx[y][x - 1],
                                                                   s.vx[y][x + 1]);
                else
                    s.cy[high ? TY + 1 : 0][lx] = flatten_coeff_1d(gamma, s.P[y - 2][x], s.P[y - 1][x], s.P[y][x],
                                                                   s.P[y + 1][x], s.P[y + 2][x], s.vy[y - 1][x],
                                                                   s.vy[y + 1][x]);
            }
            __syncthreads();   // S2
            if (writes) {
                double x = 1.0;
                x = lesser(x, lesser(s.cx[ty][tx], lesser(s.cx[ty][tx + 1], s.cx[ty][tx + 2])));
                x = lesser(x, lesser(s.cy[ty][tx], lesser(s.cy[ty + 1][tx], s.cy[ty + 2][tx])));
                x = lesser(x, lesser(cz_prev, lesser(cz_cur, cz_next)));
                chi[g.at(gi, gj, k)] = x;
            }
        }
        cz_prev = cz_cur;
        cz_cur = cz_next;
        __syncthreads();   // S3: plane arrays and ring slot k-1 free for the next step
    }
}

// ---------------------------------------------------------------------------------------------
// fused stage
// ---------------------------------------------------------------------------------------------
struct HydroSmem {
    double ring[RING][5][TY][TX];                   // (rho, vx, vy, vz, P), planes k-1..k+3
    union {
        double W[5][TY + 2 * HALO][TX + 2 * HALO];  // plane k with star halo (phase P)
        struct {
            double fx[5][TY][TX];                   // x flux at faces 1..TX   (phases F, U)
            double fy[5][TY][TX];                   // y flux at faces 1..TY
        } fl;
    };
    double hiX[5][TY][TX + 1];                      // high-x face state of cells -1..TX-1
    double hiY[5][TY + 1][TX];                      // high-y face state of cells -1..TY-1
    double loXe[5][TY];                             // low-x face state of cell TX
    double loYe[5][TX];                             // low-y face state of cell TY
};

__global__ void __launch_bounds__(NT, 2) hydro_stage_kernel(Geom g, double gamma, double dtdx, int stage, CHydro5 U,
                                                            CHydro5 U0, const double *__restrict__ chi, Hydro5 out,
                                                            int lz, Counters *ctr)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    HydroSmem &s = *reinterpret_cast<HydroSmem *>(smem_raw);
    const int tx = threadIdx.x, ty = threadIdx.y, t = ty * TX + tx;
    const int i0 = (int)blockIdx.x * TX, j0 = (int)blockIdx.y * TY;
    const int k0 = (int)blockIdx.z * lz;
    const int k1 = min(k0 + lz, g.nz);
    const int gi = i0 + tx, gj = j0 + ty;
    const bool own_ok = in_array(g, gi, gj);
    const bool active = gi < g.nx && gj < g.ny;
    const bool chi_ok = gi <= g.nx && gj <= g.ny;     // chi is defined on -1..n

    int hx = 0, hy = 0;
    const bool is_halo = t < N_HALO;
    if (is_halo) halo_cell(t, hx, hy);
    const bool halo_ok = is_halo && in_array(g, i0 + hx, j0 + hy);

    int ex = 0, ey = 0; bool e_along_x = false, e_high = false;
    const bool is_edge = t < N_EDGE;
    if (is_edge) edge_cell(t, ex, ey, e_along_x, e_high);
    const bool edge_chi_ok = is_edge && i0 + ex <= g.nx && j0 + ey <= g.ny;

    int bad = 0;
    // prologue: planes k0-3..k0 of the own columns
    for (int p = k0 - 3; p <= k0; ++p) {
        const Cons5 u = own_ok ? load_cons(U, g.at(gi, gj, p)) : benign_cons();
        const Prim w = cons_to_prim(gamma, u.r, u.mx, u.my, u.mz, u.e);
        const int sl = ring_slot(p);
        s.ring[sl][0][ty][tx] = w.rho; s.ring[sl][1][ty][tx] = w.vx; s.ring[sl][2][ty][tx] = w.vy;
        s.ring[sl][3][ty][tx] = w.vz; s.ring[sl][4][ty][tx] = w.P;
        if (p == k0 && active && (!(w.rho > 0.0) || !(w.P > 0.0))) ++bad;
    }
    Cons5 pend_own = own_ok ? load_cons(U, g.at(gi, gj, k0 + 1)) : benign_cons();
    Cons5 pend_halo = benign_cons();
    double chi_zn = chi_ok ? chi[g.at(gi, gj, k0 - 1)] : 1.0;   // chi of the cell whose z states come next
    double chi_c = 1.0;                                         // chi of the own cell in plane k
    double chi_e = 1.0;                                         // chi of this thread's edge cell in plane k
    double hiZ[5], FzLo[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { hiZ[v] = 0.0; FzLo[v] = 0.0; }

    for (int k = k0 - 2; k < k1; ++k) {
        // ---- commit the loads issued during the previous step --------------------------------
        {
            const Prim w = cons_to_prim(gamma, pend_own.r, pend_own.mx, pend_own.my, pend_own.mz, pend_own.e);
            const int sl = ring_slot(k + 3);
            s.ring[sl][0][ty][tx] = w.rho; s.ring[sl][1][ty][tx] = w.vx; s.ring[sl][2][ty][tx] = w.vy;
            s.ring[sl][3][ty][tx] = w.vz; s.ring[sl][4][ty][tx] = w.P;
            if (active && k + 3 > k0 && k + 3 < k1 && (!(w.rho > 0.0) || !(w.P > 0.0))) ++bad;
        }
        if (k >= k0) {
            if (is_halo) {
                const Prim w = cons_to_prim(gamma, pend_halo.r, pend_halo.mx, pend_halo.my, pend_halo.mz, pend_halo.e);
                s.W[0][hy + HALO][hx + HALO] = w.rho; s.W[1][hy + HALO][hx + HALO] = w.vx;
                s.W[2][hy + HALO][hx + HALO] = w.vy; s.W[3][hy + HALO][hx + HALO] = w.vz;
                s.W[4][hy + HALO][hx + HALO] = w.P;
            }
            const int sl = ring_slot(k);
#pragma unroll
            for (int v = 0; v < 5; ++v) s.W[v][ty + HALO][tx + HALO] = s.ring[sl][v][ty][tx];
        }
        __syncthreads();   // S1
        // ---- issue the loads of the next step -------------------------------------------------
        const double chi_z = chi_zn;          // chi of cell k+1 (own column)
        double chi_e_next = 1.0;
        if (k + 1 < k1) {
            pend_own = own_ok ? load_cons(U, g.at(gi, gj, k + 4)) : benign_cons();
            chi_zn = chi_ok ? chi[g.at(gi, gj, k + 2)] : 1.0;
            if (k + 1 >= k0) {
                pend_halo = halo_ok ? load_cons(U, g.at(i0 + hx, j0 + hy, k + 1)) : benign_cons();
                chi_e_next = edge_chi_ok ? chi[g.at(i0 + ex, j0 + ey, k + 1)] : 1.0;
            }
        }
        // ---- phase P: PPM face states ---------------------------------------------------------
        double loZn[5], hiZn[5];
        {
            const int s0 = ring_slot(k - 1), s1 = ring_slot(k), s2 = ring_slot(k + 1), s3 = ring_slot(k + 2),
                      s4 = ring_slot(k + 3);
            const int sl[5] = {s0, s1, s2, s3, s4};
            ppm_cell([&](int v, int m) { return s.ring[sl[m]][v][ty][tx]; }, chi_z, loZn, hiZn);
        }
        double loX[5], loY[5];
        if (k >= k0) {
            double hi[5];
            const int y = ty + HALO, x = tx + HALO;
            ppm_cell([&](int v, int m) { return s.W[v][y][x + m - 2]; }, chi_c, loX, hi);
#pragma unroll
            for (int v = 0; v < 5; ++v) s.hiX[v][ty][tx + 1] = hi[v];
            ppm_cell([&](int v, int m) { return s.W[v][y + m - 2][x]; }, chi_c, loY, hi);
#pragma unroll
            for (int v = 0; v < 5; ++v) s.hiY[v][ty + 1][tx] = hi[v];
            if (is_edge) {
                double lo[5];
                const int yy = ey + HALO, xx = ex + HALO;
                if (e_along_x) {
                    ppm_cell([&](int v, int m) { return s.W[v][yy][xx + m - 2]; }, chi_e, lo, hi);
#pragma unroll
                    for (int v = 0; v < 5; ++v) {
                        if (e_high) s.loXe[v][ey] = lo[v];
                        else        s.hiX[v][ey][0] = hi[v];
                    }
                } else {
                    ppm_cell([&](int v, int m) { return s.W[v][yy + m - 2][xx]; }, chi_e, lo, hi);
#pragma unroll
                    for (int v = 0; v < 5; ++v) {
                        if (e_high) s.loYe[v][ex] = lo[v];
                        else        s.hiY[v][0][ex] = hi[v];
                    }
                }
            }
        }
        __syncthreads();   // S2: face states visible; plane W no longer read
        // ---- phase F: Riemann fluxes -----------------------------------------------------------
        double FzHi[5], FxLo[5], FyLo[5];
        Cons5 uc = benign_cons(), u0 = benign_cons();
        if (k >= k0 - 1) face_flux<2>(gamma, hiZ, loZn, FzHi);     // face k+1/2
        if (k >= k0) {
            if (active) {
                const int cidx = g.at(gi, gj, k);
                uc = load_cons(U, cidx);
                if (stage == 1) u0 = load_cons(U0, cidx);
            }
            double L[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) L[v] = s.hiX[v][ty][tx];
            face_flux<0>(gamma, L, loX, FxLo);                        // face tx (low x face of the own cell)
#pragma unroll
            for (int v = 0; v < 5; ++v) L[v] = s.hiY[v][ty][tx];
            face_flux<1>(gamma, L, loY, FyLo);
            if (tx >= 1) {
#pragma unroll
                for (int v = 0; v < 5; ++v) s.fl.fx[v][ty][tx - 1] = FxLo[v];
            }
            if (ty >= 1) {
#pragma unroll
                for (int v = 0; v < 5; ++v) s.fl.fy[v][ty - 1][tx] = FyLo[v];
            }
            if (t < TX + TY) {      // the faces at the high end of the tile
                double R[5], F[5];
                if (t < TY) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) { L[v] = s.hiX[v][t][TX]; R[v] = s.loXe[v][t]; }
                    face_flux<0>(gamma, L, R, F);
#pragma unroll
                    for (int v = 0; v < 5; ++v) s.fl.fx[v][t][TX - 1] = F[v];
                } else {
                    const int cx = t - TY;
#pragma unroll
                    for (int v = 0; v < 5; ++v) { L[v] = s.hiY[v][TY][cx]; R[v] = s.loYe[v][cx]; }
                    face_flux<1>(gamma, L, R, F);
#pragma unroll
                    for (int v = 0; v < 5; ++v) s.fl.fy[v][TY - 1][cx] = F[v];
                }
            }
        }
        __syncthreads();   // S3: fluxes visible
        // ---- phase U: divergence and stage update ----------------------------------------------
        if (k >= k0 && active) {
            const double ucv[5] = {uc.r, uc.mx, uc.my, uc.mz, uc.e};
            const double u0v[5] = {u0.r, u0.mx, u0.my, u0.mz, u0.e};
            double res[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                const double div = ((s.fl.fx[v][ty][tx] - FxLo[v]) + (s.fl.fy[v][ty][tx] - FyLo[v])) + (FzHi[v] - FzLo[v]);
                const double us = ucv[v] - dtdx * div;
                res[v] = stage == 0 ? us : 0.5 * u0v[v] + 0.5 * us;
            }
            const int cidx = g.at(gi, gj, k);
            out.rho[cidx] = res[0]; out.mx[cidx] = res[1]; out.my[cidx] = res[2]; out.mz[cidx] = res[3];
            out.E[cidx] = res[4];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) { FzLo[v] = FzHi[v]; hiZ[v] = hiZn[v]; }
        chi_c = chi_z;
        chi_e = chi_e_next;
        __syncthreads();   // S4: flux buffers (aliasing plane W) and ring slot k-1 free
    }
    if (bad) atomicAdd((unsigned long long *)&ctr->bad_state, (unsigned long long)bad);
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static int chunk_length(int nz_planes, int tiles_xy)
{
    // enough CTAs to fill 148 SMs x 2 several times over, chunks not shorter than 16 planes
    int lz = 32;
    while (lz > 16 && (long long)tiles_xy * ((nz_planes + lz - 1) / lz) < 148 * 2 * 4) lz -= 8;
    if (lz > nz_planes) lz = nz_planes;
    return lz < 1 ? 1 : lz;
}

int launch_flatten_march(const Geom &g, double gamma, CHydro5 U, double *chi, cudaStream_t st)
{
    const int bx = (g.nx + 2 + TX - 1) / TX, by = (g.ny + 2 + TY - 1) / TY;
    const int lz = chunk_length(g.nz + 2, bx * by);
    dim3 grid(bx, by, (g.nz + 2 + lz - 1) / lz), block(TX, TY);
    flatten_march_kernel<<<grid, block, 0, st>>>(g, gamma, U, chi, lz);
    return 1;
}

int launch_hydro_stage(const Geom &g, double gamma, double dtdx, int stage, CHydro5 U, CHydro5 U0, const double *chi,
                       Hydro5 out, Counters *ctr, cudaStream_t st)
{
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(hydro_stage_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HydroSmem));
        configured = true;
    }
    const int bx = (g.nx + TX - 1) / TX, by = (g.ny + TY - 1) / TY;
    const int lz = chunk_length(g.nz, bx * by);
    dim3 grid(bx, by, (g.nz + lz - 1) / lz), block(TX, TY);
    hydro_stage_kernel<<<grid, block, sizeof(HydroSmem), st>>>(g, gamma, dtdx, stage, U, U0, chi, out, lz, ctr);
    return 1;
}

}  // namespace qk
