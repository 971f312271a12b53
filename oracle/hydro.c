/* hydro.c -- CPU ORACLE (test infrastructure): PPM-MOL hydro step of PAPER.md:120-172.
 * See qk_oracle.h for the role of this code.  Every formula below is written in the
 * evaluation order DESIGN.md section 3 fixes; no FMA contraction (-ffp-contract=off).
 * The `omp parallel for` lines only deal independent cells / faces out to threads (every loop body writes its own
 * cell and reads arrays finished by an earlier loop): the arithmetic per cell, and so every result bit, is the
 * same for any thread count (tests/test_oracle_hydro.py::test_thread_count_does_not_change_a_bit). */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "qk_oracle.h"

#define NG ORC_NG

static double min2(double a, double b) { return a < b ? a : b; }
static double max2(double a, double b) { return a > b ? a : b; }
static double clamp01(double x) { return min2(max2(x, 0.0), 1.0); }

/* rho, v = (rho v)/rho, P = (gamma-1)(E - rho v^2/2).
 * Kinetic energy summed as (vx^2+vy^2)+vz^2 (x<->y symmetric, H10). */
void orc_cons_to_prim(double gamma, const double U[5], double W[5])
{
    double rho = U[0];
    double vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
    double ke = 0.5 * rho * ((vx * vx + vy * vy) + vz * vz);
    W[0] = rho; W[1] = vx; W[2] = vy; W[3] = vz;
    W[4] = (gamma - 1.0) * (U[4] - ke);
}

/* monotonized-central slope (Van Leer 1977) of cell averages */
double orc_mc_slope(double qm1, double q0, double qp1)
{
    double dl = q0 - qm1, dr = qp1 - q0;
    if (dl * dr <= 0.0) return 0.0;
    double dc = 0.5 * (qp1 - qm1);
    double lim = min2(fabs(dc), min2(2.0 * fabs(dl), 2.0 * fabs(dr)));
    return dc > 0.0 ? lim : -lim;
}

/* PLM: q_{j-+1/2} = q_j -+ s/2 with s the monotonized-central slope of (q_{j-1}, q_j, q_{j+1}). */
void orc_plm_faces(const double q[5], double *q_minus, double *q_plus)
{
    double s = orc_mc_slope(q[1], q[2], q[3]);
    *q_minus = q[2] - 0.5 * s;
    *q_plus = q[2] + 0.5 * s;
}

/* reconstruction selected by the flags: PPM (default) or PLM */
void orc_faces(unsigned flags, const double q[5], double *q_minus, double *q_plus)
{
    if (flags & ORC_FLAG_PLM) orc_plm_faces(q, q_minus, q_plus);
    else orc_ppm_faces(q, q_minus, q_plus);
}

/* Face states of the centre cell q[2] from q[0..4] = q_{j-2..j+2}.
 * (a) eq 22 with each bracket mirror-symmetric about its interface;
 * (b) both states clamped to [min,max] of the cell and its two neighbours;
 * (c) CW84 parabola check: extremum -> MC-limited linear profile (Balsara 2017),
 *     overshoot -> CW84 eq 1.10 on the affected side.  No flattening here. */
void orc_ppm_faces(const double q[5], double *q_minus, double *q_plus)
{
    const double c7 = 7.0 / 12.0, c1 = 1.0 / 12.0;
    double qc = q[2];
    double qm = c7 * (q[1] + q[2]) - c1 * (q[3] + q[0]);   /* interface j-1/2 */
    double qp = c7 * (q[2] + q[3]) - c1 * (q[4] + q[1]);   /* interface j+1/2 */
    double lo = min2(q[1], min2(q[2], q[3]));
    double hi = max2(q[1], max2(q[2], q[3]));
    qm = min2(max2(qm, lo), hi);
    qp = min2(max2(qp, lo), hi);
    double dm = qc - qm, dp = qp - qc;
    if (dm * dp <= 0.0) {
        double s = orc_mc_slope(q[1], q[2], q[3]);
        qm = qc - 0.5 * s;
        qp = qc + 0.5 * s;
    } else if (fabs(dm) >= 2.0 * fabs(dp)) {
        qm = qc - 2.0 * dp;
    } else if (fabs(dp) >= 2.0 * fabs(dm)) {
        qp = qc + 2.0 * dm;
    }
    *q_minus = qm; *q_plus = qp;
}

/* One-directional flattening coefficient chi~_d of the centre cell from P[0..4] and the
 * normal velocity vn[0..4] at j-2..j+2.  PAPER.md:166 names Miller & Colella (2002) and
 * prints no formula: this is the reading of SURVEY 8(c) H6 / DESIGN.md (PARITY UNPINNED). */
double orc_flatten_1d(double gamma, const double P[5], const double vn[5])
{
    double a1 = fabs(P[3] - P[1]);
    double a2 = fabs(P[4] - P[0]);
    double chi_min;
    if (a2 == 0.0) chi_min = (a1 == 0.0) ? 1.0 : 0.0;      /* 0/0: none; x/0: full */
    else           chi_min = clamp01((0.85 - a1 / a2) / 0.10);
    if (!(vn[3] < vn[1])) return 1.0;                       /* not compressive */
    double Z = a1 / (gamma * P[2]);
    return max2(chi_min, clamp01((0.75 - Z) / 0.5));
}

/* HLLC flux with Toro's PVRS wavespeeds.  W = (rho, u_n, u_t1, u_t2, p),
 * F = (mass, normal momentum, t1 momentum, t2 momentum, energy).  The star state is
 * written r*[...] with r = (S_K-u_K)/(S_K-S*) so that an isolated stationary contact
 * gives bit-exact zero mass and energy flux. */
void orc_hllc(double gamma, const double WL[5], const double WR[5], double F[5])
{
    double rL = WL[0], uL = WL[1], pL = WL[4];
    double rR = WR[0], uR = WR[1], pR = WR[4];
    double aL = sqrt(gamma * pL / rL), aR = sqrt(gamma * pR / rR);
    double rbar = 0.5 * (rL + rR), abar = 0.5 * (aL + aR);
    double ppv = 0.5 * (pL + pR) - 0.5 * (uR - uL) * rbar * abar;
    double ps = max2(0.0, ppv);
    double g2 = (gamma + 1.0) / (2.0 * gamma);
    double qL = (ps <= pL) ? 1.0 : sqrt(1.0 + g2 * (ps / pL - 1.0));
    double qR = (ps <= pR) ? 1.0 : sqrt(1.0 + g2 * (ps / pR - 1.0));
    double SL = uL - aL * qL, SR = uR + aR * qR;
    double mL = rL * (SL - uL), mR = rR * (SR - uR);
    double Ss = (pR - pL + uL * mL - uR * mR) / (mL - mR);
    /* F_L (S_L>=0) | F*_L (S*>=0) | F*_R (S_R>0) | F_R, tested in that order */
    int left, supersonic;
    if (SL >= 0.0)      { left = 1; supersonic = 1; }
    else if (Ss >= 0.0) { left = 1; supersonic = 0; }
    else if (SR > 0.0)  { left = 0; supersonic = 0; }
    else                { left = 0; supersonic = 1; }
    const double *W = left ? WL : WR;
    double SK = left ? SL : SR;
    double r = W[0], u = W[1], v = W[2], w = W[3], p = W[4];
    double E = p / (gamma - 1.0) + 0.5 * r * (u * u + (v * v + w * w));
    double U[5]  = { r, r * u, r * v, r * w, E };
    double FK[5] = { r * u, r * u * u + p, r * u * v, r * u * w, u * (E + p) };
    if (supersonic) { for (int n = 0; n < 5; ++n) F[n] = FK[n]; return; }
    double fac = (SK - u) / (SK - Ss);
    double Us[5];
    Us[0] = fac * r;
    Us[1] = fac * (r * Ss);
    Us[2] = fac * U[2];
    Us[3] = fac * U[3];
    Us[4] = fac * (E + (Ss - u) * (r * Ss + p / (SK - u)));
    for (int n = 0; n < 5; ++n) F[n] = FK[n] + SK * (Us[n] - U[n]);
}

/* div[n][cell] = ((dFx + dFy) + dFz) of the ghost-filled conserved state U */
static int hydro_divergence(const orc_grid *g, double *const U[5], double *div[5])
{
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const long long SX = 1, SY = nx + 2 * NG, SZ = (long long)(nx + 2 * NG) * (ny + 2 * NG);
    const long long ntot = orc_ncells_total(g);
    const long long strides[3] = { SX, SY, SZ };
    const int nn[3] = { nx, ny, nz };
    double *W[5], *chi, *chid[3], *flux[5], *wl[5], *wr[5];
    int rc = 0;
    for (int n = 0; n < 5; ++n) {
        W[n] = (double *)malloc(ntot * sizeof(double));
        flux[n] = (double *)malloc(ntot * sizeof(double));
        wl[n] = (double *)malloc(ntot * sizeof(double));
        wr[n] = (double *)malloc(ntot * sizeof(double));
    }
    chi = (double *)malloc(ntot * sizeof(double));
    for (int d = 0; d < 3; ++d) chid[d] = (double *)malloc(ntot * sizeof(double));

    /* 1. primitives everywhere (ghosts included) */
#pragma omp parallel for schedule(static) reduction(max : rc) if (ntot > ORC_OMP_MIN)
    for (long long c = 0; c < ntot; ++c) {
        double Uc[5] = { U[0][c], U[1][c], U[2][c], U[3][c], U[4][c] }, Wc[5];
        orc_cons_to_prim(g->gamma, Uc, Wc);
        for (int n = 0; n < 5; ++n) W[n][c] = Wc[n];
        if (!(Wc[0] > 0.0) || !(Wc[4] > 0.0)) rc = 5;
    }
    /* 2. flattening: chi~_d where the +-2 stencil fits, then min over directions and the
     *    two neighbours along each direction (multidimensional) */
#define CIDX(i, j, k) (((long long)((k) + NG) * (ny + 2 * NG) + ((j) + NG)) * (nx + 2 * NG) + ((i) + NG))
    for (int d = 0; d < 3; ++d) {
        long long s = strides[d];
        for (long long c = 0; c < ntot; ++c) chid[d][c] = 1.0;
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = -NG; k < nz + NG; ++k)
            for (int j = -NG; j < ny + NG; ++j)
                for (int i = -NG; i < nx + NG; ++i) {
                    int pos = d == 0 ? i : (d == 1 ? j : k);
                    if (pos < -NG + 2 || pos > nn[d] + NG - 3) continue;
                    long long c = CIDX(i, j, k);
                    double P[5], vn[5];
                    for (int m = 0; m < 5; ++m) { P[m] = W[4][c + (m - 2) * s]; vn[m] = W[1 + d][c + (m - 2) * s]; }
                    chid[d][c] = orc_flatten_1d(g->gamma, P, vn);
                }
    }
    for (long long c = 0; c < ntot; ++c) chi[c] = 1.0;
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
    for (int k = -1; k <= nz; ++k)
        for (int j = -1; j <= ny; ++j)
            for (int i = -1; i <= nx; ++i) {
                long long c = CIDX(i, j, k);
                double x = 1.0;
                for (int d = 0; d < 3; ++d) {
                    long long s = strides[d];
                    x = min2(x, min2(chid[d][c - s], min2(chid[d][c], chid[d][c + s])));
                }
                chi[c] = x;
            }
    /* 3.-4. per direction: PPM face states of cells -1..n, flatten, HLLC at faces 0..n */
    for (int n = 0; n < 5; ++n) memset(div[n], 0, ntot * sizeof(double));
    for (int d = 0; d < 3; ++d) {
        long long s = strides[d];
        int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        int lo[3] = { 0, 0, 0 }, hi[3] = { nx, ny, nz };
        lo[d] = -1; hi[d] = nn[d] + 1;
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i) {
                    long long c = CIDX(i, j, k);
                    for (int n = 0; n < 5; ++n) {
                        double q[5], qm, qp;
                        for (int m = 0; m < 5; ++m) q[m] = W[n][c + (m - 2) * s];
                        orc_faces(g->flags, q, &qm, &qp);
                        wl[n][c] = q[2] + chi[c] * (qm - q[2]);    /* flatten toward the average */
                        wr[n][c] = q[2] + chi[c] * (qp - q[2]);
                    }
                }
        lo[d] = 0;                                   /* face at the low side of cells 0..n */
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i) {
                    long long c = CIDX(i, j, k);
                    double WL[5] = { wr[0][c - s], wr[1 + d][c - s], wr[1 + t1][c - s], wr[1 + t2][c - s], wr[4][c - s] };
                    double WR[5] = { wl[0][c], wl[1 + d][c], wl[1 + t1][c], wl[1 + t2][c], wl[4][c] };
                    double F[5];
                    orc_hllc(g->gamma, WL, WR, F);
                    flux[0][c] = F[0]; flux[1 + d][c] = F[1]; flux[1 + t1][c] = F[2];
                    flux[1 + t2][c] = F[3]; flux[4][c] = F[4];
                }
        /* accumulate: after d=0 div=dFx; d=1 div=dFx+dFy; d=2 div=(dFx+dFy)+dFz */
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    long long c = CIDX(i, j, k);
                    for (int n = 0; n < 5; ++n) {
                        double dF = flux[n][c + s] - flux[n][c];
                        div[n][c] = (d == 0) ? dF : div[n][c] + dF;
                    }
                }
    }
#undef CIDX
    for (int n = 0; n < 5; ++n) { free(W[n]); free(flux[n]); free(wl[n]); free(wr[n]); }
    free(chi);
    for (int d = 0; d < 3; ++d) free(chid[d]);
    return rc;
}

/* SSP-RK2 (Shu & Osher 1988):
 *   U1 = Un - (dt/dx) div(Un);  U2 = U1 - (dt/dx) div(U1);  Un+1 = 0.5 Un + 0.5 U2.
 * Ghosts are filled before each stage. */
int orc_hydro_step(orc_grid *g, double dt)
{
    const long long ntot = orc_ncells_total(g);
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    double *div[5], *U0[5], *U[5];
    int rc = 0;
    const double dtdx = dt / g->dx;
    for (int n = 0; n < 5; ++n) {
        div[n] = (double *)malloc(ntot * sizeof(double));
        U0[n] = (double *)malloc(ntot * sizeof(double));
        U[n] = g->f[ORC_RHO + n];
    }
    orc_fill_boundary(g, ORC_FILL_HYDRO);
    for (int n = 0; n < 5; ++n) memcpy(U0[n], U[n], ntot * sizeof(double));
    for (int stage = 0; stage < 2; ++stage) {
        if (stage == 1) orc_fill_boundary(g, ORC_FILL_HYDRO);
        int r = hydro_divergence(g, U, div);
        if (r) rc = r;
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    long long c = ((long long)(k + NG) * (ny + 2 * NG) + (j + NG)) * (nx + 2 * NG) + (i + NG);
                    for (int n = 0; n < 5; ++n) {
                        double us = U[n][c] - dtdx * div[n][c];
                        U[n][c] = (stage == 0) ? us : 0.5 * U0[n][c] + 0.5 * us;
                    }
                }
    }
    for (int n = 0; n < 5; ++n) { free(div[n]); free(U0[n]); }
    return rc;
}
