/* radiation.c -- CPU ORACLE (test infrastructure): explicit RSLA transport of (E_r, F_r),
 * PAPER.md:174-196 (eq 11-12, 23-25).  See qk_oracle.h for the role of this code. */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "qk_oracle.h"

#define NG ORC_NG

static double min2(double a, double b) { return a < b ? a : b; }
static double max2(double a, double b) { return a > b ? a : b; }

/* Levermore (1984) Eddington factor, eq 24 */
double orc_eddington_factor(double f)
{
    double f2 = f * f;
    return (3.0 + 4.0 * f2) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f2));
}

/* Column n of the Eddington tensor T = (1-chi)/2 I + (3chi-1)/2 nn (eq 23)
 * for reduced flux fvec.  |f| is clamped to 1 for the closure only;
 * n = f/|f| (eq 25); the nn term is dropped when the flux is exactly zero. */
void orc_closure(const double fvec[3], int n, double T_col[3], double *chi_out)
{
    double fsq = (fvec[0] * fvec[0] + fvec[1] * fvec[1]) + fvec[2] * fvec[2];
    double fmag = sqrt(fsq);
    double fc = min2(fmag, 1.0);
    double chi = orc_eddington_factor(fc);
    double a = 0.5 * (1.0 - chi), b = 0.5 * (3.0 * chi - 1.0);
    for (int i = 0; i < 3; ++i) T_col[i] = (i == n) ? a : 0.0;
    if (fmag > 0.0) {
        double nh[3] = { fvec[0] / fmag, fvec[1] / fmag, fvec[2] / fmag };
        for (int i = 0; i < 3; ++i) T_col[i] = T_col[i] + b * (nh[i] * nh[n]);
    }
    if (chi_out) *chi_out = chi;
}

/* Minerbo (1978) maximum-entropy closure in the polynomial form used throughout the transport literature
 * (PAPER.md:196 names the closure, prints no formula; V3): chi(0) = 1/3, chi(1) = 1. */
double orc_minerbo_factor(double f)
{
    double f2 = f * f;
    return 1.0 / 3.0 + (2.0 / 15.0) * (f2 * ((3.0 - f) + 3.0 * f2));
}

/* closure selected by the flags: Levermore (eq 23-25, default) or the Eddington approximation chi = 1/3,
 * i.e. P_r = E_r/3 I whatever the flux ("any local closure f -> chi") */
void orc_closure_k(unsigned flags, const double fvec[3], int n, double T_col[3], double *chi_out)
{
    if (flags & ORC_FLAG_EDDINGTON) {
        double chi = 1.0 / 3.0;
        double a = 0.5 * (1.0 - chi);
        for (int i = 0; i < 3; ++i) T_col[i] = (i == n) ? a : 0.0;     /* (3chi-1)/2 = 0: no n n term */
        if (chi_out) *chi_out = chi;
        return;
    }
    if (flags & ORC_FLAG_MINERBO) {     /* as orc_closure with chi from orc_minerbo_factor */
        double fsq = (fvec[0] * fvec[0] + fvec[1] * fvec[1]) + fvec[2] * fvec[2];
        double fmag = sqrt(fsq);
        double chi = orc_minerbo_factor(min2(fmag, 1.0));
        double a = 0.5 * (1.0 - chi), b = 0.5 * (3.0 * chi - 1.0);
        for (int i = 0; i < 3; ++i) T_col[i] = (i == n) ? a : 0.0;
        if (fmag > 0.0) {
            double nh[3] = { fvec[0] / fmag, fvec[1] / fmag, fvec[2] / fmag };
            for (int i = 0; i < 3; ++i) T_col[i] = T_col[i] + b * (nh[i] * nh[n]);
        }
        if (chi_out) *chi_out = chi;
        return;
    }
    orc_closure(fvec, n, T_col, chi_out);
}

static void rad_phys_flux_k(unsigned flags, double c, double c_hat, const double S[4], int n, double G[4], double *Tnn)
{
    double T[3];
    orc_closure_k(flags, &S[1], n, T, NULL);
    double Fn = (c * S[0]) * S[1 + n];
    double cc = (c * c_hat) * S[0];
    G[0] = (c_hat / c) * Fn;
    for (int i = 0; i < 3; ++i) G[1 + i] = cc * T[i];
    if (Tnn) *Tnn = T[n];
}

/* Physical flux through a face with normal n of the state S = (E_r, f_x, f_y, f_z):
 * (c_hat/c) F_n for E_r and c c_hat E_r T_in for F_i (eq 11-12). */
void orc_rad_phys_flux(double c, double c_hat, const double S[4], int n, double G[4], double *Tnn)
{
    double T[3];
    orc_closure(&S[1], n, T, NULL);
    double Fn = (c * S[0]) * S[1 + n];
    double cc = (c * c_hat) * S[0];
    G[0] = (c_hat / c) * Fn;
    for (int i = 0; i < 3; ++i) G[1 + i] = cc * T[i];
    if (Tnn) *Tnn = T[n];
}

/* HLL flux with wavespeeds +-S, S = max(c_hat sqrt(Tnn_L), c_hat sqrt(Tnn_R), s_floor c_hat), s_floor = 0.1,
 * Eddington factors frozen.  With S_L = -S_R the HLL formula is
 * G = (G_L+G_R)/2 - (S/2)(U_R-U_L).  Optical-depth correction: the E_r
 * dissipation is scaled by eps = min(1, 1/tau_face); it is disabled for the face when
 * either HLL star state it implies violates E*>0, |F*|<=cE*.  Forms are DESIGN.md
 * readings R5/R6 (PARITY UNPINNED).  Returns 1 if the guard fired. */
int orc_rad_hll_floor(double c, double c_hat, const double SL[4], const double SR[4], int n,
                      double tau_face, unsigned flags, double s_floor, double G[4])
{
    double GL[4], GR[4], TL, TR;
    rad_phys_flux_k(flags, c, c_hat, SL, n, GL, &TL);
    rad_phys_flux_k(flags, c, c_hat, SR, n, GR, &TR);
    double S = max2(max2(c_hat * sqrt(TL), c_hat * sqrt(TR)), s_floor * c_hat);
    double UL[4] = { SL[0], (c * SL[0]) * SL[1], (c * SL[0]) * SL[2], (c * SL[0]) * SL[3] };
    double UR[4] = { SR[0], (c * SR[0]) * SR[1], (c * SR[0]) * SR[2], (c * SR[0]) * SR[3] };
    double diss = 0.5 * S;
    for (int m = 1; m < 4; ++m) G[m] = 0.5 * (GL[m] + GR[m]) - diss * (UR[m] - UL[m]);
    double eps = 1.0;
    if (flags & ORC_FLAG_TAU_CORR) eps = min2(1.0, 1.0 / tau_face);
    G[0] = 0.5 * (GL[0] + GR[0]) - (eps * diss) * (UR[0] - UL[0]);
    if (eps < 1.0) {
        double EsL = UL[0] + (G[0] - GL[0]) / (-S), EsR = UR[0] + (G[0] - GR[0]) / S;
        double FL[3], FR[3];
        for (int m = 0; m < 3; ++m) {
            FL[m] = UL[1 + m] + (G[1 + m] - GL[1 + m]) / (-S);
            FR[m] = UR[1 + m] + (G[1 + m] - GR[1 + m]) / S;
        }
        double f2L = (FL[0] * FL[0] + FL[1] * FL[1]) + FL[2] * FL[2];
        double f2R = (FR[0] * FR[0] + FR[1] * FR[1]) + FR[2] * FR[2];
        double cEL = c * EsL, cER = c * EsR;
        int bad = !(EsL > 0.0) || !(EsR > 0.0) || (f2L > cEL * cEL) || (f2R > cER * cER);
        if (bad) {
            G[0] = 0.5 * (GL[0] + GR[0]) - diss * (UR[0] - UL[0]);
            return 1;
        }
    }
    return 0;
}

/* the same with the floor of reading R5, 0.1 c_hat */
int orc_rad_hll(double c, double c_hat, const double SL[4], const double SR[4], int n,
                double tau_face, unsigned flags, double G[4])
{
    return orc_rad_hll_floor(c, c_hat, SL, SR, n, tau_face, flags, 0.1, G);
}

/* div[m][cell] = ((dGx + dGy) + dGz) for the ghost-filled radiation state R=(E_r,F_x,F_y,F_z) */
static int rad_divergence(orc_grid *g, double *const R[4], double *div[4])
{
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const long long SY = nx + 2 * NG, SZ = (long long)(nx + 2 * NG) * (ny + 2 * NG);
    const long long ntot = orc_ncells_total(g);
    const long long strides[3] = { 1, SY, SZ };
    const int nn[3] = { nx, ny, nz };
    const double *rho = g->f[ORC_RHO], *kR = g->f[ORC_KR];
    double *S[4], *sl[4], *sr[4], *flux[4];
    int rc = 0;
    for (int m = 0; m < 4; ++m) {
        S[m] = (double *)malloc(ntot * sizeof(double));
        sl[m] = (double *)malloc(ntot * sizeof(double));
        sr[m] = (double *)malloc(ntot * sizeof(double));
        flux[m] = (double *)malloc(ntot * sizeof(double));
    }
    /* reconstruct in E_r and the reduced flux f = F_r/(c E_r) */
#pragma omp parallel for schedule(static) if (ntot > ORC_OMP_MIN)
    for (long long cidx = 0; cidx < ntot; ++cidx) {
        double E = R[0][cidx], cE = g->c * E;
        S[0][cidx] = E;
        for (int m = 1; m < 4; ++m) S[m][cidx] = R[m][cidx] / cE;
    }
#define CIDX(i, j, k) (((long long)((k) + NG) * (ny + 2 * NG) + ((j) + NG)) * (nx + 2 * NG) + ((i) + NG))
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                if (!(R[0][CIDX(i, j, k)] > 0.0)) rc = 5;      /* needs E_r > 0 */
    for (int m = 0; m < 4; ++m) memset(div[m], 0, ntot * sizeof(double));
    for (int d = 0; d < 3; ++d) {
        long long s = strides[d];
        int lo[3] = { 0, 0, 0 }, hi[3] = { nx, ny, nz };
        lo[d] = -1; hi[d] = nn[d] + 1;
        long long nfall = 0, nguard = 0;
#pragma omp parallel for collapse(3) schedule(static) reduction(+ : nfall) if (ntot > ORC_OMP_MIN)
        for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i) {
                    long long c = CIDX(i, j, k);
                    double lo4[4], hi4[4];
                    for (int m = 0; m < 4; ++m) {
                        double q[5];
                        for (int t = 0; t < 5; ++t) q[t] = S[m][c + (t - 2) * s];
                        orc_faces(g->flags, q, &lo4[m], &hi4[m]); /* no flattening */
                    }
                    /* first-order fallback per face state when |f|>1 (or E_r<=0) */
                    double f2 = (lo4[1] * lo4[1] + lo4[2] * lo4[2]) + lo4[3] * lo4[3];
                    if (f2 > 1.0 || !(lo4[0] > 0.0)) {
                        for (int m = 0; m < 4; ++m) lo4[m] = S[m][c];
                        nfall++;
                    }
                    f2 = (hi4[1] * hi4[1] + hi4[2] * hi4[2]) + hi4[3] * hi4[3];
                    if (f2 > 1.0 || !(hi4[0] > 0.0)) {
                        for (int m = 0; m < 4; ++m) hi4[m] = S[m][c];
                        nfall++;
                    }
                    for (int m = 0; m < 4; ++m) { sl[m][c] = lo4[m]; sr[m][c] = hi4[m]; }
                }
        lo[d] = 0;
#pragma omp parallel for collapse(3) schedule(static) reduction(+ : nguard) if (ntot > ORC_OMP_MIN)
        for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i) {
                    long long c = CIDX(i, j, k);
                    double SL[4] = { sr[0][c - s], sr[1][c - s], sr[2][c - s], sr[3][c - s] };
                    double SR[4] = { sl[0][c], sl[1][c], sl[2][c], sl[3][c] };
                    double tau = (0.5 * (kR[c - s] * rho[c - s] + kR[c] * rho[c])) * g->dx;
                    double G[4];
                    nguard += orc_rad_hll_floor(g->c, g->c_hat, SL, SR, d, tau, g->flags, g->s_floor, G);
                    for (int m = 0; m < 4; ++m) flux[m][c] = G[m];
                }
        g->fallback_states += nfall; g->guard_faces += nguard;
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    long long c = CIDX(i, j, k);
                    for (int m = 0; m < 4; ++m) {
                        double dG = flux[m][c + s] - flux[m][c];
                        div[m][c] = (d == 0) ? dG : div[m][c] + dG;
                    }
                }
    }
#undef CIDX
    for (int m = 0; m < 4; ++m) { free(S[m]); free(sl[m]); free(sr[m]); free(flux[m]); }
    return rc;
}

/* kappa = kappa0 (rho/rho0)^e (T/T0)^(texp2/2) (orc_opacity_density_part, orc_temp_power) for the interior cells,
 * from the density and gas temperature the hydro step / the last exchange left (opacities are static during the
 * transport part of a radiation subcycle) */
static void apply_opacity_law(orc_grid *g)
{
    if (!(g->opac_rho0 > 0.0)) return;
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                long long c = ((long long)(k + NG) * (g->ny + 2 * NG) + (j + NG)) * (g->nx + 2 * NG) + (i + NG);
                double rho = g->f[ORC_RHO][c], kp, kr;
                orc_opacity_density_part(g, rho, &kp, &kr);
                if (g->opac_texp2 != 0) {
                    double m[3] = { g->f[ORC_MX][c], g->f[ORC_MY][c], g->f[ORC_MZ][c] };
                    double tp = orc_temp_power(orc_gas_temperature(g, rho, m, g->f[ORC_E][c]), g->opac_T0, g->opac_texp2);
                    kp = kp * tp; kr = kr * tp;
                }
                g->f[ORC_KP][c] = kp; g->f[ORC_KR][c] = kr;
            }
}

/* one radiation subcycle of transport: the same SSP-RK2 as hydro */
int orc_rad_transport(orc_grid *g, double dt)
{
    apply_opacity_law(g);
    const long long ntot = orc_ncells_total(g);
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    double *div[4], *R0[4], *R[4];
    const double dtdx = dt / g->dx;
    int rc = 0;
    g->fallback_states = 0; g->guard_faces = 0;
    for (int m = 0; m < 4; ++m) {
        div[m] = (double *)malloc(ntot * sizeof(double));
        R0[m] = (double *)malloc(ntot * sizeof(double));
        R[m] = g->f[ORC_ER + m];
    }
    /* rho and kappa_R ghosts feed tau_face at the domain faces */
    orc_fill_boundary(g, ORC_FILL_RAD);
    orc_fill_field(g, ORC_RHO);
    orc_fill_field(g, ORC_KR);
    for (int m = 0; m < 4; ++m) memcpy(R0[m], R[m], ntot * sizeof(double));
    for (int stage = 0; stage < 2; ++stage) {
        if (stage == 1) orc_fill_boundary(g, ORC_FILL_RAD);
        int r = rad_divergence(g, R, div);
        if (r) rc = r;
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    long long c = ((long long)(k + NG) * (ny + 2 * NG) + (j + NG)) * (nx + 2 * NG) + (i + NG);
                    for (int m = 0; m < 4; ++m) {
                        double us = R[m][c] - dtdx * div[m][c];
                        R[m][c] = (stage == 0) ? us : 0.5 * R0[m][c] + 0.5 * us;
                    }
                }
    }
    for (int m = 0; m < 4; ++m) { free(div[m]); free(R0[m]); }
    return rc;
}
