/* exchange.c -- CPU ORACLE (test infrastructure): per-cell implicit matter-radiation
 * coupling, PAPER.md:198-265 (eq 26-43).  See qk_oracle.h for the role of this code.
 *
 * Readings: X1 eq 28 is taken as R = dt rho kappa_P c_hat (a_r T^4 - E_r)
 * (the printed "4 pi B - c_hat E_r" is dimensionally inconsistent with eq 15-16 and with
 * its own Jacobian eq 30, 32; 4 pi B = c a_r T^4 and the RSLA factor c_hat/c multiplies it).
 * X2 C_v is the volumetric heat capacity dE_g/dT.  X5 converge-then-polish stop rule unless
 * ORC_FLAG_NEWTON_LITERAL. */
#include <math.h>
#include <stdlib.h>
#include "qk_oracle.h"

#define NG ORC_NG

/* T and C_v = dE_g/dT from the gas internal energy density */
static void eos_T_Cv(const orc_grid *g, double rho, double Eg, double *T, double *Cv)
{
    if (g->eos == ORC_EOS_ALPHA_T3) {          /* eq 55: E_g = alpha T^4/4, C_v = alpha T^3 */
        double t = sqrt(sqrt(4.0 * Eg / g->alpha));
        *T = t; *Cv = g->alpha * (t * t * t);
    } else {                                    /* ideal gas: E_g = rho kB/(mu mH) T/(gamma-1) */
        double cv = rho * g->kB_mu / (g->gamma - 1.0);
        *Cv = cv; *T = Eg / cv;
    }
}

/* (T/T0)^(n2/2) for an integer n2 by repeated multiplication, one square root when n2 is odd and one division
 * when it is negative -- no pow(), so that the CUDA path can reproduce every bit (X14). */
double orc_temp_power(double T, double T0, int n2)
{
    int a = n2 < 0 ? -n2 : n2;
    double q = T / T0, p = 1.0;
    for (int m = 0; m < a / 2; ++m) p = p * q;
    if (a & 1) p = p * sqrt(q);
    return n2 < 0 ? 1.0 / p : p;
}

/* density part kappa0 (rho/rho0)^e of the opacity law, integer e by repeated multiplication */
void orc_opacity_density_part(const orc_grid *g, double rho, double *kP, double *kR)
{
    const int n = g->opac_exp < 0 ? -g->opac_exp : g->opac_exp;
    double q = g->opac_exp < 0 ? g->opac_rho0 / rho : rho / g->opac_rho0;
    double kp = g->opac_kP0, kr = g->opac_kR0;
    for (int m = 0; m < n; ++m) { kp = kp * q; kr = kr * q; }
    *kP = kp; *kR = kr;
}

/* gas temperature of a cell from its conserved state (PAPER.md:204 and the equation of state) */
double orc_gas_temperature(const orc_grid *g, double rho, const double m[3], double E)
{
    double msq = (m[0] * m[0] + m[1] * m[1]) + m[2] * m[2];
    double Eg = E - 0.5 * msq / rho, T, Cv;
    eos_T_Cv(g, rho, Eg, &T, &Cv);
    return T;
}

/* Updates (m, E, Er, F) of one cell over dt.  With a temperature-dependent opacity law (orc_set_opacity_law_T,
 * texp2 != 0) kP and kR are the density parts of the law: kappa_P follows the Newton iterate's temperature and
 * enters the Jacobian through d kappa_P / dT (eq 33), kappa_F ~ kappa_R is evaluated at the updated
 * gas temperature.  Returns 0 ok, 4 Newton failure, 5 bad state. */
int orc_exchange_cell(const orc_grid *g, double dt, double rho, double m[3], double *E,
                      double *Er, double F[3], double kP, double kR, int *iters)
{
    const double c = g->c, ch = g->c_hat, coc = c / ch;
    const double S = g->S_src;
    int rc = 0;
    double msq0 = (m[0] * m[0] + m[1] * m[1]) + m[2] * m[2];
    double Ekin0 = 0.5 * msq0 / rho;
    double Eg0 = *E - Ekin0;
    double Er0 = *Er;
    double Etot = Eg0 + coc * (Er0 + S);        /* eq 38 */
    double coef = dt * rho * kP * ch;           /* dt rho kappa_P c_hat */
    const int kT = (g->opac_rho0 > 0.0) && (g->opac_texp2 != 0);   /* kappa(rho, T) law */
    double Eg = Eg0, Erad = Er0;
    int it = 0, done = 0;
    const int literal = (g->flags & ORC_FLAG_NEWTON_LITERAL) != 0;
    while (it < g->newton_maxit) {
        double T, Cv;
        eos_T_Cv(g, rho, Eg, &T, &Cv);
        double T2 = T * T;
        double T4 = T2 * T2;
        double dcoef_dT = 0.0;
        if (kT) {                                                 /* kappa_P at the iterate's temperature */
            double kPT = kP * orc_temp_power(T, g->opac_T0, g->opac_texp2);
            coef = dt * rho * kPT * ch;
            double dkP_dT = (0.5 * (double)g->opac_texp2) * kPT / T;
            if (!(g->flags & ORC_FLAG_NO_DKAPPA_DT)) dcoef_dT = dt * rho * dkP_dT * ch;
        }
        double R = coef * (g->a_rad * T4 - Erad);                 /* eq 28 (reading X1) */
        double FG = (Eg - Eg0) + coc * R;                         /* eq 26 */
        double FR = (Erad - Er0) - (R + S);                       /* eq 27 */
        int conv = (fabs(FG / Etot) < g->newton_tol) && (fabs(coc * FR / Etot) < g->newton_tol); /* eq 36-37 */
        if (conv && literal) { done = 1; break; }
        double dRdEg = coef * (4.0 * g->a_rad * (T2 * T)) / Cv;   /* eq 33, dkappa/dT = 0 */
        if (kT) dRdEg = (coef * (4.0 * g->a_rad * (T2 * T)) + dcoef_dT * (g->a_rad * T4 - Erad)) / Cv;   /* eq 33 */
        double dFGdEg = 1.0 + coc * dRdEg;                        /* eq 29 */
        double dFGdEr = -(coc * coef);                            /* eq 30 */
        double dFRdEg = -dRdEg;                                   /* eq 31 */
        double dFRdEr = 1.0 + coef;                               /* eq 32 */
        double eta = -dFRdEg / dFGdEg;
        double dEr = -(FR + eta * FG) / (dFRdEr + eta * dFGdEr);  /* eq 34 */
        double dEg = -(FG + dEr * dFGdEr) / dFGdEg;               /* eq 35 */
        Erad = Erad + dEr;
        Eg = Eg + dEg;
        ++it;
        if (conv) { done = 1; break; }
    }
    if (!done) rc = 4;
    if (iters) *iters = it;
    /* eq 39-41 with kappa_F ~ kappa_R */
    if (kT) {                                                     /* kappa_F at the updated temperature */
        double T, Cv;
        eos_T_Cv(g, rho, Eg, &T, &Cv);
        kR = kR * orc_temp_power(T, g->opac_T0, g->opac_texp2);
    }
    double denom = 1.0 + rho * kR * ch * dt;
    double F1[3], m1[3];
    for (int i = 0; i < 3; ++i) F1[i] = F[i] / denom;
    if (g->flags & ORC_FLAG_STATIC_MATTER) {                       /* drop all v/c terms */
        *E = Eg + Ekin0;
        *Er = Erad;
    } else {
        for (int i = 0; i < 3; ++i) m1[i] = m[i] - (F1[i] - F[i]) / (ch * c);
        double msq1 = (m1[0] * m1[0] + m1[1] * m1[1]) + m1[2] * m1[2];
        double dEkin = 0.5 * (msq1 - msq0) / rho;
        *E = Eg + (Ekin0 + dEkin);                                 /* eq 42 */
        *Er = Erad - (ch / c) * dEkin;                             /* eq 43 */
        for (int i = 0; i < 3; ++i) m[i] = m1[i];
    }
    for (int i = 0; i < 3; ++i) F[i] = F1[i];
    if (!(Eg > 0.0) || !(*Er > 0.0)) rc = rc ? rc : 5;
    return rc;
}

int orc_exchange(orc_grid *g, double dt)
{
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const long long ntot = orc_ncells_total(g);
    const int kT = (g->opac_rho0 > 0.0) && (g->opac_texp2 != 0);
    long long fail = 0, tot = 0, bad = 0; int mx = 0;
#pragma omp parallel for collapse(3) schedule(static) reduction(+ : fail, tot, bad) reduction(max : mx) if (ntot > ORC_OMP_MIN)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                long long cidx = ((long long)(k + NG) * (ny + 2 * NG) + (j + NG)) * (nx + 2 * NG) + (i + NG);
                double m[3] = { g->f[ORC_MX][cidx], g->f[ORC_MY][cidx], g->f[ORC_MZ][cidx] };
                double F[3] = { g->f[ORC_FX][cidx], g->f[ORC_FY][cidx], g->f[ORC_FZ][cidx] };
                double E = g->f[ORC_E][cidx], Er = g->f[ORC_ER][cidx];
                double kP = g->f[ORC_KP][cidx], kR = g->f[ORC_KR][cidx];
                int it = 0;
                orc_grid cell = *g;                              /* per-cell copy of the parameters: carries S */
                cell.S_src = dt * g->f[ORC_SRC][cidx];           /* energy added during the substep (X13) */
                if (kT) orc_opacity_density_part(g, g->f[ORC_RHO][cidx], &kP, &kR);
                int r = orc_exchange_cell(&cell, dt, g->f[ORC_RHO][cidx], m, &E, &Er, F, kP, kR, &it);
                if (r == 4) ++fail;
                if (r == 5) ++bad;
                tot += it; if (it > mx) mx = it;
                g->f[ORC_MX][cidx] = m[0]; g->f[ORC_MY][cidx] = m[1]; g->f[ORC_MZ][cidx] = m[2];
                g->f[ORC_FX][cidx] = F[0]; g->f[ORC_FY][cidx] = F[1]; g->f[ORC_FZ][cidx] = F[2];
                g->f[ORC_E][cidx] = E; g->f[ORC_ER][cidx] = Er;
            }
    g->newton_fail_cells = fail; g->newton_total_iters = tot; g->newton_max_iters = mx;
    g->bad_state_cells = bad;
    return fail ? 4 : (bad ? 5 : 0);
}
