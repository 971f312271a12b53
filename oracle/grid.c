/* grid.c -- CPU ORACLE (test infrastructure): storage, ghost fill, CFL, step drivers.
 * See qk_oracle.h for the role of this code.  Citations: /root/reference/PAPER.md. */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "qk_oracle.h"

static long long sx(const orc_grid *g) { (void)g; return 1; }
static long long sy(const orc_grid *g) { return (long long)(g->nx + 2 * ORC_NG); }
static long long sz(const orc_grid *g) { return (long long)(g->nx + 2 * ORC_NG) * (g->ny + 2 * ORC_NG); }

long long orc_ncells_total(const orc_grid *g)
{
    return (long long)(g->nx + 2 * ORC_NG) * (g->ny + 2 * ORC_NG) * (g->nz + 2 * ORC_NG);
}

/* index of cell (i,j,k), interior 0..n-1, ghosts -4..-1 and n..n+3 */
static long long idx(const orc_grid *g, int i, int j, int k)
{
    return ((long long)(k + ORC_NG) * (g->ny + 2 * ORC_NG) + (j + ORC_NG)) * (g->nx + 2 * ORC_NG) + (i + ORC_NG);
}

orc_grid *orc_create(int nx, int ny, int nz, double dx, double gamma, double c_hat, double c, int bc)
{
    orc_grid *g = (orc_grid *)calloc(1, sizeof(orc_grid));
    if (!g) return NULL;
    g->nx = nx; g->ny = ny; g->nz = nz;
    g->dx = dx; g->gamma = gamma; g->c_hat = c_hat; g->c = c; g->bc = bc;
    for (int f = 0; f < 6; ++f) g->face_bc[f] = bc;
    g->a_rad = 1.0; g->kB_mu = 1.0;
    g->cfl = 0.3; g->newton_tol = 1e-10; g->newton_maxit = 400; g->nsub_max = 10;
    g->flags = 0;                    /* optical-depth correction off: DESIGN.md R6 */
    g->s_floor = 0.1;                /* wavespeed floor of reading R5, in units of c_hat */
    g->eos = ORC_EOS_IDEAL; g->alpha = 0.0; g->S_src = 0.0;
    long long n = orc_ncells_total(g);
    for (int f = 0; f < ORC_NFIELDS; ++f) {
        g->f[f] = (double *)calloc((size_t)n, sizeof(double));
        if (!g->f[f]) { orc_destroy(g); return NULL; }
    }
    return g;
}

void orc_destroy(orc_grid *g)
{
    if (!g) return;
    for (int f = 0; f < ORC_NFIELDS; ++f) free(g->f[f]);
    free(g);
}

void orc_set_constants(orc_grid *g, double a_rad, double kB_mu) { g->a_rad = a_rad; g->kB_mu = kB_mu; }

void orc_set_params(orc_grid *g, double cfl, double newton_tol, int newton_maxit, int nsub_max, unsigned flags)
{
    g->cfl = cfl; g->newton_tol = newton_tol; g->newton_maxit = newton_maxit;
    g->nsub_max = nsub_max; g->flags = flags;
}

void orc_set_eos(orc_grid *g, int eos, double alpha) { g->eos = eos; g->alpha = alpha; }

/* Density power-law opacities of the paper's tests: kappa = kappa0 (rho/rho0)^e with integer e
 * (rho kappa ~ rho^2, e = 1; kappa ~ 1/rho, e = -1).  rho0 = 0 switches the law off
 * (opacities are then the fields the caller set).  DESIGN.md X14. */
void orc_set_opacity_law(orc_grid *g, double kP0, double kR0, double rho0, int exponent)
{
    g->opac_kP0 = kP0; g->opac_kR0 = kR0; g->opac_rho0 = rho0; g->opac_exp = exponent;
    g->opac_T0 = 1.0; g->opac_texp2 = 0;
}

/* ... times (T/T0)^(texp2/2), T the gas temperature: half-integer powers such as Kramers' T^-3.5 (texp2 = -7).
 * The exchange then treats kappa_P implicitly, with the d kappa_P/dT term of eq 33, and evaluates
 * kappa_F at the updated temperature. */
void orc_set_opacity_law_T(orc_grid *g, double kP0, double kR0, double rho0, int exponent, double T0, int texp2)
{
    orc_set_opacity_law(g, kP0, kR0, rho0, exponent);
    g->opac_T0 = T0; g->opac_texp2 = texp2;
}

/* floor of the HLL wavespeed in units of c_hat (reading R5: 0.1); exposed for the sensitivity pin only */
void orc_set_wavespeed_floor(orc_grid *g, double s_floor) { g->s_floor = s_floor; }

/* worker threads of the `omp parallel for` loops (results do not depend on it) */
#ifdef _OPENMP
#include <omp.h>
void orc_set_threads(int n) { omp_set_num_threads(n < 1 ? 1 : n); }
int  orc_get_threads(void) { return omp_get_max_threads(); }
#else
void orc_set_threads(int n) { (void)n; }
int  orc_get_threads(void) { return 1; }
#endif

void orc_set_field(orc_grid *g, int field, const double *interior)
{
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i)
                g->f[field][idx(g, i, j, k)] = interior[((long long)k * g->ny + j) * g->nx + i];
}

void orc_get_field(const orc_grid *g, int field, double *interior)
{
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i)
                interior[((long long)k * g->ny + j) * g->nx + i] = g->f[field][idx(g, i, j, k)];
}

void orc_get_raw(const orc_grid *g, int field, double *with_ghosts)
{
    memcpy(with_ghosts, g->f[field], (size_t)orc_ncells_total(g) * sizeof(double));
}

void orc_set_raw(orc_grid *g, int field, const double *with_ghosts)
{
    memcpy(g->f[field], with_ghosts, (size_t)orc_ncells_total(g) * sizeof(double));
}

void orc_get_info(const orc_grid *g, long long *out7)
{
    out7[0] = g->last_nsub; out7[1] = g->newton_fail_cells; out7[2] = g->newton_max_iters;
    out7[3] = g->newton_total_iters; out7[4] = g->bad_state_cells; out7[5] = g->fallback_states;
    out7[6] = g->guard_faces;
}

/* source index along one axis for a ghost index (PAPER.md:293,572 periodic; 464 outflow; 408 reflecting).
 * Outflow is read as zero-gradient: copy of the nearest interior cell (H15).
 * Reflecting: the mirror image about the wall, ghost -1 <- cell 0, -2 <- 1, n <- n-1, ... (B1). */
static int src_index(int i, int n, int bc)
{
    if (i >= 0 && i < n) return i;
    if (bc == ORC_BC_PERIODIC) { int m = i % n; if (m < 0) m += n; return m; }
    if (bc == ORC_BC_REFLECTING) {
        int m = i < 0 ? -1 - i : 2 * n - 1 - i;
        return m < 0 ? 0 : (m > n - 1 ? n - 1 : m);        /* boxes thinner than the ghost width */
    }
    return i < 0 ? 0 : n - 1;
}

/* vector component a field carries (0,1,2) or -1 for a scalar: at a reflecting wall normal to axis a the
 * a-component of the momentum and of the radiation flux changes sign in the image cell */
static int field_component(int field)
{
    switch (field) {
    case ORC_MX: case ORC_FX: return 0;
    case ORC_MY: case ORC_FY: return 1;
    case ORC_MZ: case ORC_FZ: return 2;
    default: return -1;
    }
}

int orc_set_face_bc(orc_grid *g, const int bc6[6])
{
    for (int a = 0; a < 3; ++a)
        if ((bc6[2 * a] == ORC_BC_PERIODIC) != (bc6[2 * a + 1] == ORC_BC_PERIODIC)) return 1;
    for (int f = 0; f < 6; ++f) g->face_bc[f] = bc6[f];
    return 0;
}

static void fill_one(orc_grid *g, double *a, int comp)
{
    /* every ghost cell (faces, edges, corners) <- the interior cell its three axis indices map to, each axis by the
     * rule of the face the index lies beyond; equivalent to filling x, then y, then z in sequence.  A ghost cell
     * beyond a FIXED face is left as the caller stored it. */
    const int n[3] = { g->nx, g->ny, g->nz };
    const long long ntot = orc_ncells_total(g);
#pragma omp parallel for collapse(3) schedule(static) if (ntot > ORC_OMP_MIN)
    for (int k = -ORC_NG; k < g->nz + ORC_NG; ++k)
        for (int j = -ORC_NG; j < g->ny + ORC_NG; ++j)
            for (int i = -ORC_NG; i < g->nx + ORC_NG; ++i) {
                const int idx3[3] = { i, j, k };
                int src[3], fixed = 0, flip = 0, ghost = 0;
                for (int ax = 0; ax < 3; ++ax) {
                    int v = idx3[ax];
                    src[ax] = v;
                    if (v >= 0 && v < n[ax]) continue;
                    ghost = 1;
                    int bc = g->face_bc[2 * ax + (v < 0 ? 0 : 1)];
                    if (bc == ORC_BC_FIXED) { fixed = 1; continue; }
                    src[ax] = src_index(v, n[ax], bc);
                    if (bc == ORC_BC_REFLECTING && comp == ax) flip = !flip;
                }
                if (!ghost || fixed) continue;
                double val = a[idx(g, src[0], src[1], src[2])];
                a[idx(g, i, j, k)] = flip ? -val : val;
            }
}

void orc_fill_field(orc_grid *g, int field) { fill_one(g, g->f[field], field_component(field)); }

void orc_fill_boundary(orc_grid *g, int which)
{
    if (which & ORC_FILL_HYDRO) for (int f = ORC_RHO; f <= ORC_E; ++f) fill_one(g, g->f[f], field_component(f));
    if (which & ORC_FILL_RAD)   for (int f = ORC_ER; f <= ORC_FZ; ++f) fill_one(g, g->f[f], field_component(f));
    if (which & 4)              for (int f = ORC_KP; f <= ORC_KR; ++f) fill_one(g, g->f[f], -1);
}

/* eq 21: dt = CFL dx / max(|v| + c_s), |v| the vector magnitude
 * (PAPER.md:142).  If c_hat > 0 the result is also limited so that the number of
 * radiation substeps stays <= N_sub,max: dt <= nsub_max CFL dx / c_hat. */
double orc_cfl_dt(orc_grid *g)
{
    double smax = 0.0;
    long long bad = 0;
    const long long ntot = orc_ncells_total(g);
#pragma omp parallel for collapse(3) schedule(static) reduction(max : smax) reduction(+ : bad) if (ntot > ORC_OMP_MIN)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                long long c = idx(g, i, j, k);
                double U[5] = { g->f[ORC_RHO][c], g->f[ORC_MX][c], g->f[ORC_MY][c], g->f[ORC_MZ][c], g->f[ORC_E][c] };
                double W[5];
                orc_cons_to_prim(g->gamma, U, W);
                if (!(W[0] > 0.0) || !(W[4] > 0.0)) { ++bad; continue; }
                double vmag = sqrt((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]);
                double cs = sqrt(g->gamma * W[4] / W[0]);
                double s = vmag + cs;
                if (s > smax) smax = s;
            }
    g->bad_state_cells = bad;
    if (bad) return NAN;
    double dt = g->cfl * g->dx / smax;
    if (g->c_hat > 0.0) {
        double dtr = (double)g->nsub_max * (g->cfl * g->dx / g->c_hat);
        if (dtr < dt) dt = dtr;
    }
    return dt;
}

/* number of radiation substeps for a hydro step dt */
int orc_nsub_for(const orc_grid *g, double dt)
{
    double ratio = dt * g->c_hat / (g->cfl * g->dx);
    int n = (int)ceil(ratio * (1.0 - 1e-12));
    return n < 1 ? 1 : n;
}

int orc_rad_step(orc_grid *g, double dt)
{
    int rc = orc_rad_transport(g, dt);
    if (rc) return rc;
    return orc_exchange(g, dt);                 /* once per subcycle */
}

/* operator-split cycle: hydro, then N_sub x (transport, exchange) */
int orc_rhd_step(orc_grid *g, double dt)
{
    int nsub = orc_nsub_for(g, dt);
    if (nsub > g->nsub_max) return 1;
    int rc = orc_hydro_step(g, dt);
    if (rc) return rc;
    double dts = dt / (double)nsub;
    long long fail = 0, tot = 0, fb = 0, gf = 0; int mx = 0;
    for (int s = 0; s < nsub; ++s) {
        rc = orc_rad_step(g, dts);
        fail += g->newton_fail_cells; tot += g->newton_total_iters;
        fb += g->fallback_states; gf += g->guard_faces;
        if (g->newton_max_iters > mx) mx = g->newton_max_iters;
        if (rc) break;
    }
    g->last_nsub = nsub; g->newton_fail_cells = fail; g->newton_total_iters = tot;
    g->newton_max_iters = mx; g->fallback_states = fb; g->guard_faces = gf;
    (void)sx; (void)sy; (void)sz;
    return rc;
}
