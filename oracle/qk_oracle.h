/* qk_oracle.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow fp64 C restatement of the per-timestep uniform-grid
 * cell update of Wibking & Krumholz, "QUOKKA" (arXiv:2110.01792), written from
 * /root/reference/PAPER.md (cited below as PAPER.md:<line>) and from the readings
 * listed in DESIGN.md section 3.  It exists so that the CUDA path can be checked
 * against something that is not itself.  It shares no code with the CUDA path and
 * neither includes nor links anything under paper_2110_01792_b200/.  Only tests/,
 * __graft_entry__.smoke() and the cpu_baseline / --impl reference legs of bench.py
 * may load it.  Build: gcc -O2 -ffp-contract=off (no FMA contraction).
 *
 * Pins (tests/test_oracle_*.py) and which function each pins:
 *   orc_ppm_faces, orc_hllc, orc_hydro_step : sound-wave errors printed at PAPER.md:299,
 *        stationary contact, Sod vs exact Riemann solution, advected
 *        wave order, conservation, equilibrium invariance, x<->y symmetry
 *   orc_closure                             : chi(0)=1/3, chi(1)=1, trace T = 1
 *   orc_plm_faces (ORC_FLAG_PLM)            : exact on linear data, zero slope at extrema, second-order
 *        advected wave, conservation, contact preservation
 *   ORC_FLAG_EDDINGTON                      : T = I/3 for every f; linear wave speed c_hat/sqrt(3)
 *   orc_rad_step (transport)                : linear wave speed c_hat/sqrt(3), streaming
 *        top-hat causality/positivity, conservation, split-diffusion factor
 *   orc_exchange_cell                       : eq 57 relaxation to 1e-5,
 *        bisection solution of the backward-Euler quartic, F_r decay closed form
 *   default radiation flux (plain HLL, eps = 1)     : the radiation pressure tube, "better than 0.2 per cent"
 *        (PAPER.md:484-494), which the opt-in optical-depth correction (ORC_FLAG_TAU_CORR, reading R6) misses
 *   kappa(rho, T), eq 33 with d kappa_P/dT           : bisection of the backward-Euler scalar equation, Newton
 *        iteration counts against the Jacobian without the term, kappa_F at the updated temperature
 *   PARITY UNPINNED (oracle<->GPU agreement only): the shock-flattening
 *        constants (PAPER.md:166 prints no formula), the VALUE 0.1 of the wavespeed floor (its reach is pinned:
 *        it binds only for |f| > 0.99 grazing the face), the form of the opt-in optical-depth correction and of
 *        its causality guard (PAPER.md:180-182 print no formula), the Minerbo polynomial (literature form).
 */
#ifndef QK_ORACLE_H
#define QK_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_NG 4          /* ghost zones per side (BASELINE.json config 1) */
#define ORC_NFIELDS 12    /* rho mx my mz E Er Fx Fy Fz kappaP kappaR src  */
#define ORC_OMP_MIN 4096  /* boxes (ghosts included) below this many cells stay on one thread: the `omp parallel for`
                             lines deal independent cells out to threads and change no result */

enum { ORC_RHO = 0, ORC_MX, ORC_MY, ORC_MZ, ORC_E, ORC_ER, ORC_FX, ORC_FY, ORC_FZ,
       ORC_KP, ORC_KR,
       ORC_SRC };   /* radiation energy source rate per cell: S of eq 27 is dt * src (reading X13) */
enum { ORC_BC_PERIODIC = 0, ORC_BC_OUTFLOW = 1,
       ORC_BC_REFLECTING = 2,
       ORC_BC_FIXED = 3 };       /* Dirichlet: the ghost cells keep the values the caller stored (orc_set_raw);
                                    PAPER.md:492, 518, 528; inflow boundaries 422, 464, 476 (B2) */  /* solid wall: mirror image, normal momentum / flux component negated */
enum { ORC_FLAG_TAU_CORR = 1, ORC_FLAG_STATIC_MATTER = 2, ORC_FLAG_NEWTON_LITERAL = 4,
       ORC_FLAG_PLM = 8,          /* piecewise-linear reconstruction with the MC limiter */
       ORC_FLAG_EDDINGTON = 16,   /* Eddington approximation chi = 1/3 (P_r = E_r/3)  */
       ORC_FLAG_MINERBO = 32,     /* Minerbo (1978) closure in its usual polynomial form
                                     chi = 1/3 + (2/15) f^2 (3 - f + 3 f^2): approximate, NOT printed in PAPER.md (V3) */
       ORC_FLAG_NO_DKAPPA_DT = 64 }; /* oracle only: drop the d kappa_P/dT term of eq 33 from the Jacobian (the pin that
                                        shows the term speeds up Newton's iteration compares against this) */
enum { ORC_EOS_IDEAL = 0, ORC_EOS_ALPHA_T3 = 1 };   /* eq 55, PAPER.md:424 (oracle only) */
enum { ORC_FILL_HYDRO = 1, ORC_FILL_RAD = 2, ORC_FILL_ALL = 7 }; /* bit 4: opacities */

typedef struct orc_grid {
    int nx, ny, nz;                 /* interior cells                                  */
    double dx, gamma, c_hat, c;
    int bc;                         /* boundary given to orc_create: all six faces       */
    int face_bc[6];                 /* per face: x-lo, x-hi, y-lo, y-hi, z-lo, z-hi      */
    double a_rad, kB_mu;            /* radiation constant, k_B/(mu m_H)                */
    double cfl, newton_tol;
    int newton_maxit, nsub_max;
    unsigned flags;
    int opac_exp; double opac_kP0, opac_kR0, opac_rho0;   /* opacity law (orc_set_opacity_law), opac_rho0 = 0: fields */
    int opac_texp2; double opac_T0;                       /* ... times (T/T0)^(opac_texp2/2) (orc_set_opacity_law_T)  */
    double s_floor;                                       /* HLL wavespeed floor / c_hat (reading R5: 0.1)           */
    int eos; double alpha;          /* ORC_EOS_ALPHA_T3: E_g = alpha T^4 / 4           */
    double S_src;                   /* S of eq 27 for the cell orc_exchange_cell is called on; orc_exchange sets it
                                       to dt * f[ORC_SRC][cell] (0 in every BASELINE config)                  */
    double *f[ORC_NFIELDS];         /* (nz+8)(ny+8)(nx+8) each, x fastest              */
    /* diagnostics of the last call */
    int last_nsub;
    long long newton_fail_cells;
    int newton_max_iters;
    long long newton_total_iters;
    long long bad_state_cells;
    long long fallback_states;      /* first-order fallbacks            */
    long long guard_faces;          /* faces where the tau correction was disabled     */
} orc_grid;

orc_grid *orc_create(int nx, int ny, int nz, double dx, double gamma, double c_hat, double c, int bc);
void   orc_destroy(orc_grid *g);
long long orc_ncells_total(const orc_grid *g);
void   orc_set_constants(orc_grid *g, double a_rad, double kB_mu);
void   orc_set_params(orc_grid *g, double cfl, double newton_tol, int newton_maxit, int nsub_max, unsigned flags);
void   orc_set_eos(orc_grid *g, int eos, double alpha);
void   orc_set_opacity_law(orc_grid *g, double kP0, double kR0, double rho0, int exponent);
void   orc_set_opacity_law_T(orc_grid *g, double kP0, double kR0, double rho0, int exponent, double T0, int texp2);
void   orc_set_wavespeed_floor(orc_grid *g, double s_floor);
void   orc_set_threads(int n);
int    orc_get_threads(void);
int    orc_set_face_bc(orc_grid *g, const int bc6[6]);   /* 0 ok, 1 if periodic is not on both faces of an axis */
void   orc_set_field(orc_grid *g, int field, const double *interior);
void   orc_get_field(const orc_grid *g, int field, double *interior);
void   orc_get_raw(const orc_grid *g, int field, double *with_ghosts);
void   orc_set_raw(orc_grid *g, int field, const double *with_ghosts);
void   orc_get_info(const orc_grid *g, long long *out7);

void   orc_fill_boundary(orc_grid *g, int which);
void   orc_fill_field(orc_grid *g, int field);
double orc_cfl_dt(orc_grid *g);
int    orc_hydro_step(orc_grid *g, double dt);
int    orc_rad_transport(orc_grid *g, double dt);      /* RK2 transport only          */
int    orc_exchange(orc_grid *g, double dt);           /* eq 26-43 over all cells     */
int    orc_rad_step(orc_grid *g, double dt);           /* transport + exchange        */
int    orc_rhd_step(orc_grid *g, double dt);
int    orc_nsub_for(const orc_grid *g, double dt);

/* building blocks, exported so the pins can reach them one by one */
void   orc_cons_to_prim(double gamma, const double U[5], double W[5]);
void   orc_ppm_faces(const double q[5], double *q_minus, double *q_plus);
void   orc_plm_faces(const double q[5], double *q_minus, double *q_plus);
void   orc_faces(unsigned flags, const double q[5], double *q_minus, double *q_plus);
double orc_mc_slope(double qm1, double q0, double qp1);
double orc_flatten_1d(double gamma, const double P[5], const double vn[5]);
void   orc_hllc(double gamma, const double WL[5], const double WR[5], double F[5]);
double orc_eddington_factor(double f);
double orc_minerbo_factor(double f);
void   orc_closure(const double fvec[3], int n, double T_col[3], double *chi_out);
void   orc_closure_k(unsigned flags, const double fvec[3], int n, double T_col[3], double *chi_out);
void   orc_rad_phys_flux(double c, double c_hat, const double S[4], int n, double G[4], double *Tnn);
int    orc_rad_hll(double c, double c_hat, const double SL[4], const double SR[4], int n,
                   double tau_face, unsigned flags, double G[4]);
int    orc_rad_hll_floor(double c, double c_hat, const double SL[4], const double SR[4], int n,
                         double tau_face, unsigned flags, double s_floor, double G[4]);
double orc_temp_power(double T, double T0, int n2);
void   orc_opacity_density_part(const orc_grid *g, double rho, double *kP, double *kR);
double orc_gas_temperature(const orc_grid *g, double rho, const double m[3], double E);
int    orc_exchange_cell(const orc_grid *g, double dt, double rho, double m[3], double *E,
                         double *Er, double F[3], double kP, double kR, int *iters);

#ifdef __cplusplus
}
#endif
#endif
