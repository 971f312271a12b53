// qk_math.cuh -- per-cell / per-face arithmetic of the cell update, device inline functions.
//
// Every formula is written in the evaluation order DESIGN.md section 3 fixes, and the library is
// built with -fmad=false (the paper needs it too), so that sums, products, IEEE
// divisions and square roots round exactly as stated there.  min/max are spelled as
// comparisons (a < b ? a : b) so that ties and signed zeros resolve by the written order.
//
// Citations: PAPER.md:<line> of /root/reference/PAPER.md; H*/R*/X* = readings in DESIGN.md.
#pragma once

#ifndef QK_HD
#ifdef __CUDACC__
#define QK_HD __host__ __device__ __forceinline__
#else
#define QK_HD inline
#endif
#endif

#include <math.h>

namespace qk {

QK_HD double lesser(double a, double b) { return a < b ? a : b; }
QK_HD double greater(double a, double b) { return a > b ? a : b; }
QK_HD double unit_clamp(double x) { return lesser(greater(x, 0.0), 1.0); }

// ---------------------------------------------------------------------------------------------
// Hydro
// ---------------------------------------------------------------------------------------------

struct Prim { double rho, vx, vy, vz, P; };

// Conserved -> primitive.  |v|^2 grouped (vx^2+vy^2)+vz^2 (H10).
QK_HD Prim cons_to_prim(double gamma, double rho, double mx, double my, double mz, double E)
{
    Prim w;
    w.rho = rho;
    w.vx = mx / rho;
    w.vy = my / rho;
    w.vz = mz / rho;
    const double v2 = (w.vx * w.vx + w.vy * w.vy) + w.vz * w.vz;
    const double ekin = 0.5 * rho * v2;
    w.P = (gamma - 1.0) * (E - ekin);
    return w;
}

// Monotonized-central slope of three cell averages (used at extrema).
QK_HD double mc_slope(double qW, double qC, double qE)
{
    const double dW = qC - qW, dE = qE - qC;
    if (dW * dE <= 0.0) return 0.0;
    const double dC = 0.5 * (qE - qW);
    const double bound = lesser(fabs(dC), lesser(2.0 * fabs(dW), 2.0 * fabs(dE)));
    return dC > 0.0 ? bound : -bound;
}

// PPM face states of cell j from the five averages q_{j-2..j+2} = (a, b, c, d, e):
// eq 22 interface values with mirror-symmetric brackets, three-cell clamp
// (H3), then the parabola check: extremum -> MC-limited line (H4), one-sided
// overshoot -> CW84 correction (H5).  qlo = state at j-1/2, qhi = state at j+1/2.
// eq 22 interface value between the cells m and p, with their outer neighbours mm (beyond m) and pp (beyond p)
QK_HD double ppm_interface(double mm, double m, double p, double pp)
{
    return (7.0 / 12.0) * (m + p) - (1.0 / 12.0) * (pp + mm);
}

// Limiting steps of PPM for one cell (b, c, d) given the two raw interface values of eq 22.
template <bool BRANCHLESS>
QK_HD void ppm_limit_t(double lo_face, double hi_face, double b, double c, double d, double &qlo, double &qhi)
{
    const double floor3 = lesser(b, lesser(c, d));
    const double ceil3 = greater(b, greater(c, d));
    lo_face = lesser(greater(lo_face, floor3), ceil3);
    hi_face = lesser(greater(hi_face, floor3), ceil3);
    const double below = c - lo_face, above = hi_face - c;
    if (BRANCHLESS) {
    // same values as the branches below, written as selects so that the variables of a cell
    // interleave in the fp64 pipe (no divergent control flow)
    const double s = mc_slope(b, c, d);
    const bool extremum = below * above <= 0.0;
    const double ab = fabs(below), aa = fabs(above);
    const bool fix_lo = ab >= 2.0 * aa;
    const bool fix_hi = !fix_lo && (aa >= 2.0 * ab);
    const double lo_fix = c - 2.0 * above, hi_fix = c + 2.0 * below;
    const double lo_ext = c - 0.5 * s, hi_ext = c + 0.5 * s;
    qlo = extremum ? lo_ext : (fix_lo ? lo_fix : lo_face);
    qhi = extremum ? hi_ext : (fix_hi ? hi_fix : hi_face);
    return;
    }
    if (below * above <= 0.0) {
        const double s = mc_slope(b, c, d);
        lo_face = c - 0.5 * s;
        hi_face = c + 0.5 * s;
    } else if (fabs(below) >= 2.0 * fabs(above)) {
        lo_face = c - 2.0 * above;
    } else if (fabs(above) >= 2.0 * fabs(below)) {
        hi_face = c + 2.0 * below;
    }
    qlo = lo_face;
    qhi = hi_face;
}

template <bool BRANCHLESS>
QK_HD void ppm_face_states_t(double a, double b, double c, double d, double e, double &qlo, double &qhi)
{
    ppm_limit_t<BRANCHLESS>(ppm_interface(a, b, c, d), ppm_interface(b, c, d, e), b, c, d, qlo, qhi);
}

QK_HD void ppm_face_states(double a, double b, double c, double d, double e, double &qlo, double &qhi)
{
    ppm_face_states_t<false>(a, b, c, d, e, qlo, qhi);
}

// One-directional shock-flattening coefficient of cell j from the pressures P_{j-2..j+2}
// and the normal velocities at j-1, j+1 (constants are reading H6).
QK_HD double flatten_coeff_1d(double gamma, double Pm2, double Pm1, double P0, double Pp1, double Pp2,
                              double vn_m1, double vn_p1)
{
    if (!(vn_p1 < vn_m1)) return 1.0;          // expanding flow: nothing below is needed
    const double near = fabs(Pp1 - Pm1);
    // Weak jump: near < 0.2499 gamma P0 makes near / (gamma P0) < 0.25, hence (0.75 - strength) / 0.5 > 1, its
    // clamp exactly 1 and the result max(steep, 1) = 1 whatever `steep` is -- the value the full evaluation
    // below returns, without its three divisions.  (Only genuine shocks get past this line.)
    if (near < 0.2499 * (gamma * P0)) return 1.0;
    const double far = fabs(Pp2 - Pm2);
    double steep;
    if (far == 0.0) steep = (near == 0.0) ? 1.0 : 0.0;
    else            steep = unit_clamp((0.85 - near / far) / 0.10);
    const double strength = near / (gamma * P0);
    return greater(steep, unit_clamp((0.75 - strength) / 0.5));
}

// HLLC flux with Toro's PVRS wave speeds.  States are (rho, u_n, u_t1, u_t2, p);
// the flux comes back as (mass, normal, t1, t2 momentum, energy).
struct Flux5 { double m, pn, pt1, pt2, e; };

QK_HD Flux5 hllc_flux(double gamma, double rL, double uL, double vL, double wL, double pL,
                      double rR, double uR, double vR, double wR, double pR)
{
    const double aL = sqrt(gamma * pL / rL), aR = sqrt(gamma * pR / rR);
    const double rho_bar = 0.5 * (rL + rR), a_bar = 0.5 * (aL + aR);
    const double p_pvrs = 0.5 * (pL + pR) - 0.5 * (uR - uL) * rho_bar * a_bar;
    const double p_star = greater(0.0, p_pvrs);
    const double g2 = (gamma + 1.0) / (2.0 * gamma);
    const double qL = (p_star <= pL) ? 1.0 : sqrt(1.0 + g2 * (p_star / pL - 1.0));
    const double qR = (p_star <= pR) ? 1.0 : sqrt(1.0 + g2 * (p_star / pR - 1.0));
    const double SL = uL - aL * qL, SR = uR + aR * qR;
    const double mdotL = rL * (SL - uL), mdotR = rR * (SR - uR);
    const double S_star = (pR - pL + uL * mdotL - uR * mdotR) / (mdotL - mdotR);

    // upwind side K and whether the star region is crossed:
    // F_L (S_L >= 0) | F*_L (S* >= 0) | F*_R (S_R > 0) | F_R
    bool from_left, star;
    if (SL >= 0.0)          { from_left = true;  star = false; }
    else if (S_star >= 0.0) { from_left = true;  star = true;  }
    else if (SR > 0.0)      { from_left = false; star = true;  }
    else                    { from_left = false; star = false; }

    const double r = from_left ? rL : rR, u = from_left ? uL : uR, v = from_left ? vL : vR;
    const double w = from_left ? wL : wR, p = from_left ? pL : pR, SK = from_left ? SL : SR;
    const double E = p / (gamma - 1.0) + 0.5 * r * (u * u + (v * v + w * w));
    const double Um = r, Upn = r * u, Upt1 = r * v, Upt2 = r * w;
    Flux5 F;
    F.m = r * u;
    F.pn = r * u * u + p;
    F.pt1 = r * u * v;
    F.pt2 = r * u * w;
    F.e = u * (E + p);
    if (star) {
        const double ratio = (SK - u) / (SK - S_star);
        const double Sm = ratio * r;
        const double Spn = ratio * (r * S_star);
        const double Spt1 = ratio * Upt1;
        const double Spt2 = ratio * Upt2;
        const double Se = ratio * (E + (S_star - u) * (r * S_star + p / (SK - u)));
        F.m = F.m + SK * (Sm - Um);
        F.pn = F.pn + SK * (Spn - Upn);
        F.pt1 = F.pt1 + SK * (Spt1 - Upt1);
        F.pt2 = F.pt2 + SK * (Spt2 - Upt2);
        F.e = F.e + SK * (Se - E);
    }
    return F;
}

// ---------------------------------------------------------------------------------------------
// Radiation transport
// ---------------------------------------------------------------------------------------------

// Levermore (1984) Eddington factor, eq 24.
QK_HD double eddington_factor(double f)
{
    const double f2 = f * f;
    return (3.0 + 4.0 * f2) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f2));
}

// Minerbo (1978) closure in its customary polynomial form (V3): chi(0) = 1/3, chi(1) = 1.
QK_HD double minerbo_factor(double f)
{
    const double f2 = f * f;
    return 1.0 / 3.0 + (2.0 / 15.0) * (f2 * ((3.0 - f) + 3.0 * f2));
}

// Physical flux of the face state (E, f_x, f_y, f_z) through a face with normal n (0,1,2):
// (c_hat/c) F_n for E_r and c c_hat E_r T_in for F_i (eq 11-12), with
// T = (1-chi)/2 I + (3chi-1)/2 n n (eq 23), |f| clamped to 1 for the closure only (R4),
// n = f/|f| (eq 25), isotropic when f = 0.  Returns T_nn in Tnn.
struct Rad4 { double e, x, y, z; };

// CL = closure: 0 Levermore (eq 24), 1 Eddington approximation chi = 1/3 (the n n term vanishes),
// 2 Minerbo
template <int CL = 0>
QK_HD Rad4 rad_physical_flux(double c, double c_hat, double E, double fx, double fy, double fz, int n,
                             double &Tnn)
{
    const double fsq = (fx * fx + fy * fy) + fz * fz;
    const double fmag = CL == 1 ? 0.0 : sqrt(fsq);
    const double chi = CL == 1 ? 1.0 / 3.0 : (CL == 2 ? minerbo_factor(lesser(fmag, 1.0)) : eddington_factor(lesser(fmag, 1.0)));
    const double iso = 0.5 * (1.0 - chi), aniso = 0.5 * (3.0 * chi - 1.0);
    double Tx = (n == 0) ? iso : 0.0, Ty = (n == 1) ? iso : 0.0, Tz = (n == 2) ? iso : 0.0;
    if (fmag > 0.0) {
        const double nx = fx / fmag, ny = fy / fmag, nz = fz / fmag;
        const double nn = (n == 0) ? nx : ((n == 1) ? ny : nz);
        Tx = Tx + aniso * (nx * nn);
        Ty = Ty + aniso * (ny * nn);
        Tz = Tz + aniso * (nz * nn);
    }
    const double fn = (n == 0) ? fx : ((n == 1) ? fy : fz);
    const double Fn = (c * E) * fn;
    const double cc = (c * c_hat) * E;
    Rad4 G;
    G.e = (c_hat / c) * Fn;
    G.x = cc * Tx;
    G.y = cc * Ty;
    G.z = cc * Tz;
    Tnn = (n == 0) ? Tx : ((n == 1) ? Ty : Tz);
    return G;
}

// HLL flux between face states L and R = (E, f) with S_R = -S_L = S =
// max(c_hat sqrt(Tnn_L), c_hat sqrt(Tnn_R), 0.1 c_hat) (R5); the E_r
// dissipation is scaled by min(1, 1/tau_face) (R6) unless a star state it
// implies is non-causal.  `guard` is set to 1 when the correction was disabled for the face.
template <int CL = 0>
QK_HD Rad4 rad_hll_flux(double c, double c_hat, double EL, double fxL, double fyL, double fzL,
                        double ER, double fxR, double fyR, double fzR, int n, double tau_face,
                        bool tau_corr, int &guard)
{
    double TL, TR;
    const Rad4 GL = rad_physical_flux<CL>(c, c_hat, EL, fxL, fyL, fzL, n, TL);
    const Rad4 GR = rad_physical_flux<CL>(c, c_hat, ER, fxR, fyR, fzR, n, TR);
    const double S = greater(greater(c_hat * sqrt(TL), c_hat * sqrt(TR)), 0.1 * c_hat);
    const double FxL = (c * EL) * fxL, FyL = (c * EL) * fyL, FzL = (c * EL) * fzL;
    const double FxR = (c * ER) * fxR, FyR = (c * ER) * fyR, FzR = (c * ER) * fzR;
    const double half_S = 0.5 * S;
    Rad4 G;
    G.x = 0.5 * (GL.x + GR.x) - half_S * (FxR - FxL);
    G.y = 0.5 * (GL.y + GR.y) - half_S * (FyR - FyL);
    G.z = 0.5 * (GL.z + GR.z) - half_S * (FzR - FzL);
    double eps = 1.0;
    if (tau_corr) eps = lesser(1.0, 1.0 / tau_face);
    G.e = 0.5 * (GL.e + GR.e) - (eps * half_S) * (ER - EL);
    guard = 0;
    if (eps < 1.0) {
        const double EsL = EL + (G.e - GL.e) / (-S), EsR = ER + (G.e - GR.e) / S;
        const double xL = FxL + (G.x - GL.x) / (-S), xR = FxR + (G.x - GR.x) / S;
        const double yL = FyL + (G.y - GL.y) / (-S), yR = FyR + (G.y - GR.y) / S;
        const double zL = FzL + (G.z - GL.z) / (-S), zR = FzR + (G.z - GR.z) / S;
        const double F2L = (xL * xL + yL * yL) + zL * zL;
        const double F2R = (xR * xR + yR * yR) + zR * zR;
        const double cEL = c * EsL, cER = c * EsR;
        const bool acausal = !(EsL > 0.0) || !(EsR > 0.0) || (F2L > cEL * cEL) || (F2R > cER * cER);
        if (acausal) {
            G.e = 0.5 * (GL.e + GR.e) - half_S * (ER - EL);
            guard = 1;
        }
    }
    return G;
}

// ---------------------------------------------------------------------------------------------
// Matter-radiation exchange (eq 26-43)
// ---------------------------------------------------------------------------------------------

// (T/T0)^(n2/2), integer n2: repeated multiplication, one square root for odd n2, one division for n2 < 0 --
// no pow(), so the bits are reproducible (X14)
QK_HD double temperature_power(double T, double T0, int n2)
{
    const int a = n2 < 0 ? -n2 : n2;
    const double q = T / T0;
    double p = 1.0;
    for (int m = 0; m < a / 2; ++m) p = p * q;
    if (a & 1) p = p * sqrt(q);
    return n2 < 0 ? 1.0 / p : p;
}

// density part kappa0 (rho/rho0)^e of the opacity law, integer e
QK_HD void opacity_density_part(double rho, double kP0, double kR0, double rho0, int e, double &kP, double &kR)
{
    const double q = e < 0 ? rho0 / rho : rho / rho0;
    const int n = e < 0 ? -e : e;
    double kp = kP0, kr = kR0;
    for (int m = 0; m < n; ++m) { kp = kp * q; kr = kr * q; }
    kP = kp; kR = kr;
}

struct ExchangeConsts {
    double c, c_hat, a_rad, kB_mu, gamma, tol;
    // kappa(rho, T) law (qk_set_opacity_law_T): kappa_P follows the Newton iterate's temperature with the
    // d kappa_P/dT term of eq 33; kappa_F ~ kappa_R is taken at the updated temperature
    bool kappa_T;
    int texp2, opac_exp;
    double T0, kP0, kR0, rho0;
    double alpha;          // eos_alpha_t3: E_g = alpha T^4 / 4, C_v = alpha T^3 (eq 55)
    bool eos_alpha_t3;
    int maxit;
    bool literal_stop, static_matter;
};

// The decision |x / y| < tol of eq 36-37, taken without the division wherever it cannot matter: with
// b = fl(tol |y|) = tol |y| (1 + d), |d| <= 2^-53 (b normal), |x| < b/2 implies fl(|x|/|y|) <= tol (1 + d)(1 + d')/2 < tol
// and |x| > 2b implies fl(|x|/|y|) >= 2 tol (1 - 2^-52) > tol (rounding is monotone); only inside the factor-4 band
// around the threshold -- or when b is not a normal positive number (y zero, tiny, NaN; tol <= 0) -- is the quotient
// formed.  Same decision as fabs(x / y) < tol for every input; saves two of the seven divisions of a Newton iteration.
QK_HD bool below_tolerance(double x, double y, double tol)
{
    const double a = fabs(x), b = tol * fabs(y);
    if (b >= 1e-290) {
        if (a < 0.5 * b) return true;
        if (a > 2.0 * b) return false;
    }
    return fabs(x / y) < tol;
}

// Backward-Euler update of one cell over dt.  In/out: m (gas momentum), E, Er, F.  Returns 0,
// 4 (Newton cap reached) or 5 (non-positive E_g or E_r afterwards); iters = Newton updates.
template <bool KT>
QK_HD int exchange_cell(const ExchangeConsts &k, double dt, double rho, double &mx, double &my, double &mz,
                        double &E, double &Er, double &Fx, double &Fy, double &Fz, double kappaP, double kappaR,
                        double S, int &iters)
{
    const double c_ratio = k.c / k.c_hat;
    const double m2_old = (mx * mx + my * my) + mz * mz;
    const double Ekin_old = 0.5 * m2_old / rho;
    const double Eg_old = E - Ekin_old;
    const double Er_old = Er;
    const double Etot = Eg_old + c_ratio * (Er_old + S);        // eq 38
    double coef = dt * rho * kappaP * k.c_hat;                  // dt rho kappa_P c_hat (X1)
    const double Cv_ideal = rho * k.kB_mu / (k.gamma - 1.0);    // volumetric heat capacity (X2)
    double Eg = Eg_old, Erad = Er_old;
    int it = 0;
    bool finished = false;
    while (it < k.maxit) {
        double T, Cv;
        if (k.eos_alpha_t3) {                                             // eq 55
            T = sqrt(sqrt(4.0 * Eg / k.alpha));
            Cv = k.alpha * (T * T * T);
        } else {
            Cv = Cv_ideal;
            T = Eg / Cv;
        }
        const double T2 = T * T;
        const double T4 = T2 * T2;
        double dcoef_dT = 0.0;
        if (KT) {
            const double kPT = kappaP * temperature_power(T, k.T0, k.texp2);
            coef = dt * rho * kPT * k.c_hat;
            const double dkP_dT = (0.5 * (double)k.texp2) * kPT / T;
            dcoef_dT = dt * rho * dkP_dT * k.c_hat;
        }
        const double R = coef * (k.a_rad * T4 - Erad);                    // eq 28 (X1)
        const double FG = (Eg - Eg_old) + c_ratio * R;                    // eq 26
        const double FR = (Erad - Er_old) - (R + S);                      // eq 27
        const bool converged = below_tolerance(FG, Etot, k.tol) && below_tolerance(c_ratio * FR, Etot, k.tol);  // eq 36-37
        if (converged && k.literal_stop) { finished = true; break; }
        double dR_dEg = coef * (4.0 * k.a_rad * (T2 * T)) / Cv;           // eq 33 with d kappa/dT = 0
        if (KT) dR_dEg = (coef * (4.0 * k.a_rad * (T2 * T)) + dcoef_dT * (k.a_rad * T4 - Erad)) / Cv;   // eq 33
        const double dFG_dEg = 1.0 + c_ratio * dR_dEg;                    // eq 29
        const double dFG_dEr = -(c_ratio * coef);                         // eq 30
        const double dFR_dEg = -dR_dEg;                                   // eq 31
        const double dFR_dEr = 1.0 + coef;                                // eq 32
        const double eta = -dFR_dEg / dFG_dEg;
        const double dEr = -(FR + eta * FG) / (dFR_dEr + eta * dFG_dEr);  // eq 34
        const double dEg = -(FG + dEr * dFG_dEr) / dFG_dEg;               // eq 35
        Erad = Erad + dEr;
        Eg = Eg + dEg;
        ++it;
        if (converged) { finished = true; break; }                        // converge-then-polish (X5)
    }
    int rc = finished ? 0 : 4;
    iters = it;
    // eq 39-41 with kappa_F ~ kappa_R, at the updated gas temperature
    if (KT) {
        const double T = k.eos_alpha_t3 ? sqrt(sqrt(4.0 * Eg / k.alpha)) : Eg / Cv_ideal;
        kappaR = kappaR * temperature_power(T, k.T0, k.texp2);
    }
    const double damp = 1.0 + rho * kappaR * k.c_hat * dt;
    const double Fx1 = Fx / damp, Fy1 = Fy / damp, Fz1 = Fz / damp;
    if (k.static_matter) {                                                // PAPER.md:440 (X11)
        E = Eg + Ekin_old;
        Er = Erad;
    } else {
        const double mx1 = mx - (Fx1 - Fx) / (k.c_hat * k.c);
        const double my1 = my - (Fy1 - Fy) / (k.c_hat * k.c);
        const double mz1 = mz - (Fz1 - Fz) / (k.c_hat * k.c);
        const double m2_new = (mx1 * mx1 + my1 * my1) + mz1 * mz1;
        const double dEkin = 0.5 * (m2_new - m2_old) / rho;
        E = Eg + (Ekin_old + dEkin);                                      // eq 42
        Er = Erad - (k.c_hat / k.c) * dEkin;                              // eq 43
        mx = mx1; my = my1; mz = mz1;
    }
    Fx = Fx1; Fy = Fy1; Fz = Fz1;
    if (!(Eg > 0.0) || !(Er > 0.0)) rc = rc ? rc : 5;
    return rc;
}

}  // namespace qk
