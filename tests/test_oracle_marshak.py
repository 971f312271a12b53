"""The paper's Marshak wave on the oracle, with every printed parameter: rho = 10, kappa_P = kappa_R =
577, T_0 = 1e4 K, a half-isotropic inflow of radiation temperature 3.481334e6 K at the left face, C_v = alpha T^3 with
alpha = 4 a_r / epsilon, epsilon = 1 (eq 55), domain [0, 3.466205e-3] cm = 20 mean free paths, N_x = 400, c_hat = c, run to
t = tau / (epsilon c rho kappa) with tau = 10.

The paper compares with the Su & Olson (1996) semi-analytic solution OF THE DIFFUSION APPROXIMATION "in the region where
F_r << c E_r".  Those tables are not in this container and are not reproduced; the same diffusion problem is instead
solved here by an independent finite-difference solver (`diffusion_reference`, Crank-Nicolson; it shares nothing with
the oracle): with u = E_r / a_r T_H^4, v = (T / T_H)^4, x in mean free paths, t in 1/(c rho kappa),

    u_t = u_xx / 3 + (v - u),    v_t = epsilon (u - v),    u - (2/3) u_x = 1 at x = 0  (Marshak condition: the incoming
    partial current (c/4) E_r + F_r/2 equals that of the hohlraum, with F_r = -(c/3) dE_r/dx),  u -> 0 far away.

Reading B3: the paper does not say how the "half-isotropic flux with a radiation temperature" is imposed.
Here the cells beyond the face are Dirichlet cells (QK_BC_FIXED) that hold the hohlraum's radiation, E_r = a_r T_H^4,
F_r = 0.  That reading lands within 1 % of the diffusion solution where the paper says the two should agree; the two
other obvious candidates do not (recorded below)."""
import numpy as np
from scipy.linalg import solve_banded

import oracle as O

C_LIGHT, A_RAD = 2.99792458e10, 7.5657e-15
RHO, KAPPA, T_INIT, T_HOHL, LENGTH, TAU_END = 10.0, 577.0, 1e4, 3.481334e6, 3.466205e-3, 10.0


def diffusion_reference(tau_end=TAU_END, xmax=40.0, n=4000, nt=4000, eps=1.0):
    """the diffusion problem of the header on a cell-centred grid, Crank-Nicolson in u with v advanced by the trapezoidal
    rule and eliminated; returns x (mean free paths), u, v"""
    dx, dt, D = xmax / n, tau_end / nt, 1.0 / 3.0
    x = (np.arange(n) + 0.5) * dx
    u, v = np.zeros(n), np.zeros(n)
    # left face: u_f - (2/3) u_x = 1 with u_f = u_0 - u_x dx/2  =>  u_x = (u_0 - 1) / (2/3 + dx/2); right face: u = 0
    aL = 1.0 / (2.0 / 3.0 + dx / 2.0)
    lo, up, di = np.full(n, -D / dx ** 2), np.full(n, -D / dx ** 2), np.full(n, 2 * D / dx ** 2)
    di[0], di[-1] = D / dx ** 2 + D * aL / dx, 3 * D / dx ** 2
    src = np.zeros(n)
    src[0] = D * aL / dx

    def L(w):                                   # minus the diffusion operator
        out = di * w
        out[1:] += lo[1:] * w[:-1]
        out[:-1] += up[:-1] * w[1:]
        return out
    h = 0.5 * eps * dt
    g = h / (1 + h)                             # v1 = A + g u1,  A = (v0 (1 - h) + h u0) / (1 + h)
    ab = np.zeros((3, n))
    ab[0, 1:], ab[2, :-1] = 0.5 * up[:-1], 0.5 * lo[1:]
    ab[1] = 1.0 / dt + 0.5 * di + 0.5 * (1 - g)
    for _ in range(nt):
        A = (v * (1 - h) + h * u) / (1 + h)
        u1 = solve_banded((1, 1), ab, u / dt - 0.5 * L(u) + src + 0.5 * (A + v - u))
        v = A + g * u1
        u = u1
    return x, u, v


def marshak_setup(N=400, reading="bath"):
    """raw fields (with ghost cells) and parameters; `reading` = what the cells beyond the left face hold:
    'bath' E_r = a T_H^4, F_r = 0 (B3);  'beam' E_r = a T_H^4, F_r = c E_r / 2;  'hemisphere' E_r = a T_H^4 / 2, F_r = c a T_H^4 / 4"""
    dx = LENGTH / N
    alpha = 4.0 * A_RAD                                         # epsilon = 1
    Einc, E0 = A_RAD * T_HOHL ** 4, A_RAD * T_INIT ** 4
    Eg, Fg = {"bath": (Einc, 0.0), "beam": (Einc, 0.5 * C_LIGHT * Einc), "hemisphere": (0.5 * Einc, 0.25 * C_LIGHT * Einc)}[reading]
    i = np.arange(-4, N + 4)
    one = np.ones(N + 8)
    raw = {0: RHO * one, 4: (alpha * T_INIT ** 4 / 4) * one, 5: np.where(i < 0, Eg, E0), 6: np.where(i < 0, Fg, 0.0),
           9: KAPPA * one, 10: KAPPA * one}
    raw = {f: np.ascontiguousarray(np.broadcast_to(raw.get(f, 0 * one), (9, 9, N + 8))) for f in range(11)}
    t_end = TAU_END / (C_LIGHT * RHO * KAPPA)
    nsteps = int(np.ceil(t_end / (0.4 * dx / C_LIGHT)))        # CFL 0.4, a whole number of equal steps
    return dict(N=N, dx=dx, alpha=alpha, raw=raw, dt=t_end / nsteps, nsteps=nsteps, Einc=Einc,
                x=(np.arange(N) + 0.5) * dx * RHO * KAPPA)


def run_oracle(reading="bath", N=400):
    s = marshak_setup(N, reading)
    g = O.Grid(N, 1, 1, s["dx"], 5.0 / 3.0, c_hat=C_LIGHT, c=C_LIGHT)
    g.set_constants(A_RAD, 1.0)
    g.set_params(cfl=0.4, flags=O.FLAG_STATIC_MATTER)
    g.set_eos(O.EOS_ALPHA_T3, s["alpha"])
    g.set_face_bc([O.BC_FIXED, O.BC_OUTFLOW, 0, 0, 0, 0])
    for f, a in s["raw"].items():
        g.set_raw(f, a)
    threads = O.get_threads()
    O.set_threads(1)                    # one row of cells
    try:
        for _ in range(s["nsteps"]):
            assert g.rad_step(s["dt"]) == 0
    finally:
        O.set_threads(threads)
    out = {k: g.get_state(f).ravel() for k, f in (("E", 4), ("Er", 5), ("Fx", 6))}
    info = g.info()
    g.close()
    return s, out, info


def marshak_deviation(s, out, ref):
    """u, v of a run and their relative deviation from the diffusion reference at the run's cell centres"""
    xr, ur, vr = ref
    u, v = out["Er"] / s["Einc"], out["E"] / (s["alpha"] * T_HOHL ** 4 / 4)
    return u, v, np.abs(u / np.interp(s["x"], xr, ur) - 1), np.abs(v / np.interp(s["x"], xr, vr) - 1)


def check_marshak(s, out, ref):
    """the pins shared with the GPU test"""
    u, v, du, dv = marshak_deviation(s, out, ref)
    x = s["x"]
    f = np.abs(out["Fx"]) / (C_LIGHT * out["Er"])
    near = x < 1.0
    assert f[near].max() < 0.26                                    # the region where diffusion is a fair approximation
    assert du[near][1:].max() < 0.012 and dv[near][1:].max() < 0.012, (du[near].max(), dv[near].max())
    assert du[0] < 0.03 and dv[0] < 0.03                           # the cell on the face: 2 %
    mid = x < 2.0
    assert du[mid].max() < 0.035 and dv[mid].max() < 0.04
    # ahead of x = c t = 10 mean free paths nothing has arrived (the diffusion solution has no such front)
    ahead = x > TAU_END + 1.5
    assert np.abs(out["Er"][ahead] / (A_RAD * T_INIT ** 4) - 1).max() < 1e-6
    assert np.all(np.diff(u) <= 0) and np.all(np.diff(u)[u[1:] > 1e-6] < 0)      # a monotone wave,
    assert np.all(v <= u * (1 + 1e-12))                                          # the gas lagging the radiation
    return du, dv


def test_diffusion_reference_is_converged_and_sane():
    x, u, v = diffusion_reference()
    x2, u2, v2 = diffusion_reference(n=8000, nt=8000)
    assert np.abs(np.interp(x, x2, u2) - u).max() < 2e-4 and np.abs(np.interp(x, x2, v2) - v).max() < 2e-4
    assert np.all(np.diff(u) < 0) and np.all(v <= u) and 0 < u[0] < 1
    # long after the wave has passed everything sits at the hohlraum temperature: u = v = 1 solves the problem
    xs, us, vs = diffusion_reference(tau_end=2000.0, xmax=5.0, n=100, nt=4000)
    assert us[0] > 0.8 and vs[0] > 0.8          # (a 5 mfp slab with u = 0 behind it stays below 1: only the trend is asserted)
    # without coupling to the gas (eps = 0) and early on, the surface value follows from the Marshak condition: u(0) < 1
    x0, u0, v0 = diffusion_reference(eps=0.0)
    assert np.all(v0 == 0.0) and u0[0] < u[0] + 1.0


def test_marshak_wave_matches_the_diffusion_solution_where_it_should():
    ref = diffusion_reference()
    s, out, info = run_oracle("bath")
    assert s["nsteps"] == 500 and info["newton_fail_cells"] == 0 and info["fallback_states"] == 0
    du, dv = check_marshak(s, out, ref)
    # the two other candidate readings of "half-isotropic flux with a radiation temperature", for the record
    for reading, lo, hi in (("beam", 0.9, 1.3), ("hemisphere", 0.03, 0.07)):
        s2, out2, _ = run_oracle(reading)
        _, _, du2, _ = marshak_deviation(s2, out2, ref)
        assert lo < du2[s2["x"] < 1.0].max() < hi, (reading, du2[s2["x"] < 1.0].max())
