"""Pins for the matter-radiation exchange part of the CPU oracle (oracle/exchange.c).  CPU only."""
import numpy as np

import oracle as O

# cgs constants for the PAPER.md:444 problem
C_LIGHT = 2.99792458e10
A_RAD = 7.5657e-15


def _cell_grid(c, c_hat, gamma=5 / 3, flags=0, tol=1e-10):
    g = O.Grid(1, 1, 1, 1.0, gamma, c_hat=c_hat, c=c)
    g.set_params(newton_tol=tol, flags=flags)
    return g


def _cell(g, dt, rho, m, E, Er, F, kP, kR):
    L = O.lib()
    m = np.array(m, dtype=float); F = np.array(F, dtype=float)
    Ea, Era = np.array([E], dtype=float), np.array([Er], dtype=float)
    it = np.zeros(1, dtype=np.int32)
    rc = L.orc_exchange_cell(g.h, dt, rho, m, Ea, Era, F, kP, kR, it)
    return rc, m, Ea[0], Era[0], F, int(it[0])


def test_relaxation_matches_eq57():
    """rho=1e-7, kappa_P=1, E_r=1e12, E_g=1e2, C_v = alpha T^3 (eq 55),
    dt=1e-8: T(t) agrees with eq 57 to better than 1e-5 at each step, with c_hat = 0.1 c and c;
    T_eq follows eq 58 and the RSLA/physical ratio is (2/(1+c_hat/c))^(1/4) for alpha = 4 a_r."""
    rho, kap, dt = 1e-7, 1.0, 1e-8
    alpha = 4.0 * A_RAD                       # eq 55 with epsilon = 1
    Teq = {}
    for ratio in (0.1, 1.0):
        c, ch = C_LIGHT, ratio * C_LIGHT
        g = _cell_grid(c, ch)
        g.set_constants(A_RAD, 1.0)
        g.set_eos(O.EOS_ALPHA_T3, alpha)
        Eg, Er = 1e2, 1e12
        E0 = Eg + (c / ch) * Er
        Et0 = E0 / (A_RAD + (ch / c) * alpha / 4.0)
        T0_4 = 4.0 * Eg / alpha
        lam = (4.0 / alpha) * (A_RAD + (ch / c) * alpha / 4.0) * kap * rho * c
        worst, t = 0.0, 0.0
        for n in range(150000):
            rc, _, Eg, Er, _, it = _cell(g, dt, rho, [0, 0, 0], Eg, Er, [0, 0, 0], kap, kap)
            assert rc == 0
            t += dt
            T4 = (T0_4 - (ch / c) * Et0) * np.exp(-lam * t) + (ch / c) * Et0      # eq 57
            T = (4.0 * Eg / alpha) ** 0.25
            worst = max(worst, abs(T / T4 ** 0.25 - 1.0))
            assert abs((Eg + (c / ch) * Er) / E0 - 1.0) < 1e-12
        assert worst < 1e-5, worst
        assert lam * t > 4.5
        Teq[ratio] = ((ch / c) * Et0) ** 0.25                                      # eq 58
        assert abs(T / Teq[ratio] - 1.0) < 1e-2
    assert abs(Teq[0.1] / Teq[1.0] - (2.0 / 1.1) ** 0.25) < 1e-9               # "approximately 20 per cent"


def test_backward_euler_quartic_by_bisection():
    """Ideal gas: eq 26-27 with S=0 conserve E_g + (c/c_hat)E_r, leaving one scalar quartic in T;
    its root by bisection must equal the Newton result."""
    rng = np.random.default_rng(6)
    gamma, c, ch, a = 5 / 3, 17.0, 1.7, 1.3
    g = _cell_grid(c, ch, gamma, flags=O.FLAG_STATIC_MATTER, tol=1e-10)
    g.set_constants(a, 0.9)
    for _ in range(40):
        rho = np.exp(rng.standard_normal()); T0 = np.exp(rng.standard_normal())
        Er0 = a * T0 ** 4 * np.exp(2 * rng.standard_normal())
        kap = 10 ** rng.uniform(-2, 3); dt = 10 ** rng.uniform(-3, 0)
        Cv = rho * 0.9 / (gamma - 1)
        Eg0 = Cv * T0
        rc, _, E1, Er1, _, it = _cell(g, dt, rho, [0, 0, 0], Eg0, Er0, [0, 0, 0], kap, 0.0)
        assert rc == 0 and it <= 20
        k = dt * rho * kap * ch
        tot = Eg0 + (c / ch) * Er0

        def resid(Eg):                       # F_R with E_r eliminated
            Er = (tot - Eg) * (ch / c)
            return (Er - Er0) - k * (a * (Eg / Cv) ** 4 - Er)
        lo, hi = 0.0, tot
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if resid(mid) > 0:               # resid decreases with Eg
                lo = mid
            else:
                hi = mid
        Eg_b = 0.5 * (lo + hi)
        assert abs(E1 - Eg_b) < 1e-12 * tot, (E1, Eg_b)
        assert abs((E1 + (c / ch) * Er1) - tot) < 1e-13 * tot


def test_flux_decay_and_momentum_exchange_closed_form():
    """eq 39-41: F^n = F^0/(1+rho kappa c_hat dt)^n and the gas gains (F^0-F^n)/(c c_hat)."""
    c, ch = 10.0, 2.0
    g = _cell_grid(c, ch)
    rho, kR, dt = 1.7, 3.0, 0.05
    m, F = np.array([0.1, -0.2, 0.3]), np.array([1.0, 2.0, -3.0])
    m0, F0 = m.copy(), F.copy()
    E, Er = 5.0, 4.0
    for n in range(1, 6):
        rc, m, E, Er, F, _ = _cell(g, dt, rho, m, E, Er, F, 0.0, kR)
        assert rc == 0
        assert np.allclose(F, F0 / (1 + rho * kR * ch * dt) ** n, rtol=1e-14)
        assert np.allclose(m, m0 + (F0 - F) / (c * ch), rtol=1e-14)
        assert np.allclose(m + F / (c * ch), m0 + F0 / (c * ch), rtol=1e-15)   # momentum conserved
    # kappa_P = 0: internal energy untouched, work term moves energy between E and E_r (eq 42-43)
    Ekin0 = 0.5 * (m0 @ m0) / rho
    Ekin = 0.5 * (m @ m) / rho
    assert abs((E - Ekin) - (5.0 - Ekin0)) < 1e-14
    assert abs((E + (c / ch) * Er) - (5.0 + (c / ch) * 4.0)) < 1e-13


def test_static_matter_flag_keeps_gas_at_rest():
    g = _cell_grid(1.0, 0.1, flags=O.FLAG_STATIC_MATTER)
    rc, m, E, Er, F, _ = _cell(g, 0.1, 1.0, [0, 0, 0], 1.5, 0.3, [0.1, 0.0, 0.2], 5.0, 5.0)
    assert rc == 0 and np.all(m == 0) and np.allclose(F, np.array([0.1, 0, 0.2]) / (1 + 5.0 * 0.1 * 0.1))


def test_equilibrium_cell_bitwise_invariant():
    """T_gas = T_rad, v = 0, F = 0: R = 0 exactly, nothing changes."""
    g = _cell_grid(3.0, 0.3)
    rho, T = 2.0, 1.5
    Cv = rho * 1.0 / (5 / 3 - 1)
    Eg = Cv * T
    Er = 1.0 * ((Eg / Cv) * (Eg / Cv)) ** 2
    rc, m, E1, Er1, F, it = _cell(g, 0.2, rho, [0, 0, 0], Eg, Er, [0, 0, 0], 4.0, 4.0)
    assert rc == 0 and E1 == Eg and Er1 == Er and it == 1


def test_literal_stop_rule_stalls_polish_does_not():
    """DESIGN.md X5: with the printed rule (test before update) a cell already inside the
    tolerance is frozen; converge-then-polish still applies the Newton update."""
    out = {}
    for flags in (O.FLAG_NEWTON_LITERAL, 0):
        g = _cell_grid(1.0, 1.0, flags=flags | O.FLAG_STATIC_MATTER)
        Cv = 1.0 / (5 / 3 - 1)
        Eg = Cv * 1.0
        Er = 1.0 * (1 + 1e-9)                 # tiny disequilibrium
        rc, _, E1, Er1, _, it = _cell(g, 1e-3, 1.0, [0, 0, 0], Eg, Er, [0, 0, 0], 1.0, 1.0)
        out[flags & 4] = (E1 - Eg, it)
    assert out[4] == (0.0, 0) and out[0][0] > 0 and out[0][1] == 1


def test_rhd_conservation_3d():
    """Periodic box, full cycle: sums of rho, rho v + F_r/(c c_hat), E + (c/c_hat) E_r are
    constant to round-off."""
    from paper_2110_01792_b200 import inputs
    p, f = inputs.ragged_rhd(shape=(8, 9, 10), seed=21)
    g = O.Grid(p["nx"], p["ny"], p["nz"], p["dx"], p["gamma"], c_hat=p["c_hat"], c=p["c"], bc=p["bc"])
    g.set_constants(p["a_rad"], p["kB_mu"])
    g.set_params(flags=p["flags"])
    g.set_all(f)
    c, ch = p["c"], p["c_hat"]

    def totals():
        s = g.get_all()
        return [s["rho"].sum(), *(s["m" + a].sum() + s["F" + a].sum() / (c * ch) for a in "xyz"),
                s["E"].sum() + (c / ch) * s["Er"].sum()]
    t0 = totals()
    scale = [abs(t0[0]), *(3 * [np.abs(f["mx"]).sum()]), abs(t0[4])]
    for _ in range(3):
        dt = g.cfl_dt()
        assert g.rhd_step(dt) == 0
    info = g.info()
    assert info["newton_fail_cells"] == 0 and info["nsub"] >= 1
    for a, b, s in zip(t0, totals(), scale):
        assert abs(a - b) < 1e-12 * s, (a, b)


def test_source_term_of_eq27():
    """PAPER.md:215 (eq 27, 38): S adds radiation energy during the substep; reading X13: S = dt * rate(cell).
    Transparent gas (kappa_P = 0): E_r grows by exactly dt*rate per step and the gas is untouched.  Opaque gas:
    eq 26 + (c/c_hat) eq 27 give  Delta(E_g + (c/c_hat) E_r) = (c/c_hat) S  per step, whatever the Newton path."""
    c, ch = 10.0, 2.0
    n = 3
    shape = (n, n, n)
    rng = np.random.default_rng(4)
    rate = rng.uniform(0.5, 2.0, shape)
    for kappa in (0.0, 5.0):
        g = O.Grid(n, n, n, 1.0, 5.0 / 3.0, c_hat=ch, c=c)
        g.set_params(flags=O.FLAG_STATIC_MATTER)
        rho = rng.uniform(0.5, 2.0, shape)
        E0 = rng.uniform(1.0, 2.0, shape)
        Er0 = rng.uniform(0.5, 1.5, shape)
        for name, a in (("rho", rho), ("E", E0), ("Er", Er0), ("kappaP", np.full(shape, kappa)),
                        ("kappaR", np.full(shape, kappa)), ("src", rate)):
            g.set_state(O.FIELDS.index(name), a)
        dt, nsteps = 0.01, 7
        for s in range(1, nsteps + 1):
            assert g.exchange(dt) == 0
            E, Er = g.get_state(4), g.get_state(5)
            budget = (E + (c / ch) * Er) - (E0 + (c / ch) * Er0)
            assert np.abs(budget - (c / ch) * s * dt * rate).max() < 1e-13 * (c / ch) * 10
            if kappa == 0.0:
                assert np.array_equal(E, E0)
                assert np.abs(Er - (Er0 + s * dt * rate)).max() < 1e-14
        if kappa > 0.0:
            assert np.abs(g.get_state(4) - E0).max() > 1e-3      # the gas does take up part of the injected energy
        g.close()


# ------------------------------------------------------------------------------------------------
# temperature-dependent opacities: kappa_P implicit with the d kappa_P / dT term of eq 33,
# kappa_F at the updated temperature
# ------------------------------------------------------------------------------------------------
def test_temperature_power_is_the_plain_power():
    L = O.lib()
    for n2 in range(-8, 9):
        for T, T0 in ((3.7, 1.3), (0.02, 5.0), (2.75e7, 1e6)):
            assert abs(L.orc_temp_power(T, T0, n2) / (T / T0) ** (0.5 * n2) - 1.0) < 1e-14
    assert L.orc_temp_power(7.0, 2.0, 0) == 1.0


def _kT_grid(texp2, flags=0, c=50.0, ch=5.0, kP0=2.0, kR0=3.0, rho0=1.5, erho=1, T0=0.8):
    g = _cell_grid(c, ch, flags=flags, tol=1e-13)
    g.L.orc_set_opacity_law_T(g.h, kP0, kR0, rho0, erho, T0, texp2)
    return g


def test_kappa_of_T_backward_euler_by_bisection():
    """With kappa_P = kappa0 (rho/rho0)^e (T/T0)^s the backward-Euler system eq 26-27 (S = 0) still conserves
    E_g + (c/c_hat) E_r and reduces to one scalar equation in T^(t+1),
        C_v (T - T_0) + (c/c_hat) dt rho kappa_P(T) c_hat (a_r T^4 - E_r(T)) = 0,  E_r(T) from conservation,
    solved here by bisection to 1e-15.  Newton's result must agree for Kramers-like (s = -3.5), s = +1/2, s = 2, and
    kappa_F must be taken at the updated temperature: F^(t+1) = F / (1 + rho kappa_R(T^(t+1)) c_hat dt)."""
    c, ch, gamma = 50.0, 5.0, 5 / 3
    kP0, kR0, rho0, T0 = 2.0, 3.0, 1.5, 0.8
    for texp2 in (-7, 1, 4):
        for (rho, Tg, Er, dt) in ((1.0, 2.0, 0.5, 0.01), (3.0, 0.5, 4.0, 0.003), (0.7, 1.0, 1.0 + 1e-3, 10.0)):
            g = _kT_grid(texp2)
            Cv = rho / (gamma - 1.0)
            Eg0 = Cv * Tg
            kden_P, kden_R = kP0 * (rho / rho0), kR0 * (rho / rho0)
            rc, m1, E1, Er1, F1, it = _cell(g, dt, rho, [0, 0, 0], Eg0, Er, [0.3, 0.0, 0.0], kden_P, kden_R)
            assert rc == 0
            Eg1 = E1 - 0.5 * (m1 @ m1) / rho           # the damped flux pushed the gas (eq 41-42)
            Etot = Eg0 + (c / ch) * Er

            def resid(T):
                kap = kden_P * (T / T0) ** (0.5 * texp2)
                Er_T = (Etot - Cv * T) * (ch / c)
                return Cv * (T - Tg) + (c / ch) * dt * rho * kap * ch * (T ** 4 - Er_T)

            lo, hi = 1e-8, Etot / Cv
            assert resid(lo) < 0 < resid(hi)
            for _ in range(300):
                mid = 0.5 * (lo + hi)
                if resid(mid) > 0: hi = mid
                else: lo = mid
            Tnew = 0.5 * (lo + hi)
            assert abs(Eg1 / (Cv * Tnew) - 1.0) < 1e-11, (texp2, rho, Eg1 / (Cv * Tnew) - 1.0)
            assert abs((E1 + (c / ch) * Er1) / Etot - 1.0) < 1e-13
            kR_new = kden_R * (Tnew / T0) ** (0.5 * texp2)
            assert abs(F1[0] / (0.3 / (1 + rho * kR_new * ch * dt)) - 1.0) < 1e-10


def test_dkappa_dT_term_of_eq33_speeds_up_newton():
    """The Jacobian with the d kappa_P/dT term (eq 33) is the exact one: Newton then converges quadratically, while
    the Jacobian without it (ORC_FLAG_NO_DKAPPA_DT) only converges linearly -- same fixed point, more iterations."""
    rng = np.random.default_rng(8)
    tot_full = tot_frozen = 0
    for _ in range(200):
        rho, Tg = np.exp(rng.normal(0, 0.5)), 10.0 ** rng.uniform(-0.3, 0.3)
        Er = Tg ** 4 * 10.0 ** rng.uniform(-1, 1)
        dt = 10.0 ** rng.uniform(-3, 0)
        Cv = rho / (5 / 3 - 1.0)
        res = []
        for flags in (0, O.FLAG_NO_DKAPPA_DT):
            g = _kT_grid(-7, flags=flags)
            rc, _, Eg1, Er1, _, it = _cell(g, dt, rho, [0, 0, 0], Cv * Tg, Er, [0, 0, 0], 2.0 * rho / 1.5, 3.0 * rho / 1.5)
            assert rc == 0
            res.append((Eg1, it))
        assert abs(res[0][0] / res[1][0] - 1.0) < 1e-9
        tot_full += res[0][1]; tot_frozen += res[1][1]
    assert tot_full < 0.8 * tot_frozen, (tot_full, tot_frozen)


def test_kappa_law_without_T_exponent_is_the_density_law_bitwise():
    """texp2 = 0 must reproduce orc_set_opacity_law bit for bit over whole RHD steps (no stray arithmetic)."""
    from paper_2110_01792_b200 import inputs as I
    outs = []
    for use_T in (False, True):
        p, f = I.ragged_rhd(shape=(6, 7, 9))
        g = O.Grid(p["nx"], p["ny"], p["nz"], p["dx"], p["gamma"], c_hat=p["c_hat"], c=p["c"], bc=p["bc"])
        g.set_constants(p["a_rad"], p["kB_mu"]); g.set_params(flags=p["flags"]); g.set_all(f)
        if use_T: g.set_opacity_law_T(40.0, 60.0, 1.0, -1, 1.0, 0)
        else: g.set_opacity_law(40.0, 60.0, 1.0, -1)
        for _ in range(2):
            assert g.rhd_step(g.cfl_dt()) == 0
        outs.append([g.get_state(k) for k in range(11)])
        g.close()
    assert all(np.array_equal(a, b) for a, b in zip(*outs))


def test_kappa_of_T_rhd_steps_conserve_and_track_temperature():
    """Kramers-like kappa ~ rho T^-3.5 over coupled RHD steps: total energy and momentum conserved to round-off on a
    periodic box, and the stored kappa_R field equals the law at the gas temperature the subcycle started from."""
    from paper_2110_01792_b200 import inputs as I
    p, f = I.ragged_rhd(shape=(6, 7, 9))
    g = O.Grid(p["nx"], p["ny"], p["nz"], p["dx"], p["gamma"], c_hat=p["c_hat"], c=p["c"], bc=p["bc"])
    g.set_constants(p["a_rad"], p["kB_mu"]); g.set_params(flags=p["flags"]); g.set_all(f)
    g.set_opacity_law_T(30.0, 30.0, 1.0, 1, 1.0, -7)
    coc = p["c"] / p["c_hat"]
    tot0 = (g.get_state(4) + coc * g.get_state(5)).sum()
    mom0 = (g.get_state(1) + g.get_state(6) / (p["c"] * p["c_hat"])).sum()
    for _ in range(3):
        assert g.rhd_step(g.cfl_dt()) == 0
    tot1 = (g.get_state(4) + coc * g.get_state(5)).sum()
    mom1 = (g.get_state(1) + g.get_state(6) / (p["c"] * p["c_hat"])).sum()
    assert abs(tot1 / tot0 - 1) < 1e-13 and abs(mom1 - mom0) < 1e-12 * np.abs(g.get_state(1)).sum()
    assert g.info()["newton_fail_cells"] == 0
    g.close()
