"""Pins of the oracle's scheme variants: PLM reconstruction with the
monotonized-central limiter and the Eddington-approximation closure chi = 1/3
(PAPER.md:196, 528).  Each check is against something other than the oracle: exactness on linear data,
textbook limiter bounds, order of accuracy, conservation, the closed-form wave speed c_hat/sqrt(3)."""
import numpy as np

import oracle as O

G53 = 5.0 / 3.0


def _faces(fn, q):
    a = np.ascontiguousarray(q, dtype=np.float64)
    lo, hi = np.zeros(1), np.zeros(1)
    getattr(O.lib(), fn)(a, lo, hi)
    return float(lo[0]), float(hi[0])


def test_plm_faces_linear_extremum_and_limiter():
    # linear data: exact, slope = the common difference
    q = [1.0 + 0.25 * j for j in range(5)]
    lo, hi = _faces("orc_plm_faces", q)
    assert lo == q[2] - 0.125 and hi == q[2] + 0.125
    # local extremum: flat (MC slope vanishes when the one-sided differences change sign)
    assert _faces("orc_plm_faces", [0.0, 1.0, 3.0, 2.0, 0.0]) == (3.0, 3.0)
    # steep one-sided jump: slope limited to twice the smaller difference (Van Leer 1977)
    lo, hi = _faces("orc_plm_faces", [0.0, 1.0, 1.1, 9.0, 9.0])
    assert abs((hi - lo) - 2 * (1.1 - 1.0)) < 1e-15
    # gentle data: central slope
    lo, hi = _faces("orc_plm_faces", [0.0, 1.0, 2.2, 3.0, 4.0])
    assert abs((hi - lo) - 0.5 * (3.0 - 1.0)) < 1e-15
    # mirror symmetry
    rng = np.random.default_rng(3)
    for _ in range(200):
        q = rng.standard_normal(5)
        lo, hi = _faces("orc_plm_faces", q)
        hi2, lo2 = _faces("orc_plm_faces", q[::-1])
        assert lo == lo2 and hi == hi2
        assert min(q[1:4]) - 1e-15 <= lo <= max(q[1:4]) + 1e-15 and min(q[1:4]) - 1e-15 <= hi <= max(q[1:4]) + 1e-15


def _run_1d(N, prim_fn, t_end, cfl, flags, bc=O.BC_PERIODIC):
    g = O.Grid(N, 1, 1, 1.0 / N, G53, bc=bc)
    g.set_params(cfl=cfl, flags=flags)
    x = (np.arange(N) + 0.5) / N
    rho, vx, P = prim_fn(x)
    U0 = [rho, rho * vx, 0 * x, 0 * x, P / (G53 - 1) + 0.5 * rho * vx * vx]
    for k in range(5):
        g.set_state(k, U0[k].reshape(1, 1, N))
    t = 0.0
    while t < t_end * (1 - 1e-14):
        dt = min(g.cfl_dt(), t_end - t)
        assert g.hydro_step(dt) == 0
        t += dt
    U = [g.get_state(k).ravel() for k in range(5)]
    g.close()
    return U0, U


def test_plm_advected_wave_second_order_and_less_accurate_than_ppm():
    def ic(x):
        return 1.0 + 0.1 * np.sin(2 * np.pi * x), np.ones_like(x), np.ones_like(x)
    errs, errs_ppm = [], []
    for N in (16, 32, 64, 128):
        U0, U = _run_1d(N, ic, 1.0, 0.3, O.FLAG_PLM)
        errs.append(np.abs(U[0] - U0[0]).mean())
        U0, U = _run_1d(N, ic, 1.0, 0.3, 0)
        errs_ppm.append(np.abs(U[0] - U0[0]).mean())
    orders = [np.log2(errs[n] / errs[n + 1]) for n in range(3)]
    # clipping at the two extrema costs accuracy at low resolution: the order climbs towards 2
    assert orders[0] < orders[1] < orders[2] and 1.8 < orders[2] < 2.2 and orders[0] > 1.3, (errs, orders)
    assert all(e > p for e, p in zip(errs, errs_ppm)), (errs, errs_ppm)      # "PPM by default" for a reason


def test_plm_stationary_contact_exact_and_conservation():
    def ic(x):
        return np.where(x < 0.5, 1.4, 1.0), np.zeros_like(x), np.ones_like(x)
    U0, U = _run_1d(64, ic, 0.5, 0.3, O.FLAG_PLM, bc=O.BC_OUTFLOW)
    assert all(np.array_equal(a, b) for a, b in zip(U0, U))                  # HLLC keeps the contact
    rng = np.random.default_rng(11)
    shape = (6, 7, 8)
    g = O.Grid(8, 7, 6, 1.0 / 8, G53)
    g.set_params(flags=O.FLAG_PLM)
    rho = np.exp(0.3 * rng.standard_normal(shape))
    v = 0.8 * rng.standard_normal((3,) + shape)
    E = 1.0 / (G53 - 1) + 0.5 * rho * (v ** 2).sum(0)
    for k, a in enumerate([rho, rho * v[0], rho * v[1], rho * v[2], E]):
        g.set_state(k, a)
    tot0 = [g.get_state(k).sum() for k in range(5)]
    for _ in range(5):
        assert g.hydro_step(g.cfl_dt()) == 0
    tot = [g.get_state(k).sum() for k in range(5)]
    g.close()
    scale = [abs(t) + rho.sum() for t in tot0]
    assert all(abs(a - b) < 1e-13 * s for a, b, s in zip(tot, tot0, scale))


def test_eddington_closure_is_isotropic_for_every_flux():
    L = O.lib()
    rng = np.random.default_rng(5)
    for _ in range(100):
        f = rng.uniform(-1, 1, 3)
        for n in range(3):
            T, chi = np.zeros(3), np.zeros(1)
            L.orc_closure_k(O.FLAG_EDDINGTON, np.ascontiguousarray(f), n, T, chi)
            assert chi[0] == 1.0 / 3.0
            assert [T[i] for i in range(3)] == [0.5 * (1.0 - 1.0 / 3.0) if i == n else 0.0 for i in range(3)]
            assert abs(T[n] - 1.0 / 3.0) < 1e-16
            # and the default stays Levermore
            L.orc_closure_k(0, np.ascontiguousarray(f), n, T, chi)
            assert abs(chi[0] - L.orc_eddington_factor(min(1.0, float(np.sqrt((f ** 2).sum()))))) < 1e-15


def _wave_about_streaming_state(flags, f0=0.5, N=64):
    """Right-going wave of the chi = 1/3 system about a base state with reduced flux f0; error after one
    period of a c_hat/sqrt(3) wave, in units of the amplitude."""
    c, c_hat, A = 1.0, 0.1, 1e-6
    g = O.Grid(N, 1, 1, 1.0 / N, G53, c_hat=c_hat, c=c)
    g.set_params(flags=flags)
    x = (np.arange(N) + 0.5) / N
    dE = A * np.sin(2 * np.pi * x)
    E0 = 1.0 + dE
    F0 = f0 * c * 1.0 + c / np.sqrt(3.0) * dE
    for name, a in (("Er", E0), ("Fx", F0), ("rho", np.ones(N))):
        g.set_state(O.FIELDS.index(name), a.reshape(1, 1, N))
    period = 1.0 / (c_hat / np.sqrt(3.0))
    nsteps = int(np.ceil(period / (0.3 / N / c_hat)))
    for _ in range(nsteps):
        assert g.rad_transport(period / nsteps) == 0
    err = np.abs(g.get_state(5).ravel() - E0).mean() / A
    g.close()
    return err


def test_eddington_closure_makes_the_moment_system_linear():
    """With P_r = E_r/3 the moment equations (eq 11-12) are linear with characteristic speeds +-c_hat/sqrt(3)
    whatever the background flux, so a wave about a streaming state (f0 = 0.5) is back in phase after one
    period; under the Levermore closure the speeds at f0 = 0.5 differ and the same wave is not."""
    err_edd = _wave_about_streaming_state(O.FLAG_EDDINGTON)
    err_lev = _wave_about_streaming_state(0)
    assert err_edd < 3e-2, err_edd
    assert err_lev > 10 * err_edd and err_lev > 0.2, (err_lev, err_edd)


def test_eddington_linear_wave_speed():
    c, c_hat, A, N = 1.0, 0.1, 1e-6, 64
    g = O.Grid(N, 1, 1, 1.0 / N, G53, c_hat=c_hat, c=c)
    g.set_params(flags=O.FLAG_EDDINGTON | O.FLAG_PLM)
    x = (np.arange(N) + 0.5) / N
    E0 = 1.0 + A * np.sin(2 * np.pi * x)
    F0 = A * c / np.sqrt(3.0) * np.sin(2 * np.pi * x)
    for name, a in (("Er", E0), ("Fx", F0), ("rho", np.ones(N))):
        g.set_state(O.FIELDS.index(name), a.reshape(1, 1, N))
    period = 1.0 / (c_hat / np.sqrt(3.0))
    nsteps = int(np.ceil(period / (0.3 / N / c_hat)))
    for _ in range(nsteps):
        assert g.rad_transport(period / nsteps) == 0
    err = np.abs(g.get_state(5).ravel() - E0).mean() / A
    g.close()
    assert err < 2e-2, err      # back in phase after exactly one period of a c_hat/sqrt(3) wave


def test_minerbo_closure_against_its_maximum_entropy_definition():
    """Minerbo (1978): the Eddington factor of the maximum-entropy intensity I(mu) ~ exp(a mu), i.e.
    f = coth a - 1/a and chi = 1 - 2 f / a.  The oracle uses the customary polynomial form (PAPER.md:196 prints
    none, V3); it must hit the limits exactly, be monotone and realizable (f^2 <= chi <= 1) and follow
    the exact relation closely."""
    L = O.lib()
    assert L.orc_minerbo_factor(0.0) == 1.0 / 3.0 and abs(L.orc_minerbo_factor(1.0) - 1.0) < 1e-15
    fs = np.linspace(0.0, 1.0, 401)
    chi = np.array([L.orc_minerbo_factor(float(f)) for f in fs])
    assert np.all(np.diff(chi) > 0) and np.all(chi >= fs ** 2 - 1e-15) and np.all(chi <= 1 + 1e-15)
    worst = 0.0
    for f, c in zip(fs[1:-1], chi[1:-1]):
        lo, hi = 1e-8, 1e4
        for _ in range(200):                                   # invert the Langevin function by bisection
            a = 0.5 * (lo + hi)
            if 1.0 / np.tanh(a) - 1.0 / a < f:
                lo = a
            else:
                hi = a
        a = 0.5 * (lo + hi)
        worst = max(worst, abs(c - (1.0 - 2.0 * f / a)))
    assert worst < 0.011, worst
    # the closure is selected by its flag and differs from Levermore's in between
    T, ch = np.zeros(3), np.zeros(1)
    L.orc_closure_k(O.FLAG_MINERBO, np.array([0.3, 0.4, 0.0]), 0, T, ch)
    assert ch[0] == L.orc_minerbo_factor(0.5) and abs(ch[0] - L.orc_eddington_factor(0.5)) > 0.02
    assert abs(T[0] - (0.5 * (1 - ch[0]) + 0.5 * (3 * ch[0] - 1) * 0.36)) < 1e-15
