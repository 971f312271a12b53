"""Pins for the hydro part of the CPU oracle (oracle/hydro.c): what the paper and the
mathematics fix, not the oracle's own formulas.  CPU only."""
import glob
import hashlib
import json
import os

import numpy as np
import pytest

import oracle as O

G53 = 5.0 / 3.0
HERE = os.path.dirname(os.path.abspath(__file__))


def _golden(name):
    rows = []
    for line in open(os.path.join(HERE, "golden", name)):
        line = line.strip()
        if line and not line.startswith("#"):
            rows.append([float(x) for x in line.split()])
    return rows


# ---- the two long pins (PAPER.md:299 at N = 1024): minutes each, because the oracle carries the full
# ghost shell around an N x 1 x 1 box.  Their values depend on nothing but the oracle's sources and this file, so
# tests/golden/make_oracle_slow_pins.py (which calls only the functions below, i.e. only oracle/) stores them next to a
# SHA-256 of exactly those files; the tests take the stored value when the fingerprint still matches and compute it
# otherwise (any change of the oracle, of its build flags or of this file) or when QK_SLOW=1.  Either way the assertion
# against the paper's printed number runs.
def _oracle_fingerprint():
    root = os.path.dirname(HERE)
    files = sorted(glob.glob(os.path.join(root, "oracle", "*.c")) + glob.glob(os.path.join(root, "oracle", "*.h")))
    files += [os.path.join(root, "oracle", "__init__.py"), os.path.abspath(__file__)]
    h = hashlib.sha256()
    for f in files:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()


SLOW_PINS = os.path.join(HERE, "golden", "oracle_slow_pins.json")


def _slow_pin(name, compute):
    if os.environ.get("QK_SLOW") != "1":
        try:
            stored = json.load(open(SLOW_PINS))
            if stored["fingerprint"] == _oracle_fingerprint():
                return float(stored["values"][name])
        except (OSError, KeyError, ValueError):
            pass
    return compute()


def _run_1d(N, prim_fn, gamma, t_end, cfl, bc=O.BC_PERIODIC, length=1.0, x0=0.0):
    """1-D problem as an N x 1 x 1 box; prim_fn(x) -> rho, vx, P.  Returns x, U0, U."""
    dx = length / N
    g = O.Grid(N, 1, 1, dx, gamma, bc=bc)
    g.set_params(cfl=cfl)
    x = x0 + (np.arange(N) + 0.5) * dx
    rho, vx, P = prim_fn(x)
    U0 = [rho, rho * vx, 0 * x, 0 * x, P / (gamma - 1) + 0.5 * rho * vx * vx]
    for k in range(5):
        g.set_state(k, U0[k].reshape(1, 1, N))
    t = 0.0
    while t < t_end * (1 - 1e-14):
        dt = min(g.cfl_dt(), t_end - t)
        assert g.hydro_step(dt) == 0
        t += dt
    U = [g.get_state(k).ravel() for k in range(5)]
    g.close()
    return x, U0, U


def _sound_wave_error(N):
    # PAPER.md:289-297, eq 44-45
    g = O.Grid(N, 1, 1, 1.0 / N, G53)
    g.set_params(cfl=0.1)
    x = (np.arange(N) + 0.5) / N
    A, R = 1e-6, np.array([1.0, -1.0, 1.0, 1.0, 1.5])
    Ub = np.array([1.0, 0.0, 0.0, 0.0, (1.0 / G53) / (G53 - 1.0)])
    U0 = [(Ub[k] + A * R[k] * np.sin(2 * np.pi * x)).reshape(1, 1, N) for k in range(5)]
    for k in range(5):
        g.set_state(k, U0[k])
    t = 0.0
    while t < 1.0 - 1e-14:
        dt = min(g.cfl_dt(), 1.0 - t)
        g.hydro_step(dt)
        t += dt
    err = [np.abs(g.get_state(k) - U0[k]).mean() for k in range(5)]
    g.close()
    return float(np.sqrt(np.sum(np.square(err))))


@pytest.mark.parametrize("row", [r for r in _golden("sound_wave_paper.txt") if r[0] <= 128])
def test_sound_wave_printed_errors(row):
    """PAPER.md:299 prints 1.0e-7 (N=16), 1.6e-9 (N=128): two significant digits."""
    N, printed = int(row[0]), row[1]
    e = _sound_wave_error(N)
    assert abs(e / printed - 1.0) < 0.05, (N, e, printed)


def test_sound_wave_printed_error_1024():
    e = _slow_pin("sound_wave_error_1024", lambda: _sound_wave_error(1024))
    assert abs(e / 1.7e-11 - 1.0) < 0.05, e


def test_stationary_contact_exactly_zero():
    """rho 1.4 | 1.0, P = 1, v = 0, gamma = 1.4, to t = 2: error exactly zero."""
    def ic(x):
        return np.where(x < 0.5, 1.4, 1.0), 0 * x, np.ones_like(x)
    _, U0, U = _run_1d(64, ic, 1.4, 2.0, 0.3, bc=O.BC_OUTFLOW)
    for k in range(5):
        assert np.array_equal(U[k], U0[k]), k


# ---- exact Riemann solver (textbook: Toro, Riemann Solvers, ch. 4), written for the test ----
def _exact_riemann(rl, ul, pl, rr, ur, pr, g, xi):
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)

    def fK(p, rk, pk, ak):
        if p > pk:
            A, B = 2 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * np.sqrt(A / (p + B)), np.sqrt(A / (p + B)) * (1 - 0.5 * (p - pk) / (B + p))
        return 2 * ak / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1 / (rk * ak) * (p / pk) ** (-(g + 1) / (2 * g))
    p = 0.5 * (pl + pr)
    for _ in range(100):
        f1, d1 = fK(p, rl, pl, al)
        f2, d2 = fK(p, rr, pr, ar)
        pn = max(1e-12, p - (f1 + f2 + ur - ul) / (d1 + d2))
        if abs(pn - p) < 1e-15 * p:
            p = pn
            break
        p = pn
    ps = p
    us = 0.5 * (ul + ur) + 0.5 * (fK(ps, rr, pr, ar)[0] - fK(ps, rl, pl, al)[0])
    rho, u, P = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    for n, s in enumerate(xi):
        if s <= us:  # left of contact
            if ps > pl:
                sl = ul - al * np.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                if s <= sl:
                    rho[n], u[n], P[n] = rl, ul, pl
                else:
                    rho[n] = rl * ((ps / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pl + 1))
                    u[n], P[n] = us, ps
            else:
                shl, asl = ul - al, al * (ps / pl) ** ((g - 1) / (2 * g))
                stl = us - asl
                if s <= shl:
                    rho[n], u[n], P[n] = rl, ul, pl
                elif s >= stl:
                    rho[n], u[n], P[n] = rl * (ps / pl) ** (1 / g), us, ps
                else:
                    cc = 2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)
                    rho[n], u[n], P[n] = rl * cc ** (2 / (g - 1)), 2 / (g + 1) * (al + (g - 1) / 2 * ul + s), pl * cc ** (2 * g / (g - 1))
        else:
            if ps > pr:
                sr = ur + ar * np.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                if s >= sr:
                    rho[n], u[n], P[n] = rr, ur, pr
                else:
                    rho[n] = rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1))
                    u[n], P[n] = us, ps
            else:
                shr, asr = ur + ar, ar * (ps / pr) ** ((g - 1) / (2 * g))
                strr = us + asr
                if s >= shr:
                    rho[n], u[n], P[n] = rr, ur, pr
                elif s <= strr:
                    rho[n], u[n], P[n] = rr * (ps / pr) ** (1 / g), us, ps
                else:
                    cc = 2 / (g + 1) - (g - 1) / ((g + 1) * ar) * (ur - s)
                    rho[n], u[n], P[n] = rr * cc ** (2 / (g - 1)), 2 / (g + 1) * (-ar + (g - 1) / 2 * ur + s), pr * cc ** (2 * g / (g - 1))
    return rho, u, P, ps, us


def test_exact_riemann_solver_star_values():
    """The test's own exact solver reproduces the textbook Sod star state."""
    _, _, _, ps, us = _exact_riemann(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4, np.array([0.0]))
    assert abs(ps - 0.30313) < 1e-5 and abs(us - 0.92745) < 1e-5


def test_sod_against_exact_solution():
    """Sod tube (north_star pin): L1 error vs the exact Riemann solution falls ~first order and
    the star-region plateau is reproduced; no undershoot below the right state."""
    def ic(x):
        return np.where(x < 0.5, 1.0, 0.125), 0 * x, np.where(x < 0.5, 1.0, 0.1)
    errs = []
    for N in (100, 200, 400):
        x, _, U = _run_1d(N, ic, 1.4, 0.2, 0.3, bc=O.BC_OUTFLOW)
        rho_ex, u_ex, p_ex, ps, us = _exact_riemann(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4, (x - 0.5) / 0.2)
        errs.append(np.abs(U[0] - rho_ex).mean())
        assert U[0].min() >= 0.125 - 1e-12
        if N == 400:
            plateau = (x > 0.5 + us * 0.2 + 0.03) & (x < 0.5 + 1.75216 * 0.2 - 0.03)   # between contact and shock
            assert np.abs(U[0][plateau] - 0.26557).max() < 2e-3
            vel = U[1] / U[0]
            assert np.abs(vel[plateau] - 0.92745).max() < 2e-3
    assert errs[0] < 6e-3 and errs[2] < 1.5e-3, errs
    assert 1.6 < errs[0] / errs[1] < 2.6 and 1.6 < errs[1] / errs[2] < 2.6, errs


def _strong_shock_rel_error():
    def ic(x):
        return np.where(x < 2.0, 10.0, 1.0), 0 * x, np.where(x < 2.0, 100.0, 1.0)
    g = 1.4
    x, _, U = _run_1d(1000, ic, g, 0.4, 0.1, bc=O.BC_OUTFLOW, length=5.0)
    r, u, p, _, _ = _exact_riemann(10.0, 0.0, 100.0, 1.0, 0.0, 1.0, g, (x - 2.0) / 0.4)
    Uex = [r, r * u, p / (g - 1) + 0.5 * r * u * u]
    num = np.sqrt(np.mean([np.abs(U[k] - Uex[n]).mean() ** 2 for n, k in enumerate((0, 1, 4))]))
    den = np.sqrt(np.mean([np.abs(Uex[n]).mean() ** 2 for n in range(3)]))
    return float(num / den)


def test_strong_shock_tube_error_scale():
    """(rho,p) = (10,100)|(1,1), 1000 cells on [0,5], x0=2, t=0.4, CFL 0.1;
    relative rms-of-L1 error printed as 1.12e-3 (gamma not printed; 1.4 assumed: weak pin, ~1e-3)."""
    rel = _slow_pin("strong_shock_rel_error", _strong_shock_rel_error)
    # paper: 1.12e-3 (gamma = 1.4 gives 1.19e-3 here, gamma = 5/3 1.31e-3); within 20 % of the printed value -- without
    # flattening the paper reports "unacceptably large post-shock oscillations", so this holds the H6 constants to scale
    assert 0.9e-3 < rel < 1.35e-3, rel


SLOW_SHOCK = dict(gamma=1.4, L=(3.86, -3.1266, 27.0913), R=(1.0, -3.44, 8.4168), speed=0.1096)


def slow_shock_ic(x):
    g = SLOW_SHOCK["gamma"]
    (rl, ml, el), (rr, mr, er) = SLOW_SHOCK["L"], SLOW_SHOCK["R"]
    pl, pr = (g - 1) * (el - 0.5 * ml * ml / rl), (g - 1) * (er - 0.5 * mr * mr / rr)
    left = x < 0.5
    return np.where(left, rl, rr), np.where(left, ml / rl, mr / rr), np.where(left, pl, pr)


def shock_position(x, rho, level):
    """where rho falls through `level`, linearly interpolated between cell centres (last crossing from the left)"""
    j = np.nonzero(rho > level)[0][-1]
    return x[j] + (rho[j] - level) / (rho[j] - rho[j + 1]) * (x[j + 1] - x[j])


def test_slow_moving_shock_speed():
    """PAPER.md:357-366 (Jin & Liu parameters, gamma = 1.4, CFL 0.2): 'the shock jump moving to the right with a
    velocity v_shock = 0.1096', ~250 steps per cell.  The density jump's midpoint travels at that speed (between t = 1
    and t = 2, after the start-up waves of the rounded printed states have left), the post-shock oscillation the
    paper describes stays at the per-cent level with flattening, and nothing overshoots on the pre-shock side."""
    N = 100
    gamma = SLOW_SHOCK["gamma"]
    g = O.Grid(N, 1, 1, 1.0 / N, gamma, bc=O.BC_OUTFLOW)
    g.set_params(cfl=0.2)
    x = (np.arange(N) + 0.5) / N
    rho, vx, P = slow_shock_ic(x)
    for k, a in enumerate([rho, rho * vx, 0 * x, 0 * x, P / (gamma - 1) + 0.5 * rho * vx * vx]):
        g.set_state(k, a.reshape(1, 1, N))
    threads = O.get_threads()
    O.set_threads(1)                   # one row of cells, ~5000 steps: the thread team would cost more than the loops
    pos, t, steps = [], 0.0, 0
    try:
        for t_end in (1.0, 2.0):
            while t < t_end * (1 - 1e-14):
                dt = min(g.cfl_dt(), t_end - t)
                assert g.hydro_step(dt) == 0
                t += dt
                steps += 1
            U = [g.get_state(0).ravel()]
            pos.append(shock_position(x, U[0], 0.5 * (SLOW_SHOCK["L"][0] + SLOW_SHOCK["R"][0])))
    finally:
        O.set_threads(threads)
        g.close()
    assert 200 < steps / (N * (pos[1] - 0.5)) < 300          # "~250 timesteps to move across a single cell"
    speed = pos[1] - pos[0]
    assert abs(speed - SLOW_SHOCK["speed"]) < 0.5 / N, (pos, speed)
    post = U[0][x < pos[1] - 0.05]
    assert np.abs(post / SLOW_SHOCK["L"][0] - 1.0).max() < 0.02
    pre = U[0][x > pos[1] + 0.03]
    assert np.abs(pre - 1.0).max() < 1e-6


def test_advected_wave_second_order():
    """Smooth advected density wave (config 1 without noise): L1 order ~2."""
    def ic(x):
        return 1.0 + 0.1 * np.sin(2 * np.pi * x), np.ones_like(x), np.ones_like(x)
    errs = []
    for N in (16, 32, 64, 128):
        _, U0, U = _run_1d(N, ic, G53, 1.0, 0.3)
        errs.append(np.abs(U[0] - U0[0]).mean())
    orders = [np.log2(errs[n] / errs[n + 1]) for n in range(3)]
    assert all(1.7 < o < 2.6 for o in orders), (errs, orders)


def _random_box(shape, seed, gamma=G53, mach=1.0):
    rng = np.random.default_rng(seed)
    rho = np.exp(0.3 * rng.standard_normal(shape))
    v = [mach * rng.standard_normal(shape) for _ in range(3)]
    P = np.exp(0.3 * rng.standard_normal(shape))
    E = P / (gamma - 1) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    return [rho, rho * v[0], rho * v[1], rho * v[2], E]


def test_conservation_periodic():
    """Flux-form update: sums of rho, rho v, E constant to round-off on a periodic grid."""
    shape = (10, 12, 14)
    g = O.Grid(shape[2], shape[1], shape[0], 1.0 / 14, G53)
    U0 = _random_box(shape, 3, mach=0.5)
    for k in range(5):
        g.set_state(k, U0[k])
    for _ in range(5):
        assert g.hydro_step(g.cfl_dt()) == 0
    for k in range(5):
        s0, s1 = U0[k].sum(), g.get_state(k).sum()
        scale = np.abs(U0[k]).sum()
        assert abs(s1 - s0) < 1e-13 * scale, (k, s0, s1)
    assert not np.array_equal(g.get_state(0), U0[0])


def test_uniform_state_bitwise_invariant():
    shape = (6, 7, 9)
    g = O.Grid(shape[2], shape[1], shape[0], 0.1, G53)
    vals = [1.3, 0.0, 0.0, 0.0, 2.7]
    for k in range(5):
        g.set_state(k, np.full(shape, vals[k]))
    for _ in range(3):
        g.hydro_step(g.cfl_dt())
    for k in range(5):
        assert np.array_equal(g.get_state(k), np.full(shape, vals[k]))


def test_xy_symmetry_bitwise():
    """with fluxes added symmetrically and no FMA an x<->y symmetric state
    stays exactly symmetric."""
    n = 12
    shape = (6, n, n)
    rng = np.random.default_rng(5)
    def sym(a):
        return 0.5 * (a + a.transpose(0, 2, 1))
    rho = sym(np.exp(0.4 * rng.standard_normal(shape)))
    P = sym(np.exp(0.4 * rng.standard_normal(shape)))
    a = rng.standard_normal(shape)
    vx, vy = a, a.transpose(0, 2, 1).copy()
    vz = sym(rng.standard_normal(shape))
    E = P / (G53 - 1) + 0.5 * rho * ((vx * vx + vy * vy) + vz * vz)
    U0 = [rho, rho * vx, rho * vy, rho * vz, E]
    assert np.array_equal(U0[1], U0[2].transpose(0, 2, 1)) and np.array_equal(E, E.transpose(0, 2, 1))
    g = O.Grid(n, n, 6, 1.0 / n, G53)
    for k in range(5):
        g.set_state(k, U0[k])
    for _ in range(6):
        g.hydro_step(g.cfl_dt())
    U = [g.get_state(k) for k in range(5)]
    assert np.array_equal(U[0], U[0].transpose(0, 2, 1))
    assert np.array_equal(U[1], U[2].transpose(0, 2, 1))
    assert np.array_equal(U[3], U[3].transpose(0, 2, 1))
    assert np.array_equal(U[4], U[4].transpose(0, 2, 1))
    assert not np.array_equal(U[0], rho)


def test_direction_permutation_of_1d_problem():
    """The same 1-D shock tube run along x, y and z gives the same profile (index mapping)."""
    N = 48
    prof = []
    for axis in range(3):
        dims = [1, 1, 1]
        dims[axis] = N
        g = O.Grid(dims[0], dims[1], dims[2], 1.0 / N, 1.4, bc=O.BC_OUTFLOW)
        x = (np.arange(N) + 0.5) / N
        rho = np.where(x < 0.5, 1.0, 0.125)
        P = np.where(x < 0.5, 1.0, 0.1)
        shp = (dims[2], dims[1], dims[0])
        g.set_state(0, rho.reshape(shp))
        g.set_state(4, (P / 0.4).reshape(shp))
        for _ in range(20):
            g.hydro_step(0.2 / N)
        prof.append([g.get_state(k).ravel() for k in (0, 1 + axis, 4)])
        others = [g.get_state(1 + a) for a in range(3) if a != axis]
        assert all(np.all(o == 0) for o in others)
    for axis in (1, 2):
        for a, b in zip(prof[0], prof[axis]):
            assert np.allclose(a, b, rtol=0, atol=1e-14)


def test_hllc_consistency_and_upwinding():
    L = O.lib()
    rng = np.random.default_rng(0)
    F = np.zeros(5)
    for _ in range(50):
        W = np.array([np.exp(rng.standard_normal()), *rng.standard_normal(3), np.exp(rng.standard_normal())])
        L.orc_hllc(1.4, W, W, F)
        r, u, v, w, p = W
        E = p / 0.4 + 0.5 * r * (u * u + (v * v + w * w))
        phys = np.array([r * u, r * u * u + p, r * u * v, r * u * w, u * (E + p)])
        assert np.allclose(F, phys, rtol=1e-14, atol=1e-14)
    # supersonic to the right: pure left flux
    WL = np.array([1.0, 5.0, 0.1, 0.2, 1.0]); WR = np.array([0.5, 4.0, 0.0, 0.0, 0.7])
    L.orc_hllc(1.4, WL, WR, F)
    r, u, v, w, p = WL
    E = p / 0.4 + 0.5 * r * (u * u + (v * v + w * w))
    assert np.array_equal(F, np.array([r * u, r * u * u + p, r * u * v, r * u * w, u * (E + p)]))
    # mirror symmetry: reflecting the problem flips the sign of mass/energy flux
    F2 = np.zeros(5)
    WLm, WRm = WR.copy(), WL.copy()
    WLm[1] *= -1; WRm[1] *= -1
    L.orc_hllc(1.4, WLm, WRm, F2)
    assert np.allclose(F2[[0, 4]], -F[[0, 4]], rtol=1e-14) and np.isclose(F2[1], F[1], rtol=1e-14)


def test_ppm_properties():
    L = O.lib()
    qm, qp = np.zeros(1), np.zeros(1)
    # eq 22 on a parabola's cell averages is exact at the interface for smooth monotone data
    xs = np.arange(-2, 3, dtype=float)
    avg = lambda a, b, c, x: a * (x * x + 1 / 12.0) + b * x + c     # cell average of a x^2 + b x + c, width 1
    q = avg(0.05, 1.0, 3.0, xs)
    L.orc_ppm_faces(q, qm, qp)
    assert abs(qm[0] - (0.05 * 0.25 - 0.5 + 3.0)) < 1e-14 and abs(qp[0] - (0.05 * 0.25 + 0.5 + 3.0)) < 1e-14
    # mirror symmetry, bitwise
    rng = np.random.default_rng(1)
    for _ in range(200):
        q = rng.standard_normal(5)
        L.orc_ppm_faces(q, qm, qp)
        a, b = qm[0], qp[0]
        L.orc_ppm_faces(q[::-1].copy(), qm, qp)
        assert a == qp[0] and b == qm[0]
        lo, hi = q[1:4].min(), q[1:4].max()
        assert lo - 1e-15 <= a <= hi + 1e-15 and lo - 1e-15 <= b <= hi + 1e-15
    # local extremum of the averages -> flat (MC slope 0)
    q = np.array([0.0, 1.0, 2.0, 1.0, 0.0])
    L.orc_ppm_faces(q, qm, qp)
    assert qm[0] == 2.0 and qp[0] == 2.0
    # CW84 overshoot: steep on the right -> left state pulled to q - 2 dp, parabola monotone
    q = np.array([0.0, 0.0, 0.1, 1.0, 1.0])
    L.orc_ppm_faces(q, qm, qp)
    dm, dp = q[2] - qm[0], qp[0] - q[2]
    assert dm * dp >= 0 and abs(dp) <= 2 * abs(dm) + 1e-15 and abs(dm) <= 2 * abs(dp) + 1e-15
    assert L.orc_mc_slope(0.0, 1.0, 4.0) == 2.0 and L.orc_mc_slope(0.0, 1.0, 0.5) == 0.0
    assert L.orc_mc_slope(0.0, 1.0, 2.0) == 1.0


def test_flattening_limits():
    L = O.lib()
    g = 1.4
    smooth = np.array([1.0, 1.01, 1.02, 1.03, 1.04])
    v_div = np.array([0.0, 0.1, 0.2, 0.3, 0.4])
    v_conv = v_div[::-1].copy()
    assert L.orc_flatten_1d(g, smooth, v_conv) == 1.0       # weak gradient: no flattening
    shock = np.array([1.0, 1.0, 5.0, 10.0, 10.0])
    assert L.orc_flatten_1d(g, shock, v_conv) == 0.0        # strong, compressive, narrow: full
    assert L.orc_flatten_1d(g, shock, v_div) == 1.0         # expanding: none
    assert L.orc_flatten_1d(g, np.ones(5), v_conv) == 1.0   # 0/0


def test_cfl_dt_eq21():
    """eq 21 with the vector magnitude (footnote 3)."""
    g = O.Grid(4, 4, 4, 0.25, G53)
    shape = (4, 4, 4)
    rho, P = 2.0, 3.0
    v = np.array([1.0, 1.0, 1.0]) / np.sqrt(3.0)
    g.set_state(0, np.full(shape, rho))
    for a in range(3):
        g.set_state(1 + a, np.full(shape, rho * v[a]))
    g.set_state(4, np.full(shape, P / (G53 - 1) + 0.5 * rho * 1.0))
    dt = g.cfl_dt()
    assert abs(dt - 0.3 * 0.25 / (1.0 + np.sqrt(G53 * P / rho))) < 1e-15


def test_thread_count_does_not_change_a_bit():
    """oracle loops over cells are dealt out to threads (omp parallel for): per-cell arithmetic is untouched, so one
    thread and all threads give identical bits and identical integer diagnostics (CPU baseline)."""
    from paper_2110_01792_b200 import inputs as I
    n0 = O.get_threads()
    outs = []
    try:
        for nt in (1, max(2, n0)):
            O.set_threads(nt)
            p, f = I.ragged_rhd(shape=(14, 15, 17), tau_corr=True)
            g = O.Grid(p["nx"], p["ny"], p["nz"], p["dx"], p["gamma"], c_hat=p["c_hat"], c=p["c"], bc=p["bc"])
            g.set_constants(p["a_rad"], p["kB_mu"]); g.set_params(flags=p["flags"]); g.set_all(f)
            assert g.L.orc_ncells_total(g.h) > 4096          # above ORC_OMP_MIN: the parallel regions are active
            for _ in range(2):
                assert g.rhd_step(g.cfl_dt()) == 0
            outs.append(([g.get_state(k) for k in range(9)], g.info()))
            g.close()
    finally:
        O.set_threads(n0)
    assert all(np.array_equal(a, b) for a, b in zip(outs[0][0], outs[1][0])) and outs[0][1] == outs[1][1]
