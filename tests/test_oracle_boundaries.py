"""Pins of the oracle's per-face boundaries and of the Dirichlet ("fixed") type the paper uses for inflow and
prescribed-state boundaries.  Checked against the definition (brute-force
image map), against invariants (a uniform stream through fixed faces stays uniform bit for bit), against the
equivalent outflow run (a shock tube whose ends have not been reached yet) and against the streaming limit
(a beam entering through a fixed face fills the box behind a front moving at c_hat)."""
import numpy as np

import oracle as O

NG = 4
G53 = 5.0 / 3.0


def _img(v, n, bc):
    if 0 <= v < n:
        return v, False, False
    if bc == O.BC_FIXED:
        return v, True, False
    if bc == O.BC_PERIODIC:
        return v % n, False, False
    if bc == O.BC_OUTFLOW:
        return (0 if v < 0 else n - 1), False, False
    m = -1 - v if v < 0 else 2 * n - 1 - v
    return min(max(m, 0), n - 1), False, True


def test_mixed_face_boundaries_brute_force():
    nz, ny, nx = 5, 6, 7
    faces = [O.BC_FIXED, O.BC_OUTFLOW, O.BC_PERIODIC, O.BC_PERIODIC, O.BC_REFLECTING, O.BC_FIXED]
    rng = np.random.default_rng(2)
    g = O.Grid(nx, ny, nz, 0.1, G53, c_hat=1.0, c=10.0)
    g.set_face_bc(faces)
    shape_g = (nz + 2 * NG, ny + 2 * NG, nx + 2 * NG)
    before = []
    for f in range(9):
        a = rng.standard_normal(shape_g)
        g.set_raw(f, a)
        before.append(a)
    g.fill_boundary(O.FILL_ALL)
    comp = {1: 0, 2: 1, 3: 2, 6: 0, 7: 1, 8: 2}            # field -> axis (0 = x) of its vector component
    n = (nx, ny, nz)
    for f in range(9):
        raw = g.get_raw(f).reshape(shape_g)
        for K in range(-NG, nz + NG):
            for J in range(-NG, ny + NG):
                for Ii in range(-NG, nx + NG):
                    src, fixed, sign = [], False, 1.0
                    for ax, v in enumerate((Ii, J, K)):
                        lohi = 0 if v < 0 else 1
                        m, fx, refl = _img(v, n[ax], faces[2 * ax + lohi])
                        fixed |= fx
                        if refl and comp.get(f) == ax:
                            sign = -sign
                        src.append(m)
                    here = raw[K + NG, J + NG, Ii + NG]
                    if fixed:
                        assert here == before[f][K + NG, J + NG, Ii + NG]
                    else:
                        assert here == sign * before[f][src[2] + NG, src[1] + NG, src[0] + NG]
    g.close()
    h = O.Grid(4, 4, 4, 0.1, G53)
    try:
        h.set_face_bc([O.BC_PERIODIC, O.BC_OUTFLOW, 0, 0, 0, 0])
        raise SystemError("periodic on one face only must be refused")
    except AssertionError:
        pass
    h.close()


def _raw_uniform(g, values):
    shape_g = (g.nz + 2 * NG, g.ny + 2 * NG, g.nx + 2 * NG)
    for f, v in enumerate(values):
        g.set_raw(f, np.full(shape_g, v))


def test_uniform_supersonic_stream_through_fixed_faces_is_invariant():
    g = O.Grid(12, 5, 4, 0.1, G53)
    g.set_face_bc([O.BC_FIXED, O.BC_FIXED, O.BC_PERIODIC, O.BC_PERIODIC, O.BC_OUTFLOW, O.BC_OUTFLOW])
    rho, vx, P = 1.3, 4.0, 0.7                              # Mach ~ 4.2
    U = [rho, rho * vx, 0.0, 0.0, P / (G53 - 1) + 0.5 * rho * vx * vx]
    _raw_uniform(g, U)
    for _ in range(10):
        assert g.hydro_step(g.cfl_dt()) == 0
    for f in range(5):
        assert np.all(g.get_state(f) == U[f])
    g.close()


def test_shock_tube_with_fixed_ends_equals_outflow_until_the_waves_arrive():
    N = 96
    x = (np.arange(-NG, N + NG) + 0.5) / N
    rho = np.where(x < 0.5, 1.0, 0.125)
    P = np.where(x < 0.5, 1.0, 0.1)
    shape_g = (1 + 2 * NG, 1 + 2 * NG, N + 2 * NG)
    res = []
    for bc in (O.BC_FIXED, O.BC_OUTFLOW):
        g = O.Grid(N, 1, 1, 1.0 / N, 1.4)
        g.set_face_bc([bc, bc, O.BC_PERIODIC, O.BC_PERIODIC, O.BC_PERIODIC, O.BC_PERIODIC])
        for f, a in enumerate([rho, 0 * x, 0 * x, 0 * x, P / 0.4]):
            g.set_raw(f, np.broadcast_to(a, shape_g).copy())
        t = 0.0
        while t < 0.15:                                      # fastest wave 1.75: travels 0.26 < 0.5
            dt = g.cfl_dt()
            assert g.hydro_step(dt) == 0
            t += dt
        res.append([g.get_state(f) for f in range(5)])
        g.close()
    assert all(np.array_equal(a, b) for a, b in zip(*res))
    assert np.abs(res[0][1]).max() > 0.1


def test_beam_entering_through_a_fixed_face_streams_at_c_hat():
    """Inflow boundary of the paper's streaming tests: ghost cells hold E_r = 1, F_r = c E_r;
    the interior starts almost empty.  The beam fills the box behind a front that moves at c_hat."""
    N, c, c_hat = 128, 1.0, 0.25
    g = O.Grid(N, 1, 1, 1.0 / N, G53, c_hat=c_hat, c=c)
    g.set_params(flags=0)
    g.set_face_bc([O.BC_FIXED, O.BC_OUTFLOW, O.BC_PERIODIC, O.BC_PERIODIC, O.BC_PERIODIC, O.BC_PERIODIC])
    shape_g = (1 + 2 * NG, 1 + 2 * NG, N + 2 * NG)
    i = np.arange(-NG, N + NG)
    Er = np.where(i < 0, 1.0, 1e-8)
    for name, a in (("Er", Er), ("Fx", c * Er), ("rho", np.ones_like(Er))):
        g.set_raw(O.FIELDS.index(name), np.broadcast_to(a, shape_g).copy())
    dt, nsteps = 0.3 / N / c_hat, 200
    for _ in range(nsteps):
        assert g.rad_transport(dt) == 0
    E = g.get_state(5).ravel()
    x = (np.arange(N) + 0.5) / N
    front = c_hat * nsteps * dt                             # 0.47
    assert np.abs(E[x < front - 0.1] - 1.0).max() < 2e-2    # filled with the inflow state
    assert E[x > front + 0.1].max() < 1e-3                  # nothing ahead of the front
    half = x[np.nonzero(E > 0.5)[0][-1]]
    assert abs(half - front) < 0.03
    g.close()


def test_density_power_law_opacities():
    """kappa = kappa0 (rho/rho0)^e (PAPER.md:464 e = 1, PAPER.md:528 e = -1).  With e = -1 the extinction rho kappa is
    the same everywhere whatever the density field, so the radiation evolves as in a uniform medium of the same
    rho kappa; with e = 1 in a uniform medium of density 2 rho0 the law is the constant field 2 kappa0, bit for bit."""
    N, c, c_hat = 64, 1.0, 0.5
    x = (np.arange(N) + 0.5) / N
    E0 = 1.0 + np.exp(-((x - 0.5) / 0.08) ** 2)

    def run(rho, law=None, kfield=None, nsteps=40):
        g = O.Grid(N, 1, 1, 1.0 / N, G53, c_hat=c_hat, c=c)
        g.set_params(flags=O.FLAG_STATIC_MATTER | O.FLAG_TAU_CORR)
        for name, a in (("rho", rho), ("E", 1.5 * rho), ("Er", E0)):
            g.set_state(O.FIELDS.index(name), a.reshape(1, 1, N))
        if law:
            g.set_opacity_law(*law)
        else:
            g.set_state(O.FIELDS.index("kappaR"), np.full((1, 1, N), kfield))
        for _ in range(nsteps):
            assert g.rad_step(0.3 / N / c_hat) == 0
        out = g.get_state(5).ravel(), g.get_state(10).ravel()
        g.close()
        return out

    wavy = 1.0 + 0.5 * np.sin(2 * np.pi * x)
    Er_law, kR = run(wavy, law=(0.0, 50.0, 1.0, -1))
    assert np.abs(kR * wavy - 50.0).max() < 1e-13 * 50
    Er_uni, _ = run(np.ones(N), kfield=50.0)
    assert np.abs(Er_law - Er_uni).max() < 1e-12 and np.abs(Er_uni - E0).max() > 0.05
    Er_a, kR_a = run(np.full(N, 2.0), law=(0.0, 50.0, 1.0, 1))
    Er_b, _ = run(np.full(N, 2.0), kfield=100.0)
    assert np.all(kR_a == 100.0) and np.array_equal(Er_a, Er_b)
