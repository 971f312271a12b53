"""Pins of the oracle's reflecting (solid-wall) boundary, used by the paper's implosion, Su-Olson and shadow
tests.  Checked against what a wall means: the ghost image is the mirror image with
the normal vector component negated (brute force), a closed box conserves mass and energy, a box with walls
equals one half of a mirror-symmetric periodic box of twice the size, and an x<->y-symmetric initial state
stays bitwise symmetric (the paper's claim for its implosion run)."""
import numpy as np

import oracle as O

G14 = 1.4
NG = 4


def test_ghost_image_is_the_mirror_image_with_normal_component_negated():
    nz, ny, nx = 5, 6, 7
    rng = np.random.default_rng(1)
    g = O.Grid(nx, ny, nz, 0.1, G14, c_hat=1.0, c=10.0, bc=O.BC_REFLECTING)
    data = [rng.standard_normal((nz, ny, nx)) for _ in range(9)]
    for f, a in enumerate(data):
        g.set_state(f, a)
    g.fill_boundary(O.FILL_ALL)
    comp = {1: 2, 2: 1, 3: 0, 6: 2, 7: 1, 8: 0}          # field -> numpy axis of its vector component
    for f, a in enumerate(data):
        raw = g.get_raw(f).reshape(nz + 2 * NG, ny + 2 * NG, nx + 2 * NG)
        for K in range(-NG, nz + NG):
            for J in range(-NG, ny + NG):
                for Ii in range(-NG, nx + NG):
                    idx, sign = [], 1.0
                    for axis, (v, n) in enumerate(((K, nz), (J, ny), (Ii, nx))):
                        m = v if 0 <= v < n else (-1 - v if v < 0 else 2 * n - 1 - v)
                        if m != v and comp.get(f) == axis:
                            sign = -sign
                        idx.append(m)
                    assert raw[K + NG, J + NG, Ii + NG] == sign * a[tuple(idx)], (f, K, J, Ii)
    g.close()


def _blob(n, seed=0):
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")
    rho = 1.0 + 0.5 * np.exp(-((X - 0.35) ** 2 + (Y - 0.4) ** 2) / 0.02)
    P = 1.0 + 2.0 * np.exp(-((X - 0.6) ** 2 + (Y - 0.3) ** 2) / 0.01)
    return rho, P


def _set2d(g, rho, vx, vy, P, gamma, nz=2):
    E = P / (gamma - 1) + 0.5 * rho * (vx ** 2 + vy ** 2)
    for f, a in enumerate([rho, rho * vx, rho * vy, 0 * rho, E]):
        g.set_state(f, np.repeat(a[None], nz, axis=0))


def test_closed_box_conserves_mass_and_energy_and_walls_hold():
    n = 24
    rho, P = _blob(n)
    g = O.Grid(n, n, 2, 1.0 / n, G14, bc=O.BC_REFLECTING)
    _set2d(g, rho, 0 * rho, 0 * rho, P, G14)
    m0, e0 = g.get_state(0).sum(), g.get_state(4).sum()
    for _ in range(30):
        assert g.hydro_step(g.cfl_dt()) == 0
    assert abs(g.get_state(0).sum() - m0) < 1e-13 * m0 and abs(g.get_state(4).sum() - e0) < 1e-13 * e0
    assert np.abs(g.get_state(1)).max() > 1e-2             # the gas did move
    assert np.all(g.get_state(3) == 0.0)                   # nothing leaks into the uniform direction
    g.close()


def test_wall_equals_half_of_a_mirror_symmetric_periodic_box():
    """Solution in [0,1]^2 with walls = lower-left quadrant of the periodic solution in [0,2]^2 whose initial state
    is the mirror extension (to round-off: the scheme is mirror symmetric only up to the rounding of HLLC's S*)."""
    n = 16
    rho, P = _blob(n)
    g = O.Grid(n, n, 2, 1.0 / n, G14, bc=O.BC_REFLECTING)
    _set2d(g, rho, 0 * rho, 0 * rho, P, G14)
    ext = lambda a: np.block([[a, a[:, ::-1]], [a[::-1, :], a[::-1, ::-1]]])     # noqa: E731
    h = O.Grid(2 * n, 2 * n, 2, 1.0 / n, G14, bc=O.BC_PERIODIC)
    _set2d(h, ext(rho), 0 * ext(rho), 0 * ext(rho), ext(P), G14)
    for _ in range(12):
        dt = g.cfl_dt()
        assert abs(h.cfl_dt() - dt) < 1e-13 * dt
        assert g.hydro_step(dt) == 0 and h.hydro_step(dt) == 0
    for f in range(5):
        a, b = g.get_state(f)[0], h.get_state(f)[0][:n, :n]
        assert np.abs(a - b).max() < 1e-12 * max(1.0, np.abs(b).max()), f
    g.close(), h.close()


def test_diagonal_symmetry_stays_bitwise_in_a_reflecting_box():
    """with contraction off the implosion problem stays exactly symmetric about the diagonal."""
    n = 20
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")
    inside = X + Y < 0.5                                    # Liska-Wendroff-like corner triangle
    rho = np.where(inside, 0.125, 1.0)
    P = np.where(inside, 0.14, 1.0)
    g = O.Grid(n, n, 2, 1.0 / n, G14, bc=O.BC_REFLECTING)
    _set2d(g, rho, 0 * rho, 0 * rho, P, G14)
    for _ in range(25):
        assert g.hydro_step(g.cfl_dt()) == 0
    r, mx, my, E = (g.get_state(f)[0] for f in (0, 1, 2, 4))
    assert np.array_equal(r, r.T) and np.array_equal(E, E.T) and np.array_equal(mx, my.T)
    assert np.abs(mx).max() > 0.05
    g.close()


def test_radiation_in_a_mirror_box_keeps_its_energy():
    n = 32
    c, c_hat = 1.0, 0.2
    g = O.Grid(n, 1, 1, 1.0 / n, 5.0 / 3.0, c_hat=c_hat, c=c, bc=O.BC_REFLECTING)
    g.set_params(flags=0)
    x = (np.arange(n) + 0.5) / n
    E0 = 1.0 + np.exp(-((x - 0.7) / 0.08) ** 2)
    for name, a in (("Er", E0), ("Fx", 0.3 * c * E0), ("rho", np.ones(n))):
        g.set_state(O.FIELDS.index(name), a.reshape(1, 1, n))
    dt = 0.3 / n / c_hat
    for _ in range(200):                                    # several wall bounces
        assert g.rad_transport(dt) == 0
    E, F = g.get_state(5).ravel(), g.get_state(6).ravel()
    assert abs(E.sum() - E0.sum()) < 1e-12 * E0.sum()
    assert E.min() > 0 and np.all(np.abs(F) <= c * E)
    assert F.sum() < 0.9 * (0.3 * c * E0).sum()             # the walls took up momentum: the net flux sloshes back
    g.close()
