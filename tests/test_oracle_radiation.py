"""Pins for the radiation transport part of the CPU oracle (oracle/radiation.c).  CPU only."""
import os

import numpy as np

import oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))


def test_closure_values_and_identities():
    """eq 23-25: chi(0)=1/3, chi(1)=1, chi(0.9) by hand; trace T = 1;
    T_nn = chi along the flux; isotropic when F = 0."""
    L = O.lib()
    for line in open(os.path.join(HERE, "golden", "closure_values.txt")):
        if line.strip() and not line.startswith("#"):
            f, chi = (float(x) for x in line.split())
            assert abs(L.orc_eddington_factor(f) - chi) < 2e-6
    rng = np.random.default_rng(2)
    T = np.zeros(3); chi = np.zeros(1)
    for _ in range(100):
        n = rng.standard_normal(3); n /= np.linalg.norm(n)
        fmag = rng.uniform(0, 1.3)
        f = fmag * n
        cols = []
        for d in range(3):
            L.orc_closure(f, d, T, chi)
            cols.append(T.copy())
        Tm = np.array(cols)
        assert abs(np.trace(Tm) - 1.0) < 1e-14
        assert np.allclose(Tm, Tm.T, atol=1e-15)
        assert abs(n @ Tm @ n - chi[0]) < 1e-14
        assert abs(chi[0] - L.orc_eddington_factor(min(fmag, 1.0))) < 1e-14   # clamp for the closure only
        t = np.cross(n, rng.standard_normal(3)); t /= np.linalg.norm(t)
        assert abs(t @ Tm @ t - 0.5 * (1 - chi[0])) < 1e-14
    L.orc_closure(np.zeros(3), 1, T, chi)
    assert np.array_equal(T, np.array([0.0, 1.0 / 3.0, 0.0])) or np.allclose(T, [0, 1 / 3, 0], atol=1e-16)


def test_hll_consistency_bitwise():
    L = O.lib()
    rng = np.random.default_rng(3)
    G, Gp, Tnn = np.zeros(4), np.zeros(4), np.zeros(1)
    for _ in range(50):
        n = rng.standard_normal(3); n /= np.linalg.norm(n)
        S = np.array([np.exp(rng.standard_normal()), *(rng.uniform(0, 0.99) * n)])
        for d in range(3):
            L.orc_rad_phys_flux(1.0, 0.1, S, d, Gp, Tnn)
            L.orc_rad_hll(1.0, 0.1, S, S, d, 5.0, O.FLAG_TAU_CORR, G)
            assert np.array_equal(G, Gp)
            # eq 11: E_r flux is (c_hat/c) F_n
            assert abs(Gp[0] - 0.1 * S[0] * S[1 + d]) < 1e-15


def _rad_grid(N, c, c_hat, bc=O.BC_PERIODIC, flags=0, dx=None):
    g = O.Grid(N, 1, 1, dx or 1.0 / N, 5.0 / 3.0, c_hat=c_hat, c=c, bc=bc)
    g.set_params(flags=flags)
    return g


def _set1d(g, N, **kw):
    for name, a in kw.items():
        g.set_state(O.FIELDS.index(name), np.asarray(a, dtype=float).reshape(1, 1, N))


def test_linear_wave_speed_and_order():
    """Small-amplitude wave about an isotropic field travels at c_hat*sqrt(chi(0)) = c_hat/sqrt(3)
    (eq 11-12 with eq 24); error after one period converges at second order."""
    c, c_hat, A = 1.0, 0.1, 1e-6
    errs = []
    for N in (16, 32, 64, 128):
        g = _rad_grid(N, c, c_hat)
        x = (np.arange(N) + 0.5) / N
        E0 = 1.0 + A * np.sin(2 * np.pi * x)
        F0 = A * c / np.sqrt(3.0) * np.sin(2 * np.pi * x)
        _set1d(g, N, Er=E0, Fx=F0, rho=np.ones(N))
        period = 1.0 / (c_hat / np.sqrt(3.0))
        nsteps = int(np.ceil(period / (0.3 / N / c_hat)))
        for _ in range(nsteps):
            assert g.rad_transport(period / nsteps) == 0
        errs.append(np.abs(g.get_state(5).ravel() - E0).mean() / A)
    orders = [np.log2(errs[n] / errs[n + 1]) for n in range(3)]
    assert errs[-1] < 2e-3 and all(1.6 < o < 2.7 for o in orders), (errs, orders)


def test_streaming_tophat_causal_positive_conservative():
    """f = 1 top-hat: moves at c_hat, E_r > 0, |F| <= cE_r, sum conserved."""
    c, c_hat, N = 1.0, 0.1, 128
    g = _rad_grid(N, c, c_hat)
    x = (np.arange(N) + 0.5) / N
    E0 = np.where((x > 0.2) & (x < 0.4), 1.0, 1e-3)
    _set1d(g, N, Er=E0, Fx=c * E0, rho=np.ones(N))
    dt = 0.3 / N / c_hat
    nsteps = 100
    for _ in range(nsteps):
        assert g.rad_transport(dt) == 0
    E, F = g.get_state(5).ravel(), g.get_state(6).ravel()
    assert E.min() > 0 and np.all(np.abs(F) <= c * E * (1 + 1e-12))
    assert abs(E.sum() - E0.sum()) < 1e-12 * E0.sum()
    centroid0 = (x * (E0 - 1e-3)).sum() / (E0 - 1e-3).sum()
    centroid = (x * (E - 1e-3)).sum() / (E - 1e-3).sum()
    assert abs((centroid - centroid0) - c_hat * nsteps * dt) < 0.01


def test_transport_conservation_3d_periodic():
    shape = (8, 9, 10)
    rng = np.random.default_rng(4)
    c, c_hat = 1.0, 0.1
    g = O.Grid(shape[2], shape[1], shape[0], 0.1, 5 / 3, c_hat=c_hat, c=c)
    E = np.exp(0.3 * rng.standard_normal(shape))
    n = rng.standard_normal((3,) + shape); n /= np.sqrt((n ** 2).sum(0))
    f = rng.uniform(0, 0.8, shape)
    g.set_state(0, np.ones(shape)); g.set_state(5, E)
    for a in range(3):
        g.set_state(6 + a, f * c * E * n[a])
    g.set_state(10, 10.0 ** rng.uniform(-1, 2, shape))
    sums0 = [g.get_state(k).sum() for k in range(5, 9)]
    for _ in range(4):
        assert g.rad_transport(0.3 * 0.1 / c_hat) == 0
    for k in range(4):
        assert abs(g.get_state(5 + k).sum() - sums0[k]) < 1e-12 * np.abs(g.get_state(5 + k)).sum()
    assert g.get_state(5).min() > 0


def test_uniform_radiation_bitwise_invariant():
    shape = (5, 6, 7)
    g = O.Grid(7, 6, 5, 0.1, 5 / 3, c_hat=0.1, c=1.0, bc=O.BC_OUTFLOW)
    g.set_state(0, np.ones(shape)); g.set_state(5, np.full(shape, 0.7)); g.set_state(10, np.full(shape, 3.0))
    g.set_state(7, np.full(shape, 0.2))
    for _ in range(3):
        g.rad_transport(0.3)
    assert np.array_equal(g.get_state(5), np.full(shape, 0.7))
    assert np.array_equal(g.get_state(7), np.full(shape, 0.2))


def test_split_scheme_diffusion_factor():
    """kappa_P = 0, kappa_R > 0, tau_cell >> 1: transport + backward-Euler flux damping after
    each full RK2 substep (eq 39) diffuses a Gaussian with
    D_eff = D (1 + rho kappa_R c_hat dt / 2), D = c_hat/(3 rho kappa_R): the excess over D is a
    property of the Lie splitting at fixed CFL and pins the ordering 'exchange once per subcycle'."""
    c, c_hat, N = 1.0, 1.0, 128
    dx = 1.0 / N
    for tau_cell, lo, hi in ((10.0, 2.2, 2.8), (100.0, 13.0, 18.0)):
        g = _rad_grid(N, c, c_hat, flags=O.FLAG_TAU_CORR | O.FLAG_STATIC_MATTER)
        x = (np.arange(N) + 0.5) / N
        s0 = 0.06
        E0 = 1.0 + np.exp(-0.5 * ((x - 0.5) / s0) ** 2)
        kap = tau_cell / dx
        _set1d(g, N, Er=E0, rho=np.ones(N), kappaR=np.full(N, kap), E=np.ones(N))
        dt = 0.3 * dx / c_hat
        D = c_hat / (3.0 * kap)
        nsteps = 400
        for _ in range(nsteps):
            assert g.rad_step(dt) == 0
        E = g.get_state(5).ravel() - 1.0
        var = ((x - 0.5) ** 2 * E).sum() / E.sum()
        ratio = (var - s0 ** 2) / (2 * D * nsteps * dt)
        assert lo < ratio < hi, (tau_cell, ratio, 1 + 0.5 * kap * c_hat * dt)
