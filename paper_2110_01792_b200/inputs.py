"""Seeded synthetic inputs shared by the oracle tests, the GPU parity
tests and bench.py.  This module holds none of the method's arithmetic: it only draws
numbers and shapes them like the paper's uniform-grid workloads (Sedov blast,
PAPER.md:572-574; radiating shell) and like BASELINE.json's configs.
The same host arrays are handed to the oracle and to the CUDA library.

Every generator returns (params, fields): params is a dict for qk_init / qk_set_* and
fields maps field name -> float64 array of shape (nz, ny, nx), x fastest.
"""
from __future__ import annotations

import numpy as np

FIELDS = ["rho", "mx", "my", "mz", "E", "Er", "Fx", "Fy", "Fz", "kappaP", "kappaR"]
BC_PERIODIC, BC_OUTFLOW, BC_REFLECTING, BC_FIXED = 0, 1, 2, 3
FLAG_TAU_CORR, FLAG_STATIC_MATTER, FLAG_NEWTON_LITERAL = 1, 2, 4
FLAG_PLM, FLAG_EDDINGTON, FLAG_MINERBO = 8, 16, 32     # scheme variants


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _centres(n, lo=0.0, hi=1.0):
    return lo + (np.arange(n) + 0.5) * ((hi - lo) / n)


def spectral_field(rng, shape, kmin=1, kmax=16, slope=-2.0):
    """White N(0,1) noise filtered to |k|^slope on integer wavenumbers kmin<=|k|<=kmax,
    zero mean, unit variance (BASELINE.json config 2: 'power spectrum k^-2 on modes 1..16')."""
    nz, ny, nx = shape
    w = rng.standard_normal(shape)
    wk = np.fft.rfftn(w)
    kz = np.fft.fftfreq(nz, 1.0 / nz)[:, None, None]
    ky = np.fft.fftfreq(ny, 1.0 / ny)[None, :, None]
    kx = np.fft.rfftfreq(nx, 1.0 / nx)[None, None, :]
    kk = np.sqrt(kx * kx + ky * ky + kz * kz)
    filt = np.zeros_like(kk)
    m = (kk >= kmin) & (kk <= kmax)
    filt[m] = kk[m] ** slope
    out = np.fft.irfftn(wk * filt, s=shape, axes=(0, 1, 2))
    out -= out.mean()
    out /= out.std()
    return np.ascontiguousarray(out)


def _zeros(shape):
    return np.zeros(shape, dtype=np.float64)


def _hydro_fields(rho, vx, vy, vz, P, gamma):
    E = P / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return {"rho": rho, "mx": rho * vx, "my": rho * vy, "mz": rho * vz, "E": E}


def _fill_missing(fields, shape):
    for name in FIELDS:
        if name not in fields:
            fields[name] = _zeros(shape)
        fields[name] = np.ascontiguousarray(fields[name], dtype=np.float64)
    return fields


def config1(n=32, seed=1001, noise=1e-3):
    """BASELINE.json configs[0]: advected density wave + velocity noise, periodic, gamma=5/3."""
    shape = (n, n, n)
    gamma = 5.0 / 3.0
    rng = _rng(seed)
    x = _centres(n)[None, None, :]
    rho = np.broadcast_to(1.0 + 0.1 * np.sin(2.0 * np.pi * x), shape).copy()
    vx = 1.0 + noise * rng.standard_normal(shape)
    vy = noise * rng.standard_normal(shape)
    vz = noise * rng.standard_normal(shape)
    P = np.ones(shape)
    params = dict(nx=n, ny=n, nz=n, dx=1.0 / n, gamma=gamma, c_hat=0.0, c=0.0, bc=BC_PERIODIC,
                  cfl=0.3, flags=0, name="config1_hydro_wave")
    return params, _fill_missing(_hydro_fields(rho, vx, vy, vz, P, gamma), shape)


def config2(n=256, seed=1002, mach=2.0, kmax=16, shape=None):
    """BASELINE.json configs[1]: supersonic-turbulence-like state, periodic, gamma=5/3."""
    shape = shape or (n, n, n)
    gamma = 5.0 / 3.0
    rng = _rng(seed)
    kmax = min(kmax, max(1, min(shape) // 4))
    s = 0.5 * spectral_field(rng, shape, kmax=kmax)
    rho = np.exp(s - 0.125)
    v = [spectral_field(rng, shape, kmax=kmax) for _ in range(3)]
    rms = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    scale = mach * np.sqrt(gamma) / rms
    P = np.ones(shape)
    params = dict(nx=shape[2], ny=shape[1], nz=shape[0], dx=1.0 / shape[2], gamma=gamma, c_hat=0.0, c=0.0,
                  bc=BC_PERIODIC, cfl=0.3, flags=0, name="config2_hydro_turbulence")
    return params, _fill_missing(_hydro_fields(rho, v[0] * scale, v[1] * scale, v[2] * scale, P, gamma), shape)


def config3(n=128, seed=1003, shape=None, tau_corr=False):
    """BASELINE.json configs[2]: radiation only, static matter, outflow, c=1, c_hat=0.1.
    tau_corr=True switches on the optical-depth correction of reading R6 (off by default: DESIGN.md section 3)."""
    shape = shape or (n, n, n)
    gamma = 5.0 / 3.0
    rng = _rng(seed)
    dx = 1.0 / shape[2]
    c, c_hat = 1.0, 0.1
    rho = np.ones(shape)
    Er = 10.0 ** rng.uniform(-2.0, 0.0, shape)
    f = rng.uniform(0.0, 0.9, shape)
    nvec = [rng.standard_normal(shape) for _ in range(3)]
    norm = np.sqrt(nvec[0] ** 2 + nvec[1] ** 2 + nvec[2] ** 2)
    tau = 10.0 ** rng.uniform(-3.0, 2.0, shape)
    kappa = tau / (rho * dx)
    fields = {"rho": rho, "mx": _zeros(shape), "my": _zeros(shape), "mz": _zeros(shape),
              "E": np.full(shape, 1.5), "Er": Er,
              "Fx": f * c * Er * nvec[0] / norm, "Fy": f * c * Er * nvec[1] / norm,
              "Fz": f * c * Er * nvec[2] / norm, "kappaP": kappa, "kappaR": kappa.copy()}
    params = dict(nx=shape[2], ny=shape[1], nz=shape[0], dx=dx, gamma=gamma, c_hat=c_hat, c=c,
                  bc=BC_OUTFLOW, cfl=0.3, a_rad=1.0, kB_mu=1.0,
                  flags=FLAG_STATIC_MATTER | (FLAG_TAU_CORR if tau_corr else 0), name="config3_radiation_static")
    return params, _fill_missing(fields, shape)


def config4(n=256, seed=1004, kmax=16, shape=None, chat_ratio=0.01, tau_corr=False):
    """BASELINE.json configs[3]/[4]: coupled RHD, periodic, c/c_s ~ 100, c_hat/c = 0.01."""
    shape = shape or (n, n, n)
    gamma = 5.0 / 3.0
    rng = _rng(seed)
    dx = 1.0 / shape[2]
    kmax = min(kmax, max(1, min(shape) // 4))
    c = 100.0 * np.sqrt(gamma)
    c_hat = chat_ratio * c      # BASELINE configs[3]: c_hat/c = 0.01 (N_sub = 1); larger ratios force subcycling
    rho = np.exp(0.5 * spectral_field(rng, shape, kmax=kmax) - 0.125)
    tf = spectral_field(rng, shape, kmax=kmax)
    ranks = np.empty(tf.size, dtype=np.float64)
    ranks[np.argsort(tf, axis=None, kind="stable")] = (np.arange(tf.size) + 0.5) / tf.size
    T = 0.5 * 4.0 ** ranks.reshape(shape)
    v = [spectral_field(rng, shape, kmax=kmax) for _ in range(3)]
    rms = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    scale = np.sqrt(gamma) / rms
    vx, vy, vz = v[0] * scale, v[1] * scale, v[2] * scale
    a_rad, kB_mu = 1.0, 1.0
    E = rho * kB_mu * T / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    Er = a_rad * T ** 4 * np.maximum(0.1, 1.0 + 0.1 * rng.standard_normal(shape))
    tau = 10.0 ** rng.uniform(-2.0, 2.0, shape)
    kappa = tau / (rho * dx)
    fields = {"rho": rho, "mx": rho * vx, "my": rho * vy, "mz": rho * vz, "E": E, "Er": Er,
              "kappaP": kappa, "kappaR": kappa.copy()}
    params = dict(nx=shape[2], ny=shape[1], nz=shape[0], dx=dx, gamma=gamma, c_hat=c_hat, c=c,
                  bc=BC_PERIODIC, cfl=0.3, a_rad=a_rad, kB_mu=kB_mu, flags=FLAG_TAU_CORR if tau_corr else 0,
                  name="config4_rhd")
    return params, _fill_missing(fields, shape)


def config5(n=512, seed=1005):
    p, f = config4(n=n, seed=seed)
    p["name"] = "config5_rhd_512"
    return p, f


def sedov(n=256):
    """The paper's hydro benchmark: [-1,1]^3 periodic, rho=1, v=0, P=10 (r<0.1) else 0.1."""
    shape = (n, n, n)
    gamma = 5.0 / 3.0
    x = _centres(n, -1.0, 1.0)
    r2 = x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2
    P = np.where(r2 < 0.01, 10.0, 0.1)
    z = _zeros(shape)
    params = dict(nx=n, ny=n, nz=n, dx=2.0 / n, gamma=gamma, c_hat=0.0, c=0.0, bc=BC_PERIODIC,
                  cfl=0.25, flags=0, name="sedov")
    return params, _fill_missing(_hydro_fields(np.ones(shape), z, z.copy(), z.copy(), P, gamma), shape)


def su_olson(n=1500):
    """The paper's Su-Olson problem (eq 56) with every printed parameter: a_r = c = 1, no reduced
    speed of light, kappa_P = kappa_R = 1, rho = 1, gas at rest (v/c terms dropped), source Q a_r T_H^4 = 1 in
    0 <= x < x_0 = 0.5 while t < t_0 = 10, initial E_g = E_r = 1e-10, reflecting walls on [0, 30], N_x = 1500, CFL 0.4,
    heat capacity C_v = alpha T^3 with alpha = 4 a_r / epsilon, epsilon = 1 (eq 55).  One row of cells in y and z.
    Returns (params, fields, extra): extra holds what the generic setters do not (source rate, EOS, end time)."""
    shape = (1, 1, n)
    L, x0, t0 = 30.0, 0.5, 10.0
    dx = L / n
    x = _centres(n, 0.0, L)
    e0 = 1e-10
    fields = {"rho": np.ones(shape), "E": np.full(shape, e0), "Er": np.full(shape, e0),
              "kappaP": np.ones(shape), "kappaR": np.ones(shape)}
    src = np.where(x < x0, 1.0 / (2.0 * x0), 0.0).reshape(shape)
    params = dict(nx=n, ny=1, nz=1, dx=dx, gamma=5.0 / 3.0, c_hat=1.0, c=1.0, bc=BC_REFLECTING, cfl=0.4,
                  a_rad=1.0, kB_mu=1.0, flags=FLAG_STATIC_MATTER, name="su_olson")
    extra = dict(src=np.ascontiguousarray(src), eos_alpha=4.0, t_end=t0, x0=x0, dt=0.4 * dx / 1.0, e_init=e0, length=L)
    return params, _fill_missing(fields, shape), extra


def ragged_hydro(shape=(19, 22, 37), seed=7, bc=BC_PERIODIC, mach=1.5):
    """Small non-cubic, non-multiple-of-tile box with shocks: several tiles and a ragged tail."""
    p, f = config2(seed=seed, mach=mach, kmax=3, shape=shape)
    p["bc"] = bc
    p["name"] = "ragged_hydro"
    return p, f


def ragged_rhd(shape=(18, 21, 35), seed=11, bc=BC_PERIODIC, tau_corr=False):
    p, f = config4(seed=seed, kmax=3, shape=shape, tau_corr=tau_corr)
    p["bc"] = bc
    p["name"] = "ragged_rhd"
    return p, f


CONFIGS = {"config1": config1, "config2": config2, "config3": config3, "config4": config4,
           "config5": config5, "sedov": sedov}
