"""CPU ORACLE (test infrastructure, not the product).

ctypes loader for the plain-C restatement of the paper's cell update in this folder
(qk_oracle.h, grid.c, hydro.c, radiation.c, exchange.c).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package; nothing under paper_2110_01792_b200/ does, and this package imports
nothing from there.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = ["grid.c", "hydro.c", "radiation.c", "exchange.c"]
_LIB = os.path.join(_HERE, "libqk_oracle.so")

NG = 4
FIELDS = ["rho", "mx", "my", "mz", "E", "Er", "Fx", "Fy", "Fz", "kappaP", "kappaR", "src"]
BC_PERIODIC, BC_OUTFLOW, BC_REFLECTING, BC_FIXED = 0, 1, 2, 3
FLAG_TAU_CORR, FLAG_STATIC_MATTER, FLAG_NEWTON_LITERAL = 1, 2, 4
FLAG_PLM, FLAG_EDDINGTON, FLAG_MINERBO, FLAG_NO_DKAPPA_DT = 8, 16, 32, 64
EOS_IDEAL, EOS_ALPHA_T3 = 0, 1
FILL_HYDRO, FILL_RAD, FILL_ALL = 1, 2, 7


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (no FMA contraction) -fopenmp (independent cells dealt out to
    threads; no result bit depends on the thread count) -> libqk_oracle.so"""
    srcs = [os.path.join(_HERE, s) for s in _SRCS]
    deps = srcs + [os.path.join(_HERE, "qk_oracle.h")]
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(d) for d in deps)):
        return _LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-fopenmp", "-shared", "-fPIC",
           "-o", _LIB] + srcs + ["-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    # idle worker threads sleep instead of spinning, so that several processes using the oracle at once (pytest-xdist,
    # a test next to a bench) do not starve each other; read by libgomp when it is loaded
    os.environ.setdefault("OMP_WAIT_POLICY", "passive")
    L = C.CDLL(build())
    d, i, p, u = C.c_double, C.c_int, C.c_void_p, C.c_uint
    dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
    sig = {
        "orc_create": (p, [i, i, i, d, d, d, d, i]),
        "orc_destroy": (None, [p]),
        "orc_ncells_total": (C.c_longlong, [p]),
        "orc_set_constants": (None, [p, d, d]),
        "orc_set_params": (None, [p, d, d, i, i, u]),
        "orc_set_eos": (None, [p, i, d]),
        "orc_set_opacity_law": (None, [p, d, d, d, i]),
        "orc_set_opacity_law_T": (None, [p, d, d, d, i, d, i]),
        "orc_set_wavespeed_floor": (None, [p, d]),
        "orc_set_threads": (None, [i]),
        "orc_get_threads": (i, []),
        "orc_rad_hll_floor": (i, [d, d, dp, dp, i, d, u, d, dp]),
        "orc_temp_power": (d, [d, d, i]),
        "orc_set_face_bc": (i, [p, np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")]),
        "orc_set_field": (None, [p, i, dp]),
        "orc_get_field": (None, [p, i, dp]),
        "orc_get_raw": (None, [p, i, dp]),
        "orc_set_raw": (None, [p, i, dp]),
        "orc_get_info": (None, [p, np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")]),
        "orc_fill_boundary": (None, [p, i]),
        "orc_fill_field": (None, [p, i]),
        "orc_cfl_dt": (d, [p]),
        "orc_hydro_step": (i, [p, d]),
        "orc_rad_transport": (i, [p, d]),
        "orc_exchange": (i, [p, d]),
        "orc_rad_step": (i, [p, d]),
        "orc_rhd_step": (i, [p, d]),
        "orc_nsub_for": (i, [p, d]),
        "orc_cons_to_prim": (None, [d, dp, dp]),
        "orc_ppm_faces": (None, [dp, dp, dp]),
        "orc_plm_faces": (None, [dp, dp, dp]),
        "orc_closure_k": (None, [u, dp, i, dp, dp]),
        "orc_mc_slope": (d, [d, d, d]),
        "orc_flatten_1d": (d, [d, dp, dp]),
        "orc_hllc": (None, [d, dp, dp, dp]),
        "orc_eddington_factor": (d, [d]),
        "orc_minerbo_factor": (d, [d]),
        "orc_closure": (None, [dp, i, dp, dp]),
        "orc_rad_phys_flux": (None, [d, d, dp, i, dp, dp]),
        "orc_rad_hll": (i, [d, d, dp, dp, i, d, u, dp]),
        "orc_exchange_cell": (i, [p, d, d, dp, dp, dp, dp, d, d, np.ctypeslib.ndpointer(dtype=np.int32)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


class Grid:
    """One uniform box with 4 ghost zones, advanced by the oracle."""

    def __init__(self, nx, ny, nz, dx, gamma, c_hat=0.0, c=0.0, bc=BC_PERIODIC):
        self.L = lib()
        self.nx, self.ny, self.nz = nx, ny, nz
        self.h = self.L.orc_create(nx, ny, nz, dx, gamma, c_hat, c, bc)
        if not self.h:
            raise MemoryError("orc_create failed")

    def close(self):
        if self.h:
            self.L.orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # parameters
    def set_constants(self, a_rad, kB_mu):
        self.L.orc_set_constants(self.h, a_rad, kB_mu)

    def set_params(self, cfl=0.3, newton_tol=1e-10, newton_maxit=400, nsub_max=10, flags=0):
        self.L.orc_set_params(self.h, cfl, newton_tol, newton_maxit, nsub_max, flags)

    def set_opacity_law(self, kP0, kR0, rho0, exponent):
        self.L.orc_set_opacity_law(self.h, kP0, kR0, rho0, exponent)

    def set_opacity_law_T(self, kP0, kR0, rho0, exponent, T0, texp2):
        """kappa = kappa0 (rho/rho0)^exponent (T/T0)^(texp2/2)"""
        self.L.orc_set_opacity_law_T(self.h, kP0, kR0, rho0, exponent, T0, texp2)

    def set_wavespeed_floor(self, s_floor):
        self.L.orc_set_wavespeed_floor(self.h, s_floor)

    def set_face_bc(self, bc6):
        """Per-face boundary types (x-lo, x-hi, y-lo, y-hi, z-lo, z-hi)."""
        rc = self.L.orc_set_face_bc(self.h, np.ascontiguousarray(bc6, dtype=np.int32))
        assert rc == 0, "periodic must be set on both faces of an axis"

    def set_eos(self, eos, alpha=0.0):
        self.L.orc_set_eos(self.h, eos, alpha)

    # state
    def set_state(self, field, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == (self.nz, self.ny, self.nx), a.shape
        self.L.orc_set_field(self.h, field, a)

    def get_state(self, field):
        out = np.empty((self.nz, self.ny, self.nx), dtype=np.float64)
        self.L.orc_get_field(self.h, field, out)
        return out

    def get_raw(self, field):
        out = np.empty((self.nz + 2 * NG, self.ny + 2 * NG, self.nx + 2 * NG), dtype=np.float64)
        self.L.orc_get_raw(self.h, field, out)
        return out

    def set_raw(self, field, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == (self.nz + 2 * NG, self.ny + 2 * NG, self.nx + 2 * NG)
        self.L.orc_set_raw(self.h, field, a)

    def set_all(self, fields: dict):
        for name, a in fields.items():
            self.set_state(FIELDS.index(name), a)

    def get_all(self, names=None):
        names = names or FIELDS
        return {n: self.get_state(FIELDS.index(n)) for n in names}

    def info(self):
        out = np.zeros(7, dtype=np.int64)
        self.L.orc_get_info(self.h, out)
        keys = ["nsub", "newton_fail_cells", "newton_max_iters", "newton_total_iters",
                "bad_state_cells", "fallback_states", "guard_faces"]
        return dict(zip(keys, (int(v) for v in out)))

    # operations
    def fill_boundary(self, which=FILL_ALL):
        self.L.orc_fill_boundary(self.h, which)

    def cfl_dt(self):
        return float(self.L.orc_cfl_dt(self.h))

    def hydro_step(self, dt):
        return int(self.L.orc_hydro_step(self.h, dt))

    def rad_transport(self, dt):
        return int(self.L.orc_rad_transport(self.h, dt))

    def exchange(self, dt):
        return int(self.L.orc_exchange(self.h, dt))

    def rad_step(self, dt):
        return int(self.L.orc_rad_step(self.h, dt))

    def rhd_step(self, dt):
        return int(self.L.orc_rhd_step(self.h, dt))

    def nsub_for(self, dt):
        return int(self.L.orc_nsub_for(self.h, dt))


def set_threads(n):
    """worker threads of the oracle's loops over cells (no result depends on it)"""
    lib().orc_set_threads(int(n))


def get_threads():
    return int(lib().orc_get_threads())
