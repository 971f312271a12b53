"""Helpers for the parity tests: build the oracle grid and the CUDA context from the same seeded
host arrays (paper_2110_01792_b200.inputs) and compare them in the norm DESIGN.md section 3 states:
per variable, max |difference| over interior cells divided by max |value|, the three momentum
components pooled and the three radiation-flux components pooled."""
import numpy as np

import oracle as O
from paper_2110_01792_b200 import binding as B

GROUPS = {"rho": ["rho"], "mom": ["mx", "my", "mz"], "E": ["E"], "Er": ["Er"], "Frad": ["Fx", "Fy", "Fz"]}
HYDRO = ["rho", "mom", "E"]
RAD = ["Er", "Frad"]
TOL_ONE_STEP = 1e-12     # BASELINE.json north_star: relative 1e-12 after one step
TOL_100_STEPS = 1e-9     # ... and 1e-9 after 100 steps


def make_oracle(params, fields):
    g = O.Grid(params["nx"], params["ny"], params["nz"], params["dx"], params["gamma"],
               c_hat=params.get("c_hat", 0.0), c=params.get("c", 0.0), bc=params.get("bc", 0))
    if "a_rad" in params:
        g.set_constants(params["a_rad"], params["kB_mu"])
    g.set_params(cfl=params.get("cfl", 0.3), flags=params.get("flags", 0))
    g.set_all(fields)
    return g


def make_gpu(params, fields, path=None, **kw):
    """path: qk_set_flatten_path (1 two passes, 2 one pass; None = the library's choice by box size)"""
    ctx = B.from_params(params, fields, **kw)
    if path is not None:
        ctx.qk_set_flatten_path(path)
    return ctx


def rel_errors(ref: dict, got: dict, groups=None):
    out = {}
    for gname in (groups or GROUPS):
        names = GROUPS[gname]
        num = max(float(np.max(np.abs(ref[n] - got[n]))) for n in names)
        den = max(float(np.max(np.abs(ref[n]))) for n in names)
        out[gname] = num / den if den > 0 else num
    return out


def assert_parity(ref, got, tol, groups=None, what=""):
    errs = rel_errors(ref, got, groups)
    bad = {k: v for k, v in errs.items() if not (v <= tol)}
    assert not bad, "%s: relative max-norm error above %g: %s (all: %s)" % (what, tol, bad, errs)
    return errs


def assert_bitwise(ref, got, names, what=""):
    """every listed field equal bit for bit (+0 == -0 counts as equal, NaN as different): the number of mismatching
    cells is reported, so 'bit-identical' is asserted, not inferred from a tolerance"""
    mism = count_mismatch(ref, got, names)
    assert not any(mism.values()), "%s: cells that differ from the oracle: %s" % (what, mism)
    return mism


def count_mismatch(ref, got, names):
    return {n: int(np.count_nonzero(ref[n] != got[n])) for n in names}


def sub_box(fields, lo, size):
    """Periodic sub-box [lo, lo+size) of every field (modular indices, so it may straddle the wrap)."""
    out = {}
    for name, a in fields.items():
        idx = [(lo[d] + np.arange(size[d])) % a.shape[d] for d in range(3)]
        out[name] = np.ascontiguousarray(a[np.ix_(*idx)])
    return out
