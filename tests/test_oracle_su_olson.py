"""The paper's Su-Olson problem (eq 56) on the oracle, with every printed parameter.  The paper
compares with the semi-analytic transport / diffusion tables of Su & Olson (1997), which are not in this container
 and are not reproduced here; what the paper's text and the equations do fix is pinned instead:

* the energy budget: the walls reflect and c_hat = c, so eq 26 + eq 27 + the flux form of eq 11 give
  sum (E_g + E_r) dx = initial + integral of S dx dt = 30 * 2e-10 + Q a_r T_H^4 x_0 t = 5 at t = t_0 = 10, to round-off --
  a source applied twice per step, to the wrong cells, scaled by c/c_hat or leaking through the wall misses it;
* causality: beyond x_0 + c t the radiation is still at its initial value;
* the gas lags the radiation while the source is on (E_g = a_r T^4 <= E_r), E_r falls monotonically away from the source,
  and at t = 10 the source region is the brightest, the medium far from it still dark ("radiation penetrating a cold
  medium").
"""
import numpy as np

import oracle as O
from paper_2110_01792_b200 import inputs as I


def su_olson_oracle(n, nsteps=None):
    params, fields, extra = I.su_olson(n)
    g = O.Grid(params["nx"], 1, 1, params["dx"], params["gamma"], c_hat=params["c_hat"], c=params["c"], bc=params["bc"])
    g.set_constants(params["a_rad"], params["kB_mu"])
    g.set_params(cfl=params["cfl"], flags=params["flags"])
    g.set_eos(O.EOS_ALPHA_T3, extra["eos_alpha"])
    g.set_all(fields)
    g.set_state(O.FIELDS.index("src"), extra["src"])
    steps = int(round(extra["t_end"] / extra["dt"])) if nsteps is None else nsteps
    threads = O.get_threads()
    O.set_threads(1)                   # one row of cells: the thread team costs more than the loop (no result depends on it)
    try:
        for _ in range(steps):
            assert g.rad_step(extra["dt"]) == 0
    finally:
        O.set_threads(threads)
    out = {k: g.get_state(O.FIELDS.index(k)).ravel() for k in ("E", "Er", "Fx", "mx")}
    info = g.info()
    g.close()
    return params, extra, steps, out, info


def check_su_olson(params, extra, steps, out, info):
    """the pins of the header, shared with the GPU test (which passes the CUDA path's arrays)"""
    dx, n = params["dx"], params["nx"]
    t = steps * extra["dt"]
    x = (np.arange(n) + 0.5) * dx
    Eg, Er = out["E"], out["Er"]
    budget = float(np.sum(Eg + Er, dtype=np.longdouble)) * dx
    expect = 2.0 * extra["e_init"] * extra["length"] + 1.0 * extra["x0"] * t       # S = Q a_r T_H^4 = 1 on [0, x_0)
    assert abs(budget - expect) < 1e-12 * expect, (budget, expect)
    assert info["newton_fail_cells"] == 0 and info["fallback_states"] == 0
    assert np.all(out["mx"] == 0.0)                                   # gas at rest: v/c terms dropped
    ahead = x > extra["x0"] + params["c"] * t + 1.5                   # 1.5 = 75 cells: the PPM stencil's numerical precursor
    assert ahead.any() and np.abs(Er[ahead] - extra["e_init"]).max() < 1e-6 * extra["e_init"]
    assert np.abs(Eg[ahead] - extra["e_init"]).max() < 1e-6 * extra["e_init"]
    lit = Er > 1e-6
    assert np.all(Eg[lit] <= Er[lit] * (1 + 1e-12))                   # the gas lags the radiation while the source is on
    outside = x > extra["x0"]
    assert np.all(np.diff(Er[outside & lit]) < 0.0) and np.all(Er > 0.0) and np.all(Eg > 0.0)
    assert np.all(np.abs(out["Fx"]) <= params["c"] * Er * (1 + 1e-12))
    return budget, Er


def test_su_olson_energy_budget_causality_and_shape():
    # the paper's grid and timestep, a fifth of its run (t = 2: every pin holds at any time; the run to t_0 = 10 is
    # tests/test_gpu_parity.py's, on the CUDA path, with the same checks)
    assert int(round(I.su_olson(1500)[2]["t_end"] / I.su_olson(1500)[2]["dt"])) == 1250
    params, extra, steps, out, info = su_olson_oracle(1500, 250)
    budget, Er = check_su_olson(params, extra, steps, out, info)
    # brightest in the source region, energy a mean free path (= 1) out, dark far away; most of what was injected is
    # still within x < 5
    assert Er.argmax() == 0 and Er[int(1.0 / params["dx"])] > 0.05 * Er[0] and Er[int(9.0 / params["dx"])] < 1e-3 * Er[0]
    near = (np.arange(params["nx"]) + 0.5) * params["dx"] < 5.0
    assert float(np.sum((out["E"] + Er)[near])) * params["dx"] > 0.9 * budget


def test_su_olson_converges_with_resolution():
    """self-convergence where no table is available: N = 300 -> 600 -> 1200 (the source edge x_0 on a cell face in each)
    at t = 0.96 (24, 48, 96 steps at the problem's CFL number), E_r at fixed points (x = 0.25, 1.0): the differences
    shrink"""
    pts = (0.25, 1.0)
    vals = []
    for n in (300, 600, 1200):
        params, fields, extra = I.su_olson(n)
        steps = 24 * n // 300
        assert abs(steps * extra["dt"] - 0.96) < 1e-12
        p, e, s, out, info = su_olson_oracle(n, steps)
        x = (np.arange(n) + 0.5) * p["dx"]
        vals.append([np.interp(q, x, out["Er"]) for q in pts])
    d1 = np.abs(np.array(vals[1]) - np.array(vals[0]))
    d2 = np.abs(np.array(vals[2]) - np.array(vals[1]))
    assert np.all(d2 < 0.7 * d1), (d1, d2)
