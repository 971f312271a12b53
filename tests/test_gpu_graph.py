"""Replayable step (qk_graph_capture / qk_graph_launch, include/qk.h): one qk_hydro_step_cfl or qk_rhd_step_cfl
recorded as a CUDA graph.  The replay must be the ordinary step bit for bit -- and therefore the oracle's -- with the
same counters and the same device-resident timestep; a recording made for other parameters must be refused."""
import numpy as np
import pytest

import parity_util as P
from paper_2110_01792_b200 import binding as B
from paper_2110_01792_b200 import inputs as I

pytestmark = pytest.mark.gpu

HYD = I.FIELDS[:5]
RADF = I.FIELDS[:9]


def _on_side_stream(params, fields):
    """a context whose stream can be captured (the legacy default stream cannot)"""
    import torch
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ctx = P.make_gpu(params, fields)
    return ctx, s


@pytest.mark.parametrize("gen", [I.config1, I.ragged_hydro], ids=["config1_32", "ragged"])
def test_graph_hydro_replay_is_the_ordinary_step_and_the_oracle(gen):
    import torch
    params, fields = gen()
    nsteps = 6
    g = P.make_oracle(params, fields)
    dts = []
    for _ in range(nsteps):
        dts.append(g.cfl_dt())
        assert g.hydro_step(dts[-1]) == 0
    with P.make_gpu(params, fields) as a:
        for _ in range(nsteps):
            a.qk_hydro_step_cfl()
        ref = a.get_all(HYD)
        dt_a, launches_a = a.qk_last_dt(), a.qk_launch_count()
    ctx, s = _on_side_stream(params, fields)
    with ctx, torch.cuda.stream(s):
        ctx.qk_graph_capture(B.QK_GRAPH_HYDRO)              # recorded before any step: nothing runs, state untouched
        P.assert_bitwise({n: fields[n] for n in HYD}, ctx.get_all(HYD), HYD, "capture must not touch the state")
        ctx.qk_graph_launch(2)                              # first step ordinary (fresh state), second a replay
        for _ in range(nsteps - 2):
            ctx.qk_graph_launch(1)
        got = ctx.get_all(HYD)
        assert ctx.qk_last_dt() == dt_a == dts[-1]
        info = ctx.qk_last_info()
        assert info["status"] == 0 and info["bad_state_cells"] == 0
        assert ctx.qk_launch_count() == launches_a
    P.assert_bitwise(ref, got, HYD, "graph replay vs qk_hydro_step_cfl")
    P.assert_bitwise(g.get_all(HYD), got, HYD, "graph replay vs oracle")
    g.close()


@pytest.mark.parametrize("chat_mult,bc", [(1.0, 0), (6.0, 0), (1.0, 2)], ids=["nsub1", "nsub_gt_1", "reflecting"])
def test_graph_rhd_replay_is_the_ordinary_step_and_the_oracle(chat_mult, bc):
    import torch
    params, fields = I.ragged_rhd()
    params["c_hat"] = params["c_hat"] * chat_mult
    params["bc"] = bc
    nsteps = 4
    with P.make_gpu(params, fields) as a:
        nsub = a.qk_nsub_for(a.qk_cfl_dt())
        assert (nsub > 1) == (chat_mult > 1.0)
        infos = []
        for _ in range(nsteps):
            a.qk_rhd_step_cfl(nsub)
            infos.append(a.qk_last_info())
        ref = a.get_all(RADF)
        dt_a = a.qk_last_dt()
    g = P.make_oracle(params, fields)
    for _ in range(nsteps):
        dt = g.cfl_dt()
        assert g.nsub_for(dt) == nsub                       # the pair qk_cfl_dt + qk_rhd_step takes the same substeps
        assert g.rhd_step(dt) == 0
    ctx, s = _on_side_stream(params, fields)
    with ctx, torch.cuda.stream(s):
        ctx.qk_hydro_step_cfl()                             # leave valid caches, then put the initial state back:
        ctx.set_all(fields)                                 # the caches are invalid again, the recording is still good
        ctx.qk_graph_capture(B.QK_GRAPH_RHD, nsub)
        ctx.qk_graph_launch(nsteps)
        got = ctx.get_all(RADF)
        info = ctx.qk_last_info()
        assert ctx.qk_last_dt() == dt_a
        for key in ("nsub", "newton_total_iters", "newton_max_iters", "fallback_states", "guard_faces", "status"):
            assert info[key] == infos[-1][key], key
    P.assert_bitwise(ref, got, RADF, "graph replay vs qk_rhd_step_cfl")
    P.assert_bitwise(g.get_all(RADF), got, RADF, "graph replay vs oracle")
    g.close()


def test_graph_refusals():
    import torch
    params, fields = I.config1(n=16)
    with P.make_gpu(params, fields) as ctx:                 # legacy default stream: cannot be captured
        with pytest.raises(B.QkError):
            ctx.qk_graph_launch(1)                          # nothing recorded
        if torch.cuda.current_stream().cuda_stream == 0:
            with pytest.raises(B.QkError):
                ctx.qk_graph_capture(B.QK_GRAPH_HYDRO)
        ctx.qk_hydro_step_cfl()                             # the context still works after the refused capture
        assert ctx.qk_last_info()["status"] == 0
    ctx, s = _on_side_stream(params, fields)
    with ctx, torch.cuda.stream(s):
        with pytest.raises(B.QkError):
            ctx.qk_graph_capture(B.QK_GRAPH_RHD, 1)         # no radiation constants on this context
        ctx.qk_graph_capture(B.QK_GRAPH_HYDRO)
        ctx.qk_graph_launch(3)
        ctx.qk_set_params(cfl=0.2)                          # recorded with CFL 0.3: stale
        with pytest.raises(B.QkError):
            ctx.qk_graph_launch(1)
        ctx.qk_graph_capture(B.QK_GRAPH_HYDRO)
        ctx.qk_graph_launch(1)
        dt_graph = ctx.qk_last_dt()
        ctx.qk_graph_free()
        with pytest.raises(B.QkError):
            ctx.qk_graph_launch(1)
        assert dt_graph > 0.0 and np.isfinite(dt_graph)
