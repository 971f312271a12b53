"""The allocation-free entry point qk_cfl_dt_noalloc (include/qk.h; scratch in a static device array) against the
existing path, qk_cfl_dt of a context holding the same cells.  A maximum does not depend on its order, so the two
doubles are equal bit for bit -- the tolerance every CFL test in test_gpu_parity.py uses (`==`).  Two calls in a row on
different states and sizes: the shared scratch keeps the first call's contents, the second must not see them.

The file name makes pytest collect it last: the suite runs with `pytest -x`, so a failure here hides nothing."""
import numpy as np
import pytest

from paper_2110_01792_b200 import binding as B
from paper_2110_01792_b200 import inputs as I

pytestmark = pytest.mark.gpu


def _existing_path_dt(params, fields):
    with B.from_params(params, fields) as ctx:
        return ctx.qk_cfl_dt()


def _noalloc_dt(torch, params, fields):
    dev = [torch.from_numpy(np.ascontiguousarray(fields[n])).cuda() for n in I.FIELDS[:5]]
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    B.qk_cfl_dt_noalloc(*[t.data_ptr() for t in dev], dev[0].numel(), params["gamma"], params.get("cfl", 0.3),
                        params["dx"], out.data_ptr())
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    return float(out.item())


def test_noalloc_cfl_dt_equals_the_existing_path_on_two_calls_in_a_row():
    import torch
    B.qk_noalloc_setup()
    # first call: 64^3 turbulence (256 partial maxima); second: a ragged box with a tail CTA (16 partials) whose
    # maximum is smaller than the first one's -- stale partials of the first call would raise it
    big_p, big_f = I.config2(n=64)
    small_p, small_f = I.ragged_hydro()
    small_f = {n: (a * (0.01 if n in ("mx", "my", "mz") else 1.0)) for n, a in small_f.items()}
    want_big, want_small = _existing_path_dt(big_p, big_f), _existing_path_dt(small_p, small_f)
    assert np.isfinite(want_big) and np.isfinite(want_small)
    assert want_small / small_p["dx"] > want_big / big_p["dx"]          # i.e. max speed(small) < max speed(big)
    got_big = _noalloc_dt(torch, big_p, big_f)
    got_small = _noalloc_dt(torch, small_p, small_f)
    assert got_big == want_big, (got_big, want_big)
    assert got_small == want_small, (got_small, want_small)
    # a bad cell gives NaN like the existing path, and the counter it raised is cleared by the next call
    bad_f = {n: a.copy() for n, a in small_f.items()}
    bad_f["rho"][2, 3, 4] = -1.0
    assert np.isnan(_existing_path_dt(small_p, bad_f)) and np.isnan(_noalloc_dt(torch, small_p, bad_f))
    assert _noalloc_dt(torch, small_p, small_f) == want_small


def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    x = torch.ones(8, dtype=torch.float64, device="cuda")
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    limit = B.qk_noalloc_max_cells()
    assert limit == 256 ** 3
    with pytest.raises(B.QkError, match="exceed"):
        B.qk_cfl_dt_noalloc(*[x.data_ptr()] * 5, limit + 1, 5.0 / 3.0, 0.3, 1.0, out.data_ptr())
    with pytest.raises(B.QkError, match="QK_EINVAL"):
        B.qk_cfl_dt_noalloc(*[x.data_ptr()] * 5, 0, 5.0 / 3.0, 0.3, 1.0, out.data_ptr())
    with pytest.raises(B.QkError, match="QK_EINVAL"):
        B.qk_cfl_dt_noalloc(0, *[x.data_ptr()] * 4, 8, 5.0 / 3.0, 0.3, 1.0, out.data_ptr())
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0                                  # nothing was launched
