"""bench.py prints ONE JSON line with the keys the driver reads (both arms)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True,
                       cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _run(["--impl", "reference", "--steps", "1", "--warmup", "1", "--ref-size", "16"])
    assert d["impl"] == "reference" and d["value"] > 0 and d["unit"] == "cell-updates/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and "workload" in d["config"]


@pytest.mark.gpu
def test_own_arm_line_has_the_contract_keys():
    d = _run(["--size", "32", "--steps", "3", "--warmup", "3", "--rhd-steps", "2", "--ref-size", "16"])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["scaling"] == "weak" and d["n_gpus"] == 1
    assert d["gpu_launches"] > 0 and d["value"] > 0 and "workload" in d["config"]
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] == 5 * 32 ** 3 * 8 == d["e2e"]["d2h_bytes_per_step"]
    r = d["roofline"]
    assert r["bound"] == "alu" and 0 < r["frac"] < 1 and abs(r["achieved"] / r["peak"] - r["frac"]) < 1e-9
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert d["rhd"]["value"] > 0 and d["rhd"]["nsub"] >= 1 and d["rhd"]["roofline_exchange"]["bound"] == "hbm"
    assert "traffic_source" in r and 0 < d["roofline_step"]["frac_alu"] < 1 and 0 < d["roofline_step"]["frac_hbm"] < 1
    assert d["device_dt"]["value"] > 0 and d["rhd"]["device_dt"]["value"] > 0 and d["rhd"]["e2e"]["value"] > 0
    assert d["cpu_baseline"]["one_core"]["cores"] == 1 and d["cpu_baseline"]["cores"] >= 1
    if d["clocks"] is not None:
        assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])


@pytest.mark.gpu
def test_own_arm_two_ranks_decomposed_box_runs_under_torchrun():
    """`bench.py --gpus 2` as the driver launches it, except for `--backend gloo` so that both ranks can share the one
    GPU of this box: the decomposed path (peer-mapped exchange across processes, global dt, max over ranks) runs, rank 0
    alone prints the line, and the line says how the halos travelled.  The timings of two time-slicing ranks mean
    nothing and are not looked at."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--size", "32",
           "--steps", "3", "--warmup", "3", "--rhd-steps", "2", "--no-cpu-baseline", "--backend", "gloo"]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, timeout=600,
                       env=dict(os.environ, OMP_NUM_THREADS="1", GLOO_SOCKET_IFNAME="lo"))
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    lines = [l for l in r.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1, lines
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["value"] > 0 and d["gpu_launches"] > 0
    assert "z-slab decomposition" in d["config"]["parallelism"] and "peer-mapped" in d["halo"]["exchange"]
    assert d["e2e"]["value"] > 0 and d["rhd"]["value"] > 0
