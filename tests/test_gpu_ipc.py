"""The peer-mapped halo exchange across PROCESSES (CUDA IPC handles), on the one GPU this box has: `world` processes,
one z slab each, neighbours' storage opened with cudaIpcOpenMemHandle, halos pushed by kernels on side streams, arrival
a stream memory operation -- the path `torchrun bench.py --gpus N` takes.  The glued slabs must be the single box, bit
for bit.  (The in-process form of the same exchange is in test_gpu_parity.py; the host-side logic on gloo in
test_decomp_gloo.py.)  No kernel here waits on another rank: B200_PROFILING.md's rule about spinning kernels on a shared
GPU does not apply to stream memory operations, and the ranks are bounded by a timeout all the same."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2110_01792_b200 import inputs as I
import parity_util as P

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _run_ranks(kind, gen_name, bc, nsteps, world, outdir, limit=240):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   GLOO_SOCKET_IFNAME="lo", OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, os.path.join(HERE, "ipc_rank.py"), kind, gen_name, str(bc),
                                       str(nsteps), str(outdir)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT))
    outs = []
    try:
        for p in procs:
            o, _ = p.communicate(timeout=limit)
            outs.append(o.decode(errors="replace"))
    finally:
        for p in procs:                 # exact PIDs only
            if p.poll() is None:
                p.kill()
                p.wait()
    for r, p in enumerate(procs):
        assert p.returncode == 0, "rank %d exited %s:\n%s" % (r, p.returncode, outs[r][-3000:] if r < len(outs) else "")
    return [np.load(os.path.join(outdir, "rank%d.npz" % r)) for r in range(world)]


@pytest.mark.parametrize("kind,gen_name,world,bc", [("hydro", "ragged_hydro", 2, I.BC_PERIODIC),
                                                    ("rhd", "ragged_rhd", 2, I.BC_PERIODIC),
                                                    ("hydro", "ragged_hydro", 3, I.BC_OUTFLOW)],
                         ids=["hydro_x2_periodic", "rhd_x2_periodic", "hydro_x3_outflow"])
def test_ipc_peer_exchange_between_processes_is_bitwise_the_single_box(kind, gen_name, world, bc, tmp_path):
    params, fields = getattr(I, gen_name)(bc=bc)
    nsteps = 3 if kind == "hydro" else 2
    names = I.FIELDS[:5] if kind == "hydro" else I.FIELDS[:9]
    with P.make_gpu(params, fields) as ctx:
        for _ in range(nsteps):
            dt = ctx.qk_cfl_dt()
            ctx.qk_hydro_step(dt) if kind == "hydro" else ctx.qk_rhd_step(dt)
        single = ctx.get_all(names)
        info1 = ctx.qk_last_info()
    parts = _run_ranks(kind, gen_name, bc, nsteps, world, tmp_path)
    for r, p in enumerate(parts):
        assert bool(p["attached"]), "rank %d could not attach its neighbours: %s" % (r, p["error"])
        assert int(p["status"]) == info1["status"]
    glued = {n: np.concatenate([parts[r][n] for r in range(world)], axis=0) for n in names}
    P.assert_bitwise(single, glued, names, "IPC peer exchange %s x%d" % (kind, world))
    if kind == "rhd":
        assert sum(int(p["newton"]) for p in parts) == info1["newton_total_iters"]
