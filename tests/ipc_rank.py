"""One rank of the multi-process peer-mapped exchange test (tests/test_gpu_ipc.py starts `world` of these, all on
cuda:0, rendezvous over gloo on 127.0.0.1).  Each rank owns one z slab, publishes the handle of its storage
(qk_halo_export), opens its neighbours' handles with CUDA IPC (qk_set_halo_peers), steps with the reduced dt and writes
its slab to <outdir>/rank<r>.npz.  Nothing here spins on the device: arrival of a halo is a stream memory operation of
the driver on the receiving rank's stream."""
import os
import sys

import numpy as np


def main():
    kind, gen_name, bc, nsteps, outdir = sys.argv[1], sys.argv[2], int(sys.argv[3]), int(sys.argv[4]), sys.argv[5]
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), ".."))
    import torch
    import torch.distributed as dist
    from paper_2110_01792_b200 import binding as B, decomp as D, inputs as I

    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    params, fields = getattr(I, gen_name)(bc=bc)
    k0, nz = D.slab_extent(params["nz"], rank, world)
    local = {n: np.ascontiguousarray(a[k0:k0 + nz]) for n, a in fields.items()}
    names = I.FIELDS[:5] if kind == "hydro" else I.FIELDS[:9]
    with B.from_params(dict(params, nz=nz), local) as ctx:
        px = D.PeerExchange(ctx, rank, world, params["bc"] == I.BC_PERIODIC)
        attached = bool(px.ok)
        err = repr(px.error)
        if attached:
            for _ in range(nsteps):
                dt = px.global_dt(ctx.qk_cfl_dt())
                ctx.qk_hydro_step(dt) if kind == "hydro" else ctx.qk_rhd_step(dt)
            out = ctx.get_all(names)
            info = ctx.qk_last_info()
            dist.barrier()                 # nobody unmaps a neighbour that may still be pushing
            px.detach()
        else:
            out, info = {}, {}
    np.savez(os.path.join(outdir, "rank%d.npz" % rank), attached=attached, error=err,
             newton=int(info.get("newton_total_iters", 0)), status=int(info.get("status", -1)), **out)
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
