"""N>1 host logic on CPU: the z-slab halo-exchange plan of paper_2110_01792_b200.decomp driven over
torch.distributed (gloo, world_size 2 and 3) with a numpy stand-in for the device context.  The ghost
zones every rank ends up with must equal, bit for bit, the corresponding part of the ORACLE's ghost fill of
the undecomposed box (periodic and outflow), and the global timestep must be the minimum over ranks."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2110_01792_b200 import decomp as D  # noqa: E402

NG = 4


class NumpyCtx:
    """Stand-in with the four halo entry points of the binding, on host arrays."""

    def __init__(self, fields, bc):
        self.f, self.bc = fields, bc
        self.nz, self.ny, self.nx = (s - 2 * NG for s in fields[0].shape)
        self.faces, self.fn = 0, None

    def qk_set_halo_exchange(self, faces, fn):
        self.faces, self.fn = faces, fn

    def qk_halo_doubles(self):
        return NG * self.ny * self.nx

    def new_buffer(self, n):
        return torch.empty(n, dtype=torch.float64)

    def _planes(self, face, ghost):
        if face == D.FACE_ZLO:
            k0 = 0 if ghost else NG
        else:
            k0 = NG + self.nz if ghost else self.nz
        return slice(k0, k0 + NG)

    def qk_halo_pack(self, face, buf):
        v = buf.numpy().reshape(len(self.f), NG, self.ny, self.nx)
        for n, a in enumerate(self.f):
            v[n] = a[self._planes(face, False), NG:-NG, NG:-NG]

    def qk_halo_unpack(self, face, buf):
        v = buf.numpy().reshape(len(self.f), NG, self.ny, self.nx)
        for n, a in enumerate(self.f):
            a[self._planes(face, True), NG:-NG, NG:-NG] = v[n]

    def fill(self):
        if self.fn:
            self.fn(len(self.f))
        for a in self.f:
            for axis, n in ((2, self.nx), (1, self.ny), (0, self.nz)):
                lo_ext = axis == 0 and (self.faces & D.FACE_ZLO)
                hi_ext = axis == 0 and (self.faces & D.FACE_ZHI)
                for g in range(NG):
                    dst_lo, dst_hi = [slice(None)] * 3, [slice(None)] * 3
                    src_lo, src_hi = [slice(None)] * 3, [slice(None)] * 3
                    dst_lo[axis], dst_hi[axis] = g, NG + n + g
                    if self.bc == 0:    # periodic
                        src_lo[axis], src_hi[axis] = NG + (g - NG) % n, NG + g % n
                    else:               # outflow: nearest interior cell
                        src_lo[axis], src_hi[axis] = NG, NG + n - 1
                    if not lo_ext:
                        a[tuple(dst_lo)] = a[tuple(src_lo)]
                    if not hi_ext:
                        a[tuple(dst_hi)] = a[tuple(src_hi)]


def _worker(rank, world, port, bc, shape, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle as O
        nzg, ny, nx = shape
        rng = np.random.Generator(np.random.PCG64(5))
        glob = [rng.standard_normal(shape) for _ in range(3)]
        # reference: the oracle's ghost fill of the whole box
        g = O.Grid(nx, ny, nzg, 1.0 / nx, 5.0 / 3.0, bc=bc)
        ref = []
        for f, a in enumerate(glob):
            g.set_state(f, a)
        g.fill_boundary(O.FILL_HYDRO)
        for f in range(3):
            ref.append(g.get_raw(f).reshape(nzg + 2 * NG, ny + 2 * NG, nx + 2 * NG))
        g.close()
        k0, nz = D.slab_extent(nzg, rank, world)
        local = []
        for a in glob:
            s = np.full((nz + 2 * NG, ny + 2 * NG, nx + 2 * NG), np.nan)
            s[NG:-NG, NG:-NG, NG:-NG] = a[k0:k0 + nz]
            local.append(s)
        ctx = NumpyCtx(local, bc)
        ex = D.SlabExchange(ctx, rank, world, periodic=(bc == 0), transport=D.TorchTransport())
        for _ in range(2):          # twice: buffers are reused
            ctx.fill()
            ex.check()
        ok = all(np.array_equal(local[f], ref[f][k0:k0 + nz + 2 * NG]) for f in range(3))
        dt = ex.global_dt(0.25 + rank)
        nan_dt = ex.global_dt(float("nan") if rank == world - 1 else 1.0)
        expected_faces = (0 if D.neighbours(rank, world, bc == 0)[0] is None else 1) | \
                         (0 if D.neighbours(rank, world, bc == 0)[1] is None else 2)
        out[rank] = (ok, dt, nan_dt != nan_dt, ex.faces == expected_faces, ex.calls)
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("bc", [0, 1], ids=["periodic", "outflow"])
def test_slab_halo_exchange_matches_global_fill(world, bc):
    out = mp.Manager().dict()
    mp.spawn(_worker, args=(world, _free_port(), bc, (13, 6, 7), out), nprocs=world, join=True)
    assert len(out) == world
    for rank in range(world):
        ok, dt, nan_seen, faces_ok, calls = out[rank]
        assert ok, "rank %d: ghost zones differ from the global fill" % rank
        assert dt == 0.25 and nan_seen and faces_ok and calls == 2


def test_slab_extents_and_neighbours():
    for nzg, world in ((13, 3), (256, 8), (9, 2), (4, 1)):
        ext = [D.slab_extent(nzg, r, world) for r in range(world)]
        assert ext[0][0] == 0 and sum(n for _, n in ext) == nzg
        assert all(ext[r][0] + ext[r][1] == ext[r + 1][0] for r in range(world - 1))
        assert max(n for _, n in ext) - min(n for _, n in ext) <= 1
    assert D.neighbours(0, 1, True) == (None, None)
    assert D.neighbours(0, 2, True) == (1, 1) and D.neighbours(1, 2, True) == (0, 0)
    assert D.neighbours(0, 3, False) == (None, 1) and D.neighbours(2, 3, False) == (1, None)
    assert D.neighbours(0, 4, True) == (3, 1)


# ------------------------------------------------------------------------------------------------
# the peer-mapped plan (decomp.PeerExchange): handles cross ranks once, then every rank writes its boundary planes
# straight into its neighbours' ghost planes and raises their arrival counters.  Stand-in: the "device storage" of a
# rank is a POSIX shared-memory block, the handle is its name, a push is a numpy copy into the neighbour's block.
# ------------------------------------------------------------------------------------------------
class ShmPeerCtx(NumpyCtx):
    def __init__(self, shape3, nfields, bc, rank):
        from multiprocessing import shared_memory
        self.shape3 = shape3
        n = nfields * int(np.prod(shape3)) + 2
        self.shm = shared_memory.SharedMemory(create=True, size=8 * n, name="qk_peer_test_%d_%d" % (os.getppid(), rank))
        flat = np.ndarray((n,), dtype=np.float64, buffer=self.shm.buf)
        flat[:] = 0.0
        fields = [flat[f * int(np.prod(shape3)):(f + 1) * int(np.prod(shape3))].reshape(shape3) for f in range(nfields)]
        self.arrive = flat[-2:]                     # [from lo neighbour, from hi neighbour]
        super().__init__(fields, bc)
        self.peers, self.epoch, self.opened = [None, None], 0, []

    def qk_halo_export(self):
        return (self.shm.name, self.shape3, len(self.f))

    def qk_set_halo_peers(self, lo, hi):
        from multiprocessing import shared_memory
        self.faces = 0
        for side, h in enumerate((lo, hi)):
            if h is None:
                continue
            name, shape3, nf = h
            shm = shared_memory.SharedMemory(name=name)
            self.opened.append(shm)
            flat = np.ndarray((nf * int(np.prod(shape3)) + 2,), dtype=np.float64, buffer=shm.buf)
            fields = [flat[f * int(np.prod(shape3)):(f + 1) * int(np.prod(shape3))].reshape(shape3) for f in range(nf)]
            self.peers[side] = (fields, flat[-2:], shape3[0] - 2 * NG)
            self.faces |= D.FACE_ZHI if side else D.FACE_ZLO

    def fill(self):
        import time
        self.epoch += 1
        for side, p in enumerate(self.peers):
            if p is None:
                continue
            fields, arrive, nz_nb = p
            for mine, theirs in zip(self.f, fields):
                if side == 0:       # my low planes -> the low neighbour's HIGH ghost planes
                    theirs[NG + nz_nb:NG + nz_nb + NG, NG:-NG, NG:-NG] = mine[NG:2 * NG, NG:-NG, NG:-NG]
                else:               # my high planes -> the high neighbour's LOW ghost planes
                    theirs[0:NG, NG:-NG, NG:-NG] = mine[self.nz:self.nz + NG, NG:-NG, NG:-NG]
            arrive[1 if side == 0 else 0] = self.epoch      # I am the HIGH neighbour of my low peer
        for side, p in enumerate(self.peers):
            t0 = time.time()
            while p is not None and self.arrive[side] < self.epoch:
                assert time.time() - t0 < 60, "peer never arrived"
                time.sleep(0.001)
        super().fill()

    def close(self):
        self.f, self.arrive, self.peers = None, None, None
        for s in self.opened:
            s.close()
        self.shm.close()
        self.shm.unlink()


def _peer_worker(rank, world, port, bc, shape, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle as O
        nzg, ny, nx = shape
        rng = np.random.Generator(np.random.PCG64(6))
        glob = [rng.standard_normal(shape) for _ in range(2)]
        g = O.Grid(nx, ny, nzg, 1.0 / nx, 5.0 / 3.0, bc=bc)
        for f, a in enumerate(glob):
            g.set_state(f, a)
        g.fill_boundary(O.FILL_HYDRO)
        ref = [g.get_raw(f) for f in range(2)]
        g.close()
        k0, nz = D.slab_extent(nzg, rank, world)
        ctx = ShmPeerCtx((nz + 2 * NG, ny + 2 * NG, nx + 2 * NG), 2, bc, rank)
        for f, a in enumerate(glob):
            ctx.f[f][:] = np.nan
            ctx.f[f][NG:-NG, NG:-NG, NG:-NG] = a[k0:k0 + nz]
        ex = D.PeerExchange(ctx, rank, world, periodic=(bc == 0))
        for _ in range(3):
            ctx.fill()
            dist.barrier()          # a rank must not start the next push while a neighbour still reads (on the device the
                                    # RK stage structure gives this order: DESIGN.md section 8)
        ok = all(np.array_equal(ctx.f[f], ref[f][k0:k0 + nz + 2 * NG]) for f in range(2))
        dt = ex.global_dt(1.5 - 0.25 * rank)
        dist.barrier()
        ctx.close()
        out[rank] = (ok, dt)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("bc", [0, 1], ids=["periodic", "outflow"])
def test_peer_exchange_plan_matches_global_fill(world, bc):
    out = mp.Manager().dict()
    mp.spawn(_peer_worker, args=(world, _free_port(), bc, (14, 5, 6), out), nprocs=world, join=True)
    for rank in range(world):
        ok, dt = out[rank]
        assert ok, "rank %d: ghost zones differ from the global fill" % rank
        assert dt == 1.5 - 0.25 * (world - 1)
