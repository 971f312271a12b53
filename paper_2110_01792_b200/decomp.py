"""z-slab domain decomposition of one global box over the ranks of a torch.distributed job
(the paper's pattern: one ghost exchange per RK stage plus a min-reduction of the
timestep).

Host-side plumbing only: which faces border a neighbour, who the neighbours are, the order of the
sends and receives, the reduction of dt.  Two ways to move the halos: `PeerExchange` (the fast path: the library
writes boundary planes straight into the neighbours' peer-mapped ghost planes on a side stream and overlaps the
transfer with the interior work of the stage; Python only introduces the ranks to each other once) and
`SlabExchange` (portable: a callback per ghost fill packs, sends with torch.distributed point-to-point operations
and unpacks; it is what the CPU tests drive over gloo).  The halo planes themselves are packed / unpacked by
kernels of the library (qk_halo_pack / qk_halo_unpack) and moved by torch.distributed point-to-point
operations (NCCL over NVLink on GPUs, gloo on CPU in the tests).  `SlabExchange` works with any
object that has qk_set_halo_exchange / qk_halo_doubles / qk_halo_pack / qk_halo_unpack and a
`new_buffer(ndoubles)` method, so the CPU tests drive it with a numpy stand-in.
"""
from __future__ import annotations

FACE_ZLO, FACE_ZHI = 1, 2


def slab_extent(nz_global: int, rank: int, world: int):
    """(first plane, number of planes) of rank's slab: planes are dealt out as evenly as possible,
    the first nz_global % world ranks get one more."""
    base, extra = divmod(nz_global, world)
    n = base + (1 if rank < extra else 0)
    k0 = rank * base + min(rank, extra)
    return k0, n


def neighbours(rank: int, world: int, periodic: bool):
    """(lower neighbour, upper neighbour) along z, None at a physical boundary."""
    if world == 1:
        return None, None
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return lo, hi


class TorchTransport:
    """Moves (send_lo, send_hi) to the neighbours and fills (recv_lo, recv_hi) with torch.distributed
    point-to-point operations.  With two ranks and periodic boundaries both neighbours are the same
    peer: messages between one pair of ranks match in posting order, so the sends are posted high
    face first and the receives low face first (my low ghost planes are the peer's high planes)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group

    def device_stream(self):
        """raw handle of the stream NCCL orders its point-to-point operations against (None on CPU backends)"""
        import torch
        if self.dist.get_backend(self.group) != "nccl":
            return None
        return int(torch.cuda.current_stream().cuda_stream)

    def exchange(self, lo, hi, send_lo, send_hi, recv_lo, recv_hi):
        dist = self.dist
        ops = []
        if hi is not None:
            ops.append(dist.P2POp(dist.isend, send_hi, hi, self.group))
        if lo is not None:
            ops.append(dist.P2POp(dist.isend, send_lo, lo, self.group))
        if lo is not None:
            ops.append(dist.P2POp(dist.irecv, recv_lo, lo, self.group))
        if hi is not None:
            ops.append(dist.P2POp(dist.irecv, recv_hi, hi, self.group))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()

    def min_over_ranks(self, x: float) -> float:
        import torch
        dist = self.dist
        dev = "cuda" if dist.get_backend(self.group) == "nccl" else "cpu"
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MIN, group=self.group)
        return float(t.item())


class SlabExchange:
    """Attaches the halo exchange of one rank's slab to a context."""

    def __init__(self, ctx, rank: int, world: int, periodic: bool, transport):
        self.ctx, self.transport = ctx, transport
        self.lo, self.hi = neighbours(rank, world, periodic)
        self.faces = (FACE_ZLO if self.lo is not None else 0) | (FACE_ZHI if self.hi is not None else 0)
        self.per_field = ctx.qk_halo_doubles()
        self.buffers = {}
        self.calls = 0
        self.bytes_sent = 0
        self.error = None
        ctx.qk_set_halo_exchange(self.faces, self._on_fill if self.faces else None)

    def _bufs(self, nfields):
        if nfields not in self.buffers:
            n = nfields * self.per_field
            self.buffers[nfields] = tuple(self.ctx.new_buffer(n) for _ in range(4))
        return self.buffers[nfields]

    def _on_fill(self, nfields):
        # called by the library before every ghost fill; exceptions cannot cross the C frame: a non-zero return
        # makes the step call fail and later step calls return QK_EINVAL until the exchange is attached again
        try:
            # the point-to-point operations order against torch's current stream, pack / unpack against the context's
            # stream: they must be the same one
            sp = getattr(self.ctx, "stream_ptr", None)
            ts = self.transport.device_stream() if hasattr(self.transport, "device_stream") else None
            if sp is not None and ts is not None:
                assert ts == sp, "halo exchange: torch's current stream is not the context's stream"
            send_lo, send_hi, recv_lo, recv_hi = self._bufs(nfields)
            if self.lo is not None:
                self.ctx.qk_halo_pack(FACE_ZLO, send_lo)
            if self.hi is not None:
                self.ctx.qk_halo_pack(FACE_ZHI, send_hi)
            self.transport.exchange(self.lo, self.hi, send_lo, send_hi, recv_lo, recv_hi)
            if self.lo is not None:
                self.ctx.qk_halo_unpack(FACE_ZLO, recv_lo)
            if self.hi is not None:
                self.ctx.qk_halo_unpack(FACE_ZHI, recv_hi)
            self.calls += 1
            self.bytes_sent += 8 * nfields * self.per_field * ((self.lo is not None) + (self.hi is not None))
            return 0
        except BaseException as e:      # noqa: BLE001 -- re-raised by check() on the Python side
            if self.error is None:
                self.error = e
            return 1                    # the library aborts the step (QK_EINVAL) instead of running on stale ghosts

    def check(self):
        if self.error is not None:
            e, self.error = self.error, None
            raise e

    def global_dt(self, local_dt: float) -> float:
        """eq 21 over the whole box: the minimum of the ranks' local timesteps (NaN propagates)."""
        if local_dt != local_dt:
            local_dt = float("-inf")
        dt = self.transport.min_over_ranks(local_dt)
        return float("nan") if dt == float("-inf") else dt

    def detach(self):
        self.ctx.qk_set_halo_exchange(0, None)


class PeerExchange:
    """Peer-mapped halo exchange (qk_halo_export / qk_set_halo_peers): every rank publishes a handle of its storage,
    picks up its neighbours' handles and attaches them; from then on the stage path never enters Python.
    `gather(obj) -> list of objects by rank` is how handles cross ranks (torch.distributed.all_gather_object by
    default); `min_reduce(x) -> float` reduces the timestep."""

    def __init__(self, ctx, rank: int, world: int, periodic: bool, gather=None, min_reduce=None, barrier=None):
        self.ctx = ctx
        self.lo, self.hi = neighbours(rank, world, periodic)
        if gather is None:
            import torch.distributed as dist

            def gather(obj):
                out = [None] * dist.get_world_size()
                dist.all_gather_object(out, obj)
                return out
            barrier = barrier or dist.barrier
        self.min_reduce = min_reduce or TorchTransport().min_over_ranks
        handles = gather(ctx.qk_halo_export())
        self.error = None
        try:
            ctx.qk_set_halo_peers(handles[self.lo] if self.lo is not None else None,
                                  handles[self.hi] if self.hi is not None else None)
        except Exception as e:      # e.g. no IPC handle for this kind of allocation, no stream memory operations
            self.error = e
        # nobody steps before everybody has attached (the arrival counters restart at attach); the reduction is the
        # barrier, and if any rank failed every rank detaches so that the caller can fall back to SlabExchange
        self.ok = self.min_reduce(0.0 if self.error else 1.0) > 0.5
        if not self.ok:
            try:
                ctx.qk_set_halo_peers(None, None)
            except Exception:
                pass
        elif barrier is not None:
            barrier()

    def global_dt(self, local_dt: float) -> float:
        if local_dt != local_dt:
            local_dt = float("-inf")
        dt = self.min_reduce(local_dt)
        return float("nan") if dt == float("-inf") else dt

    def check(self):
        pass

    def detach(self):
        self.ctx.qk_set_halo_peers(None, None)
