"""z-slab decomposition over ranks (the paper splits along x and overlaps the halo exchange with the
bulk propagate on separate streams, Fig. 3-4 -- with x-fastest storage the contiguous cut is
along z).  One process per GPU, one `Slab` per process; the 26 population-rows per direction and step travel with
torch.distributed point-to-point calls (NCCL over NVLink on GPUs; gloo in the CPU tests of the host logic).

Only marshalling and scheduling live here: packing, unpacking and stepping are lbm_slab_* calls of the library.
"""
from __future__ import annotations


def partition(Lz: int, world: int, min_rows: int = 6):
    """Rows [z0, z0 + nz) of rank r, r = 0 .. world-1: contiguous, balanced to within one row, bottom first."""
    if world < 1 or Lz < world * min_rows:
        raise ValueError(f"cannot cut {Lz} rows into {world} slabs of at least {min_rows} rows")
    base, extra = divmod(Lz, world)
    out, z0 = [], 0
    for r in range(world):
        nz = base + (1 if r < extra else 0)
        out.append((z0, nz))
        z0 += nz
    return out


def exchange_messages(send_up, send_dn, recv_below, recv_above, rank: int, world: int, group=None):
    """Posts the four transfers of one step and returns the requests: `send_up` goes to rank + 1 (which receives it in
    its `recv_below`), `send_dn` to rank - 1 (its `recv_above`).  The walls have no neighbour: rank 0 neither sends
    down nor receives from below, rank world-1 neither sends up nor receives from above.  Tag-free: every pair
    exchanges exactly one message per direction and step, posted in the same order on both sides."""
    import torch.distributed as dist
    ops = []
    if rank + 1 < world:
        ops.append(dist.P2POp(dist.isend, send_up, rank + 1, group))
        ops.append(dist.P2POp(dist.irecv, recv_above, rank + 1, group))
    if rank > 0:
        ops.append(dist.P2POp(dist.isend, send_dn, rank - 1, group))
        ops.append(dist.P2POp(dist.irecv, recv_below, rank - 1, group))
    return dist.batch_isend_irecv(ops) if ops else []


class SlabRing:
    """The slab of this rank plus its message buffers.  `step(n)`: pairs of steps with the two-step kernel (6 whole
    ghost rows per open side and pair), an odd last step -- or every step with `fused=False` -- with the one-step
    kernel (26 population-rows per open side).  Either way the exchange hides behind the bulk (PAPER.md:116-118,
    Fig. 4): pack on the exchange stream, the interior rows -- which read no ghost row -- on the main stream while the
    messages travel, unpack, then the edge rows.

    Transport: NCCL moves the device buffers directly.  With any other backend (gloo: the CPU tests, and two ranks
    sharing one GPU in tests/test_gpu_slab_ring.py) the messages are staged through pinned host buffers; the schedule
    of kernels and streams is the same."""

    def __init__(self, Lx: int, Lz: int, tau: float, g: float, rank: int, world: int, wall_kind: int = 0,
                 T_wall=(1.0, 1.0), device="cuda", group=None):
        import torch
        import torch.distributed as dist

        from . import Slab
        self.rank, self.world, self.group = rank, world, group
        self.z0, self.nz = partition(Lz, world)[rank]
        self.slab = Slab(Lx, Lz, self.z0, self.nz, tau, g, wall_kind=wall_kind, T_wall=T_wall, device=device)
        # device messages: [send up, send down, received from below, received from above], one-step and two-step sizes
        self.msg = [self.slab.new_message() for _ in range(4)]
        self.msg2 = [self.slab.new_message(True) for _ in range(4)]
        self.staged = world > 1 and dist.get_backend(group) != "nccl"
        if self.staged:
            self.host = [torch.empty(m.shape, dtype=m.dtype).pin_memory() for m in self.msg]
            self.host2 = [torch.empty(m.shape, dtype=m.dtype).pin_memory() for m in self.msg2]
        self.xs = torch.cuda.Stream(device=self.slab.device)

    def _post(self, dev, host):
        """Starts the transfers of the packed messages `dev[0:2]` (on the exchange stream); returns the requests."""
        import torch
        s = self.slab
        with torch.cuda.stream(self.xs):
            if not self.staged:
                return exchange_messages(dev[0], dev[1], dev[2], dev[3], self.rank, self.world, self.group)
            if s.open_above:
                host[0].copy_(dev[0], non_blocking=True)
            if s.open_below:
                host[1].copy_(dev[1], non_blocking=True)
        self.xs.synchronize()                                    # the host copies are complete before gloo reads them
        return exchange_messages(host[0], host[1], host[2], host[3], self.rank, self.world, self.group)

    def _arrived(self, reqs, dev, host):
        """Waits for the transfers; afterwards the received messages are (or will be, in stream order) in `dev[2:4]`."""
        import torch
        s = self.slab
        with torch.cuda.stream(self.xs):
            for r in reqs:
                r.wait()
            if self.staged:
                if s.open_below:
                    dev[2].copy_(host[2], non_blocking=True)
                if s.open_above:
                    dev[3].copy_(host[3], non_blocking=True)

    def step(self, n: int = 1, fused: bool = True):
        import torch
        s = self.slab
        main, xs = torch.cuda.current_stream(s.device), self.xs
        pairs = n // 2 if fused else 0
        for k in range(n - pairs):                               # `pairs` double steps, then single steps
            two = k < pairs
            dev, host = (self.msg2, getattr(self, "host2", None)) if two else (self.msg, getattr(self, "host", None))
            pack, unpack = (s.pack2, s.unpack2) if two else (s.pack, s.unpack)
            xs.wait_stream(main)
            if s.open_above:
                pack(1, dev[0], stream=xs)
            if s.open_below:
                pack(0, dev[1], stream=xs)
            if two:
                main.wait_stream(xs)                             # pack2 refreshes the wrap columns the interior's boxes read
                s.step2_part(s.INTERIOR, stream=main)            # overlaps the exchange
            else:
                s.step_part(s.INTERIOR, stream=main)
            reqs = self._post(dev, host)
            self._arrived(reqs, dev, host)
            if s.open_below:
                unpack(0, dev[2], stream=xs)
            if s.open_above:
                unpack(1, dev[3], stream=xs)
            main.wait_stream(xs)
            if two:
                s.step2_part(s.EDGES, stream=main)
            else:
                s.step_part(s.EDGES, stream=main)

    def close(self):
        self.slab.close()
