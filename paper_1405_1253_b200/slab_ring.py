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
    ghost rows per open side and pair, exchanged before the launch: a few microseconds beside milliseconds), an odd
    last step -- or every step with `fused=False` -- with the one-step kernel: pack on the exchange stream, interior
    rows on the main stream while the messages travel, unpack, edge rows (interior first)."""

    def __init__(self, Lx: int, Lz: int, tau: float, g: float, rank: int, world: int, wall_kind: int = 0,
                 T_wall=(1.0, 1.0), device="cuda", group=None):
        import torch

        from . import Slab
        self.rank, self.world, self.group = rank, world, group
        self.z0, self.nz = partition(Lz, world)[rank]
        self.slab = Slab(Lx, Lz, self.z0, self.nz, tau, g, wall_kind=wall_kind, T_wall=T_wall, device=device)
        self.send_up, self.send_dn, self.recv_below, self.recv_above = (self.slab.new_message() for _ in range(4))
        self.send2_up, self.send2_dn, self.recv2_below, self.recv2_above = (self.slab.new_message(True) for _ in range(4))
        self.xs = torch.cuda.Stream(device=self.slab.device)

    def step(self, n: int = 1, fused: bool = True):
        import torch
        s = self.slab
        main = torch.cuda.current_stream(s.device)
        pairs = n // 2 if fused else 0
        for _ in range(pairs):
            if s.open_above:
                s.pack2(1, self.send2_up, stream=main)
            if s.open_below:
                s.pack2(0, self.send2_dn, stream=main)
            for r in exchange_messages(self.send2_up, self.send2_dn, self.recv2_below, self.recv2_above, self.rank,
                                       self.world, self.group):
                r.wait()
            if s.open_below:
                s.unpack2(0, self.recv2_below, stream=main)
            if s.open_above:
                s.unpack2(1, self.recv2_above, stream=main)
            s.step2(stream=main)
        for _ in range(n - 2 * pairs):
            self.xs.wait_stream(main)
            with torch.cuda.stream(self.xs):
                if s.open_above:
                    s.pack(1, self.send_up, stream=self.xs)
                if s.open_below:
                    s.pack(0, self.send_dn, stream=self.xs)
                reqs = exchange_messages(self.send_up, self.send_dn, self.recv_below, self.recv_above, self.rank,
                                         self.world, self.group)
            s.step_part(s.INTERIOR, stream=main)                 # overlaps the exchange
            with torch.cuda.stream(self.xs):
                for r in reqs:
                    r.wait()
                if s.open_below:
                    s.unpack(0, self.recv_below, stream=self.xs)
                if s.open_above:
                    s.unpack(1, self.recv_above, stream=self.xs)
            main.wait_stream(self.xs)
            s.step_part(s.EDGES, stream=main)

    def close(self):
        self.slab.close()
