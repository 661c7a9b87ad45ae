"""Time-slab decomposition of the even-odd dslash over several GPUs (next row f3).

One process per GPU (torch.distributed, NCCL); rank r owns the global time slices [r T/N, (r+1) T/N) as a local
lattice of T/N + 2 slices whose first and last slice are ghosts.  Everything arithmetic stays in the CUDA kernels
(lqcd_dslash_eo_range); this module is plumbing only: which slices a rank holds, where the global boundary phase
cuts it (lqcd_set_time_slab), and the ghost exchange -- plain copies of whole time slices, which are contiguous
byte ranges of the native layout.  Links need no exchange: every rank packs the links of its own slices, ghosts
included.  The paper's own multi-device scheme is host-mediated; this is the natural
sharding named in SURVEY.md sec. 8(e).  Not used by bench.py (north_star: single GPU); covered by a
single-GPU emulation of N ranks (tests/test_gpu_slab.py) and a world-size-2 gloo test of the exchange.
"""
from __future__ import annotations

from . import Context


class TimeSlab:
    """Rank `rank` of `world` in a decomposition of a lattice of global extents dims = (X, Y, Z, T) along t."""

    def __init__(self, dims, precision, recon, bc, rank, world):
        X, Y, Z, T = (int(d) for d in dims)
        if T % world or (T // world) % 2 or T // world < 2:
            raise ValueError("T / world must be an even number of time slices")
        self.global_dims, self.rank, self.world = (X, Y, Z, T), int(rank), int(world)
        self.Tl = T // world
        self.t0 = self.rank * self.Tl
        self.local_dims = (X, Y, Z, self.Tl + 2)
        self.ctx = Context(self.local_dims, precision, recon, bc)
        # the global t boundary lies between the last slice of the last rank and the first slice of rank 0
        self.ctx.set_time_slab(self.Tl if self.rank == self.world - 1 else -1, 1 if self.rank == 0 else -1)
        self.slice_bytes = self.ctx.time_slice_bytes()
        if self.slice_bytes == 0:
            raise ValueError("time slices are not whole 32-site tiles (or precision 16): no slab path for this lattice")

    # ---- bookkeeping -------------------------------------------------------------------------------------
    def time_indices(self):
        """Global t of the local slices 0 .. Tl + 1 (ghosts wrap around the global lattice)."""
        T = self.global_dims[3]
        return [(self.t0 - 1 + k) % T for k in range(self.Tl + 2)]

    def local_parity(self, global_parity):
        """Local slice 1 is global slice t0 (even), so a site's local and global parities differ by one."""
        return int(global_parity) ^ ((self.t0 - 1) & 1)

    def left(self):
        return (self.rank - 1) % self.world

    def right(self):
        return (self.rank + 1) % self.world

    def slice_view(self, field, tl):
        """Bytes of local time slice tl of a native half spinor held in a flat uint8 tensor."""
        return field[tl * self.slice_bytes:(tl + 1) * self.slice_bytes]

    # ---- ghost exchange ----------------------------------------------------------------------------------
    def exchange(self, field, dist):
        """Fill the ghost slices of `field` (flat uint8 tensor, native half spinor of this slab) from the ring
        neighbours with torch.distributed point-to-point copies; blocks until they have arrived."""
        if self.world == 1:
            self.slice_view(field, 0).copy_(self.slice_view(field, self.Tl))
            self.slice_view(field, self.Tl + 1).copy_(self.slice_view(field, 1))
            return
        ops = [dist.P2POp(dist.isend, self.slice_view(field, 1), self.left()),
               dist.P2POp(dist.isend, self.slice_view(field, self.Tl), self.right()),
               dist.P2POp(dist.irecv, self.slice_view(field, self.Tl + 1), self.right()),
               dist.P2POp(dist.irecv, self.slice_view(field, 0), self.left())]
        for req in dist.batch_isend_irecv(ops):
            req.wait()

    # ---- the operator ------------------------------------------------------------------------------------
    def dslash_eo(self, out, gauge, inp, global_out_parity, exchange, stream=None):
        """out = H in on this rank's interior slices.  `exchange(field)` fills the ghosts of `inp` (self.exchange
        bound to a process group, or an emulation); the slices that do not touch a ghost are launched first, so
        with an asynchronous exchange on another stream they overlap it."""
        lp = self.local_parity(global_out_parity)
        if self.Tl > 2:
            self.ctx.dslash_eo_range(out, gauge, inp, lp, 2, self.Tl, stream)
        exchange(inp)
        self.ctx.dslash_eo_range(out, gauge, inp, lp, 1, 2, stream)
        self.ctx.dslash_eo_range(out, gauge, inp, lp, self.Tl, self.Tl + 1, stream)


def exchange_emulated(slabs, fields):
    """All ranks in one process (one GPU): copy the boundary slices between the slabs' fields directly."""
    n = len(slabs)
    for r, s in enumerate(slabs):
        left, right = fields[(r - 1) % n], fields[(r + 1) % n]
        s.slice_view(fields[r], 0).copy_(slabs[(r - 1) % n].slice_view(left, s.Tl))
        s.slice_view(fields[r], s.Tl + 1).copy_(slabs[(r + 1) % n].slice_view(right, 1))
