"""Time-slab decomposition of the even-odd dslash over several GPUs (next row f3).

One process per GPU (torch.distributed); rank r owns the global time slices [r T/N, (r+1) T/N) as a local lattice of
exactly those slices (T/N even, so local and global site parities agree).  Everything arithmetic stays in the CUDA
kernels (csrc/slab_kernels.cuh): the face projection to half spinors, the stores into the neighbours' halo buffers, the
boundary sites that consume them.  This module is plumbing only: which slices a rank holds, where the global boundary
phase cuts it (lqcd_set_time_slab), the buffers, the streams and events that order push / interior / boundary, and the
transport of the projected faces (12 reals per face site, 786 KB per face in fp32 at 32^3 x 64):

  PeerMemoryTransport   the B200 path: halo buffers and flags live in NVLink-mapped symmetric memory
                        (torch.distributed._symmetric_memory); lqcd_slab_push_faces stores the projected faces straight
                        into the neighbours' buffers and publishes an epoch, lqcd_dslash_eo_slab acquires it on the
                        device -- projection, transfer and consumption without a host round trip or a library collective
  SendRecvTransport     projected faces into local send buffers, then ncclSend / ncclRecv between ring neighbours
                        (torch.distributed P2P ops: NCCL on GPUs, gloo in the CPU tests) on a side stream, an event
                        orders the boundary launches after the receives
  LocalRingTransport    all ranks in one process on one GPU (tests, single-GPU emulation): "peer" pointers are the other
                        slabs' buffers, ordering by stream order

The paper's own multi-device scheme is host-mediated; this is the natural sharding named in
SURVEY.md sec. 8(e).  The headline bench stays "replicas only" (north_star: single GPU); bench.py's `slab` leg times this
path when WORLD_SIZE > 1.
"""
from __future__ import annotations

from . import Context


class TimeSlab:
    """Rank `rank` of `world` in a decomposition of a lattice of global extents dims = (X, Y, Z, T) along t."""

    def __init__(self, dims, precision, recon, bc, rank, world):
        X, Y, Z, T = (int(d) for d in dims)
        if T % world or (T // world) % 2 or T // world < 4:
            raise ValueError("T / world must be an even number of time slices, at least 4")
        self.global_dims, self.rank, self.world = (X, Y, Z, T), int(rank), int(world)
        self.Tl = T // world
        self.t0 = self.rank * self.Tl
        self.local_dims = (X, Y, Z, self.Tl)
        self.ctx = Context(self.local_dims, precision, recon, bc)
        # the global t boundary lies between the last slice of the last rank and the first slice of rank 0
        self.ctx.set_time_slab(self.Tl - 1 if self.rank == self.world - 1 else -1, 0 if self.rank == 0 else -1)
        self.halo_bytes = self.ctx.halo_bytes()
        if self.halo_bytes == 0:
            raise ValueError("no slab path for this context (precision 16 / half links)")
        self.face_sites = X * Y * Z // 2

    # ---- bookkeeping -------------------------------------------------------------------------------------
    def time_indices(self):
        """Global t of the local slices 0 .. Tl - 1."""
        return list(range(self.t0, self.t0 + self.Tl))

    def below(self):
        return (self.rank - 1) % self.world

    def above(self):
        return (self.rank + 1) % self.world

    def t_below(self):
        """Global t of the last slice of the rank below: its t links are the backward t links of local slice 0."""
        return (self.t0 - 1) % self.global_dims[3]

    def pack_gauge(self, native, U_local, Ut_below, stream=None):
        """U_local: canonical links [4][Tl][Z][Y][X][3][3] of the own slices; Ut_below: canonical [Z][Y][X][3][3] t links of
        global slice t_below() (device tensors)."""
        self.ctx.pack_gauge_slab(native, U_local, Ut_below, stream)

    # ---- the operator ------------------------------------------------------------------------------------
    def dslash_eo(self, out, gauge, inp, out_parity, transport, stream=None):
        """out = H in on this rank's slices.  Enqueue only: the faces are projected and pushed on the transport's side
        stream while the interior slices (which read no halo) run on `stream`; the two boundary slices follow once the
        neighbours' faces have arrived (an event, or the device-side epoch of the peer-memory transport)."""
        import torch
        stream = stream if stream is not None else torch.cuda.current_stream()
        h = transport.push(self, inp, stream)                       # side stream: projection + transfer
        self.ctx.dslash_eo_range(out, gauge, inp, out_parity, 1, self.Tl - 1, stream)
        h.before_boundary(stream)
        kw = dict(wait_up=h.wait_up, wait_down=h.wait_down, epoch=h.epoch, stream=stream)
        self.ctx.dslash_eo_slab(out, gauge, inp, h.from_up, h.from_down, out_parity, 0, 1, **kw)
        self.ctx.dslash_eo_slab(out, gauge, inp, h.from_up, h.from_down, out_parity, self.Tl - 1, self.Tl, **kw)
        transport.after_boundary(self, stream)


class _Halos:
    """What one push hands to the boundary launches."""

    def __init__(self, from_up, from_down, event=None, wait_up=None, wait_down=None, epoch=0):
        self.from_up, self.from_down, self.event = from_up, from_down, event
        self.wait_up, self.wait_down, self.epoch = wait_up, wait_down, epoch

    def before_boundary(self, stream):
        if self.event is not None:
            stream.wait_event(self.event)


def _align(n, a=256):
    return (n + a - 1) // a * a


class LocalRingTransport:
    """All ranks of the ring in one process on one GPU: every slab's halo buffers are ordinary device tensors and the
    "peer" pointers handed to lqcd_slab_push_faces are the neighbouring slabs' buffers.  `push_all` runs every rank's
    face projection first (one stream: stream order is the synchronisation); with use_flags the device-side epoch
    protocol is exercised too -- the flags are already published when the boundary kernels start, so nothing spins."""

    def __init__(self, slabs, device, use_flags=False):
        import torch
        self.slabs, self.use_flags, self.epoch = slabs, use_flags, 0
        hb = slabs[0].halo_bytes
        self.from_up = [torch.full((hb,), 0xFF, dtype=torch.uint8, device=device) for _ in slabs]    # NaN-ish until pushed
        self.from_down = [torch.full((hb,), 0xFF, dtype=torch.uint8, device=device) for _ in slabs]
        self.flags = [torch.zeros(2, dtype=torch.int64, device=device) for _ in slabs]                 # [from_up, from_down]

    def push_all(self, inputs, stream=None):
        self.epoch += 1
        for r, s in enumerate(self.slabs):
            up, dn = s.above(), s.below()
            fu = self.flags[up][1:2] if self.use_flags else None       # my last slice is the rank above's "from_down"
            fd = self.flags[dn][0:1] if self.use_flags else None
            s.ctx.slab_push_faces(inputs[r], self.from_down[up], self.from_up[dn], fu, fd, self.epoch, stream)

    def push(self, slab, inp, stream):
        r = slab.rank
        if self.use_flags:
            return _Halos(self.from_up[r], self.from_down[r], None, self.flags[r][0:1], self.flags[r][1:2], self.epoch)
        return _Halos(self.from_up[r], self.from_down[r])

    def after_boundary(self, slab, stream):
        pass


class SendRecvTransport:
    """Faces projected into local send buffers, exchanged with the ring neighbours by torch.distributed point-to-point
    operations (ncclSend / ncclRecv on GPUs; gloo with host tensors in the CPU tests) on a side stream.  The host never
    waits with NCCL: `Work.wait()` only makes the side stream wait for NCCL's stream, and an event orders the boundary
    launches after the receives."""
    TAG_DOWNWARD, TAG_UPWARD = 1, 2     # a face travelling to the rank below / above

    def __init__(self, slab, dist, device):
        import torch
        self.dist, self.device = dist, torch.device(device)
        self.cuda = self.device.type == "cuda"
        hb = slab.halo_bytes
        mk = lambda: torch.zeros(hb, dtype=torch.uint8, device=self.device)
        self.send_up, self.send_down, self.from_up, self.from_down = mk(), mk(), mk(), mk()
        self.side = torch.cuda.Stream(self.device) if self.cuda else None
        self.use_tags = dist is not None and dist.get_backend() != "nccl"
        # a backend without device buffers (gloo: the functional test of the N > 1 path on a one-GPU box) goes through
        # pinned host copies; NCCL sends and receives the device buffers directly
        self.host_staged = self.cuda and dist is not None and dist.get_backend() != "nccl"
        if self.host_staged:
            hk = lambda: torch.zeros(hb, dtype=torch.uint8).pin_memory()
            self.h_send_up, self.h_send_down, self.h_from_up, self.h_from_down = hk(), hk(), hk(), hk()

    def exchange(self, slab):
        """send_down -> rank below (its from_up), send_up -> rank above (its from_down).  On a ring of two both
        neighbours are the same rank: NCCL pairs the operations of a peer in the order they are posted, so the sends go
        [downward, upward] and the receives [from above, from below] -- the downward face of the rank above is what
        from_up must get.  Backends with tags (gloo) carry the direction in the tag as well."""
        dist = self.dist
        if slab.world == 1:
            self.from_up.copy_(self.send_down)
            self.from_down.copy_(self.send_up)
            return
        tag = (lambda t: dict(tag=t)) if self.use_tags else (lambda t: {})
        sd, su, fu, fd = self.send_down, self.send_up, self.from_up, self.from_down
        if self.host_staged:
            import torch
            self.h_send_down.copy_(sd, non_blocking=True)
            self.h_send_up.copy_(su, non_blocking=True)
            torch.cuda.current_stream(self.device).synchronize()
            sd, su, fu, fd = self.h_send_down, self.h_send_up, self.h_from_up, self.h_from_down
        ops = [dist.P2POp(dist.isend, sd, slab.below(), **tag(self.TAG_DOWNWARD)),
               dist.P2POp(dist.isend, su, slab.above(), **tag(self.TAG_UPWARD)),
               dist.P2POp(dist.irecv, fu, slab.above(), **tag(self.TAG_DOWNWARD)),
               dist.P2POp(dist.irecv, fd, slab.below(), **tag(self.TAG_UPWARD))]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        if self.host_staged:
            self.from_up.copy_(fu, non_blocking=True)
            self.from_down.copy_(fd, non_blocking=True)

    def push(self, slab, inp, stream):
        import torch
        self.side.wait_stream(stream)          # the input is ready and the previous boundary launches have read the halos
        with torch.cuda.stream(self.side):
            slab.ctx.slab_push_faces(inp, self.send_up, self.send_down, stream=self.side)
            self.exchange(slab)
            ev = torch.cuda.Event()
            ev.record(self.side)
        return _Halos(self.from_up, self.from_down, ev)

    def after_boundary(self, slab, stream):
        pass


class PeerMemoryTransport:
    """Halo buffers and flags in NVLink-mapped symmetric memory.  Per rank: two generations (epoch parity) of
    [from_up | from_down] halo buffers and two 8-byte flags.  A push stores this rank's projected faces directly into the
    neighbours' buffers of the current generation (the face-projection kernel's own stores cross NVLink) and then
    publishes the epoch into their flags; the boundary kernel acquires this rank's own two flags on the device.  Two
    generations suffice: a rank pushes generation n + 1 only after its own boundary launches of application n
    (side.wait_stream), and a neighbour can push n + 2 only after it has consumed this rank's n + 1."""

    def __init__(self, slab, dist, device, group=None):
        import torch
        import torch.distributed._symmetric_memory as symm_mem
        self.dist, self.device = dist, torch.device(device)
        self.hb = _align(slab.halo_bytes)
        self.flag_off = 4 * self.hb
        nbytes = self.flag_off + 256
        self.buf = symm_mem.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.buf.zero_()
        self.hdl = symm_mem.rendezvous(self.buf, group if group is not None else dist.group.WORLD)
        self.ptrs = [int(p) for p in self.hdl.buffer_ptrs]
        assert self.ptrs[slab.rank] == self.buf.data_ptr()
        self.side = torch.cuda.Stream(self.device)
        self.epoch = 0
        torch.cuda.synchronize(self.device)     # this rank's flags are zero; make_transport's agreement (a collective
                                                # every rank passes) is what keeps anyone from pushing before that holds everywhere

    def _halo(self, rank, gen, which):          # which: 0 = from_up, 1 = from_down
        return self.ptrs[rank] + (2 * gen + which) * self.hb

    def _flag(self, rank, which):
        return self.ptrs[rank] + self.flag_off + 8 * which

    def push(self, slab, inp, stream):
        import torch
        self.epoch += 1
        gen, me = self.epoch & 1, slab.rank
        self.side.wait_stream(stream)
        slab.ctx.slab_push_faces(inp, self._halo(slab.above(), gen, 1), self._halo(slab.below(), gen, 0),
                                 self._flag(slab.above(), 1), self._flag(slab.below(), 0), self.epoch, stream=self.side)
        ev = None
        if slab.world == 1:                     # own faces, own flags: order by event, nothing may spin on this GPU
            ev = torch.cuda.Event()
            ev.record(self.side)
        return _Halos(self._halo(me, gen, 0), self._halo(me, gen, 1), ev, self._flag(me, 0), self._flag(me, 1), self.epoch)

    def after_boundary(self, slab, stream):
        pass


def _p2p_name(dist):
    return "ncclSend/ncclRecv" if dist.get_backend() == "nccl" else f"{dist.get_backend()} send/recv through pinned host copies (functional test path)"


def _all_ranks_ok(dist, ok, device):
    """Collective: True on every rank iff `ok` is true on every rank (MIN over the group).  The tensor lives where the
    backend can reduce it: on the GPU for NCCL, on the host otherwise."""
    import torch
    t = torch.tensor([1 if ok else 0], dtype=torch.int32, device=device if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return bool(int(t.item()))


def make_transport(slab, dist, device, kind="auto", peer_factory=None):
    """Returns (transport, name).  Collective: every rank of the group must call it with the same `kind`.

    kind = "sendrecv"  ncclSend / ncclRecv between ring neighbours (gloo through pinned host copies in the CPU tests).
    kind = "auto"      the same.  The peer-memory path has never run on two physical GPUs (every measurement of this
                       repository is single-GPU), and its boundary kernels spin on flags another GPU
                       writes, so it is not something to pick silently.
    kind = "peer"      symmetric memory + device-side epoch flags (PeerMemoryTransport), or an exception ON EVERY RANK.
    kind = "peer_or_sendrecv"  peer memory if it came up on every rank, send/recv on every rank otherwise.

    The choice is agreed on by the whole group: each rank tries to set the peer path up, then a MIN all-reduce of the
    outcome decides for all.  Without that, a rank whose rendezvous failed would post ncclSend / ncclRecv while its
    neighbours store into peer memory and spin on flags that are never written -- a hang on one side, a trap on the
    other.  (A rank that dies inside the rendezvous itself still stalls the others until the process group's timeout:
    nothing after the fact can repair that.)  peer_factory: the constructor to try, for tests."""
    if kind not in ("auto", "sendrecv", "peer", "peer_or_sendrecv"):
        raise ValueError(f"unknown transport kind {kind!r}")
    if kind in ("auto", "sendrecv"):
        return SendRecvTransport(slab, dist, device), _p2p_name(dist)
    transport, why = None, ""
    try:
        transport = (peer_factory or PeerMemoryTransport)(slab, dist, device)
    except Exception as e:  # noqa: BLE001 -- any failure of the set-up means: no peer mapping for this rank
        why = f"{type(e).__name__}: {e}"[:160]
    if _all_ranks_ok(dist, transport is not None, device):
        return transport, "peer-memory stores + device-side epoch flags (symmetric memory)"
    transport = None    # drop a mapping that came up here but not everywhere
    why = why or "set-up failed on another rank"
    if kind == "peer":
        raise RuntimeError(f"peer-memory transport unavailable on at least one rank (rank {slab.rank}: {why})")
    return SendRecvTransport(slab, dist, device), f"{_p2p_name(dist)} (peer memory unavailable: {why})"
