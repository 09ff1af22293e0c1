"""Multi-GPU ghost exchange for the stage driver: host-side plan and transport.

MeshBlocks are sharded over ranks in contiguous ranges (shard.py).  A rank keeps, behind its own
blocks, read-only MIRROR copies of the remote blocks its neighbour table refers to; before every
ghost fill the owners send what the readers need of those blocks' U~ and B~f with point-to-point
torch.distributed operations (NCCL over NVLink on GPUs, gloo in the CPU tests), after which the
unchanged single-GPU ghost fill (ak_fill_ghosts with ak_set_neighbors(..., nmb_total)) reads the
mirrors like local blocks.  What travels is the ghost SLAB of each (block, neighbour code) pair
(include/ak.h: ak_halo_pack / ak_halo_unpack): one packed buffer and one message per peer and
direction.  HaloPlan.exchange (whole blocks, nothing packed) is kept as the plain alternative.

This module holds no arithmetic and no sequencing of the method: it builds index tables and moves
bytes.  The Runge-Kutta stage loop is the library's (ak_advance_hooked calls back here before every
ghost fill); `ops` says whose loop runs, so the same plan drives the CUDA library on GPUs and, in
tests/test_multirank_cpu.py, the CPU oracle on gloo.
"""
import numpy as np

from . import shard


def slab_box(n, ng, code, fld):
    """(start, extent) per axis x, y, z of the slab of neighbour code `code` for field `fld`
    (0-4 cell fields, 5-7 B~f^x,y,z) - the index rule of include/ak.h (ak_halo_pack), host copy."""
    o = (code % 3 - 1, (code // 3) % 3 - 1, code // 9 - 1)
    box = []
    for a in range(3):
        start = n if o[a] < 0 else ng
        if fld - 5 == a:
            ext = ng if o[a] < 0 else (ng + 1 if o[a] > 0 else n + 1)
        else:
            ext = ng if o[a] != 0 else n
        box.append((start, ext))
    return box


def slab_elems(n, ng, code):
    return sum(int(np.prod([e for _, e in slab_box(n, ng, code, fld)])) for fld in range(8))


class HaloPlan:
    """Index tables of one rank for a global neighbour table nbr_global[nmb_global][27]."""

    def __init__(self, nbr_global, rank, world):
        nbr_global = np.asarray(nbr_global, dtype=np.int64).reshape(-1, 27)
        self.rank, self.world = rank, world
        nb = nbr_global.shape[0]
        self.ranges = [shard.shard_blocks(nb, r, world) for r in range(world)]
        lo, hi = self.ranges[rank]
        self.lo, self.hi, self.n_own = lo, hi, hi - lo
        owner = np.empty(nb, dtype=np.int64)
        for r, (a, b) in enumerate(self.ranges):
            owner[a:b] = r
        self.owner = owner
        mine = nbr_global[lo:hi]
        remote = sorted({int(g) for g in mine.ravel() if g >= 0 and not (lo <= g < hi)})
        self.mirrors = remote                                   # global ids, in mirror-slot order
        slot = {g: self.n_own + q for q, g in enumerate(remote)}
        local = np.full(mine.shape, -1, dtype=np.int32)
        for (m, o), g in np.ndenumerate(mine):
            if g < 0:
                continue
            local[m, o] = g - lo if lo <= g < hi else slot[int(g)]
        self.local_nbr = local
        self.n_total = self.n_own + len(remote)
        # what I receive: for each peer, the mirror slots it fills (ascending global id)
        self.recv = {}
        for g in remote:
            self.recv.setdefault(int(owner[g]), []).append(slot[g])
        # what I send: every rank derives every other rank's mirror list the same way
        self.send = {}
        for r, (a, b) in enumerate(self.ranges):
            if r == rank:
                continue
            theirs = nbr_global[a:b]
            want = sorted({int(g) for g in theirs.ravel() if lo <= g < hi})
            if want:
                self.send[r] = [g - lo for g in want]
        # slabs: (block, neighbour code) pairs, ordered by (global id, code) on both ends
        self.send_pairs, self.recv_pairs = {}, {}
        for (m, o), g in np.ndenumerate(mine):
            if o != 13 and g >= 0 and not (lo <= g < hi):
                self.recv_pairs.setdefault(int(owner[g]), set()).add((int(g), o))
        for r, (a, b) in enumerate(self.ranges):
            if r == rank:
                continue
            for (m, o), g in np.ndenumerate(nbr_global[a:b]):
                if o != 13 and lo <= g < hi:
                    self.send_pairs.setdefault(r, set()).add((int(g), o))
        self.send_pairs = {r: sorted(v) for r, v in sorted(self.send_pairs.items())}
        self.recv_pairs = {r: sorted(v) for r, v in sorted(self.recv_pairs.items())}
        self._slot = slot
        self._tables = {}

    def slab_tables(self, n, ng=4):
        """(send_desc, send_seg, recv_desc, recv_seg) for blocks of n^3: desc = int64 [ndesc][3] =
        block index in the local arrays, neighbour code, offset in the rank's send (receive) buffer;
        seg[peer] = (start, length) of that peer's contiguous part of the buffer, in doubles."""
        key = (n, ng)
        if key not in self._tables:
            out = []
            for pairs, index in ((self.send_pairs, lambda g: g - self.lo), (self.recv_pairs, lambda g: self._slot[g])):
                desc, seg, off = [], {}, 0
                for peer, lst in pairs.items():
                    start = off
                    for g, code in lst:
                        desc.append((index(g), code, off))
                        off += slab_elems(n, ng, code)
                    seg[peer] = (start, off - start)
                out += [np.array(desc, dtype=np.int64).reshape(-1, 3), seg]
            self._tables[key] = tuple(out)
        return self._tables[key]

    def refresh(self, ops, U, Bf):
        """Refresh what the ghost fill reads of the mirror blocks: pack -> one message per peer ->
        unpack.  ops: n; halo_buffers(nsend, nrecv) -> (sendbuf, recvbuf) 1-D float64 tensors;
        pack(desc, U, Bf, sendbuf); unpack(desc, recvbuf, U, Bf)."""
        if self.world == 1 or (not self.send_pairs and not self.recv_pairs):
            return
        import torch.distributed as dist
        sdesc, sseg, rdesc, rseg = self.slab_tables(ops.n)
        nsend = sum(l for _, l in sseg.values()); nrecv = sum(l for _, l in rseg.values())
        sendbuf, recvbuf = ops.halo_buffers(nsend, nrecv)
        ops.pack(sdesc, U, Bf, sendbuf)
        p2p = [dist.P2POp(dist.isend, sendbuf[a:a + l], peer) for peer, (a, l) in sseg.items()]
        p2p += [dist.P2POp(dist.irecv, recvbuf[a:a + l], peer) for peer, (a, l) in rseg.items()]
        for w in dist.batch_isend_irecv(p2p):
            w.wait()
        ops.unpack(rdesc, recvbuf, U, Bf)

    def exchange(self, fields):
        """Refresh the mirror blocks of every tensor in `fields` ([n_total, ...], block-major)."""
        if self.world == 1 or (not self.send and not self.recv):
            return
        import torch.distributed as dist
        ops = []
        for t in fields:
            for peer, blocks in sorted(self.send.items()):
                for b in blocks:
                    ops.append(dist.P2POp(dist.isend, t[b], peer))
            for peer, slots in sorted(self.recv.items()):
                for s in slots:
                    ops.append(dist.P2POp(dist.irecv, t[s], peer))
        for w in dist.batch_isend_irecv(ops):
            w.wait()


def advance(plan, ops, integrator, nsteps, dt, U, Bf, whole_blocks=False):
    """nsteps steps of SSP-RK<integrator> over this rank's blocks with a mirror refresh before every ghost
    fill.  The stage sequence (fill -> rhs with the stage's FOFC blend -> Shu-Osher update, with CT) is
    not written here: it lives behind the boundary (ak_advance_hooked; the oracle's orc_advance_hooked in
    the CPU tests), which calls back into `refresh` at the right places.
    ops: advance(integrator, nsteps, dt, U, Bf, refresh), and what HaloPlan.refresh needs.
    whole_blocks: refresh the mirrors with HaloPlan.exchange instead of ghost slabs."""
    refresh = (lambda: plan.exchange(list(U) + list(Bf))) if whole_blocks else (lambda: plan.refresh(ops, U, Bf))
    ops.advance(integrator, nsteps, dt, U, Bf, refresh)


class AkOps:
    """`ops` for the CUDA library: U, Bf, W are lists of device tensors with plan.n_total blocks; the
    context was created with nmb = plan.n_own on torch's current stream (the point-to-point
    operations order themselves against that stream)."""

    def __init__(self, ctx, plan, bc, W, dU, E, flag=None):
        from . import ak
        self.ak, self.ctx, self.bc = ak, ctx, bc
        self.W, self.dU, self.E, self.flag = W, dU, E, flag
        self.n = int(W[0].shape[1]) - 8
        self._bufs, self._desc = None, {}
        ak.ak_set_neighbors(ctx, plan.local_nbr, plan.n_total)

    def halo_buffers(self, nsend, nrecv):
        import torch
        if self._bufs is None or self._bufs[0].numel() != nsend or self._bufs[1].numel() != nrecv:
            dev = self.W[0].device
            self._bufs = (torch.empty(nsend, dtype=torch.float64, device=dev),
                          torch.empty(nrecv, dtype=torch.float64, device=dev))
        return self._bufs

    def _dev_desc(self, desc):
        import torch
        key = id(desc)
        if key not in self._desc:
            self._desc[key] = (desc, torch.from_numpy(desc).to(self.W[0].device))     # keeps desc alive
        return self._desc[key][1]

    def pack(self, desc, U, Bf, buf):
        if len(desc):
            self.ak.ak_halo_pack(self.ctx, self._dev_desc(desc), U, Bf, buf)

    def unpack(self, desc, buf, U, Bf):
        if len(desc):
            self.ak.ak_halo_unpack(self.ctx, self._dev_desc(desc), buf, U, Bf)

    def advance(self, integrator, nsteps, dt, U, Bf, refresh):
        self.ak.ak_advance_hooked(self.ctx, integrator, nsteps, dt, self.bc, U, Bf, self.W, self.flag, refresh)
