"""Multi-GPU ghost exchange for the stage driver: host-side plan and transport.

MeshBlocks are sharded over ranks in contiguous ranges (shard.py).  A rank keeps, behind its own
blocks, read-only MIRROR copies of the remote blocks its neighbour table refers to; before every
ghost fill the owners send those blocks' U~ and B~f (a block is one contiguous chunk of each
block-major array, so there is nothing to pack) with point-to-point torch.distributed operations
(NCCL over NVLink on GPUs, gloo in the CPU tests), after which the unchanged single-GPU ghost fill
(ak_fill_ghosts with ak_set_neighbors(..., nmb_total)) reads them like local blocks.  Whole blocks
travel instead of ghost slabs: simple and exact; slab packing is the optimisation left open.

This module holds no arithmetic of the method: it builds index tables, moves bytes and sequences
calls.  The stage operations are passed in (`ops`), so the same loop drives the CUDA library on
GPUs and, in tests/test_multirank_cpu.py, the CPU oracle on gloo.
"""
import numpy as np

from . import shard


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


# Shu-Osher weights: U <- a U0 + b (U + dt L(U))
RK_A = {1: (0.0,), 2: (0.0, 0.5), 3: (0.0, 0.75, 1.0 / 3.0)}
RK_B = {1: (1.0,), 2: (1.0, 0.5), 3: (1.0, 0.25, 2.0 / 3.0)}


def advance(plan, ops, integrator, nsteps, dt, U, Bf):
    """The loop of ak_advance with a mirror refresh before every ghost fill.
    ops: fill(U, Bf); rhs(U, Bf, U0_or_None, a, b, dt) -> (dU, E); update(a, b, dt, U0, B0, U, Bf, dU, E);
         snapshot(U, Bf) -> (U0, B0) copies of the owned blocks' state."""
    U0 = B0 = None
    for _ in range(nsteps):
        for s in range(integrator):
            a, b = RK_A[integrator][s], RK_B[integrator][s]
            plan.exchange(list(U) + list(Bf))
            ops.fill(U, Bf)
            dU, E = ops.rhs(U, Bf, None if s == 0 else U0, a, b, dt)
            if s == 0 and integrator > 1:
                U0, B0 = ops.snapshot(U, Bf)
            if s == 0:
                ops.update(0.0, 1.0, dt, U, Bf, U, Bf, dU, E)
            else:
                ops.update(a, b, dt, U0, B0, U, Bf, dU, E)
    plan.exchange(list(U) + list(Bf))
    ops.fill(U, Bf)


class AkOps:
    """`ops` for the CUDA library: U, Bf, W are lists of device tensors with plan.n_total blocks; the
    context was created with nmb = plan.n_own."""

    def __init__(self, ctx, plan, bc, W, dU, E, flag=None):
        from . import ak
        self.ak, self.ctx, self.bc = ak, ctx, bc
        self.W, self.dU, self.E, self.flag = W, dU, E, flag
        ak.ak_set_neighbors(ctx, plan.local_nbr, plan.n_total)

    def fill(self, U, Bf):
        self.ak.ak_fill_ghosts(self.ctx, self.bc, U, Bf)

    def rhs(self, U, Bf, U0, a, b, dt):
        self.ak.ak_set_fofc_blend(self.ctx, U0, a, b)
        self.ak.ak_rhs(self.ctx, U, Bf, self.W, 0, dt, self.dU, self.E, self.flag, None)
        self.ak.ak_set_fofc_blend(self.ctx, None)
        return self.dU, self.E

    def snapshot(self, U, Bf):
        return [u.clone() for u in U], [b.clone() for b in Bf]

    def update(self, a, b, dt, U0, B0, U, Bf, dU, E):
        self.ak.ak_stage_update(self.ctx, a, b, dt, U0, B0, U, Bf, dU, E)
