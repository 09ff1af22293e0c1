"""world_size-2 gloo test of the multi-GPU host logic: block sharding covers the
batch without overlap, the per-rank results of a sharded stage equal the single-process stage
(blocks are independent: no collective on the data path), and timings reduce as the max."""
import os
import socket

import numpy as np
import pytest
import sys
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2409_10384_b200 import shard, workloads as wl


def test_shard_blocks_partition():
    for nmb in (1, 2, 7, 8, 768):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                lo, hi = shard.shard_blocks(nmb, r, world)
                assert 0 <= lo <= hi <= nmb
                got += list(range(lo, hi))
            assert got == list(range(nmb))
            sizes = [shard.shard_blocks(nmb, r, world) for r in range(world)]
            assert max(h - l for l, h in sizes) - min(h - l for l, h in sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_blocks(4, 2, 2)
    ids = np.arange(10)
    assert np.array_equal(shard.rank_block_ids(ids, 1, 2, strong=False), ids)
    assert np.array_equal(shard.rank_block_ids(ids, 1, 2, strong=True), ids[5:])


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ids, out):
    from oracle import pyoracle as orc
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = shard.rank_block_ids(ids, rank, world, strong=True)
        w = wl.make_blocks("C1", blocks=mine)
        r = orc.rhs(orc.make_params(**w["params"]), w["dx"], w["U"], w["Bf"], w["adm"], w["dt_fofc"])
        # gather per-rank results on rank 0 (reporting only; the stage itself never communicates)
        payload = dict(ids=mine, dD=r["dU"][0], Ez=r["E"][2], flag=r["flag"])
        gathered = [None] * world if rank == 0 else None
        dist.gather_object(payload, gathered, dst=0)
        tmax = shard.reduce_max(10.0 + rank)
        zsum = shard.reduce_sum(len(mine))
        if rank == 0:
            out.put((gathered, tmax, zsum))
    finally:
        dist.destroy_process_group()


def test_sharded_stage_equals_single_process():
    from oracle import pyoracle as orc
    orc.build()
    ids = np.array([0, 3, 7])
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, ids, q)) for r in range(world)]
    for p in procs:
        p.start()
    gathered, tmax, zsum = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert tmax == 11.0 and zsum == 3.0
    w = wl.make_blocks("C1", blocks=ids)
    ref = orc.rhs(orc.make_params(**w["params"]), w["dx"], w["U"], w["Bf"], w["adm"], w["dt_fofc"])
    seen = []
    for part in gathered:
        for local, b in enumerate(part["ids"]):
            g = int(np.where(ids == b)[0][0])
            seen.append(int(b))
            assert np.array_equal(part["dD"][local], ref["dU"][0][g])
            assert np.array_equal(part["Ez"][local], ref["E"][2][g])
            assert np.array_equal(part["flag"][local], ref["flag"][g])
    assert sorted(seen) == sorted(ids.tolist())


# ---------------------------------------------------------------- halo exchange across ranks
def _eight_block_domain():
    """the periodic 12^3 domain of T27 as 2x2x2 blocks of 6^3 (identical in every process)."""
    import stagekit as sk
    from oracle import pyoracle as orc
    N, n, NG = 12, 6, 4
    d = 1.0 / N

    def prim(x, y, z):
        rho = 1.0 + 0.3 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) + 0.2 * np.sin(2 * np.pi * z)
        rho = np.where((abs(x - 0.3) < 0.1) & (abs(y - 0.6) < 0.1) & (abs(z - 0.5) < 0.1), 1e-3 * rho, rho)
        o = np.ones_like(x)
        return rho, [0.3 * np.sin(2 * np.pi * y) * o, -0.2 * o, 0.25 * np.cos(2 * np.pi * x) * o], 0.6 * o

    def A(comp, x, y, z):
        return 0.1 * np.sin(2 * np.pi * (x + 2 * y)) if comp == 2 else 0.05 * np.cos(2 * np.pi * z) * (comp == 0) + 0 * x
    blocks = []
    for bz in range(2):
        for by in range(2):
            for bx in range(2):
                blocks.append(sk.build_block(n, d, (bx * n * d, by * n * d, bz * n * d), sk.flat_metric, prim,
                                             A_fn=A, gamma_ad=5.0 / 3.0))
    cat = lambda key, q: np.ascontiguousarray(np.concatenate([b[key][q] for b in blocks], axis=0))
    p = dict(n=n, gamma_ad=5.0 / 3.0, rho_atm=1e-10, T_atm=1e-8, recon=2, riemann=1, fofc=1, dmp_M=1.2)
    return dict(U=[cat("U", v) for v in range(5)], Bf=[cat("Bf", c) for c in range(3)],
                adm=[cat("adm", q) for q in range(16)], dx=np.full((8, 3), d), p=p, dt=0.15 * d)


def numpy_slabs(desc, fields, buf, n, unpack, ng=4):
    """pack/unpack by numpy slicing: the eight boxes of every (block, code) pair, k-major, in order."""
    from paper_2409_10384_b200 import halo
    for blk, code, off in desc:
        for fld in range(8):
            (sx, ex), (sy, ey), (sz, ez) = halo.slab_box(n, ng, int(code), fld)
            view = fields[fld][blk, sz:sz + ez, sy:sy + ey, sx:sx + ex]
            cnt = ex * ey * ez
            if unpack:
                view[...] = buf[off:off + cnt].reshape(ez, ey, ex)
            else:
                buf[off:off + cnt] = view.reshape(-1)
            off += cnt


class _OracleOps:
    """halo.advance `ops` backed by the CPU oracle (numpy views of the CPU tensors)."""

    def __init__(self, par, plan, dx, adm, bc, n):
        from oracle import pyoracle as orc
        self.orc, self.par, self.plan, self.dx, self.adm, self.bc, self.n = orc, par, plan, dx, adm, bc, n

    def halo_buffers(self, nsend, nrecv):
        return torch.zeros(nsend, dtype=torch.float64), torch.zeros(nrecv, dtype=torch.float64)

    def pack(self, desc, U, Bf, buf):
        numpy_slabs(desc, [u.numpy() for u in U] + [b.numpy() for b in Bf], buf.numpy(), self.n, unpack=False)

    def unpack(self, desc, buf, U, Bf):
        numpy_slabs(desc, [u.numpy() for u in U] + [b.numpy() for b in Bf], buf.numpy(), self.n, unpack=True)

    def advance(self, integrator, nsteps, dt, U, Bf, refresh):
        # U, Bf: n_total blocks (own + mirrors), numpy views of the CPU tensors, advanced in place
        self.orc.advance_hooked(self.par, self.dx, integrator, nsteps, dt, self.bc, self.plan.local_nbr,
                                [u.numpy() for u in U], [b.numpy() for b in Bf], self.adm, refresh)


def _halo_worker(rank, world, port, out, whole_blocks=False):
    from oracle import pyoracle as orc
    from paper_2409_10384_b200 import halo
    from test_oracle_exchange import lattice_nbr
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dom = _eight_block_domain()
        nbr = lattice_nbr((2, 2, 2), (True, True, True))
        plan = halo.HaloPlan(nbr, rank, world)
        lo, hi = plan.lo, plan.hi

        def with_mirrors(a):
            # mirrors start as NaN: anything the ghost fill reads of them must have been delivered
            t = torch.full((plan.n_total,) + a.shape[1:], float("nan"), dtype=torch.float64)
            t[:plan.n_own] = torch.from_numpy(a[lo:hi])
            return t
        U = [with_mirrors(u) for u in dom["U"]]; Bf = [with_mirrors(b) for b in dom["Bf"]]
        par = orc.make_params(nmb=plan.n_own, **dom["p"])
        ops = _OracleOps(par, plan, dom["dx"][lo:hi], [np.ascontiguousarray(a[lo:hi]) for a in dom["adm"]], (0, 0, 0),
                         dom["p"]["n"])
        halo.advance(plan, ops, 3, 2, dom["dt"], U, Bf, whole_blocks=whole_blocks)
        payload = dict(lo=lo, hi=hi, U=[u[:plan.n_own].numpy().copy() for u in U],
                       Bf=[b[:plan.n_own].numpy().copy() for b in Bf], mirrors=plan.mirrors)
        gathered = [None] * world if rank == 0 else None
        dist.gather_object(payload, gathered, dst=0)
        if rank == 0:
            out.put(gathered)
    finally:
        dist.destroy_process_group()


def test_halo_plan_tables():
    from paper_2409_10384_b200 import halo
    from test_oracle_exchange import lattice_nbr
    nbr = lattice_nbr((2, 2, 2), (True, True, True))
    plans = [halo.HaloPlan(nbr, r, 2) for r in range(2)]
    for r, pl in enumerate(plans):
        other = plans[1 - r]
        assert pl.n_own == 4 and pl.mirrors == list(range(other.lo, other.hi))     # 2x2x2 periodic: all remote
        assert sorted(pl.send[1 - r]) == [g - pl.lo for g in other.mirrors]
        assert len(pl.recv[1 - r]) == len(other.send[r])
        # every table entry resolves to the right global block
        glob = list(range(pl.lo, pl.hi)) + pl.mirrors
        for m in range(pl.n_own):
            for o in range(27):
                if o != 13:
                    assert glob[pl.local_nbr[m, o]] == nbr[pl.lo + m, o]
    one = halo.HaloPlan(nbr, 0, 1)
    assert one.n_total == 8 and not one.send and not one.recv and np.array_equal(one.local_nbr, nbr)


@pytest.mark.parametrize("whole_blocks", [False, True])
def test_two_ranks_with_halo_exchange_equal_one_process(whole_blocks):
    """ghost slabs (default) and whole-block mirrors both reproduce the single-process run bit for bit."""
    from oracle import pyoracle as orc
    from test_oracle_exchange import lattice_nbr
    orc.build()
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_halo_worker, args=(r, world, port, q, whole_blocks)) for r in range(world)]
    for p in procs:
        p.start()
    gathered = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    dom = _eight_block_domain()
    nbr = lattice_nbr((2, 2, 2), (True, True, True))
    par = orc.make_params(nmb=8, **dom["p"])
    U = [u.copy() for u in dom["U"]]; Bf = [b.copy() for b in dom["Bf"]]
    orc.advance_nbr(par, dom["dx"], 3, 2, dom["dt"], (0, 0, 0), nbr, U, Bf, dom["adm"], nthreads=4)
    for part in gathered:
        lo, hi = part["lo"], part["hi"]
        for v in range(5):
            assert np.array_equal(part["U"][v], U[v][lo:hi]), (lo, v)
        for c in range(3):
            assert np.array_equal(part["Bf"][c], Bf[c][lo:hi]), (lo, c)


def test_slab_boxes_are_what_the_exchange_reads():
    """Pin of the slab index rule (include/ak.h, halo.slab_box) against the oracle's ghost exchange: on
    a periodic 3x3x3 lattice every element carries its own address; after orc.exchange_ghosts the
    ghosts of block 0 tell which elements of which neighbour were read.  For every neighbour code
    that set equals the slab box, except that a face field's box keeps face ie+1 along its normal
    where the offset is 0 (read only when the reader has no upper image there)."""
    from oracle import pyoracle as orc
    from paper_2409_10384_b200 import halo
    from test_oracle_exchange import lattice_nbr
    n, ng, nmb = 6, 4, 27
    nt = n + 2 * ng
    sh = orc.shapes(nmb, n)
    nbr = lattice_nbr((3, 3, 3), (True, True, True))
    keys = ["cell"] * 5 + ["xf", "yf", "zf"]
    fields = []
    for k in keys:
        per = int(np.prod(sh[k][1:]))
        fields.append((np.arange(nmb)[:, None] * 1e6 + np.arange(per)[None, :]).reshape(sh[k]).astype(np.float64))
    before = [f.copy() for f in fields]
    orc.exchange_ghosts(orc.make_params(nmb=nmb, n=n), nbr, (0, 0, 0), fields[:5], fields[5:])
    code_of = {int(nbr[0, c]): c for c in range(27) if c != 13}
    assert len(code_of) == 26
    for fld, k in enumerate(keys):
        shape = sh[k][1:]
        got = fields[fld][0]
        changed = got != before[fld][0]
        src_blk = (got[changed] // 1e6).astype(int)
        src_idx = (got[changed] % 1e6).astype(int)
        assert 0 not in set(src_blk.tolist())
        for blk, code in code_of.items():
            read = set(src_idx[src_blk == blk].tolist())
            (sx, ex), (sy, ey), (sz, ez) = halo.slab_box(n, ng, code, fld)
            box = np.zeros(shape, dtype=bool)
            box[sz:sz + ez, sy:sy + ey, sx:sx + ex] = True
            boxset = set(np.flatnonzero(box).tolist())
            assert read <= boxset, (fld, code)
            extra = boxset - read
            if fld < 5:
                assert not extra, (fld, code)
            else:
                a = fld - 5                                              # normal axis: 0 x, 1 y, 2 z
                o = (code % 3 - 1, (code // 3) % 3 - 1, code // 9 - 1)[a]
                idx = np.array(sorted(extra), dtype=int)
                coord = np.unravel_index(idx, shape)[2 - a] if idx.size else idx
                assert (o == 0 and np.all(coord == ng + n)) or idx.size == 0, (fld, code)
        assert sum(halo.slab_elems(n, ng, c) for c in code_of.values()) > 0
