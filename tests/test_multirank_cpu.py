"""world_size-2 gloo test of the multi-GPU host logic: block sharding covers the
batch without overlap, the per-rank results of a sharded stage equal the single-process stage
(blocks are independent: no collective on the data path), and timings reduce as the max."""
import os
import socket

import numpy as np
import pytest
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
