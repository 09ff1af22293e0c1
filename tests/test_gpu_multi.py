"""Multi-GPU readiness: the halo path over NCCL.  Skipped unless
the box has at least two GPUs (this project's GPU runs have one; the same plan is exercised on two gloo
ranks against the oracle in tests/test_multirank_cpu.py and as two lock-stepped contexts on one GPU in
tests/test_gpu_driver.py).  One process per GPU; nothing here makes a kernel wait on another rank's
kernel: the point-to-point operations are NCCL's own."""
import multiprocessing as mp
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _nccl_worker(rank, world, port, out, whole_blocks):
    import torch
    import torch.distributed as dist
    from paper_2409_10384_b200 import ak, halo
    from test_multirank_cpu import _eight_block_domain
    from test_oracle_exchange import lattice_nbr
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log (transport, NVLS) stays on
    dev = torch.device("cuda", rank)
    torch.cuda.set_device(dev)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    ctx = None
    try:
        dom = _eight_block_domain()
        nbr = lattice_nbr((2, 2, 2), (True, True, True))
        plan = halo.HaloPlan(nbr, rank, world)
        lo, hi = plan.lo, plan.hi

        def with_mirrors(a):        # mirrors start as NaN: whatever the ghost fill reads must have been delivered
            t = torch.full((plan.n_total,) + a.shape[1:], float("nan"), dtype=torch.float64)
            t[:plan.n_own] = torch.from_numpy(np.ascontiguousarray(a[lo:hi]))
            return t.to(dev)
        U = [with_mirrors(u) for u in dom["U"]]; Bf = [with_mirrors(b) for b in dom["Bf"]]
        adm = [torch.from_numpy(np.ascontiguousarray(a[lo:hi])).to(dev) for a in dom["adm"]]
        sh = ak.shapes(plan.n_own, dom["p"]["n"])
        z = lambda k: torch.zeros(sh[k], dtype=torch.float64, device=dev)
        W = [z("cell") for _ in range(8)]; dU = [z("cell") for _ in range(5)]; E = [z("ex"), z("ey"), z("ez")]
        par = ak.make_params(nmb=plan.n_own, device=rank, stream=torch.cuda.current_stream(dev).cuda_stream, **dom["p"])
        ctx = ak.ak_create(par, dom["dx"][lo:hi])
        ak.ak_set_metric(ctx, adm)
        ops = halo.AkOps(ctx, plan, (0, 0, 0), W, dU, E)
        halo.advance(plan, ops, 3, 2, dom["dt"], U, Bf, whole_blocks=whole_blocks)
        torch.cuda.synchronize(dev)
        out.put(dict(lo=lo, hi=hi, U=[u[:plan.n_own].cpu().numpy() for u in U],
                     Bf=[b[:plan.n_own].cpu().numpy() for b in Bf]))
        dist.barrier()
    finally:
        if ctx is not None:
            ak.ak_destroy(ctx)
        dist.destroy_process_group()


@pytest.mark.parametrize("whole_blocks", [False, True])
def test_halo_advance_over_nccl_equals_oracle(whole_blocks):
    """The eight-block periodic domain evolved for two RK3 steps on two GPUs (ghost slabs packed by
    ak_halo_pack, one NCCL send/recv pair per peer, ak_halo_unpack, then the single-GPU ghost fill reading
    the mirrors; the stage loop inside ak_advance_hooked) equals the oracle's single-process run bit for
    bit.  No scaling number is taken: a correctness gate for boxes that have the GPUs."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs >= 2 GPUs (NCCL leg of the halo exchange)")
    from oracle import pyoracle as orc
    from test_multirank_cpu import _eight_block_domain
    from test_oracle_exchange import lattice_nbr
    world = 2
    ctxm = mp.get_context("spawn")
    q = ctxm.Queue()
    port = _free_port()
    procs = [ctxm.Process(target=_nccl_worker, args=(r, world, port, q, whole_blocks)) for r in range(world)]
    for p in procs:
        p.start()
    parts = [q.get(timeout=600) for _ in range(world)]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    dom = _eight_block_domain()
    nbr = lattice_nbr((2, 2, 2), (True, True, True))
    U = [u.copy() for u in dom["U"]]; Bf = [b.copy() for b in dom["Bf"]]
    orc.advance_nbr(orc.make_params(nmb=8, **dom["p"]), dom["dx"], 3, 2, dom["dt"], (0, 0, 0), nbr, U, Bf,
                    dom["adm"], nthreads=8)
    for part in parts:
        lo, hi = part["lo"], part["hi"]
        for g, o in zip(part["U"] + part["Bf"], U + Bf):
            assert np.array_equal(g, o[lo:hi])
