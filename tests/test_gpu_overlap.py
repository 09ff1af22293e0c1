"""GPU tests of round 2's boundary work: the overlapped schedule of ak_rhs (ak_set_overlap) gives the
bits of the serial schedule and of the oracle; misaligned field pointers are AK_EINVAL, not a device
fault; two live contexts of different block size share the TMA sweep instantiations safely."""
import copy

import numpy as np
import pytest

from oracle import pyoracle as orc
from paper_2409_10384_b200 import workloads as wl

import gpukit

pytestmark = pytest.mark.gpu


def _noise_batch(nblocks, n, seed0, frac=0.03):
    """a batch of independent noise blocks (floors, flags, re-fluxed faces in every block)."""
    ws = [wl.make_test_noise_block(seed=seed0 + b, n=n, frac=frac) for b in range(nblocks)]
    w = copy.deepcopy(ws[0])
    for k in ("U", "Bf", "adm"):
        w[k] = [np.concatenate([x[k][q] for x in ws], axis=0) for q in range(len(ws[0][k]))]
    w["dx"] = np.concatenate([x["dx"] for x in ws], axis=0)
    w["params"] = dict(w["params"]); w["params"]["nmb"] = nblocks
    w["dt_fofc"] = 2.0 * ws[0]["dt_fofc"]
    return w


@pytest.mark.parametrize("nchunks", [2, 3, 64])
@pytest.mark.parametrize("eos", [None, dict(K0=0.15, gammas=[1.8, 2.4, 2.1], rho_breaks=[0.3, 1.0], gamma_th=1.6)])
def test_overlapped_schedule_equals_serial_and_oracle(nchunks, eos):
    """7 blocks in 2 / 3 (uneven) / 7 (clamped from 64) chunks; WENO-Z, HLLE, FOFC + DMP."""
    import torch
    from paper_2409_10384_b200 import ak
    w = _noise_batch(7, 8, seed0=40)
    over = dict(recon=2, dmp_M=1.1)
    if eos is not None:
        over["eos_hybrid"] = eos
    U_in = [u.copy() for u in w["U"]]
    with gpukit.GpuStage(copy.deepcopy(w), **over) as a, gpukit.GpuStage(copy.deepcopy(w), **over) as b:
        a.rhs()
        ak.ak_set_overlap(b.ctx, nchunks)
        b.rhs()
        ra, rb = a.result(), b.result()
        for k in ("dU", "E", "W", "U"):
            for x, y in zip(ra[k], rb[k]):
                assert np.array_equal(x, y), k
        assert np.array_equal(ra["flag"], rb["flag"]) and np.array_equal(ra["status"], rb["status"])
        assert a.stats() == b.stats()
        fa, fb = a.flux(), b.flux()
        for x, y in zip(fa, fb):
            assert np.array_equal(x, y)
        # CT alone from the fluxes the overlapped stage left behind
        E2 = [torch.zeros_like(e) for e in b.E]
        ak.ak_emf(b.ctx, b.W, *E2)
        torch.cuda.synchronize()
        for x, y in zip(E2, b.E):
            assert torch.equal(x, y)
        # w_is_valid = 1 under overlap
        b.rhs(w_is_valid=True)
        rc = b.result()
        for k in ("dU", "E"):
            for x, y in zip(ra[k], rc[k]):
                assert np.array_equal(x, y), k
        sb = b.stats()
        assert sb["n_c2p_fail"] == 0 and sb["n_cons_floor"] == 0      # part (1) skipped: no con2prim counts
        assert sb["n_fofc_cells"] == a.stats()["n_fofc_cells"]
        # back to the serial schedule
        ak.ak_set_overlap(b.ctx, 0)
        b.rhs(w_is_valid=True)
        rd = b.result()
        for x, y in zip(ra["dU"] + ra["E"], rd["dU"] + rd["E"]):
            assert np.array_equal(x, y)
    p = dict(w["params"]); p.update(over)
    o = orc.rhs(orc.make_params(**p), w["dx"], w["U"], w["Bf"], w["adm"], w["dt_fofc"], nthreads=8)
    o["U"] = w["U"]
    gpukit.assert_parity(rb, o, U_in, label="overlap %d" % nchunks)
    assert np.count_nonzero(o["flag"]) > 0


def test_overlapped_advance_equals_serial():
    """ak_advance (RK3, stage-blended FOFC estimate) under the overlapped schedule: same bits."""
    import torch
    from paper_2409_10384_b200 import ak
    w = _noise_batch(4, 8, seed0=70, frac=0.01)
    res = []
    for nchunks in (0, 3):
        with gpukit.GpuStage(copy.deepcopy(w), recon=2, dmp_M=1.1) as g:
            ak.ak_set_overlap(g.ctx, nchunks)
            fl = torch.zeros_like(g.flag)
            ak.ak_advance(g.ctx, 3, 2, 0.02 / 8, (0, 1, 0), g.U, g.Bf, g.W, fl)
            torch.cuda.synchronize()
            res.append([t.cpu().numpy() for t in g.U + g.Bf + g.W] + [fl.cpu().numpy()])
    for x, y in zip(*res):
        assert np.array_equal(x, y)
    assert np.count_nonzero(res[0][-1]) > 0


def test_set_overlap_validation():
    from paper_2409_10384_b200 import ak
    w = wl.make_blocks("C0")
    with gpukit.GpuStage(copy.deepcopy(w)) as g:
        for bad in (-1, 65):
            assert ak.lib().ak_set_overlap(g.ctx, bad) == ak.AK_EINVAL
        assert ak.lib().ak_set_overlap(None, 2) == ak.AK_EINVAL
        ak.ak_set_overlap(g.ctx, 8)           # one block: clamps to the serial schedule
        g.rhs()
        ra = g.result()
    with gpukit.GpuStage(copy.deepcopy(w)) as h:
        h.rhs()
        rb = h.result()
    for x, y in zip(ra["dU"] + ra["E"], rb["dU"] + rb["E"]):
        assert np.array_equal(x, y)


def test_misaligned_field_pointer_is_einval():
    """base pointers 16-byte aligned, checked -> AK_EINVAL.  A view that starts one double
    into an allocation is 8-byte aligned only; the TMA bulk copies would fault on it."""
    import ctypes as C
    import torch
    from paper_2409_10384_b200 import ak
    w = wl.make_blocks("C0")
    with gpukit.GpuStage(copy.deepcopy(w)) as g:
        def off(t):                       # same shape, base address + 8 bytes
            big = torch.zeros(t.numel() + 2, dtype=t.dtype, device=t.device)
            v = big[1:1 + t.numel()].view(t.shape)
            assert v.data_ptr() % 16 == 8
            return v
        L = ak.lib()
        u, b, wp = ak._struct(ak.AkCons, g.U), ak._struct(ak.AkFaceB, g.Bf), ak._struct(ak.AkPrim, g.W)
        o = ak._struct(ak.AkRhsOut, g.dU + g.E + [g.flag, g.status, None])
        assert L.ak_rhs(g.ctx, C.byref(u), C.byref(b), C.byref(wp), 0, 0.01, C.byref(o)) == ak.AK_OK
        for which in ("U", "Bf", "W"):
            args = dict(U=list(g.U), Bf=list(g.Bf), W=list(g.W))
            args[which][1] = off(args[which][1])
            u, b, wp = ak._struct(ak.AkCons, args["U"]), ak._struct(ak.AkFaceB, args["Bf"]), ak._struct(ak.AkPrim, args["W"])
            assert L.ak_rhs(g.ctx, C.byref(u), C.byref(b), C.byref(wp), 0, 0.01, C.byref(o)) == ak.AK_EINVAL, which
            assert L.ak_con2prim(g.ctx, C.byref(u), C.byref(b), C.byref(wp), None) == ak.AK_EINVAL, which
        adm = list(g.adm); adm[7] = off(adm[7])
        s = ak._struct(ak.AkAdm, adm)
        assert L.ak_set_metric(g.ctx, C.byref(s)) == ak.AK_EINVAL
        torch.cuda.synchronize()          # nothing faulted
        g.rhs()                           # the context still works with its (aligned) arrays


def test_two_contexts_of_different_block_size_interleaved():
    """cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel function, not the context: a
    32^3 context (larger x-sweep tile), then a 16^3 context, then the 32^3 one again — same WENO-Z
    instantiations, different shared-memory needs.  (the attribute must never be lowered.)"""
    w32 = wl.make_blocks("C2", blocks=[21])
    w16 = wl.make_test_noise_block(seed=5, n=16, frac=0.01)
    with gpukit.GpuStage(copy.deepcopy(w16), recon=2) as small0:
        small0.rhs()
        r16_first = small0.result()
    with gpukit.GpuStage(copy.deepcopy(w32)) as big, gpukit.GpuStage(copy.deepcopy(w16), recon=2) as small:
        big.rhs()
        r1 = big.result()
        small.rhs()
        r16 = small.result()
        big.rhs(w_is_valid=True)
        r2 = big.result()
        small.rhs(w_is_valid=True)
    for x, y in zip(r1["dU"] + r1["E"], r2["dU"] + r2["E"]):
        assert np.array_equal(x, y)
    for x, y in zip(r16["dU"] + r16["E"], r16_first["dU"] + r16_first["E"]):
        assert np.array_equal(x, y)


def test_host_entry_without_primitives():
    """ak_rhs_host with W = NULL returns dU/dt, E, masks and floored U as before and skips the copy of the
    primitives (small batch: plain path; 32 blocks: the two-lane pipeline)."""
    import torch
    from paper_2409_10384_b200 import ak
    for w in (wl.make_test_noise_block(seed=13, n=8, frac=0.02), wl.make_blocks("C3", blocks=list(range(192, 224)))):
        with gpukit.GpuStage(copy.deepcopy(w)) as a:
            a.rhs()
            ra = a.result()
            sh = a.sh
            hU = [u.copy() for u in w["U"]]
            hdU = [np.zeros(sh["cell"]) for _ in range(5)]
            hE = [np.zeros(sh[k]) for k in ("ex", "ey", "ez")]
            hflag = np.zeros(sh["cell"], dtype=np.uint8); hst = np.zeros(sh["cell"], dtype=np.uint8)
            ak.ak_rhs_host(a.ctx, hU, w["Bf"], None, w["dt_fofc"], hdU, hE, hflag, hst)
            for x, y in zip(hdU + hE + hU, ra["dU"] + ra["E"] + ra["U"]):
                assert np.array_equal(x, y)
            assert np.array_equal(hflag, ra["flag"]) and np.array_equal(hst, ra["status"])
            # a partly filled W is a usage error
            import ctypes as C
            u, b = ak._struct(ak.AkCons, hU), ak._struct(ak.AkFaceB, w["Bf"])
            wp = ak.AkPrim(); wp.rho = hdU[0].ctypes.data
            o = ak._struct(ak.AkRhsOut, hdU + hE + [hflag, hst, None])
            assert ak.lib().ak_rhs_host(a.ctx, C.byref(u), C.byref(b), C.byref(wp), 0.01, C.byref(o)) == ak.AK_EINVAL


@pytest.mark.parametrize("name,blocks,over", [
    ("C2", [0, 21, 22, 41, 42, 63], dict()),                     # atmosphere blocks (u = 0, B = 0 exactly), star rims
    ("C1", [0, 7], dict(recon=2)),                               # static star: every velocity exactly zero
    ("C1", [0, 7], dict(recon=4, riemann=0)),
    ("C3", [192 + 21, 64 + 21, 21], dict(recon=3)),              # nothing is zero: the shortcuts never fire
    ("C2", [0, 63, 21], dict(recon=0, riemann=0)),               # donor cell + LLF through the static face flux
    ("C4", [0, 1, 300, 301], dict()),                            # rotational shift, atmosphere blocks of two sizes
])
def test_exact_shortcuts_leave_every_bit_unchanged(name, blocks, over):
    """ak_set_exact_shortcuts: skipping the reconstruction of fields that are +0.0 on a whole tile and
    running the root find of static unmagnetised cells on f(mu) = mu - const, and the static face flux on
    tiles with u = 0 and B = 0, are exact: mask 0 (full arithmetic), 1, 2, 4 and 7 give the same bits in
    every output, fluxes and the signs of their zeros included, and equal the oracle."""
    from paper_2409_10384_b200 import ak
    w = wl.make_blocks(name, blocks=blocks)
    U_in = [u.copy() for u in w["U"]]
    res = []
    for mask in (0, 1, 2, 4, 7):
        with gpukit.GpuStage(copy.deepcopy(w), **over) as g:
            ak.ak_set_exact_shortcuts(g.ctx, mask)
            g.rhs()
            res.append((g.result(), g.flux(), g.stats()))
    r0, f0, s0 = res[0]
    for r, fl, st in res[1:]:
        for k in ("dU", "E", "W", "U"):
            for x, y in zip(r0[k], r[k]):
                assert np.array_equal(x, y), k
        assert np.array_equal(r0["flag"], r["flag"]) and np.array_equal(r0["status"], r["status"])
        for x, y in zip(f0, fl):
            assert np.array_equal(x, y)
            assert np.array_equal(np.signbit(x), np.signbit(y))      # signed zeros of a static face included
        assert st == s0
    p = dict(w["params"]); p.update(over)
    o = orc.rhs(orc.make_params(**p), w["dx"], w["U"], w["Bf"], w["adm"], w["dt_fofc"], nthreads=8)
    o["U"] = w["U"]
    gpukit.assert_parity(res[-1][0], o, U_in, label=name + " shortcuts")


def test_exact_shortcuts_with_signed_zeros_and_partly_zero_fields():
    """Hand-made primitives through ak_rhs(w_is_valid = 1): u^x = -0.0 in some cells (not +0.0: must be
    reconstructed), u^z zero except one cell, B~cc zero on half the block, u^y = +0.0 everywhere.  Mask 0
    and 3 must agree bit for bit, signs of zeros in the fluxes included."""
    import torch
    from paper_2409_10384_b200 import ak
    w = wl.make_test_noise_block(seed=3, n=8, frac=0.0)
    outs = []
    for mask in (0, 7):
        with gpukit.GpuStage(copy.deepcopy(w), recon=2, dmp_M=1.1) as g:
            ak.ak_set_exact_shortcuts(g.ctx, mask)
            g.con2prim()
            nt = 16
            g.W[1].zero_(); g.W[1][0, 5:9, 3:7, 2:12] = -0.0
            g.W[2].zero_()
            g.W[3].zero_(); g.W[3][0, 8, 8, 8] = 0.01
            g.W[5][0, :, :, : nt // 2] = 0.0; g.W[6][0, : nt // 2] = 0.0; g.W[7].zero_()
            g.rhs(w_is_valid=True)
            outs.append((g.result(), g.flux()))
    (ra, fa), (rb, fb) = outs
    for x, y in zip(ra["dU"] + ra["E"] + fa, rb["dU"] + rb["E"] + fb):
        assert np.array_equal(x, y)
        assert np.array_equal(np.signbit(x), np.signbit(y))
    assert np.array_equal(ra["flag"], rb["flag"])


@pytest.mark.parametrize("over", [dict(recon=2, dmp_M=1.1), dict(recon=1, riemann=0),
                                  dict(recon=2, eos_hybrid=dict(K0=40.0, gammas=[2.0, 2.2], rho_breaks=[6.4e-4], gamma_th=2.0))])
def test_unmagnetised_moving_tiles_take_the_no_B_side_state_exactly(over):
    """side_state<.., NOB> (mask bit 2): tiles whose B components are all +0.0 while the matter moves.  Velocities
    of both signs (so that (Bv) = 0 v_x + 0 v_y + 0 v_z comes out as +0 and as -0), a slab of u = -0.0, a slab at
    rest, and one corner of the block magnetised so that the general side_state runs beside it.  Masks 0, 4 and 7
    must agree bit for bit, signs of zeros in the fluxes included."""
    from paper_2409_10384_b200 import ak
    w = wl.make_test_noise_block(seed=17, n=8, frac=0.0)
    outs = []
    for mask in (0, 4, 7):
        with gpukit.GpuStage(copy.deepcopy(w), **over) as g:
            ak.ak_set_exact_shortcuts(g.ctx, mask)
            g.con2prim()
            import torch
            sh = tuple(g.W[1].shape)
            for v in (1, 2, 3):
                u = 0.3 * (np.random.default_rng(40 + v).random(sh) - 0.5)
                u[0, :, :4, :] = -np.abs(u[0, :, :4, :])        # every component negative: (Bv) = -0
                u[0, :, 4:6, :] = -0.0
                u[0, :, 6:8, :] = 0.0
                g.W[v].copy_(torch.from_numpy(u))
            for v in (5, 6, 7): g.W[v].zero_()
            for b in g.Bf: b.zero_()
            g.W[5][0, 12:, 12:, 12:] = 1e-3                      # a magnetised corner: B~cc^x only
            g.rhs(w_is_valid=True)
            outs.append((g.result(), g.flux()))
    ra, fa = outs[0]
    assert any(np.any(np.signbit(x) & (x == 0.0)) for x in fa), "no negative zero in any flux: the case does not bite"
    for rb, fb in outs[1:]:
        for x, y in zip(ra["dU"] + ra["E"] + fa, rb["dU"] + rb["E"] + fb):
            assert np.array_equal(x, y)
            assert np.array_equal(np.signbit(x), np.signbit(y))
        assert np.array_equal(ra["flag"], rb["flag"])


def test_fused_fofc_test_and_sources_path_is_exact(monkeypatch):
    """AK_FUSE_SRC=1 (opt-in; slower on C4, DESIGN.md §6 item 21): part (6) inside the FOFC-test kernel from the
    high-order fluxes, then k_src_fix for the cells next to re-fluxed faces.  Must give the bits of the default
    path (k_div_src after the re-flux), matter epilogue included, on blocks with many flags."""
    import torch
    from paper_2409_10384_b200 import ak
    w = _noise_batch(5, 8, seed0=90)
    out = []
    for fuse in ("0", "1"):
        monkeypatch.setenv("AK_FUSE_SRC", fuse)             # read by ak_create
        with gpukit.GpuStage(copy.deepcopy(w), recon=2, dmp_M=1.1) as g:
            M = [torch.full_like(g.W[0], float("nan")) for _ in range(10)]
            ak.ak_rhs(g.ctx, g.U, g.Bf, g.W, 0, g.dt_fofc, g.dU, g.E, g.flag, g.status, matter=M)
            torch.cuda.synchronize()
            out.append((g.result(), [t.cpu().numpy() for t in M], g.stats()))
    (ra, ma, sa), (rb, mb, sb) = out
    assert np.count_nonzero(ra["flag"]) > 20 and sa == sb
    for x, y in zip(ra["dU"] + ra["E"] + ra["W"], rb["dU"] + rb["E"] + rb["W"]):
        assert np.array_equal(x, y)
    for x, y in zip(ma, mb):
        assert np.array_equal(x, y, equal_nan=True)
    assert np.array_equal(ra["flag"], rb["flag"])


def test_graph_replay_equals_plain_launches():
    """ak_set_graph: the stage replayed from a CUDA graph gives the bits of the plain launches, call after call,
    with the graph really in use (ak_graph_replays), through ak_rhs and through ak_advance (three blends per RK3
    step -> three cached graphs), and a changed argument (another output buffer, w_is_valid) is noticed."""
    import torch
    from paper_2409_10384_b200 import ak
    w = _noise_batch(3, 8, seed0=120)
    over = dict(recon=2, dmp_M=1.1)
    with gpukit.GpuStage(copy.deepcopy(w), **over) as a, gpukit.GpuStage(copy.deepcopy(w), **over) as b:
        ak.ak_set_graph(b.ctx, 1)
        for it in range(5):                    # plain, capture + replay, replay, replay, replay
            a.rhs(); b.rhs()
            ra, rb = a.result(), b.result()
            for k in ("dU", "E", "W", "U"):
                for x, y in zip(ra[k], rb[k]):
                    assert np.array_equal(x, y), (it, k)
            assert np.array_equal(ra["flag"], rb["flag"]) and np.array_equal(ra["status"], rb["status"])
            assert a.stats() == b.stats()
        assert ak.ak_graph_replays(b.ctx) == 4
        assert np.count_nonzero(ra["flag"]) > 0
        # another dU buffer: a new argument set, not a stale replay into the old buffer
        old = [t.clone() for t in b.dU]
        b.dU = [torch.zeros_like(t) for t in b.dU]            # (dU is written on interior cells only)
        for t in old:
            t.fill_(123.0)
        b.rhs()
        for x, y in zip(b.dU, a.dU):
            assert torch.equal(x, y)
        assert all(bool((t == 123.0).all()) for t in old)
        a.rhs(w_is_valid=True); b.rhs(w_is_valid=True); b.rhs(w_is_valid=True); b.rhs(w_is_valid=True)
        for x, y in zip(b.dU + b.E, a.dU + a.E):
            assert torch.equal(x, y)
        # timing on: graphs bypassed, still the same
        ak.ak_timing(b.ctx, 1); b.rhs(w_is_valid=True); ak.ak_timing(b.ctx, 0)
        for x, y in zip(b.dU + b.E, a.dU + a.E):
            assert torch.equal(x, y)
        ak.ak_set_graph(b.ctx, 0)
        b.rhs(w_is_valid=True)
        for x, y in zip(b.dU + b.E, a.dU + a.E):
            assert torch.equal(x, y)
    res = []
    for on in (0, 1):
        with gpukit.GpuStage(copy.deepcopy(w), **over) as g:
            ak.ak_set_graph(g.ctx, on)
            ak.ak_advance(g.ctx, 3, 4, 0.02 / 8, (0, 1, 0), g.U, g.Bf, g.W)
            torch.cuda.synchronize()
            res.append([t.cpu().numpy() for t in g.U + g.Bf + g.W])
            if on:
                assert ak.ak_graph_replays(g.ctx) >= 6          # 12 stages: 3 plain, then graphs
    for x, y in zip(*res):
        assert np.array_equal(x, y)
    assert ak.lib().ak_set_graph(None, 1) == ak.AK_EINVAL


def test_host_entry_sparse_writeback_of_floored_cells_into_pinned_memory():
    """ak_rhs_host, pipelined path (16 blocks), pinned U~ arrays: only the cells part (1) changed (status != 0)
    are stored back, straight into the pinned arrays; with pageable arrays U~ is copied whole.  Both must leave
    the host U~ equal to the device path's, floors present."""
    import torch
    from paper_2409_10384_b200 import ak
    w = _noise_batch(16, 8, seed0=200, frac=0.05)
    over = dict(rho_atm=3e-6, T_atm=0.6, f_thr=1.0)           # atmosphere above the low-density cells: floors fire
    with gpukit.GpuStage(copy.deepcopy(w), **over) as a:
        a.rhs()
        ra = a.result()
        assert np.count_nonzero(ra["status"]) > 50
        assert any(not np.array_equal(u, r) for u, r in zip(w["U"], ra["U"]))
        sh = a.sh
        for pinned in (True, False):
            mk = (lambda arr: torch.from_numpy(np.ascontiguousarray(arr)).pin_memory()) if pinned else \
                 (lambda arr: torch.from_numpy(np.ascontiguousarray(arr).copy()))
            hU = [mk(u) for u in w["U"]]; hB = [mk(b) for b in w["Bf"]]
            hdU = [mk(np.zeros(sh["cell"])) for _ in range(5)]
            hE = [mk(np.zeros(sh[k])) for k in ("ex", "ey", "ez")]
            hflag = mk(np.zeros(sh["cell"], dtype=np.uint8)); hst = mk(np.zeros(sh["cell"], dtype=np.uint8))
            ak.ak_rhs_host(a.ctx, hU, hB, None, w["dt_fofc"], hdU, hE, hflag, hst)
            for x, y in zip(hdU + hE + hU, ra["dU"] + ra["E"] + ra["U"]):
                assert np.array_equal(x.numpy(), y), pinned
            assert np.array_equal(hflag.numpy(), ra["flag"]) and np.array_equal(hst.numpy(), ra["status"])


@pytest.mark.parametrize("name,blocks,over", [
    ("C2", [0, 21, 22, 41, 42, 63], dict()),                 # static atmosphere blocks and blocks with moving stars
    ("C1", [0, 7], dict(recon=4, riemann=0)),                # every block static (v = 0), but magnetised near the star
    ("C4", [0, 1, 300, 301], dict(recon=0)),                 # donor cell through the light kernel
    ("C2", [0, 21, 63], dict(eos_hybrid=dict(K0=40.0, gammas=[2.0, 2.2], rho_breaks=[6.4e-4], gamma_th=2.0))),
])
def test_static_block_sweep_kernel_is_exact(monkeypatch, name, blocks, over):
    """AK_SPLIT_BLOCKS=1 (automatic only for batches of >= 2^23 stored cells, e.g. C4, where the full-batch parity
    test covers it): tiles none of whose staged rows con2prim found to hold a u^i or a face B~ other than +0.0 take
    k_flux_static, the others the general tile kernels, through the device-side tile lists of k_split_tiles.  Same
    bits as without the split and as the oracle, fluxes and the signs of their zeros included."""
    from paper_2409_10384_b200 import ak
    w = wl.make_blocks(name, blocks=blocks)
    U_in = [u.copy() for u in w["U"]]
    res = []
    for split in ("0", "1"):
        monkeypatch.setenv("AK_SPLIT_BLOCKS", split)         # read by ak_create
        with gpukit.GpuStage(copy.deepcopy(w), **over) as g:
            g.rhs()
            res.append((g.result(), g.flux(), g.stats()))
            g.rhs()                                          # a second call re-sorts the blocks: same result
            again = g.result()
            for x, y in zip(res[-1][0]["dU"] + res[-1][0]["E"], again["dU"] + again["E"]):
                assert np.array_equal(x, y)
    (r0, f0, s0), (r1, f1, s1) = res
    for k in ("dU", "E", "W", "U"):
        for x, y in zip(r0[k], r1[k]):
            assert np.array_equal(x, y), k
    assert np.array_equal(r0["flag"], r1["flag"]) and np.array_equal(r0["status"], r1["status"]) and s0 == s1
    for x, y in zip(f0, f1):
        assert np.array_equal(x, y) and np.array_equal(np.signbit(x), np.signbit(y))
    if "eos_hybrid" in over:
        return      # rho^Gamma is pow() on the device and libm's in the oracle (rounding-level differences: hybrid
                    # parity against the oracle is tests/test_gpu_eos.py's subject); split on = split off is the point here
    p = dict(w["params"]); p.update(over)
    o = orc.rhs(orc.make_params(**p), w["dx"], w["U"], w["Bf"], w["adm"], w["dt_fofc"], nthreads=8)
    o["U"] = w["U"]
    gpukit.assert_parity(r1, o, U_in, label=name + " split")


def test_tile_lists_cover_every_row_a_tile_stages(monkeypatch):
    """k_split_tiles: a tile is static only if EVERY row of cells it stages is — the 5 halo rows of a y or z tile
    included.  A static atmosphere block with single moving cells and single magnetised faces placed next to
    tile boundaries (tiles of 7 face rows starting at index 3: 3, 10, 17, 24, 31, 38) and at random: a tile list
    that forgot a halo row would hand a tile with non-zero data to the light kernel, which reads rho and P only.
    Split on must give the bits of split off with the shortcuts off, signs of zero fluxes included."""
    from paper_2409_10384_b200 import ak
    w = wl.make_blocks("C2", blocks=[0, 63])
    nt = 40
    U = [u.reshape(2, nt, nt, nt) for u in w["U"]]
    for q in (1, 2, 3): U[q][...] = 0.0                      # two blocks at rest, without field
    for b in w["Bf"]: b[...] = 0.0
    rng = np.random.default_rng(11)
    cells = [(0, 19, 9, 20), (0, 16, 30, 5), (0, 3, 3, 3), (0, 36, 36, 36), (0, 12, 24, 38), (1, 22, 2, 1), (1, 38, 17, 20)]
    # the outermost halo rows of a tile [d0, d0+7): d0-3 (7, 14, 21, 28) and d0+8 (11, 18, 25, 32), in j (y) and k (z)
    cells += [(0, 20, 7, 20), (0, 21, 20, 10), (1, 5, 14, 30), (1, 28, 33, 7), (0, 25, 11, 11), (1, 18, 9, 9), (1, 6, 32, 2)]
    cells += [(int(rng.integers(2)),) + tuple(int(x) for x in rng.integers(0, nt, 3)) for _ in range(6)]
    for q, (m, k, j, i) in enumerate(cells):
        U[1 + q % 3][m, k, j, i] = (1e-3 if q % 2 else -1e-3) * U[0][m, k, j, i]      # S~_a = +-1e-3 D~
    bx = w["Bf"][0].reshape(2, nt, nt, -1); by = w["Bf"][1].reshape(2, nt, nt + 1, nt); bz = w["Bf"][2].reshape(2, nt + 1, nt, nt)
    bx[1, 10, 10, 21] = 1e-6; by[0, 30, 17, 8] = -1e-6; bz[1, 24, 5, 33] = 1e-6; bz[0, 2, 38, 0] = -0.0
    res = []
    for split, mask in (("0", 0), ("1", 7)):
        monkeypatch.setenv("AK_SPLIT_BLOCKS", split)
        with gpukit.GpuStage(copy.deepcopy(w)) as g:
            ak.ak_set_exact_shortcuts(g.ctx, mask)
            g.rhs()
            res.append((g.result(), g.flux(), g.stats()))
    (r0, f0, s0), (r1, f1, s1) = res
    assert any(np.any(x[0, 19, 9, 20] != 0.0) for x in r0["W"][1:4])        # the poked cell does move
    for k in ("dU", "E", "W", "U"):
        for x, y in zip(r0[k], r1[k]):
            assert np.array_equal(x, y), k
    assert np.array_equal(r0["flag"], r1["flag"]) and np.array_equal(r0["status"], r1["status"]) and s0 == s1
    for x, y in zip(f0, f1):
        assert np.array_equal(x, y) and np.array_equal(np.signbit(x), np.signbit(y))


def test_create_with_rows_longer_than_a_sweep_block():
    """n + 4 > 256 threads: the tile kernels (and with them the tile lists) do not apply; ak_create must size its
    list scratch without dividing by a tile height of zero, and the context must come up and go away cleanly."""
    from paper_2409_10384_b200 import ak
    w = wl.make_blocks("C0")
    p = dict(w["params"]); p.update(nmb=1, n=254)
    par = ak.make_params(device=0, stream=0, **p)
    ctx = ak.ak_create(par, np.ones((1, 3)) * 0.01)
    ak.ak_destroy(ctx)
