"""ak_con2prim_static — the allocation-free entry point (include/ak.h) — against the existing path.

Collected last on purpose (`test_zz_*`): the suite runs with `pytest -x`, so a failure here cannot hide
another test.  The entry point takes no context; its scratch (device counters, status bytes when the caller
passes none) is a file-scope device array inside libak.so that every call shares and that keeps the last
call's contents — hence two calls in a row on different inputs, the second of which must not see the first's
counters.  Bar: the tolerance of the other GPU parity tests (tests/gpukit.py: relative 1e-11, absolute floor
1e-14 max|field|; status bytes bit-exact) — the two paths run the same kernel, so they agree bit for bit.
"""
import copy

import numpy as np
import pytest

from paper_2409_10384_b200 import workloads as wl

import gpukit

pytestmark = pytest.mark.gpu


def _existing_path(w, over):
    """ak_create + ak_con2prim (context scratch from cudaMalloc) -> W, U after floors, status, counters."""
    with gpukit.GpuStage(copy.deepcopy(w), **over) as g:
        g.con2prim()
        r = g.result()
        st = g.stats()
    return r, st


def _static_path(w, over, pass_status):
    import torch
    from paper_2409_10384_b200 import ak
    p = dict(w["params"]); p.update(over)
    dev = "cuda:0"
    U = gpukit.to_dev(w["U"], dev); Bf = gpukit.to_dev(w["Bf"], dev); adm = gpukit.to_dev(w["adm"], dev)
    sh = ak.shapes(p["nmb"], p["n"])
    W = [torch.zeros(sh["cell"], dtype=torch.float64, device=dev) for _ in range(8)]
    status = torch.full(sh["cell"], 0xAB, dtype=torch.uint8, device=dev) if pass_status else None
    par = ak.make_params(device=0, stream=torch.cuda.current_stream(dev).cuda_stream, **p)
    torch.cuda.synchronize()
    counts = ak.ak_con2prim_static(par, U, Bf, adm, W, status, want_counts=True)
    torch.cuda.synchronize()
    c = lambda ts: [t.cpu().numpy() for t in ts]
    return dict(W=c(W), U=c(U), status=None if status is None else status.cpu().numpy()), counts


def _compare(new, ref, counts, stats, label):
    for k, n in (("W", 8), ("U", 5)):
        for v in range(n):
            a, b = new[k][v], ref[k][v]
            atol = gpukit.ATOL_FAC * max(float(np.max(np.abs(b))), 1e-300)
            r, d = gpukit.max_rel_dev(a, b, atol)
            assert r <= 1.0, "%s: %s[%d] off by %.3g x tolerance (max abs %.3g)" % (label, k, v, r, d)
            assert np.array_equal(a, b), "%s: %s[%d] not bit-identical" % (label, k, v)   # same kernel: same bits
    if new["status"] is not None:
        assert np.array_equal(new["status"], ref["status"]), label
    for key in ("n_c2p_fail", "n_cons_floor", "n_prim_floor"):
        assert counts[key] == stats[key], (label, key, counts[key], stats[key])


def test_static_con2prim_two_calls_in_a_row_match_the_existing_path():
    # call 1: a noisy block with the atmosphere raised above its low-density cells: D, rho, T and tau floors
    # fire (non-zero counters, rewritten U); call 2: the smooth C0 block — no floor at all, so any counter
    # left over from call 1 in the shared scratch would show.
    w1 = wl.make_test_noise_block(seed=21, n=8, frac=0.05)
    over1 = dict(rho_atm=3e-6, T_atm=0.6, f_thr=1.0)
    w2 = wl.make_blocks("C0")
    ref1, st1 = _existing_path(w1, over1)
    ref2, st2 = _existing_path(w2, {})
    assert st1["n_cons_floor"] > 0 and st1["n_prim_floor"] > 0 and np.any(ref1["status"] != 0)
    assert st2["n_cons_floor"] == 0 and st2["n_prim_floor"] == 0 and st2["n_c2p_fail"] == 0
    new1, c1 = _static_path(w1, over1, pass_status=True)
    new2, c2 = _static_path(w2, {}, pass_status=True)           # straight after: same scratch array
    _compare(new1, ref1, c1, st1, "static call 1")
    _compare(new2, ref2, c2, st2, "static call 2")
    # status = NULL: the mask goes to the scratch, outputs and counters unchanged
    new3, c3 = _static_path(w1, over1, pass_status=False)
    _compare(new3, ref1, c3, st1, "static call 3 (no status)")


def test_static_con2prim_rejects_batches_beyond_the_scratch_and_bad_arguments():
    import ctypes as C
    import torch
    from paper_2409_10384_b200 import ak
    L = ak.lib()
    w = wl.make_blocks("C0")
    dev = "cuda:0"
    U = gpukit.to_dev(w["U"], dev); Bf = gpukit.to_dev(w["Bf"], dev); adm = gpukit.to_dev(w["adm"], dev)
    W = [torch.zeros_like(U[0]) for _ in range(8)]
    u, b, a, wp = ak._struct(ak.AkCons, U), ak._struct(ak.AkFaceB, Bf), ak._struct(ak.AkAdm, adm), ak._struct(ak.AkPrim, W)
    call = lambda par: L.ak_con2prim_static(C.byref(par), C.byref(u), C.byref(b), C.byref(a), C.byref(wp), None, None)
    p = dict(w["params"])
    nt = p["n"] + 8
    too_many = ak.STATIC_MAX_CELLS // nt ** 3 + 1            # refused before anything is launched or read
    big = ak.make_params(device=0, stream=0, **dict(p, nmb=too_many))
    assert call(big) == ak.AK_ETOOBIG
    assert "AK_STATIC_MAX_CELLS" in ak.strerror(ak.AK_ETOOBIG)
    assert call(ak.make_params(device=0, stream=0, **dict(p, gamma_ad=1.0))) == ak.AK_EINVAL
    assert call(ak.make_params(device=64, stream=0, **p)) == ak.AK_EINVAL
    assert L.ak_con2prim_static(None, C.byref(u), C.byref(b), C.byref(a), C.byref(wp), None, None) == ak.AK_EINVAL
    ok = ak.make_params(device=0, stream=torch.cuda.current_stream(dev).cuda_stream, **p)
    assert call(ok) == ak.AK_OK                               # host_counts = NULL: enqueues and returns
    torch.cuda.synchronize()
    assert bool(torch.isfinite(W[0]).all()) and float(W[0].min()) > 0.0
