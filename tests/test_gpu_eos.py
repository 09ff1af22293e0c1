"""GPU parity for the piecewise-polytropic hybrid EOS (include/ak.h ak_set_eos_hybrid; DESIGN.md
reading R29): the CUDA stage against the oracle on the same seeded inputs.  The conserved inputs are
the generators' own (built with their ideal-gas formula): for this test they are simply states, hot
enough that the thermal part of the hybrid EOS is well above round-off.  rho^Gamma is pow() on both
sides (device / libm), equal to rounding and not bit for bit, so values are held to the tolerance of
BASELINE.json and the masks are required to agree on these seeds."""
import copy

import numpy as np
import pytest

from oracle import pyoracle as orc
from paper_2409_10384_b200 import ak, workloads as wl

import gpukit
from test_gpu_parity import run_both

pytestmark = pytest.mark.gpu

# C0 has rho = 1 +- 0.1, P ~ 0.5: two segments meeting at rho = 1 are both populated
HYB_C0 = dict(K0=0.2, gammas=[2.0, 2.5], rho_breaks=[1.0], gamma_th=1.8)
HYB_3 = dict(K0=0.15, gammas=[1.8, 2.4, 2.1], rho_breaks=[0.3, 1.0], gamma_th=1.6)


@pytest.mark.parametrize("recon,riemann", [(1, 1), (2, 1), (2, 0), (4, 1)])
def test_c0_hybrid(recon, riemann):
    w = wl.make_blocks("C0")
    g, o, rep = run_both(w, want_flux=True, recon=recon, riemann=riemann, eos_hybrid=HYB_C0)
    # both segments are populated
    assert (o["W"][0] < 1.0).any() and (o["W"][0] > 1.0).any()
    # and the EOS matters: the ideal-gas stage gives other primitives
    ideal = orc.rhs(orc.make_params(**dict(w["params"], recon=recon, riemann=riemann)), w["dx"],
                    [u.copy() for u in w["U"]], w["Bf"], w["adm"], w["dt_fofc"], nthreads=4)
    assert np.max(np.abs(ideal["W"][4] - o["W"][4])) > 1e-3


@pytest.mark.parametrize("seed,dmp", [(7, 1.1), (11, 0.0)])
def test_noise_block_hybrid_flags(seed, dmp):
    w = wl.make_test_noise_block(seed=seed, n=8, frac=0.02)
    if not dmp:
        w["dt_fofc"] *= 2.0
    g, o, rep = run_both(w, want_flux=True, dmp_M=dmp, recon=2 if dmp else 1, eos_hybrid=HYB_3)
    assert np.count_nonzero(o["flag"]) > 0


def test_noise_block_hybrid_floors():
    """atmosphere raised above the low-density cells: D, rho, T and tau floors of the hybrid EOS"""
    w = wl.make_test_noise_block(seed=21, n=8, frac=0.05)
    w["dt_fofc"] *= 2.0
    g, o, rep = run_both(w, want_flux=True, recon=2, rho_atm=3e-6, T_atm=0.45, f_thr=1.0, eos_hybrid=HYB_3)
    bits = int(np.bitwise_or.reduce(o["status"].ravel()))
    assert bits & 1 and bits & 16


def test_curved_blocks_hybrid():
    """two blocks of the Kerr-Schild config (curved metric with shift, magnetised): hybrid stage"""
    w = wl.make_blocks("C3", blocks=[70, 200])
    run_both(w, want_flux=True, eos_hybrid=dict(K0=0.004, gammas=[1.5, 2.0], rho_breaks=[0.3], gamma_th=13.0 / 9))


def test_set_eos_hybrid_validation_and_reset():
    import torch
    w = wl.make_blocks("C0")
    with gpukit.GpuStage(copy.deepcopy(w)) as g:
        for bad in (dict(K0=-1.0, gammas=[2.0]), dict(K0=1.0, gammas=[1.0]), dict(K0=1.0, gammas=[2.0], gamma_th=1.0),
                    dict(K0=1.0, gammas=[2.0, 2.0], rho_breaks=[-1.0]),
                    dict(K0=1.0, gammas=[2.0, 2.0, 2.0], rho_breaks=[1.0, 0.5]),
                    dict(K0=1.0, gammas=[2.0] * 5, rho_breaks=[1.0, 2.0, 3.0, 4.0])):
            with pytest.raises(ak.AkError):
                ak.ak_set_eos_hybrid(g.ctx, bad["K0"], bad["gammas"], bad.get("rho_breaks", ()), bad.get("gamma_th", 2.0))
        # a rejected call changes nothing, and nseg = 0 returns to the ideal gas: both give the ideal stage
        g.rhs()
        a = g.result()
        ak.ak_set_eos_hybrid(g.ctx, HYB_C0["K0"], HYB_C0["gammas"], HYB_C0["rho_breaks"], HYB_C0["gamma_th"])
        ak.ak_set_eos_hybrid(g.ctx, 0.0, (), (), 2.0)
        for t, u in zip(g.U, w["U"]):
            t.copy_(torch.from_numpy(u))
        g.rhs()
        b = g.result()
    for k in ("W", "dU", "E"):
        for x, y in zip(a[k], b[k]):
            assert np.array_equal(x, y)


def test_matter_sources_and_host_entry_hybrid():
    import torch
    w = wl.make_test_noise_block(seed=5, n=8, frac=0.02)
    p = dict(w["params"], recon=2, eos_hybrid=HYB_3)
    wo = copy.deepcopy(w)
    ores = orc.rhs(orc.make_params(**p), wo["dx"], wo["U"], wo["Bf"], wo["adm"], wo["dt_fofc"], nthreads=4)
    om = orc.matter_sources(orc.make_params(**p), ores["W"], wo["adm"][:6])
    with gpukit.GpuStage(copy.deepcopy(w), recon=2, eos_hybrid=HYB_3) as g:
        # the host entry (two child contexts) must carry the EOS
        sh = g.sh
        hU = [torch.from_numpy(u.copy()).pin_memory() for u in w["U"]]
        hB = [torch.from_numpy(b.copy()).pin_memory() for b in w["Bf"]]
        hW = [torch.zeros(sh["cell"], dtype=torch.float64).pin_memory() for _ in range(8)]
        hdU = [torch.zeros(sh["cell"], dtype=torch.float64).pin_memory() for _ in range(5)]
        hE = [torch.zeros(sh[k], dtype=torch.float64).pin_memory() for k in ("ex", "ey", "ez")]
        hf = torch.zeros(sh["cell"], dtype=torch.uint8).pin_memory()
        hs = torch.zeros(sh["cell"], dtype=torch.uint8).pin_memory()
        ak.ak_rhs_host(g.ctx, hU, hB, hW, w["dt_fofc"], hdU, hE, hf, hs)
        gres = dict(W=[t.numpy() for t in hW], dU=[t.numpy() for t in hdU], E=[t.numpy() for t in hE],
                    flag=hf.numpy(), status=hs.numpy())
        gpukit.assert_parity(gres, ores, w["U"], label="host entry, hybrid")
        # matter terms from the oracle's primitives
        Wd = gpukit.to_dev(ores["W"])
        out = [torch.zeros(sh["cell"], dtype=torch.float64, device="cuda:0") for _ in range(10)]
        ak.ak_matter_sources(g.ctx, Wd, out)
        torch.cuda.synchronize()
    for q in range(10):
        r, d = gpukit.max_rel_dev(out[q].cpu().numpy(), om[q], 1e-14 * float(np.max(np.abs(om[q]))))
        assert r <= 1.0, (q, r, d)


def test_advance_hybrid_matches_oracle():
    """three RK3 steps of the periodic noise block through ak_advance with the hybrid EOS"""
    import torch
    w = wl.make_test_noise_block(seed=9, n=8, frac=0.0)
    p = dict(w["params"], recon=1, riemann=1, fofc=1, eos_hybrid=HYB_3)
    dt = 0.2 * float(w["dx"].min())
    wo = copy.deepcopy(w)
    orc.fill_ghosts(orc.make_params(**p), [0, 0, 0], wo["U"], wo["Bf"])
    w0 = copy.deepcopy(wo)
    orc.advance(orc.make_params(**p), wo["dx"], 3, 3, dt, [0, 0, 0], wo["U"], wo["Bf"], wo["adm"], nthreads=4)
    with gpukit.GpuStage(w0, recon=1, riemann=1, fofc=1, eos_hybrid=HYB_3) as g:
        ak.ak_advance(g.ctx, 3, 3, dt, [0, 0, 0], g.U, g.Bf, g.W)
        torch.cuda.synchronize()
        gU = [t.cpu().numpy() for t in g.U]; gB = [t.cpu().numpy() for t in g.Bf]
    for v in range(5):
        r, d = gpukit.max_rel_dev(gU[v], wo["U"][v], 1e-13 * float(np.max(np.abs(wo["U"][v]))))
        assert r <= 10.0, (v, r, d)        # three steps of accumulated last-place differences of pow()
    for v in range(3):
        assert np.allclose(gB[v], wo["Bf"][v], rtol=1e-10, atol=1e-13)
