"""The FMA-contracted perf build (libak_fma.so: the same sources compiled --fmad=true; SURVEY.md
section 8(d), BASELINE.json "documented differences only where fp64 FMA contraction is allowed")
against the oracle.  Contraction changes roundings, and differences of nearly equal fluxes amplify
them: measured, the build leaves BASELINE.json's tolerance (relative 1e-11) by up to ~80x on C4 and by
a few per cent on C0 — which is why it is a timed context build and not the product.  Held here: every
output within LOOSE = 1000x that tolerance (relative 1e-8) wherever the masks agree, and the masks
agree except for at most a handful of threshold cells.  The product build (libak.so, --fmad=false) is
the one every other test holds bit-identical to the oracle."""
import copy

import numpy as np
import pytest

from oracle import pyoracle as orc
from paper_2409_10384_b200 import ak, build as akbuild, workloads as wl

import gpukit

pytestmark = pytest.mark.gpu
LOOSE = 1000.0


def _assert_loose(g, o, U_in, label):
    umax = [float(np.max(np.abs(u))) for u in U_in]
    worst = 0.0
    for k, atols in (("W", [1e-14 * max(float(np.max(np.abs(x))), 1e-300) for x in o["W"]]),
                     ("dU", [1e-14 * m for m in umax]), ("E", [1e-14 * max(umax)] * 3)):
        for a, b, at in zip(g[k], o[k], atols):
            r, d = gpukit.max_rel_dev(a, b, at)
            assert r <= LOOSE, "%s: %s off by %.3g x tolerance (max abs %.3g) at %s" % (
                label, k, r, d, np.unravel_index(int(np.argmax(np.abs(a - b))), a.shape))
            worst = max(worst, r)
    return worst


@pytest.fixture()
def fma_library():
    akbuild.build(fma=True)
    ak.use_library(akbuild.SO_FMA)
    try:
        yield
    finally:
        ak.use_library(None)


def _both(w, **over):
    w = copy.deepcopy(w)
    U_in = [u.copy() for u in w["U"]]
    with gpukit.GpuStage(w, **over) as g:
        g.rhs()
        gres = g.result()
    p = dict(w["params"]); p.update(over)
    ores = orc.rhs(orc.make_params(**p), w["dx"], w["U"], w["Bf"], w["adm"], w["dt_fofc"], nthreads=8)
    ores["U"] = w["U"]
    return gres, ores, U_in


@pytest.mark.parametrize("recon", [1, 2])
def test_fma_build_c0_within_tolerance(fma_library, recon):
    g, o, U_in = _both(wl.make_blocks("C0"), recon=recon)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["flag"], o["flag"])   # smooth: nothing floored
    worst = _assert_loose(g, o, U_in, "C0, fma build")
    # contraction does change the arithmetic: not bit-identical any more
    assert any(not np.array_equal(a, b) for a, b in zip(g["dU"], o["dU"])) and worst > 0.0


def test_fma_build_star_blocks_within_tolerance(fma_library):
    w = wl.make_blocks("C1", blocks=[0, 7])
    g, o, U_in = _both(w)
    nbad = int(np.count_nonzero(g["status"] != o["status"])) + int(np.count_nonzero(g["flag"] != o["flag"]))
    assert nbad <= 4
    if nbad == 0:
        _assert_loose(g, o, U_in, "C1[0,7], fma build")


def test_fma_build_noise_block_masks(fma_library):
    """floors, flags and re-fluxed faces: a mask byte may flip only where a state sits on a threshold"""
    w = wl.make_test_noise_block(seed=7, n=8, frac=0.02)
    g, o, U_in = _both(w, dmp_M=1.1, recon=2)
    nbad = int(np.count_nonzero(g["status"] != o["status"])) + int(np.count_nonzero(g["flag"] != o["flag"]))
    assert np.count_nonzero(o["flag"]) > 0
    assert nbad <= 4
    if nbad == 0:
        # On discontinuous data a contraction can also flip a decision that no mask records (an upwind
        # side, a wave-speed clamp, a limiter branch: seen with other seeds as single cells off by
        # 1e-5), so the tail is not bounded here: 99.9 % of every output within LOOSE.
        umax = [float(np.max(np.abs(u))) for u in U_in]
        for k, atols in (("dU", [1e-14 * m for m in umax]), ("E", [1e-14 * max(umax)] * 3)):
            for a, b, at in zip(g[k], o[k], atols):
                ratio = np.abs(a - b) / (at + gpukit.RTOL * np.abs(b))
                assert np.mean(ratio <= LOOSE) >= 0.999, "%s: %.3g of the elements beyond %g x tolerance" % (
                    k, np.mean(ratio > LOOSE), LOOSE)
