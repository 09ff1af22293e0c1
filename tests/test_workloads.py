"""The seeded input generators (paper_2409_10384_b200/workloads.py): inputs are functions of
(config, seed, block ids) alone.  They hold none of the method's arithmetic; what is checked here is
only that the same request gives the same arrays whatever was generated before it in the process
(the C0 vector-potential normalisation was once fixed by whichever seed came first, which made the
inputs of a test depend on the order of the tests), and the structure BASELINE.json's configs state."""
import json
import os
import subprocess
import sys

import numpy as np

from paper_2409_10384_b200 import workloads as wl


def _digest(w):
    return [float(np.sum(a)) for a in w["U"] + w["Bf"]] + [float(np.max(np.abs(a))) for a in w["Bf"]]


def test_noise_block_does_not_depend_on_what_was_generated_before():
    # in this process: other seeds and configs first
    wl.make_test_noise_block(seed=5, n=6, frac=0.03)
    wl.make_blocks("C0")
    here = _digest(wl.make_test_noise_block(seed=7, n=8, frac=0.02))
    # in a fresh process: the request alone
    code = ("import json, numpy as np\n"
            "from paper_2409_10384_b200 import workloads as wl\n"
            "w = wl.make_test_noise_block(seed=7, n=8, frac=0.02)\n"
            "print(json.dumps([float(np.sum(a)) for a in w['U'] + w['Bf']] + "
            "[float(np.max(np.abs(a))) for a in w['Bf']]))\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(wl.__file__)))
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, check=True, cwd=root)
    fresh = json.loads(out.stdout.strip().splitlines()[-1])
    assert here == fresh


def test_same_request_same_arrays_and_seed_matters():
    a = wl.make_test_noise_block(seed=11, n=6, frac=0.02)
    b = wl.make_test_noise_block(seed=11, n=6, frac=0.02)
    c = wl.make_test_noise_block(seed=12, n=6, frac=0.02)
    for x, y in zip(a["U"] + a["Bf"], b["U"] + b["Bf"]):
        assert np.array_equal(x, y)
    assert any(not np.array_equal(x, y) for x, y in zip(a["U"], c["U"]))


def test_c0_field_strength_and_divergence():
    """BASELINE.json configs[0]: |B| ~ 0.1, face B from the curl of a vector potential (div B = 0 to round-off)."""
    w = wl.make_blocks("C0")
    n, nt = w["params"]["n"], w["params"]["n"] + 8
    bx, by, bz = w["Bf"]
    d = float(w["dx"][0, 0])
    div = ((bx[0, :, :, 1:nt + 1] - bx[0, :, :, :nt]) + (by[0, :, 1:, :] - by[0, :, :-1, :]) +
           (bz[0, 1:, :, :] - bz[0, :-1, :, :])) / d
    scale = max(float(np.max(np.abs(b))) for b in (bx, by, bz)) / d
    assert np.max(np.abs(div)) < 1e-12 * scale
    s = slice(4, 4 + n)
    rms = np.sqrt(np.mean(bx[0, s, s, 4:4 + n] ** 2 + by[0, s, 4:4 + n, s] ** 2 + bz[0, 4:4 + n, s, s] ** 2))
    assert 0.05 < rms < 0.2
