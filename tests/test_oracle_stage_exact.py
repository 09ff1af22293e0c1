"""Stage-level pins with exact expectations: T4 (uniform Minkowski), T12 (rotating frame),
T13 (FLRW), T9 (CT 1-D reduction).  DESIGN.md §5.  CPU only."""
import numpy as np
import pytest

import stagekit as sk
from oracle import pyoracle as po

N = 6


def _run(blk, dt=0.05, **kw):
    par = po.make_params(nmb=1, n=N, **kw)
    U = [u.copy() for u in blk["U"]]
    return po.rhs(par, blk["dx"], U, blk["Bf"], blk["adm"], dt, want_flux=True), par


@pytest.mark.parametrize("recon", [0, 1, 2])
@pytest.mark.parametrize("riemann", [0, 1])
def test_T4_uniform_minkowski_is_stationary(recon, riemann):
    u = [0.3, -0.2, 0.5]; B = [0.2, 0.4, -0.3]
    blk = sk.build_block(N, 0.1, (0, 0, 0), sk.flat_metric,
                         lambda x, y, z: (1.3 + 0 * x, [c + 0 * x for c in u], 0.7 + 0 * x),
                         B_uniform=B)
    r, par = _run(blk, recon=recon, riemann=riemann, fofc=1, dmp_M=1.1)
    for a in r["dU"]:
        assert np.all(a == 0.0)                       # bitwise zero
    assert not r["flag"].any() and not r["status"].any()
    W = np.sqrt(1 + sum(c * c for c in u))
    v = np.array(u) / W
    Eref = -np.cross(v, np.array(B))                  # E = -v x B (alpha=1, beta=0)
    s = slice(sk.NG, sk.NG + N); s1 = slice(sk.NG, sk.NG + N + 1)
    assert np.allclose(r["E"][0][0, s1, s1, s], Eref[0], rtol=4e-16, atol=1e-17)
    assert np.allclose(r["E"][1][0, s1, s, s1], Eref[1], rtol=4e-16, atol=1e-17)
    assert np.allclose(r["E"][2][0, s, s1, s1], Eref[2], rtol=4e-16, atol=1e-17)


def test_T12_rotating_frame():
    Om = np.array([0.03, -0.02, 0.05])

    def metric(x, y, z):
        o = np.ones_like(x); zr = np.zeros_like(x)
        beta = [Om[1] * z - Om[2] * y, Om[2] * x - Om[0] * z, Om[0] * y - Om[1] * x]
        return o, beta, [o, zr, zr, o, zr, o], [zr] * 6
    u = [0.3, -0.2, 0.5]; B = np.array([0.2, 0.4, -0.3])
    blk = sk.build_block(N, 0.25, (1.0, -2.0, 0.5), metric,
                         lambda x, y, z: (1.3 + 0 * x, [c + 0 * x for c in u], 0.7 + 0 * x),
                         B_uniform=B)
    for recon, riemann in ((1, 1), (2, 0)):
        r, par = _run(blk, recon=recon, riemann=riemann, fofc=1)
        assert not r["flag"].any()
        S = np.array([sk.interior(blk["U"][1 + c], N) for c in range(3)])
        scale = np.abs(S).max()
        # dS/dt = -Omega x S, dD/dt = dtau/dt = 0
        ref = -np.cross(Om, S, axisa=0, axisb=0, axisc=0)
        for c in range(3):
            assert np.abs(sk.interior(r["dU"][1 + c], N) - ref[c]).max() <= 2e-14 * scale * 10
        assert np.abs(sk.interior(r["dU"][0], N)).max() <= 1e-14
        assert np.abs(sk.interior(r["dU"][4], N)).max() <= 1e-14
        # induction: -curl E = -Omega x B~ on every face of the interior cells
        dBx, dBy, dBz, div = sk.curlE_div(r["E"], N, 0.25)
        refB = -np.cross(Om, B)
        for a, c in ((dBx, 0), (dBy, 1), (dBz, 2)):
            assert np.abs(a - refB[c]).max() <= 1e-13
        assert np.abs(div).max() <= 1e-13


def test_T13_flrw_expansion():
    a2, Hub = 1.7, 0.3

    def metric(x, y, z):
        o = np.ones_like(x); zr = np.zeros_like(x)
        g = [a2 * o, zr, zr, a2 * o, zr, a2 * o]
        K = [-Hub * a2 * o, zr, zr, -Hub * a2 * o, zr, -Hub * a2 * o]
        return o, [zr, zr, zr], g, K
    P0 = 0.4
    blk = sk.build_block(N, 0.2, (0, 0, 0), metric,
                         lambda x, y, z: (1.1 + 0 * x, [0 * x, 0 * x, 0 * x], P0 + 0 * x))
    r, par = _run(blk, recon=2, riemann=1, fofc=1)
    sg = a2 ** 1.5
    assert np.allclose(sk.interior(r["dU"][4], N), -3 * Hub * sg * P0, rtol=1e-14)
    for c in range(4):
        assert np.abs(sk.interior(r["dU"][c], N)).max() <= 1e-15


def test_T9_ct_reduces_to_face_emf_in_1d():
    rng = np.random.default_rng(3)
    nt = N + 2 * sk.NG
    prof = {k: rng.uniform(0.5, 1.5, nt) for k in ("rho", "P")}
    prof.update({k: rng.uniform(-0.4, 0.4, nt) for k in ("ux", "uy", "uz")})
    d = 0.1

    def prim(x, y, z):
        i = np.rint((x - 0.5 * d) / d).astype(int) + sk.NG
        return prof["rho"][i], [prof["ux"][i], prof["uy"][i], prof["uz"][i]], prof["P"][i]
    blk = sk.build_block(N, d, (0, 0, 0), sk.flat_metric, prim, B_uniform=[0.3, 0.0, 0.0])
    # add a y-field varying in x only: B~^y(i) on y-faces (still divergence-free)
    by = rng.uniform(-0.5, 0.5, nt)
    blk["Bf"][1] += by[None, None, None, :]
    blk2 = dict(blk)
    r, par = _run(blk2, recon=1, riemann=1, fofc=0)
    # U was built with By=0; rebuild consistently through con2prim inputs is not needed:
    # the identity below is a property of O8 for any y,z-uniform data.
    s = slice(sk.NG, sk.NG + N); s1 = slice(sk.NG, sk.NG + N + 1)
    Ez = r["E"][2][0, s, s1, s1]
    Fx_By = r["flux"][5][0, s, :, :][:, sk.NG - 1:sk.NG + N + 1, s1]   # F^x(B~^y), slot t1
    # E_z on x-faces = -F^x(B~^y); rows j-1 and j are identical for y-uniform data
    assert np.abs(Ez - (-Fx_By[:, 1:, :])).max() <= 1e-15


def test_T28_matter_sources_equal_projections_of_the_stress_energy_tensor():
    """E = n_mu n_nu T^{mu nu}, S_i = -gamma_i^mu n^nu T_{mu nu}, S_ij = T_ij with T^{mu nu}
    built from Eqs. 2, 7 and the full 4-metric (tests/helpers.py), random metrics with shift."""
    import helpers as H
    from oracle import pyoracle as po
    rng = np.random.default_rng(28)
    n = 2
    par = po.make_params(nmb=1, n=n, gamma_ad=5.0 / 3.0)
    sh = po.shapes(1, n)
    W = [np.zeros(sh["cell"]) for _ in range(8)]
    g6 = [np.zeros(sh["cell"]) for _ in range(6)]
    exp = [np.zeros(sh["cell"]) for _ in range(10)]
    nt = n + 8
    for k in range(nt):
        for j in range(nt):
            for i in range(0, nt, 3):
                g = H.random_spd(rng)
                alpha = rng.uniform(0.3, 1.5); beta = rng.uniform(-0.3, 0.3, 3)
                rho = 10 ** rng.uniform(-6, 0); P = rho * 10 ** rng.uniform(-3, 1)
                gm = H.sym6_to_mat(g)
                v = rng.uniform(-1, 1, 3); v *= rng.uniform(0, 0.9) / np.sqrt(v @ gm @ v)
                B = rng.uniform(-1, 1, 3) * 10 ** rng.uniform(-3, 0)
                U, F, d = H.tensor_state(alpha, beta, g, rho, v, P, B, 5.0 / 3.0)
                T, g4 = d["T"], d["g4"]
                Tdd = g4 @ T @ g4
                nl = np.array([-alpha, 0, 0, 0]); nu_ = np.concatenate([[1 / alpha], -beta / alpha])
                E = nl @ T @ nl
                Si = -(Tdd[1:, :] @ nu_)
                Sij = Tdd[1:, 1:]
                Wl = d["W"]
                vals = [rho, Wl * v[0], Wl * v[1], Wl * v[2], P] + list(d["sg"] * B)
                for q, a in enumerate(vals):
                    W[q][0, k, j, i] = a
                for q in range(6):
                    g6[q][0, k, j, i] = g[q]
                e = [E, Si[0], Si[1], Si[2]] + [Sij[a_, b_] for (a_, b_) in H.SYM]
                for q in range(10):
                    exp[q][0, k, j, i] = e[q]
    # unset cells: harmless flat-space fluid at rest
    for q, a in enumerate((1.0, 0, 0, 0, 1.0, 0, 0, 0)):
        W[q][W[0] == 0] = a
    for q, a in enumerate((1.0, 0, 0, 1.0, 0, 1.0)):
        g6[q][g6[0] == 0] = a
    out = po.matter_sources(par, W, g6)
    mask = exp[0] != 0
    for q in range(10):
        scale = np.abs(exp[0][mask]) + np.abs(exp[q][mask])
        assert np.max(np.abs(out[q][mask] - exp[q][mask]) / scale) < 1e-12, q
