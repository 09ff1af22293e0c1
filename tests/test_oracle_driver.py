"""Pins of the oracle's stage driver: ghost fill, Shu-Osher register update with the
constrained-transport update of B~f, the SSP-RK loop and the stage-blended FOFC estimate — against
numpy index primitives, closed forms, Richardson orders in dt, conservation and symmetry."""
import numpy as np
import pytest

from oracle import pyoracle as orc
from paper_2409_10384_b200 import workloads as wl

import helpers
import stagekit as sk

NG = 4


def rand_fields(n, seed):
    rng = np.random.default_rng(seed)
    sh = orc.shapes(1, n)
    U = [rng.uniform(-1, 1, sh["cell"]) for _ in range(5)]
    Bf = [rng.uniform(-1, 1, sh[k]) for k in ("xf", "yf", "zf")]
    return U, Bf, sh


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1), (1, 0, 0), (0, 1, 0)])
def test_T18_ghost_fill_equals_numpy_pad(bc):
    n = 6
    U, Bf, sh = rand_fields(n, 1)
    par = orc.make_params(nmb=1, n=n)
    U2 = [u.copy() for u in U]; B2 = [b.copy() for b in Bf]
    orc.fill_ghosts(par, bc, U2, B2)
    s = slice(NG, NG + n)
    mode = lambda d: "wrap" if bc[d] == 0 else "edge"

    def pad3(a, widths):
        # pad axis by axis (k, j, i <-> directions 2, 1, 0) so each can have its own mode
        for ax, d in ((0, 2), (1, 1), (2, 0)):
            pw = [(0, 0)] * 3
            pw[ax] = widths[ax]
            a = np.pad(a, pw, mode=mode(d))
        return a
    for v in range(5):
        exp = pad3(U[v][0, s, s, s], [(NG, NG)] * 3)
        assert np.array_equal(U2[v][0], exp)
    # faces: the n+1 faces is..ie+1 bound the interior; periodic: face ie+1 == face is
    nt = n + 2 * NG
    for d, key in enumerate(("xf", "yf", "zf")):
        ax = 2 - d                                   # array axis of the normal direction
        sl = [s, s, s]
        sl[ax] = slice(NG, NG + n + 1)
        core = Bf[d][0][tuple(sl)].copy()
        if bc[d] == 0:                               # the n distinct faces, then wrap
            idx = [slice(None)] * 3; idx[ax] = slice(0, n)
            core = core[tuple(idx)]
            widths = [(NG, NG)] * 3
            widths[ax] = (NG, NG + 1)
        else:
            widths = [(NG, NG)] * 3
        exp = pad3(core, widths)
        got = B2[d][0]
        if d == 0:
            got = got[:, :, :nt + 1]
        assert np.array_equal(got, exp), key


def test_T19_stage_update_closed_form():
    n, d = 6, 0.37
    U, Bf, sh = rand_fields(n, 2)
    U0, B0, _ = rand_fields(n, 3)
    rng = np.random.default_rng(4)
    dU = [rng.uniform(-1, 1, sh["cell"]) for _ in range(5)]
    E = [rng.uniform(-1, 1, sh[k]) for k in ("ex", "ey", "ez")]
    par = orc.make_params(nmb=1, n=n)
    a, b, dt = 0.75, 0.25, 0.013
    U2 = [u.copy() for u in U]; B2 = [x.copy() for x in Bf]
    orc.stage_update(par, np.full((1, 3), d), a, b, dt, U0, B0, U2, B2, dU, E)
    s = slice(NG, NG + n); s1 = slice(NG, NG + n + 1)
    for v in range(5):
        exp = U[v].copy()
        exp[:, s, s, s] = a * U0[v][:, s, s, s] + b * (U[v][:, s, s, s] + dt * dU[v][:, s, s, s])
        assert np.allclose(U2[v], exp, rtol=1e-15, atol=1e-16) and np.array_equal(U2[v][:, 0], U[v][:, 0])
    dBx, dBy, dBz, div = sk.curlE_div(E, n, d)      # independent curl (tests/stagekit.py)
    for comp, (dB, sl) in enumerate(((dBx, (s, s, s1)), (dBy, (s, s1, s)), (dBz, (s1, s, s)))):
        exp = Bf[comp].copy()
        idx = (slice(None),) + sl
        exp[idx] = a * B0[comp][idx] + b * (Bf[comp][idx] + dt * dB)
        assert np.allclose(B2[comp], exp, rtol=1e-13, atol=1e-14), comp
    assert np.max(np.abs(div)) < 1e-12               # curl of anything is divergence-free


def wave_block(n, recon=2, fofc=0, B0=(0.0, 0.0, 0.0)):
    """flat-space periodic block [0,1]^3: density wave advected by a uniform flow."""
    d = 1.0 / n

    def prim(x, y, z):
        rho = 1.0 + 0.2 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y)
        v = (0.4, 0.3, 0.0)
        W = 1.0 / np.sqrt(1 - sum(c * c for c in v))
        o = np.ones_like(x)
        return rho, [W * v[0] * o, W * v[1] * o, W * v[2] * o], 1.0 * o
    w = sk.build_block(n, d, (0.0, 0.0, 0.0), sk.flat_metric, prim, B_uniform=B0, gamma_ad=5.0 / 3.0)
    p = dict(nmb=1, n=n, gamma_ad=5.0 / 3.0, rho_atm=1e-10, T_atm=1e-8, recon=recon, riemann=1, fofc=fofc)
    return w, p, d


@pytest.mark.parametrize("integrator,order", [(1, 1), (2, 2), (3, 3)])
def test_T20_temporal_order_by_richardson(integrator, order):
    """Same spatial operator, dt halved twice: ||u_dt - u_dt/2|| / ||u_dt/2 - u_dt/4|| -> 2^p pins the
    Shu-Osher coefficients of SSP-RK1/2/3 and the register update."""
    n = 8
    w, p, d = wave_block(n, recon=2, fofc=0)
    par = orc.make_params(**p)
    T = 0.08
    sols = []
    for nst in (4, 8, 16):
        U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
        orc.advance(par, w["dx"], integrator, nst, T / nst, (0, 0, 0), U, Bf, w["adm"], nthreads=4)
        sols.append(sk.interior(U[0], n).copy())
    e1 = np.linalg.norm(sols[0] - sols[1]); e2 = np.linalg.norm(sols[1] - sols[2])
    assert e2 > 0
    assert abs(np.log2(e1 / e2) - order) < 0.35, (e1, e2, np.log2(e1 / e2))


def test_T20b_density_wave_is_advected():
    """SR hydro with uniform v and P: rho(x - v t) exactly; RK3 + WENO-Z error shrinks >= 12x from
    n = 8 to n = 16 (dt ~ dx), i.e. the loop evolves the right equation in the right direction."""
    errs = []
    for n in (8, 16):
        w, p, d = wave_block(n)
        par = orc.make_params(**p)
        T = 0.1
        nst = n // 2
        U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
        W, _ = orc.advance(par, w["dx"], 3, nst, T / nst, (0, 0, 0), U, Bf, w["adm"], nthreads=4)
        c = (np.arange(n) + 0.5) * d
        Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
        exact = 1.0 + 0.2 * np.sin(2 * np.pi * (X - 0.4 * T)) * np.cos(2 * np.pi * (Y - 0.3 * T))
        # the data are point-sampled, and a field whose cell averages are those samples is advected
        # exactly, so the centred values of the exact solution are the right comparison to O(dx^4)
        orc.fill_ghosts(par, (0, 0, 0), U, Bf)
        Wc, st = orc.con2prim(par, U, Bf, w["adm"][:6])
        errs.append(np.max(np.abs(sk.interior(Wc[0], n)[0] - exact)))
    assert errs[0] / errs[1] > 12.0, errs


def test_T21_periodic_conservation_and_divB_with_fofc_flags():
    w = wl.make_test_noise_block(seed=7, n=8, frac=0.02)
    n = 8
    p = dict(w["params"]); p.update(dmp_M=1.1, recon=2)
    par = orc.make_params(**p)
    U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
    orc.fill_ghosts(par, (0, 0, 0), U, Bf)            # the generator's ghosts are analytic, not periodic
    tot0 = [np.sum(sk.interior(u, n)) for u in U]
    sx = (slice(None), slice(NG, NG + n), slice(NG, NG + n), slice(NG, NG + n))
    mean0 = [np.sum(Bf[0][sx]), np.sum(Bf[1][sx]), np.sum(Bf[2][sx])]
    W, flag = orc.advance(par, w["dx"], 3, 3, 0.2 / n, (0, 0, 0), U, Bf, w["adm"], nthreads=4)
    assert np.count_nonzero(flag) > 0                 # first-order faces took part
    scale = [np.sum(np.abs(sk.interior(u, n))) for u in U]
    for v in range(5):
        assert abs(np.sum(sk.interior(U[v], n)) - tot0[v]) <= 2e-13 * max(scale[v], 1.0), v
    for c in range(3):
        assert abs(np.sum(Bf[c][sx]) - mean0[c]) <= 1e-12
    d = 1.0 / n
    s = slice(NG, NG + n); s1 = slice(NG + 1, NG + n + 1)
    div = ((Bf[0][:, s, s, s1] - Bf[0][:, s, s, s]) + (Bf[1][:, s, s1, s] - Bf[1][:, s, s, s]) +
           (Bf[2][:, s1, s, s] - Bf[2][:, s, s, s])) / d
    assert np.max(np.abs(div)) < 5e-13
    # periodic images agree bitwise: face ie+1 is face is
    assert np.array_equal(Bf[0][:, s, s, NG + n], Bf[0][:, s, s, NG])


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1)])
def test_T22_uniform_state_is_a_fixed_point(bc):
    n = 4
    prim = lambda x, y, z: (0.7 + 0 * x, [0.3 + 0 * x, -0.2 + 0 * x, 0.1 + 0 * x], 0.4 + 0 * x)
    w = sk.build_block(n, 0.25, (0, 0, 0), sk.flat_metric, prim, B_uniform=(0.3, -0.1, 0.2))
    par = orc.make_params(nmb=1, n=n, recon=1, riemann=1, fofc=1)
    U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
    orc.advance(par, w["dx"], 3, 2, 0.05, bc, U, Bf, w["adm"])
    # dU/dt and curl E vanish bit for bit (T4); the convex register combination 3/4 x + 1/4 x
    # rounds, so the state is fixed to an ulp per stage, not bitwise
    for a, b in zip(U + Bf, w["U"] + w["Bf"]):
        assert np.allclose(a, b, rtol=2e-15, atol=0)
    par1 = orc.make_params(nmb=1, n=n, recon=1, riemann=1, fofc=1)
    U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
    orc.advance(par1, w["dx"], 1, 3, 0.05, bc, U, Bf, w["adm"])      # forward Euler: a = 0, b = 1: bitwise
    for a, b in zip(U + Bf, w["U"] + w["Bf"]):
        assert np.array_equal(a, b)


def test_T23_one_euler_step_is_fill_rhs_update():
    w = wl.make_test_noise_block(seed=3, n=6, frac=0.0)
    par = orc.make_params(**w["params"])
    dt = 0.01
    U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
    orc.advance(par, w["dx"], 1, 1, dt, (0, 0, 0), U, Bf, w["adm"])
    V = [u.copy() for u in w["U"]]; Bg = [b.copy() for b in w["Bf"]]
    orc.fill_ghosts(par, (0, 0, 0), V, Bg)
    r = orc.rhs(par, w["dx"], V, Bg, w["adm"], dt)
    n = 6
    s = slice(NG, NG + n)
    for v in range(5):
        exp = V[v][:, s, s, s] + dt * r["dU"][v][:, s, s, s]
        assert np.allclose(U[v][:, s, s, s], exp, rtol=1e-15, atol=0)


def test_T24_blended_fofc_estimate():
    """fa = 0, fb = 1 reproduces the plain estimate bit for bit; fa = 1, fb = 0 makes U* = U0, whose
    flags must equal the point-level check-only con2prim of U0 (independent path)."""
    w = wl.make_test_noise_block(seed=5, n=6, frac=0.03)
    n = 6
    p = dict(w["params"])
    par = orc.make_params(**p)
    dt = 2 * w["dt_fofc"]
    U = [u.copy() for u in w["U"]]
    r0 = orc.rhs(par, w["dx"], U, w["Bf"], w["adm"], dt)
    rng = np.random.default_rng(0)
    junk = [rng.uniform(0, 1, u.shape) for u in U]
    U = [u.copy() for u in w["U"]]
    r1 = orc.rhs_blend(par, w["dx"], U, w["Bf"], w["adm"], dt, junk, 0.0, 1.0)
    assert np.array_equal(r0["flag"], r1["flag"]) and np.array_equal(r0["dU"][0], r1["dU"][0])
    # U0 with some unphysical cells
    U0 = [u.copy() for u in w["U"]]
    U0[4][0, 5, 6, 7] = -1.0; U0[0][0, 6, 6, 6] = 1e-14; U0[1][0, 7, 5, 5] = 50.0
    U = [u.copy() for u in w["U"]]
    r2 = orc.rhs_blend(par, w["dx"], U, w["Bf"], w["adm"], dt, U0, 1.0, 0.0)
    nt = n + 2 * NG
    exp = np.zeros_like(r2["flag"])
    for k in range(NG - 1, NG + n + 1):
        for j in range(NG - 1, NG + n + 1):
            for i in range(NG - 1, NG + n + 1):
                g = [a[0, k, j, i] for a in w["adm"][:6]]
                Ut = [1.0 * U0[v][0, k, j, i] + 0.0 * 0.0 for v in range(5)]
                Bc = [r2["W"][5 + c][0, k, j, i] for c in range(3)]
                st, _, _, _ = orc.con2prim_cell(par, g, Ut, Bc, check_only=True)
                exp[0, k, j, i] = st
    assert np.array_equal(r2["flag"], exp)
    assert exp[0, 5, 6, 7] & 2 and exp[0, 6, 6, 6] & 1


def test_T25_shock_tube_stays_one_dimensional_and_physical():
    """Balsara test 1 (tests/golden/balsara_table1.txt) along x with outflow in x:
    y,z-uniform data stay y,z-uniform bit for bit, density and pressure stay positive, the
    total mass changes only through the x boundaries (none before the waves arrive)."""
    n = 16
    d = 1.0 / n
    gam = 2.0

    def prim(x, y, z):
        L = x < 0.5
        return np.where(L, 1.0, 0.125), [0 * x, 0 * x, 0 * x], np.where(L, 1.0, 0.1)

    def A(comp, x, y, z):          # B~y = +-1 from A_z = -By x (piecewise), B~x = 0.5 from A_z += 0.5 y
        if comp != 2:
            return 0 * x
        By = np.where(x < 0.5, 1.0, -1.0)
        return -By * (x - 0.5) + 0.5 * y
    w = sk.build_block(n, d, (0, 0, 0), sk.flat_metric, prim, A_fn=A, gamma_ad=gam)
    par = orc.make_params(nmb=1, n=n, gamma_ad=gam, rho_atm=1e-10, T_atm=1e-8, recon=1, riemann=0, fofc=1)
    U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
    m0 = np.sum(sk.interior(U[0], n))
    W, flag = orc.advance(par, w["dx"], 2, 6, 0.25 * d, (1, 0, 0), U, Bf, w["adm"], nthreads=4)
    for a in U + list(W[:5]):
        assert np.all(a == a[:, NG:NG + 1, NG:NG + 1, :])          # uniform in y and z
    assert np.all(W[0] > 0) and np.all(W[4] > 0)
    assert abs(np.sum(sk.interior(U[0], n)) - m0) < 1e-8 * m0      # only diffusive tails reach the x boundaries
    rho = W[0][0, NG, NG, NG:NG + n]
    assert rho.max() <= 1.0 + 1e-3 and rho.min() >= 0.125 - 1e-3 and np.any((rho < 0.99) & (rho > 0.13))


def test_T29_magnetic_loop_is_advected_at_the_right_speed():
    """Loop advection: with RK3, HLLE+FOFC, WENO-Z at CFL 0.25 the loop moves with
    v = (1/1.2, 1/2.4, 0).  After t = 1.2 it has crossed the periodic box once in x and half of it
    in y, so B~x must match the initial loop displaced by n/2 cells in y (and not the undisplaced one);
    div B~ stays at round-off (paper: 7e-14 -> 3e-12 relative to max|B| at 240^2), mass is conserved,
    no B~z appears and no cell is flagged by the FOFC."""
    n = 16
    w, p, d = sk.loop_block(n)
    par = orc.make_params(**p)
    U = [u.copy() for u in w["U"]]; Bf = [b.copy() for b in w["Bf"]]
    bmax = max(np.abs(b).max() for b in Bf)
    assert abs(bmax - 1e-3) < 1e-15 and sk.divB_rel(Bf, n, d, bmax) < 1e-14
    m0 = np.sum(sk.interior(U[0], n))
    nsteps = int(np.ceil(1.2 / (0.25 * d)))
    W, flag = orc.advance(par, w["dx"], 3, nsteps, 1.2 / nsteps, (0, 0, 0), U, Bf, w["adm"], nthreads=4)
    c_moved, c_same, e_ratio = sk.loop_metrics(Bf, w["Bf"], n, n // 2)
    assert c_moved > 0.93 and c_same < 0.0
    assert 0.6 < e_ratio <= 1.0                       # diffusion only removes magnetic energy
    assert sk.divB_rel(Bf, n, d, bmax) < 1e-13
    assert abs(np.sum(sk.interior(U[0], n)) / m0 - 1.0) < 1e-13
    assert np.abs(Bf[2]).max() < 1e-15 and np.count_nonzero(flag) == 0
