"""The paper's flat-space tests run end to end on the GPU through ak_advance with the
same-level ghost exchange: properties the paper states (first-order convergence of the shock tubes,
P:196-198; the blast wave stays physical with FOFC), not element-wise parity - the
element-wise parity of ak_advance is in test_gpu_driver.py.  Exact Riemann solutions are not
available here, so convergence is measured between successive resolutions."""
import os

import numpy as np
import pytest

from paper_2409_10384_b200 import ak, workloads as wl

import gpukit
import tovkit
from test_oracle_exchange import lattice_nbr

pytestmark = pytest.mark.gpu
NG = 4
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "balsara_table1.txt")


def balsara_states(test_id):
    out = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if int(t[0]) == test_id:
            out[t[1]] = [float(x) for x in t[2:]]
    return out["L"], out["R"]


def riemann_chain(test_id, n, nbx):
    """nbx blocks of n^3 in a row along x covering [0,1], discontinuity at x = 0.5; uniform in
    y and z (each block is its own periodic neighbour there), outflow in x."""
    L, R = balsara_states(test_id)
    gam = L[0]
    nt = n + 2 * NG
    d = 1.0 / (n * nbx)
    sh = ak.shapes(nbx, n)
    U = [np.zeros(sh["cell"]) for _ in range(5)]
    Bf = [np.zeros(sh[k]) for k in ("xf", "yf", "zf")]
    for b in range(nbx):
        xc = (b * n + np.arange(nt) - NG + 0.5) * d
        left = xc < 0.5
        q = [np.where(left, L[k], R[k]) for k in range(1, 9)]          # rho P vx vy vz Bx By Bz
        rho, P, v, B = q[0], q[1], q[2:5], q[5:8]
        lor = 1.0 / np.sqrt(1.0 - (v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
        o, zr = np.ones(nt), np.zeros(nt)
        D, S, tau = wl._prim2cons_np(gam, [o, zr, zr, o, zr, o], rho, [lor * a for a in v], P, B)
        for dst, src in zip(U, (D, S[0], S[1], S[2], tau)):
            dst[b] = src[None, None, :]
        Bf[0][b] = L[6]                                                  # B^x is the same on both sides
        Bf[1][b] = B[1][None, None, :]
        Bf[2][b] = B[2][None, None, :]
    one, zero = np.ones(sh["cell"]), np.zeros(sh["cell"])
    adm = [one, zero, zero, one, zero, one, one] + [zero] * 9
    p = dict(nmb=nbx, n=n, gamma_ad=gam, rho_atm=1e-10, T_atm=1e-8, recon=1, riemann=0, fofc=0)
    return dict(U=U, Bf=Bf, adm=adm, dx=np.full((nbx, 3), d), params=p, dt_fofc=0.0), d


def run_tube(test_id, n, nbx, t_end=0.4, cfl=0.2, integrator=3, **override):
    import torch
    w, d = riemann_chain(test_id, n, nbx)
    w["params"].update(override)
    nsteps = int(np.ceil(t_end / (cfl * d)))
    w["dt_fofc"] = t_end / nsteps
    nbr = lattice_nbr((nbx, 1, 1), (False, True, True))
    with gpukit.GpuStage(w) as g:
        ak.ak_set_neighbors(g.ctx, nbr)
        gflag = torch.zeros_like(g.flag)
        ak.ak_advance(g.ctx, integrator, nsteps, t_end / nsteps, (1, 0, 0), g.U, g.Bf, g.W, gflag)
        torch.cuda.synchronize()
        W = [t.cpu().numpy() for t in g.W]
        stats = g.stats()
    s = slice(NG, NG + n)
    line = lambda a: a[:, NG, NG, s].reshape(-1)                           # the interior cells along x
    uniform = all(np.all(a[:, s, s, s] == a[:, NG:NG + 1, NG:NG + 1, s]) for a in W[:5])
    return dict(rho=line(W[0]), P=line(W[4]), ux=line(W[1]), by=line(W[6]), uniform=uniform, stats=stats,
                flagged=int(gflag.count_nonzero()))


def coarsen(a):
    return 0.5 * (a[0::2] + a[1::2])


def tube_errors(test_id, n=16, nbxs=(4, 8, 16, 32)):
    """L1 and L2 norms of rho(N) - coarsened rho(2N) for successive resolutions."""
    runs = [run_tube(test_id, n, nbx) for nbx in nbxs]
    e1, e2 = [], []
    for a, b in zip(runs[:-1], runs[1:]):
        diff = a["rho"] - coarsen(b["rho"])
        e1.append(np.mean(np.abs(diff))); e2.append(np.sqrt(np.mean(diff ** 2)))
    return runs, e1, e2


# ---------------------------------------------------------------- cylindrical blast wave
def blast_lattice(bx_field, n, nb):
    """nb x nb x 1 blocks of n^3 covering [-6,6]^2 (uniform in z): rho_in = 1e-2, P_in = 1 inside
    r_in = 0.8, ambient 1e-4 / 3e-5 outside r_out = 1, exponential decay (linear in the logarithm)
    between; B = (Bx, 0, 0); fluid at rest; Gamma = 4/3."""
    gam = 4.0 / 3.0
    nt = n + 2 * NG
    d = 12.0 / (n * nb)
    nmb = nb * nb
    sh = ak.shapes(nmb, n)
    U = [np.zeros(sh["cell"]) for _ in range(5)]
    Bf = [np.zeros(sh[k]) for k in ("xf", "yf", "zf")]
    Bf[0][:] = bx_field
    o, zr = np.ones((nt, nt)), np.zeros((nt, nt))
    for by in range(nb):
        for bx in range(nb):
            m = by * nb + bx
            xc = -6.0 + (bx * n + np.arange(nt) - NG + 0.5) * d
            yc = -6.0 + (by * n + np.arange(nt) - NG + 0.5) * d
            Y, X = np.meshgrid(yc, xc, indexing="ij")
            r = np.sqrt(X * X + Y * Y)
            f = np.clip((r - 0.8) / 0.2, 0.0, 1.0)                      # 0 inside r_in, 1 outside r_out
            rho = np.exp((1.0 - f) * np.log(1e-2) + f * np.log(1e-4))
            P = np.exp((1.0 - f) * np.log(1.0) + f * np.log(3e-5))
            D, S, tau = wl._prim2cons_np(gam, [o, zr, zr, o, zr, o], rho, [zr, zr, zr], P, [bx_field * o, zr, zr])
            for dst, src in zip(U, (D, S[0], S[1], S[2], tau)):
                dst[m] = src[None, :, :]
    one, zero = np.ones(sh["cell"]), np.zeros(sh["cell"])
    adm = [one, zero, zero, one, zero, one, one] + [zero] * 9
    p = dict(nmb=nmb, n=n, gamma_ad=gam, rho_atm=1e-10, T_atm=1e-8, f_thr=1.0, recon=2, riemann=1, fofc=1)
    return dict(U=U, Bf=Bf, adm=adm, dx=np.full((nmb, 3), d), params=p, dt_fofc=0.0), d


def run_blast(bx_field, n=20, nb=10, t_end=4.0, cfl=0.1, **override):
    import torch
    w, d = blast_lattice(bx_field, n, nb)
    w["params"].update(override)
    nsteps = int(np.ceil(t_end / (cfl * d)))
    dt = t_end / nsteps
    w["dt_fofc"] = dt
    nbr = lattice_nbr((nb, nb, 1), (False, False, True))
    s = slice(NG, NG + n)
    with gpukit.GpuStage(w) as g:
        ak.ak_set_neighbors(g.ctx, nbr)
        gflag = torch.zeros_like(g.flag)
        ak.ak_advance(g.ctx, 3, nsteps, dt, (1, 1, 0), g.U, g.Bf, g.W, gflag)
        torch.cuda.synchronize()
        W = [t.cpu().numpy() for t in g.W]
        stats = g.stats()
        flagged = int(gflag[:, s, s, s].count_nonzero())

    def plane(a):                                                          # [nb*n, nb*n] at one z
        a = a[:, NG, s, s].reshape(nb, nb, n, n)
        return a.transpose(0, 2, 1, 3).reshape(nb * n, nb * n)
    uniform_z = all(np.all(a[:, s, s, s] == a[:, NG:NG + 1, s, s]) for a in W[:5])
    return dict(rho=plane(W[0]), P=plane(W[4]), ux=plane(W[1]), uy=plane(W[2]), stats=stats, flagged=flagged,
                uniform_z=uniform_z, zones=nb * nb * n ** 3)


# ================================================================ the tests
@pytest.mark.parametrize("test_id", [1, 2, 3, 4, 5])
def test_balsara_tubes_converge_at_first_order(test_id):
    """LLF + PPM4, no FOFC, t = 0.5, the paper's resolutions 200/400/800 against its 1600-cell
    run (80 blocks of 20^3 in a row, exchanged every stage).  'Approximate first-order convergence
    for all tests' (the lowest resolutions of #3 and #5 are not yet convergent): the L1 order
    of rho between 200 and 800 cells is about one; the run stays one-dimensional bit for bit and
    needs no floor and no inversion failure ('never approaches atmosphere')."""
    runs = [run_tube(test_id, 20, nbx, t_end=0.5) for nbx in (10, 20, 40, 80)]
    ref = runs[-1]["rho"]
    err = []
    for r in runs[:-1]:
        c = ref
        while c.size > r["rho"].size:
            c = coarsen(c)
        err.append(np.mean(np.abs(r["rho"] - c)))
    order = np.log2(err[0] / err[2]) / 2.0
    assert err[0] > err[1] > err[2]
    assert 0.75 < order < 1.6, (err, order)
    for r in runs:
        st = r["stats"]
        assert r["uniform"] and np.isfinite(r["rho"]).all()
        assert st["n_c2p_fail"] == 0 and st["n_cons_floor"] == 0 and st["n_prim_floor"] == 0
        assert r["rho"].min() > 0.05 and r["P"].min() > 0.05


def _front(a, thr):
    n = a.shape[0]
    x = (np.arange(n) + 0.5) * 12.0 / n - 6.0
    return np.abs(x[a[n // 2] > thr]).max(), np.abs(x[a[:, n // 2] > thr]).max()


def test_blast_wave_moderate_field_with_fofc():
    """B_x = 0.1 (Figure 4) at the paper's 200^2 cells, HLLE + WENO-Z + RK3, CFL 0.1,
    FOFC: the state at t = 4 is physical everywhere without any floor, the front has travelled
    at nearly the speed of light (r_out + t = 5 bounds it), the solution keeps the symmetry of the data."""
    r = run_blast(0.1)
    P, rho, st = r["P"], r["rho"], r["stats"]
    assert np.isfinite(P).all() and r["uniform_z"]
    assert st["n_c2p_fail"] == 0 and st["n_cons_floor"] == 0 and st["n_prim_floor"] == 0
    assert P.min() > 1e-5 and rho.min() > 3e-5
    fx, fy = _front(P, 1e-4)
    assert 4.5 < fx <= 5.0 + 0.06 and 4.5 < fy <= 5.0 + 0.06
    assert np.abs(P - P[:, ::-1]).max() < 0.03 * P.max() and np.abs(P - P[::-1, :]).max() < 0.03 * P.max()
    assert 0.0 < r["flagged"] < 0.3 * r["zones"]


@pytest.mark.parametrize("dmp_M", [0.0, 1.1])
def test_blast_wave_strong_field_stays_physical_with_fofc(dmp_M):
    """B_x = 1 (Figure 5): with FOFC or FOFC+DMP (M = 1.1) no inversion fails and no cell
    is reset to atmosphere."""
    r = run_blast(1.0, dmp_M=dmp_M)
    assert np.isfinite(r["P"]).all() and r["stats"]["n_c2p_fail"] == 0
    assert r["rho"].min() > 1e-8 and r["P"].min() > 0.0 and r["P"].max() < 1.0
    lor = np.sqrt(1.0 + r["ux"] ** 2 + r["uy"] ** 2)
    assert lor.max() < 200.0


def test_blast_wave_strong_field_without_fofc_disintegrates():
    """'A test with WENOZ quickly disintegrated due to primitive inversion failures resetting
    the solution to atmosphere' - the same run with the FOFC switched off."""
    r = run_blast(1.0, fofc=0)
    assert r["stats"]["n_c2p_fail"] > 100
    assert int((r["rho"] <= 1.0000001e-10).sum()) > 0


# ---------------------------------------------------------------- TOV star, Cowling approximation
def run_tov(n=32, nb=2, half_width=12.8, t_end=600.0, cfl=0.4, every=10, amp=-0.024, **override):
    """central density (mean of the 8 cells around the origin) every `every` steps."""
    import torch
    w, d, M, R = tovkit.tov_lattice(ak.shapes(nb ** 3, n), n, nb, half_width, amp=amp)
    w["params"].update(override)
    dt = cfl * d
    w["dt_fofc"] = dt
    nbr = lattice_nbr((nb, nb, nb), (False, False, False))
    nchunks = int(np.ceil(t_end / (dt * every)))
    h = nb // 2
    corner = [((bz * nb + by) * nb + bx, NG + (n - 1 if bz < h else 0), NG + (n - 1 if by < h else 0),
               NG + (n - 1 if bx < h else 0)) for bz in (h - 1, h) for by in (h - 1, h) for bx in (h - 1, h)]
    idx = tuple(torch.tensor(q) for q in zip(*corner))
    t, rc = [0.0], []
    with gpukit.GpuStage(w) as g:
        ak.ak_set_neighbors(g.ctx, nbr)
        g.con2prim()
        rc.append(float(g.W[0][idx].mean()))
        mass0 = float(sum(u.sum() for u in [g.U[0][:, NG:NG + n, NG:NG + n, NG:NG + n]])) * d ** 3
        gflag = torch.zeros_like(g.flag)
        for c in range(nchunks):
            ak.ak_advance(g.ctx, 3, every, dt, (1, 1, 1), g.U, g.Bf, g.W, gflag)
            rc.append(float(g.W[0][idx].mean()))
            t.append((c + 1) * every * dt)
        torch.cuda.synchronize()
        mass1 = float(g.U[0][:, NG:NG + n, NG:NG + n, NG:NG + n].sum()) * d ** 3
        stats = g.stats()
        rho_max = float(max(x.max() for x in [g.W[0]]))
    return dict(t=np.array(t), rho_c=np.array(rc), M=M, R=R, mass0=mass0, mass1=mass1, stats=stats, rho_max=rho_max)


def peak_frequency_khz(t, y, fmin=1.0, fmax=8.0):
    """frequency of the largest spectral peak of the detrended, Hann-windowed signal (zero-padded FFT)."""
    y = y - np.polyval(np.polyfit(t, y, 1), t)
    y = y * np.hanning(y.size)
    npad = 16 * y.size
    f = np.fft.rfftfreq(npad, d=(t[1] - t[0]) * tovkit.MSUN_S) / 1e3
    a = np.abs(np.fft.rfft(y, npad))
    sel = (f > fmin) & (f < fmax)
    return float(f[sel][np.argmax(a[sel])])


def test_tov_star_stage_equals_oracle():
    """one RHS stage on the perturbed star (2x2x2 blocks of 16^3, surface and atmosphere included):
    the CUDA path equals the oracle element for element."""
    from oracle import pyoracle as orc
    n, nb = 16, 2
    w, d, M, R = tovkit.tov_lattice(ak.shapes(nb ** 3, n), n, nb, 12.8)
    w["dt_fofc"] = 0.4 * d
    U_in = [u.copy() for u in w["U"]]
    o = orc.rhs(orc.make_params(**w["params"]), w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], w["dt_fofc"])
    with gpukit.GpuStage(w) as g:
        g.rhs()
        r = g.result()
    gpukit.assert_parity(r, o, U_in, "TOV")
    assert np.count_nonzero(o["status"]) > 0                       # the atmosphere is floored


def test_tov_star_oscillates_at_the_cowling_frequencies():
    """P:254-268, Figure 7: HLLE + PPM4, CFL 0.4, rho_atm = 1e-10, f_thr = 1.01, T_atm = 1e-8, U = -0.024,
    frozen spacetime.  Here 64^3 cells of 0.4 M_sun (the paper: 0.2 with SMR and octant symmetry) as
    2x2x2 blocks with exchange, outflow boundaries at +-12.8, t = 320 M_sun (about four periods; the
    copy boundary so close to the star lets infalling atmosphere grow after t ~ 450, which the paper's
    far boundary avoids).  The central density oscillates about its initial value at the fundamental
    radial mode and its first overtone of this model in the Cowling approximation (2.706 and 4.547 kHz,
    Font et al. 2002 - 'as predicted by perturbation theory'; the paper finds them within 47 and
    20 Hz at twice the resolution and ten times the duration); FOFC changes nothing visible."""
    a = run_tov(t_end=320.0)
    b = run_tov(t_end=320.0, fofc=0)
    assert abs(a["M"] - 1.400) < 1e-3 and abs(a["R"] - 9.59) < 1e-2
    rc = a["rho_c"] / 1.28e-3
    assert abs(rc[0] - 1.0) < 5e-3 and abs(rc.mean() - 1.0) < 0.02
    assert 0.01 < rc.max() - 1.0 < 0.1 and 0.01 < 1.0 - rc.min() < 0.1
    F = peak_frequency_khz(a["t"], a["rho_c"])
    H1 = peak_frequency_khz(a["t"], a["rho_c"], 3.6, 8.0)
    assert abs(F - 2.706) < 0.15 and abs(H1 - 4.547) < 0.3, (F, H1)
    assert abs(a["mass1"] / a["mass0"] - 1.0) < 5e-4 and a["stats"]["n_c2p_fail"] == 0
    assert np.abs(a["rho_c"] - b["rho_c"]).max() < 2e-3 * 1.28e-3
