"""Pins of the oracle's piecewise-polytropic hybrid EOS (reading R29, pins T31).
None of them re-types the oracle's formulas: the cold curve is checked against the first law by
numerical quadrature, the sound speed against a numerical adiabatic derivative, the conserved
variables against the tensor definition with h = 1 + eps + P/rho, the whole path against the
(separately pinned) ideal gas in the two limits where the hybrid EOS must reduce to it, and
con2prim against prim2cons by round trip."""
import copy

import numpy as np
import pytest
from scipy import integrate

import helpers as H
from oracle import pyoracle as po
from paper_2409_10384_b200 import workloads as wl

# three segments spanning the densities of the paper's stars (rho_c = 1.28e-3)
HYB = dict(K0=100.0, gammas=[2.0, 2.6, 2.2], rho_breaks=[4e-4, 1.5e-3], gamma_th=1.75)


def _par(**kw):
    d = dict(rho_atm=1e-30, T_atm=1e-30, f_thr=1.0, eos_hybrid=HYB)
    d.update(kw)
    return po.make_params(**d)


def test_T31_cold_curve_continuity_exponents_first_law():
    par = _par()
    Pc = lambda r: po.eos_point(par, r, 1.0)[3]
    ec = lambda r: po.eos_point(par, r, 1.0)[4]
    # first segment is P = K0 rho^Gamma0 by definition
    for r in (1e-8, 3e-5, 3.9e-4):
        assert np.isclose(Pc(r), HYB["K0"] * r ** HYB["gammas"][0], rtol=1e-14)
    # P_c and eps_c continuous at the breakpoints
    for rb in HYB["rho_breaks"]:
        lo, hi = rb * (1 - 1e-13), rb * (1 + 1e-13)
        assert abs(Pc(hi) - Pc(lo)) <= 1e-11 * Pc(rb)
        assert abs(ec(hi) - ec(lo)) <= 1e-11 * ec(rb)
    # logarithmic slope = Gamma_i inside each segment
    for r, G in ((1e-4, 2.0), (8e-4, 2.6), (5e-3, 2.2)):
        sl = (np.log(Pc(r * 1.0001)) - np.log(Pc(r / 1.0001))) / (2 * np.log(1.0001))
        assert abs(sl - G) <= 1e-7
    # first law at zero temperature: eps_c(rho) = int_0^rho P_c / rho'^2 d rho'
    for r in (2e-4, 4e-4, 1e-3, 1.5e-3, 7e-3):
        pts = [b for b in HYB["rho_breaks"] if b < r]
        val, _ = integrate.quad(lambda x: Pc(x) / (x * x), 0.0, r, points=pts or None, epsabs=0, epsrel=1e-12)
        assert abs(ec(r) - val) <= 1e-10 * val


def test_T31_pressure_enthalpy_sound_speed():
    par = _par()
    rng = np.random.default_rng(31)
    for _ in range(200):
        rho = 10 ** rng.uniform(-5, -2.5)
        _, _, _, Pc, ec = po.eos_point(par, rho, 1.0)
        eps = ec * (1 + 10 ** rng.uniform(-3, 1))
        P, hm1, cs2, _, _ = po.eos_point(par, rho, eps)
        # P - P_c is the Gamma_th-law pressure of the thermal energy; h = 1 + eps + P/rho
        assert np.isclose(P - Pc, (HYB["gamma_th"] - 1) * rho * (eps - ec), rtol=1e-12)
        assert np.isclose(hm1, eps + P / rho, rtol=1e-13)
        # c_s^2 = (dP/drho at constant entropy) / h; along an adiabat d eps = P / rho^2 d rho
        def P_ad(r1):   # integrate the adiabat from rho to r1 (RK4 in eps)
            e1, r0, n = eps, rho, 8
            dr = (r1 - rho) / n
            f = lambda r, e: po.eos_point(par, r, e)[0] / (r * r)
            for _ in range(n):
                k1 = f(r0, e1); k2 = f(r0 + dr / 2, e1 + dr / 2 * k1)
                k3 = f(r0 + dr / 2, e1 + dr / 2 * k2); k4 = f(r0 + dr, e1 + dr * k3)
                e1 += dr / 6 * (k1 + 2 * k2 + 2 * k3 + k4); r0 += dr
            return po.eos_point(par, r1, e1)[0]
        d = 1e-4 * rho
        if any(abs(rho - b) < 2 * d for b in HYB["rho_breaks"]):
            continue
        dPdr = (P_ad(rho + d) - P_ad(rho - d)) / (2 * d)
        assert np.isclose(cs2, dPdr / (1 + hm1), rtol=1e-6)
        assert cs2 > 0


def test_T31_prim2cons_equals_tensor_definition():
    par = _par()
    rng = np.random.default_rng(32)
    for _ in range(200):
        g6 = H.random_spd(rng); gam = H.sym6_to_mat(g6)
        rho = 10 ** rng.uniform(-5, -2.5)
        Pc, ec = po.eos_point(par, rho, 1.0)[3:5]
        eps = ec * (1 + 10 ** rng.uniform(-2, 1))
        P = po.eos_point(par, rho, eps)[0]
        vdir = rng.normal(size=3); vdir /= np.sqrt(vdir @ gam @ vdir)
        v = vdir * rng.uniform(0, 0.95)
        B = rng.normal(size=3) * np.sqrt(rho) * 10 ** rng.uniform(-2, 0.5)
        Wl = 1 / np.sqrt(1 - v @ gam @ v)
        Uref, _, aux = H.tensor_state(1.3, rng.normal(size=3) * 0.2, g6, rho, v, P, B, None, h=1 + eps + P / rho)
        cons = po.prim2cons_eos(par, g6, [rho, *(Wl * v), P], B)
        ref = Uref[:5] / aux["sg"]
        assert np.allclose(cons, ref, rtol=1e-10, atol=1e-12 * np.abs(ref).max())


def _random_hot_state(rng, par):
    g6 = H.random_spd(rng); gam = H.sym6_to_mat(g6)
    rho = 10 ** rng.uniform(-6, -2.5)      # the causal range of this parameter set (c_s^2 < 1)
    Pc, ec = po.eos_point(par, rho, 1.0)[3:5]
    eps = ec + (ec + 1e-6) * 10 ** rng.uniform(-1, 1.5)     # hot: the thermal part survives round-off
    P = po.eos_point(par, rho, eps)[0]
    d = rng.normal(size=3); d /= np.sqrt(d @ gam @ d)
    u = d * 10 ** rng.uniform(-4, 1.3)
    bd = rng.normal(size=3); bd /= np.sqrt(bd @ gam @ bd)
    B = bd * np.sqrt(rho * 10 ** rng.uniform(-6, 2))
    return g6, gam, rho, eps, P, u, B


def test_T31_round_trip_and_master_function():
    par = _par()
    rng = np.random.default_rng(33)
    worst = 0
    for _ in range(2000):
        g6, gam, rho, eps, P, u, B = _random_hot_state(rng, par)
        _, sdet, _ = po.metric_inverse(g6)
        cons = po.prim2cons_eos(par, g6, [rho, *u, P], B)
        st, W, _, it = po.con2prim_cell(par, g6, sdet * cons, sdet * B)
        assert st == 0
        worst = max(worst, it)
        Wl = np.sqrt(1 + u @ gam @ u); B2 = B @ gam @ B
        assert abs(W[0] - rho) <= 1e-10 * rho
        assert np.sqrt((W[1:4] - u) @ gam @ (W[1:4] - u)) <= 1e-10 * np.sqrt(u @ gam @ u) * Wl ** 2
        cond = 1 + B2 / P + rho * Wl ** 2 * (1 + eps) / P
        assert abs(W[4] - P) <= 5e-11 * cond * P
        # f(mu) = 0 at mu = 1/(W h) of the state
        D, S, tau = cons[0], cons[1:4], cons[4]
        gi = np.linalg.inv(gam); r = S / D; rB = r @ B
        h = 1 + eps + P / rho
        mu = 1 / (Wl * h)
        f = po.c2p_master_eos(par, D, tau / D, r @ gi @ r, B2 / D, rB * rB / D, mu)
        assert abs(f) <= 1e-9 * mu * (1 + B2 / (rho * h)) * Wl ** 2
    assert worst <= 40


@pytest.mark.parametrize("limit", ["K0_zero", "gamma_th_equals_gamma"])
def test_T31_reduces_to_the_ideal_gas(limit):
    """K0 = 0: no cold part, T = P/rho, the ideal gas with Gamma = Gamma_th in every respect (floors
    included).  One segment with Gamma_1 = Gamma_th: P = (Gamma-1) rho eps again, only the meaning
    of T differs, so floors are kept inactive."""
    Gam = 5.0 / 3
    if limit == "K0_zero":
        hyb, tol = dict(K0=0.0, gammas=[2.5], gamma_th=Gam), 1e-13
        atm = dict(rho_atm=1e-9, T_atm=1e-6, f_thr=1.0)
    else:
        hyb, tol = dict(K0=0.3, gammas=[Gam], gamma_th=Gam), 1e-9
        atm = dict(rho_atm=1e-30, T_atm=1e-30, f_thr=1.0)
    pi = po.make_params(gamma_ad=Gam, **atm)
    ph = po.make_params(gamma_ad=1.1, eos_hybrid=hyb, **atm)     # gamma_ad must be ignored
    rng = np.random.default_rng(34)
    for it in range(400):
        g6 = H.random_spd(rng); gam = H.sym6_to_mat(g6)
        rho = 10 ** rng.uniform(-8, 0)
        Tmin = 1e-5 if limit == "K0_zero" else 0.3 * rho ** (Gam - 1) * 3   # hot: P > 3 P_c
        P = rho * max(10 ** rng.uniform(-7, 0.5), Tmin)
        d = rng.normal(size=3); d /= np.sqrt(d @ gam @ d)
        u = d * 10 ** rng.uniform(-3, 1)
        B = rng.normal(size=3) * np.sqrt(rho) * 10 ** rng.uniform(-2, 0.5)
        ci = po.prim2cons(Gam, g6, [rho, *u, P], B)
        ch = po.prim2cons_eos(ph, g6, [rho, *u, P], B)
        assert np.allclose(ch, ci, rtol=tol, atol=tol * np.abs(ci).max())
        _, sdet, _ = po.metric_inverse(g6)
        if limit == "K0_zero" and it % 4 == 0:
            ci = ci * np.array([1, 1, 1, 1, 10 ** rng.uniform(-6, 0)])   # tau floors / T floors / failures too
        si, Wi, Ui, _ = po.con2prim_cell(pi, g6, sdet * ci, sdet * B)
        sh, Wh, Uh, _ = po.con2prim_cell(ph, g6, sdet * ci, sdet * B)
        assert si == sh
        cond = (1 + (B @ gam @ B) / P + rho * (1 + u @ gam @ u) / P) if si == 0 else 1e3
        assert np.allclose(Wh, Wi, rtol=max(tol, 1e-12) * cond, atol=1e-14 * np.abs(Wi).max())
        assert np.allclose(Uh, Ui, rtol=max(tol, 1e-12) * cond, atol=1e-13 * np.abs(Ui).max())
        # one face, both solvers, with lapse and shift
        dd = it % 3
        gL = H.metric10(1.2, rng.normal(size=3) * 0.1, g6); gR = gL * (1 + 0.01 * rng.normal(size=10))
        WL = np.array([rho, *u, P, *(0.1 * rng.normal(size=2))])
        WR = WL * (1 + 0.1 * rng.uniform(-1, 1, 7))
        for rs in (0, 1):
            Fi, li = po.face_flux(pi, dd, rs, gL, gR, WL, WR, 0.05, apply_floor=True, want_lam=True)
            Fh, lh = po.face_flux(ph, dd, rs, gL, gR, WL, WR, 0.05, apply_floor=True, want_lam=True)
            assert np.allclose(Fh, Fi, rtol=100 * tol, atol=100 * tol * np.abs(Fi).max())
            assert np.allclose(lh, li, rtol=100 * tol, atol=100 * tol)


def test_T31_stage_with_K0_zero_equals_ideal_stage():
    """The whole stage (con2prim, fluxes, FOFC+DMP flags, CT, sources) on the noise block: a hybrid
    EOS without cold part gives the ideal-gas stage (same masks, dU/dt and EMFs to round-off)."""
    w = wl.make_test_noise_block(seed=11, n=8, frac=0.02)
    res = []
    for hyb in (None, dict(K0=0.0, gammas=[3.0], gamma_th=w["params"]["gamma_ad"])):
        ww = copy.deepcopy(w)
        p = dict(ww["params"]); p.update(dmp_M=1.1, recon=2, eos_hybrid=hyb, rho_atm=3e-6, T_atm=0.6, f_thr=1.0)
        if hyb:
            p["gamma_ad"] = 1.2
        res.append(po.rhs(po.make_params(**p), ww["dx"], ww["U"], ww["Bf"], ww["adm"], ww["dt_fofc"], nthreads=2))
    a, b = res
    assert np.array_equal(a["status"], b["status"]) and np.array_equal(a["flag"], b["flag"])
    assert a["flag"].any() and a["status"].any()
    for k in ("dU", "E", "W"):
        for x, y in zip(a[k], b[k]):
            assert np.allclose(y, x, rtol=1e-11, atol=1e-13 * max(np.abs(x).max(), 1e-300))


def test_T31_floors_and_atmosphere():
    par = _par(rho_atm=1e-9, T_atm=1e-4, f_thr=1.0)
    g6 = np.array([1.1, 0.05, 0, 0.9, 0.02, 1.2]); _, sdet, _ = po.metric_inverse(g6)
    Pc_atm, ec_atm = po.eos_point(par, 1e-9, 1.0)[3:5]
    # D below threshold -> atmosphere at T_atm: P = P_c(rho_atm) + rho_atm T_atm
    st, W, U, _ = po.con2prim_cell(par, g6, sdet * np.array([1e-12, 0, 0, 0, 1e-14]), [0, 0, 0])
    assert st & 1 and W[0] == 1e-9 and np.all(W[1:4] == 0) and W[4] == Pc_atm + 1e-9 * 1e-4
    assert np.isclose(U[4] / sdet, 1e-9 * (ec_atm + 1e-4 / (HYB["gamma_th"] - 1)), rtol=1e-13)
    # cold dense matter (eps = eps_c, T = 0): T floor raises P to P_c + rho T_atm, bit 16 (or the
    # equivalent tau floor, bit 2); a second pass changes nothing (a state exactly at the floor may
    # be caught again by round-off, as for the ideal gas: DESIGN.md section 4 on T_atm)
    rho = 1e-3
    Pc, ec = po.eos_point(par, rho, 1.0)[3:5]
    cons = po.prim2cons_eos(par, g6, [rho, 0.1, 0, 0, Pc], [0, 0, 0])
    st, W, U, _ = po.con2prim_cell(par, g6, sdet * cons, [0, 0, 0])
    assert st & (16 | 2) and not st & ~(16 | 2)
    assert np.isclose(W[4], Pc + rho * 1e-4, rtol=1e-9) and abs(W[0] - rho) < 1e-12
    st2, W2, U2, _ = po.con2prim_cell(par, g6, U, [0, 0, 0])
    assert st2 in (0, 16) and np.allclose(W2, W, rtol=1e-9)
    # hot matter is left alone
    P = Pc + rho * 1e-2
    cons = po.prim2cons_eos(par, g6, [rho, 0.1, 0, 0, P], [0, 0, 0])
    st, W, _, _ = po.con2prim_cell(par, g6, sdet * cons, [0, 0, 0])
    assert st == 0 and np.isclose(W[4], P, rtol=1e-10)
