"""Round-2 pins of the four oracle parts that had none ("What's weak" #2).  CPU only.

Every expectation below comes from mathematics, not from the oracle's text:
  * WENO-Z nonlinear weights: the literal alpha_k = d_k [1 + (tau_5 / (beta_k + eps))^2] of Borges et
    al. 2008 evaluated in exact rational arithmetic;
  * CT upwind sense (Gardiner & Stone 2005; "upwind constrained transport"): for a flow that is
    supersonic towards one corner the corner EMF is the EMF of the doubly-upwind cell, whatever the
    other three cells hold;
  * face-state floor ("after reconstruction"): closed-form floored states put through the
    tensor definition of the flux;
  * signal speeds with B != 0, v != 0, curved metric with shift (reading R18): a bound on, and for
    propagation perpendicular to b equal to, the extreme eigenvalues of the numerical 7x7 flux Jacobian
    built from T^{mu nu}, *F^{mu nu} (tests/helpers.py; Eqs. 2, 3, 5, 7).
Each docstring names the one-line mutation of the oracle the test was seen to fail on.
"""
import math
from fractions import Fraction as Fr

import numpy as np
import pytest

import helpers as H
import stagekit as sk
from oracle import pyoracle as po
from paper_2409_10384_b200 import workloads as wl

NG = sk.NG


# ------------------------------------------------------------------------------------------------
# (a) WENO-Z: literal nonlinear weights in exact arithmetic
# ------------------------------------------------------------------------------------------------
def _wenoz_exact(q):
    """q^+ at the right face of the centre cell, SURVEY S:408-413 as printed, in Fractions.
    beta_k: Jiang-Shu; tau_5 = |beta_0 - beta_2|; alpha_k = d_k [1 + (tau_5/(beta_k + eps))^2]."""
    qmm, qm1, q0, qp1, qpp = (Fr(float(x)) for x in q)
    eps = Fr(1e-40)
    p = [(2 * qmm - 7 * qm1 + 11 * q0) / 6, (-qm1 + 5 * q0 + 2 * qp1) / 6, (2 * q0 + 5 * qp1 - qpp) / 6]
    b = [Fr(13, 12) * (qmm - 2 * qm1 + q0) ** 2 + Fr(1, 4) * (qmm - 4 * qm1 + 3 * q0) ** 2,
         Fr(13, 12) * (qm1 - 2 * q0 + qp1) ** 2 + Fr(1, 4) * (qm1 - qp1) ** 2,
         Fr(13, 12) * (q0 - 2 * qp1 + qpp) ** 2 + Fr(1, 4) * (3 * q0 - 4 * qp1 + qpp) ** 2]
    tau5 = abs(b[0] - b[2])
    d = [Fr(1, 10), Fr(6, 10), Fr(3, 10)]
    a = [d[k] * (1 + (tau5 / (b[k] + eps)) ** 2) for k in range(3)]
    return sum(a[k] * p[k] for k in range(3)) / sum(a)


def _ulp(x):
    return math.ulp(max(abs(float(x)), 1e-300))


def _wenoz_cases():
    rng = np.random.default_rng(2409)
    cases = [np.array([0, 0, 0, 1, 1.0]), np.array([1, 1, 0, 0, 0.0]), np.array([0, 0, 1, 1, 1.0]),
             np.array([0, 1, 2, 3, 3.5]),                       # kink
             np.array([0, 1, 2, 2, 1.0]), np.array([1.0, 1.0, 1.0, 1.0, 1.0]),
             np.array([3.0, 2.0, 1.5, 1.4, 1.39])]
    for _ in range(300):                                         # O(1) random stencils
        cases.append(rng.normal(size=5))
    for _ in range(200):                                         # near-constant data: beta ~ 1e-2 .. 1e-30
        cases.append(1.0 + 10.0 ** rng.uniform(-15, -1) * rng.normal(size=5))
    for _ in range(200):                                         # tiny magnitudes: beta comparable with eps = 1e-40
        cases.append(10.0 ** rng.uniform(-22, -17) * rng.normal(size=5))
    for _ in range(100):                                         # 12 decades of contrast across the stencil
        cases.append(10.0 ** rng.uniform(-12, 0, size=5))
    return cases


def test_wenoz_weights_equal_literal_borges_formula():
    """Oracle kind 2 against alpha_k = d_k [1 + (tau_5/(beta_k + eps))^2], p = 2, eps = 1e-40, in exact
    rationals.  Licenses the oracle's one-reciprocal evaluation of the three ratios tau_5/beta_k
    (oracle/point.cpp) as a rounding-level rearrangement.  Seen to fail on: 13/12 -> 1 in beta_0;
    exponent 2 -> 1 (r0 * r0 -> r0); d = (0.1, 0.6, 0.3) -> (0.3, 0.6, 0.1); eps 1e-40 -> 1e-6;
    tau5 = |b0 - b2| -> |b0 - b1|.

    Tolerance: the candidate values p_k carry up to (2+7+11)/6 rounding errors of size ulp(max|q|) and the
    convex combination a few more: 16 ulp(max|q|) in all; the weights' own rounding (relative 1e-15) only
    moves the result by that fraction of the spread of the p_k."""
    worst = 0.0
    for q in _wenoz_cases():
        qm, qp = po.reconstruct(2, q)
        ex_p = _wenoz_exact(q)
        ex_m = _wenoz_exact(q[::-1])             # left face = mirror image ("q^- by mirror image")
        tol = 16 * _ulp(np.abs(q).max())
        for got, ex in ((qp, ex_p), (qm, ex_m)):
            err = abs(Fr(got) - ex)
            worst = max(worst, float(err / Fr(tol)))
            assert err <= tol, (q, got, float(ex))
    assert worst > 0.0


def test_wenoz_reduces_to_linear_weights_and_to_one_stencil():
    """Limits of the literal formula: beta_0 = beta_2 -> tau_5 = 0 -> the linear fifth-order weights; a
    step inside the right part of the stencil -> the smooth left stencil takes over (ENO property)."""
    q = np.array([0.0, 0.0, 0.0, 1.0, 1.0])      # step between cells i and i+1
    qm, qp = po.reconstruct(2, q)
    # only stencil 0 (cells i-2..i) is smooth: beta_0 = 0, so alpha_0 / alpha_k ~ (tau/eps)^2: q^+ = p_0 = 0
    assert abs(qp) <= 1e-30 and abs(qm) <= 1e-30
    q = np.array([1.0, 4.0, 9.0, 4.0, 1.0])      # symmetric: beta_0 = beta_2, linear weights
    _, qp = po.reconstruct(2, q)
    p = [(2 * 1 - 7 * 4 + 11 * 9) / 6, (-4 + 5 * 9 + 2 * 4) / 6, (2 * 9 + 5 * 4 - 1) / 6]
    assert abs(qp - (0.1 * p[0] + 0.6 * p[1] + 0.3 * p[2])) <= 1e-14


# ------------------------------------------------------------------------------------------------
# (b) CT: the upwind sense (Gardiner & Stone 2005)
# ------------------------------------------------------------------------------------------------
def _supersonic_block(n, comp, sa, sb, seed):
    """Flat space, uniform densitised B~, per-cell random cold states whose velocity components along
    the two axes (a, b) cyclic after `comp` are supersonic with signs (sa, sb)."""
    a, b = (comp + 1) % 3, (comp + 2) % 3
    nt = n + 2 * NG
    rng = np.random.default_rng(seed)
    v = np.zeros((3, nt, nt, nt))
    v[a] = sa * rng.uniform(0.55, 0.65, (nt, nt, nt))
    v[b] = sb * rng.uniform(0.55, 0.65, (nt, nt, nt))
    v[comp] = rng.uniform(-0.1, 0.1, (nt, nt, nt))
    lor = 1.0 / np.sqrt(1.0 - (v ** 2).sum(axis=0))
    rho = rng.uniform(0.5, 2.0, (nt, nt, nt))
    T = 10.0 ** rng.uniform(-4, -3, (nt, nt, nt))

    def prim(x, y, z):
        return rho, [lor * v[0], lor * v[1], lor * v[2]], rho * T
    Bu = np.array([0.011, -0.02, 0.015])
    w = sk.build_block(n, 0.1, (0.0, 0.0, 0.0), sk.flat_metric, prim, B_uniform=Bu, gamma_ad=5.0 / 3)
    # cell-centred EMF  E_c = -(v^a B^b - v^b B^a)  (alpha = 1, beta = 0, sqrt(gamma) = 1)
    Ec = -(v[a] * Bu[b] - v[b] * Bu[a])
    return w, Ec


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("sa,sb", [(1, 1), (-1, -1), (1, -1), (-1, 1)])
def test_ct_corner_emf_is_the_doubly_upwind_cell_for_supersonic_flow(comp, sa, sb):
    """GS05 upwinding: the gradient (E_c - E_face) that enters a corner is taken from the cell the mass
    flux comes from.  With donor-cell states and HLLE every face EMF of a flow supersonic towards
    (+a,+b) is the upwind cell's own -v x B~ (T6: all speeds > 0 => F = F^L), and the corner formula of
    S:449-453 must then collapse to the EMF of the doubly-upwind cell (ia-1, ib-1) alone:
        1/4 [e(ia-1,ib) + 2 e(ia-1,ib-1) + e(ia,ib-1)] + 1/4 [(e(ia-1,ib-1) - e(ia-1,ib-1)) ... ] = e(ia-1,ib-1)
    for ANY states in the other three cells (uniform B~, so face and cell-centred B agree).  The other
    sign pairs select (ia,ib), (ia-1,ib), (ia,ib-1).
    Seen to fail on: `wgt` in oracle/stage.cpp returning 0 for F_D > 0 and 1 for F_D < 0 (w <-> 1-w), for
    every (comp, signs); on the sign of Ebf flipped.  (A weight read at the wrong face survives here, all
    mass fluxes having one sign: that is what the shear-flow test below is for.)"""
    n = 6
    w, Ec = _supersonic_block(n, comp, sa, sb, seed=100 + 10 * comp + (sa > 0) * 2 + (sb > 0))
    par = po.make_params(nmb=1, n=n, gamma_ad=5.0 / 3, rho_atm=1e-12, T_atm=1e-10, recon=0, riemann=1, fofc=0)
    r = po.rhs(par, w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], 0.01, want_flux=True)
    assert not r["status"].any()
    a, b = (comp + 1) % 3, (comp + 2) % 3
    # mass fluxes really have the intended signs on every computed face
    for d, s in ((a, sa), (b, sb)):
        FD = r["flux"][7 * d][0]
        sl = [slice(NG - 1, NG + n + 1)] * 3          # transverse range [is-1, ie+1]
        sl[2 - d] = slice(NG - 1, NG + n + 2)         # normal range [is-1, ie+2]
        assert (s * FD[tuple(sl)] > 0).all()
    E = r["E"][comp][0]
    worst = 0.0
    for ic in range(NG, NG + n):                     # along the edge
        for ib in range(NG, NG + n + 1):
            for ia in range(NG, NG + n + 1):
                idx = [0, 0, 0]                       # (x, y, z) indices of the edge
                idx[a], idx[b], idx[comp] = ia, ib, ic
                got = E[idx[2], idx[1], idx[0]]
                cu = [0, 0, 0]                        # the doubly-upwind cell
                cu[a] = ia - 1 if sa > 0 else ia
                cu[b] = ib - 1 if sb > 0 else ib
                cu[comp] = ic
                want = Ec[cu[2], cu[1], cu[0]]
                worst = max(worst, abs(got - want))
                assert abs(got - want) <= 2e-12 * np.abs(Ec).max(), (comp, sa, sb, ia, ib, ic, got, want)
    assert worst < 2e-12 * np.abs(Ec).max()


def _shear_block(n, comp, uni, s_uni, seed, reseed_from=None, seed2=0):
    """As _supersonic_block, but only the velocity along axis `uni` (one of the two axes cyclic after
    comp) has one sign everywhere; along the other axis `alt` the sign alternates with the index along
    `uni` (a shear flow: every row keeps one sign, neighbouring rows differ).  With reseed_from = r the
    states of all cells whose uni-index is >= r are drawn again from seed2 (same signs)."""
    a, b = (comp + 1) % 3, (comp + 2) % 3
    alt = b if uni == a else a
    nt = n + 2 * NG
    ax = lambda d: 2 - d                                  # array axis of direction d ([z][y][x])
    idx_uni = np.arange(nt).reshape([nt if q == ax(uni) else 1 for q in range(3)])
    sign_alt = np.where((idx_uni // 1) % 2 == 0, 1.0, -1.0) * np.ones((nt, nt, nt))

    def draw(seed_):
        rng = np.random.default_rng(seed_)
        v = np.zeros((3, nt, nt, nt))
        v[uni] = s_uni * rng.uniform(0.55, 0.65, (nt, nt, nt))
        v[alt] = sign_alt * rng.uniform(0.55, 0.65, (nt, nt, nt))
        v[comp] = rng.uniform(-0.1, 0.1, (nt, nt, nt))
        rho = rng.uniform(0.5, 2.0, (nt, nt, nt))
        T = 10.0 ** rng.uniform(-4, -3, (nt, nt, nt))
        return v, rho, T
    v, rho, T = draw(seed)
    if reseed_from is not None:
        v2, rho2, T2 = draw(seed2)
        m = (idx_uni >= reseed_from) * np.ones((nt, nt, nt), dtype=bool)
        v = np.where(m[None], v2, v); rho = np.where(m, rho2, rho); T = np.where(m, T2, T)
    lor = 1.0 / np.sqrt(1.0 - (v ** 2).sum(axis=0))

    def prim(x, y, z):
        return rho, [lor * v[0], lor * v[1], lor * v[2]], rho * T
    return sk.build_block(n, 0.1, (0.0, 0.0, 0.0), sk.flat_metric, prim, B_uniform=np.array([0.011, -0.02, 0.015]),
                          gamma_ad=5.0 / 3)


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("which", [0, 1])
@pytest.mark.parametrize("s_uni", [1, -1])
def test_ct_corner_emf_ignores_the_downwind_row_in_a_shear_flow(comp, which, s_uni):
    """Which face's mass flux selects which gradient ("taken at x-face (i, j) for row j and at
    (i, j-1) for row j-1").  Flow supersonic along `uni` with one sign, supersonic along the other axis
    with a sign that alternates from row to row.  Information cannot travel upstream along `uni`: with
    donor cell + HLLE every face flux is its upwind cell's, and a corner EMF on the upstream side of a row
    must not change when the states of that row (and everything downstream of it) change.  If a weight
    were read from the neighbouring row's face, the gradient taken in the downwind row would no longer
    cancel its face EMF and the dependence appears.
    Seen to fail on: wp = wgt(FaD(ia, ib, ic)) (row ib instead of ib-1) and w2p = wgt(FbD(ia, ib - 1, ic))
    (face (ia, ib-1) instead of (ia-1, ib)) in oracle/stage.cpp; on w <-> 1-w."""
    n = 6
    a, b = (comp + 1) % 3, (comp + 2) % 3
    uni = (a, b)[which]
    jr = NG + 3                                              # first re-drawn row
    par = po.make_params(nmb=1, n=n, gamma_ad=5.0 / 3, rho_atm=1e-12, T_atm=1e-10, recon=0, riemann=1, fofc=0)
    E = []
    for reseed in (None, jr):
        w = _shear_block(n, comp, uni, s_uni, seed=300 + comp, reseed_from=reseed, seed2=999)
        r = po.rhs(par, w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], 0.01, want_flux=True)
        assert not r["status"].any()
        FD = r["flux"][7 * uni][0]
        sl = [slice(NG - 1, NG + n + 1)] * 3
        sl[2 - uni] = slice(NG - 1, NG + n + 2)
        assert (s_uni * FD[tuple(sl)] > 0).all()
        alt = b if uni == a else a
        FDa = r["flux"][7 * alt][0]
        sl = [slice(NG - 1, NG + n + 1)] * 3
        sl[2 - alt] = slice(NG - 1, NG + n + 2)
        assert (FDa[tuple(sl)] > 0).any() and (FDa[tuple(sl)] < 0).any()
        E.append(r["E"][comp][0])
    # edges by their index along `uni`: edge index e lies between rows e-1 and e
    ax_uni = 2 - uni
    sel = lambda arr, lo, hi: np.take(arr, np.arange(lo, hi), axis=ax_uni)
    inner = [slice(NG, NG + n + 1)] * 3
    inner[2 - comp] = slice(NG, NG + n)
    A0, A1 = E[0][tuple(inner)], E[1][tuple(inner)]          # edges of interior cells; uni-index offset NG
    k = jr - NG                                              # position of edge index jr in the cut array
    if s_uni > 0:    # rows >= jr changed; edges with index <= jr see only rows < jr
        same, diff = (sel(A0, 0, k + 1), sel(A1, 0, k + 1)), (sel(A0, k + 1, n + 1), sel(A1, k + 1, n + 1))
    else:            # flow towards -uni: edge e depends on rows >= e; edges <= jr-1... all depend on changed rows
        same, diff = None, (sel(A0, 0, n + 1), sel(A1, 0, n + 1))
    scale = np.abs(A0).max()
    if same is not None:
        assert np.abs(same[0] - same[1]).max() <= 1e-13 * scale
        assert np.abs(diff[0] - diff[1]).max() > 1e-4 * scale
    else:
        # upstream is +uni: edges with index > jr-1 ... take the mirror statement: re-draw rows < jr instead
        w = _shear_block(n, comp, uni, s_uni, seed=300 + comp)
        v0 = po.rhs(par, w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], 0.01)["E"][comp][0][tuple(inner)]
        # keep rows >= jr, replace rows < jr: build by swapping the roles of the two seeds
        w2 = _shear_block(n, comp, uni, s_uni, seed=999, reseed_from=jr, seed2=300 + comp)
        v1 = po.rhs(par, w2["dx"], [u.copy() for u in w2["U"]], w2["Bf"], w2["adm"], 0.01)["E"][comp][0][tuple(inner)]
        # edges with index >= jr see only rows >= jr (unchanged); edges below differ
        assert np.abs(sel(v0, k, n + 1) - sel(v1, k, n + 1)).max() <= 1e-13 * scale
        assert np.abs(sel(v0, 0, k) - sel(v1, 0, k)).max() > 1e-4 * scale


def test_ct_zero_mass_flux_takes_the_half_half_mean():
    """F^x_D == 0 exactly on every x-face (fluid at rest, uniform density, shift along y only), so the
    x-face weights are 1/2-1/2 and the corner value must not prefer a side: the mirror image of the
    block in x (cells i -> nt-1-i, faces i -> nt-i, B~^x -> -B~^x) must give the mirror image of the
    EMFs, E_z -> -E_z (an axial vector), at the mirrored edges.  B~^x varies from face to face in x and
    y, so E_c - E^{yf} differs between the two columns of every edge and the weights matter.
    Seen to fail on: wgt(0) = 1 (or 0) instead of 1/2 in oracle/stage.cpp."""
    n = 6
    nt = n + 2 * NG
    rng = np.random.default_rng(77)
    bxf = rng.uniform(0.5, 1.5, (nt, nt + 1))           # B~^x on x-faces: [j][i_face], uniform in z
    byf = rng.uniform(0.1, 0.3, (nt + 1, nt))           # B~^y on y-faces: [j_face][i]

    def metric(x, y, z):
        o = np.ones_like(x); zr = np.zeros_like(x)
        return o, [zr, -0.3 * o, zr], [o, zr, zr, o, zr, o], [zr] * 6

    def prim(x, y, z):
        o = np.ones_like(x)
        return o, [0 * o, 0 * o, 0 * o], 0.1 * o

    def run(mirror):
        w = sk.build_block(n, 0.1, (0, 0, 0), metric, prim, B_uniform=np.zeros(3))
        bx = -bxf[:, ::-1] if mirror else bxf
        by = byf[:, ::-1] if mirror else byf
        w["Bf"][0][0, :, :, :nt + 1] = bx[None, :, :]
        w["Bf"][1][0] = by[None, :, :]
        bcx = 0.5 * (bx[:, :-1] + bx[:, 1:]); bcy = 0.5 * (by[:-1, :] + by[1:, :])
        one = np.ones((nt, nt, nt))
        g = [one, 0 * one, 0 * one, one, 0 * one, one]
        D, S, tau = wl._prim2cons_np(2.0, g, one, [0 * one] * 3, 0.1 * one, [bcx[None] * one, bcy[None] * one, 0 * one])
        for v, a in enumerate((D, S[0], S[1], S[2], tau)):
            w["U"][v][0] = a
        par = po.make_params(nmb=1, n=n, gamma_ad=2.0, rho_atm=1e-12, T_atm=1e-10, recon=0, riemann=1, fofc=0)
        r = po.rhs(par, w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], 0.01, want_flux=True)
        assert not r["status"].any()
        s = slice(NG, NG + n)
        assert (r["flux"][0][0][s, NG:NG + n + 1, NG:NG + n + 1] == 0.0).all()      # F^x_D == 0 exactly
        assert (r["flux"][7][0][s, NG:NG + n + 1, NG - 1:NG + n + 1] > 0.0).all()   # F^y_D > 0
        return r["E"][2][0][s, NG:NG + n + 1, :nt + 1]                                # [k][j_edge][i_edge]
    a, bm = run(False), run(True)
    assert np.abs(a).max() > 0.1
    ia = np.arange(NG, NG + n + 1)
    diff = a[:, :, ia] + bm[:, :, nt - ia]
    assert np.abs(diff).max() <= 4e-16 * np.abs(a).max(), np.abs(diff).max()


# ------------------------------------------------------------------------------------------------
# (c) face-state floor
# ------------------------------------------------------------------------------------------------
def test_face_floor_closed_forms():
    """L = R, so the numerical flux is the physical flux of the (floored) state (T6), which the tensor
    definition gives for the closed-form floored state:
      rho < f_thr rho_atm          -> (rho_atm, u = 0, P = rho_atm T_atm);  B untouched;
      else T = P/rho < T_atm       -> P = rho T_atm, rho and u untouched;
      else                         -> unchanged; and apply_floor = 0 leaves all three alone.
    Seen to fail on: dropping the T branch of face_floor (oracle/point.cpp); atmosphere keeping its
    velocity (prim[1..3] not zeroed); threshold rho_atm instead of f_thr * rho_atm; P_atm = T_atm."""
    rng = np.random.default_rng(31)
    Gam, rho_atm, T_atm, f_thr = 5.0 / 3, 1e-6, 1e-3, 0.25
    par = po.make_params(gamma_ad=Gam, rho_atm=rho_atm, T_atm=T_atm, f_thr=f_thr)
    n_case = [0, 0, 0]
    for trial in range(300):
        g6 = H.random_spd(rng); gam = H.sym6_to_mat(g6)
        alpha = rng.uniform(0.4, 1.4); beta = rng.normal(size=3) * 0.2
        kind = trial % 3
        if kind == 0:      # below the density threshold (between 0.01 and 0.99 of it)
            rho = f_thr * rho_atm * rng.uniform(0.01, 0.99); P = rho * 10 ** rng.uniform(-5, 0)
        elif kind == 1:    # dense enough, too cold
            rho = rho_atm * 10 ** rng.uniform(0, 5); P = rho * T_atm * rng.uniform(0.0, 0.99)
        else:              # nothing to do (also: between f_thr rho_atm and rho_atm, warm)
            rho = f_thr * rho_atm * 10 ** rng.uniform(0.01, 5); P = rho * T_atm * 10 ** rng.uniform(0.01, 2)
        v = rng.normal(size=3); v *= rng.uniform(0.05, 0.8) / np.sqrt(v @ gam @ v)
        B = rng.normal(size=3) * np.sqrt(rho_atm) * 10 ** rng.uniform(-1, 1)
        lor = 1.0 / np.sqrt(1.0 - v @ gam @ v)
        if kind == 0:
            exp = (rho_atm, np.zeros(3), rho_atm * T_atm)
        elif kind == 1:
            exp = (rho, v, rho * T_atm)
        else:
            exp = (rho, v, P)
        n_case[kind] += 1
        _, F_exp, aux = H.tensor_state(alpha, beta, g6, exp[0], exp[1], exp[2], B, Gam)
        _, F_raw, _ = H.tensor_state(alpha, beta, g6, rho, v, P, B, Gam)
        m10 = H.metric10(alpha, beta, g6)
        sg = aux["sg"]
        for d in range(3):
            t1, t2 = (d + 1) % 3, (d + 2) % 3
            Wp = np.array([rho, *(lor * v), P, sg * B[t1], sg * B[t2]])
            for riemann in (0, 1):
                Fo = po.face_flux(par, d, riemann, m10, m10, Wp, Wp, sg * B[d], apply_floor=True)
                ref = F_exp[d][H.slots(d)]
                assert np.allclose(Fo, ref, rtol=1e-10, atol=1e-12 * np.abs(F_exp[d]).max()), (kind, d, Fo, ref)
                Fn = po.face_flux(par, d, riemann, m10, m10, Wp, Wp, sg * B[d], apply_floor=False)
                refn = F_raw[d][H.slots(d)]
                assert np.allclose(Fn, refn, rtol=1e-10, atol=1e-12 * np.abs(F_raw[d]).max())
                if kind < 2:   # the floor really changed the flux, so the comparison above discriminates
                    assert not np.allclose(Fo, refn, rtol=1e-6, atol=1e-12 * np.abs(F_raw[d]).max())
    assert min(n_case) == 100


def test_face_floor_acts_on_each_side_separately():
    """Only the side that needs it is floored: L cold, R fine  =>  flux = Riemann flux of (floored L, R),
    which for a supersonic left-to-right flow is the physical flux of the floored L state."""
    Gam, rho_atm, T_atm = 5.0 / 3, 1e-8, 1e-3
    par = po.make_params(gamma_ad=Gam, rho_atm=rho_atm, T_atm=T_atm, f_thr=1.0)
    flat = H.metric10(1.0, [0, 0, 0], [1, 0, 0, 1, 0, 1.0])
    v = np.array([0.9, 0.0, 0.0]); lor = 1 / np.sqrt(1 - v @ v)
    WL = np.array([1.0, *(lor * v), 1e-5, 0.0, 0.0])      # T = 1e-5 < T_atm
    WR = np.array([0.5, *(lor * v), 0.5 * 2e-3, 0.0, 0.0])
    F, lam = po.face_flux(par, 0, 1, flat, flat, WL, WR, 0.0, apply_floor=True, want_lam=True)
    assert lam.min() > 0
    _, FL, _ = H.tensor_state(1.0, [0, 0, 0], [1, 0, 0, 1, 0, 1.0], 1.0, v, 1.0 * T_atm, np.zeros(3), Gam)
    assert np.allclose(F, FL[0][H.slots(0)], rtol=1e-12)


# ------------------------------------------------------------------------------------------------
# (d) signal speeds with B != 0, v != 0, curved metric with shift (reading R18)
# ------------------------------------------------------------------------------------------------
def _jacobian_eigs(alpha, beta, g6, rho, v, P, B, Gam, d):
    """eigenvalues of dF^d/dU (7x7: D~, S~_i, tau~, B~^t1, B~^t2; B^d is a parameter) by central
    differences of the tensor definitions in primitive space."""
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    x0 = np.array([rho, *v, P, B[t1], B[t2]])
    sl = H.slots(d)

    def UF(x):
        Bv = np.zeros(3); Bv[d] = B[d]; Bv[t1] = x[5]; Bv[t2] = x[6]
        U, F, _ = H.tensor_state(alpha, beta, g6, x[0], x[1:4], x[4], Bv, Gam)
        return U[sl], F[d][sl]
    dU = np.zeros((7, 7)); dF = np.zeros((7, 7))
    for c in range(7):
        hstep = 1e-6 * max(abs(x0[c]), 0.1)
        xp = x0.copy(); xm = x0.copy(); xp[c] += hstep; xm[c] -= hstep
        Up, Fp = UF(xp); Um, Fm = UF(xm)
        dU[:, c] = (Up - Um) / (2 * hstep); dF[:, c] = (Fp - Fm) / (2 * hstep)
    ev = np.linalg.eigvals(dF @ np.linalg.inv(dU))
    assert np.abs(ev.imag).max() <= 1e-5, ev          # the system is hyperbolic
    return np.sort(ev.real)


def _oracle_speeds(par, alpha, beta, g6, rho, v, P, B, d):
    gam = H.sym6_to_mat(g6)
    lor = 1.0 / np.sqrt(1.0 - v @ gam @ v)
    sg = np.sqrt(np.linalg.det(gam))
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    Wp = np.array([rho, *(lor * v), P, sg * B[t1], sg * B[t2]])
    m10 = H.metric10(alpha, beta, g6)
    _, lam = po.face_flux(par, d, 1, m10, m10, Wp, Wp, sg * B[d], want_lam=True)
    return lam[0], lam[1]


def test_speeds_bound_the_flux_jacobian_spectrum_with_B_and_v():
    """lambda_- <= min eigenvalue and lambda_+ >= max eigenvalue of the 7x7 numerical dF/dU for random
    magnetised moving states in random metrics with shift (R18 is a *bound*: it replaces the quartic
    fast-wave dispersion relation by its isotropic upper envelope a^2 = c_s^2 + v_A^2 - c_s^2 v_A^2).
    Seen to fail on: a2 = cs2 (v_A dropped) in side_state (oracle/point.cpp); '- bet[d]' -> '+ bet[d]';
    gdd taken from the covariant metric; alp missing from the first term."""
    rng = np.random.default_rng(41)
    par = po.make_params(rho_atm=1e-30, T_atm=1e-30)
    slack = 0.0
    for _ in range(40):
        g6 = H.random_spd(rng); gam = H.sym6_to_mat(g6)
        alpha = rng.uniform(0.4, 1.3); beta = rng.normal(size=3) * 0.2
        Gam = rng.choice([4.0 / 3, 5.0 / 3]); par.gamma_ad = Gam
        rho = 1.0; P = 10 ** rng.uniform(-2, 0.5)
        v = rng.normal(size=3); v *= rng.uniform(0.05, 0.85) / np.sqrt(v @ gam @ v)
        B = rng.normal(size=3) * 10 ** rng.uniform(-0.7, 0.7)
        for d in range(3):
            ev = _jacobian_eigs(alpha, beta, g6, rho, v, P, B, Gam, d)
            lm, lp = _oracle_speeds(par, alpha, beta, g6, rho, v, P, B, d)
            assert lm <= ev[0] + 5e-6 and lp >= ev[-1] - 5e-6, (lm, lp, ev)
            slack = max(slack, ev[0] - lm, lp - ev[-1])
    assert slack > 1e-3        # a bound, not an identity: oblique propagation is strictly inside


def test_speeds_exact_for_propagation_perpendicular_to_b():
    """For b^mu k_mu = 0 (here B^d = 0 and B_i v^i = 0, so b^0 = 0 and b^d = 0) the fast speed in the fluid
    frame is exactly sqrt(c_s^2 + v_A^2 - c_s^2 v_A^2), so lambda_+- must EQUAL the extreme eigenvalues
    (finite-difference limited).  Seen to fail on: v_A^2 = b^2/(rho h) (b^2 missing in the denominator);
    a2 = cs2 + va2 (product term dropped); disc using v^2 in place of v^d v^d."""
    rng = np.random.default_rng(43)
    par = po.make_params(rho_atm=1e-30, T_atm=1e-30)
    for _ in range(30):
        g6 = H.random_spd(rng); gam = H.sym6_to_mat(g6)
        alpha = rng.uniform(0.4, 1.3); beta = rng.normal(size=3) * 0.2
        Gam = rng.choice([4.0 / 3, 5.0 / 3]); par.gamma_ad = Gam
        rho = 1.0; P = 10 ** rng.uniform(-2, 0.5)
        v = rng.normal(size=3); v *= rng.uniform(0.05, 0.85) / np.sqrt(v @ gam @ v)
        for d in range(3):
            e = np.zeros(3); e[d] = 1.0
            B = np.cross(e, gam @ v)                  # B^d = 0 and B^i v_i = 0
            B *= 10 ** rng.uniform(-0.5, 0.5) / np.sqrt(B @ gam @ B)
            assert abs(B[d]) < 1e-15 and abs(B @ gam @ v) < 1e-14
            ev = _jacobian_eigs(alpha, beta, g6, rho, v, P, B, Gam, d)
            lm, lp = _oracle_speeds(par, alpha, beta, g6, rho, v, P, B, d)
            assert abs(lm - ev[0]) <= 3e-6 and abs(lp - ev[-1]) <= 3e-6, (lm, lp, ev)
