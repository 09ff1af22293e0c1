"""Stage-level pins: T11 axis permutation, T14 hydrostatic second-order convergence, and the
input-generator invariants (divB~ = 0, SPD metric, subluminal velocity).  CPU only."""
import numpy as np
import pytest

import stagekit as sk
from oracle import pyoracle as po
from paper_2409_10384_b200 import workloads as wl

NG = sk.NG


# ---------------------------------------------------------------- T11
def _perm_cell(a):          # new(k,j,i) = old field at (x,y,z) -> (y,z,x): i'=k, j'=i, k'=j
    return np.ascontiguousarray(np.transpose(a, (0, 2, 3, 1)))


def _cyc_inputs(w, n):
    """relabel axes x->y->z->x: a field f'(x',y',z') = f(x=z', y=x', z=y'); vector
    components V'^{x'} = V^z ... i.e. new component c' takes old component (c'-1)."""
    nt = n + 2 * NG
    # arrays are [b,k,j,i] = [b,z,y,x]; new [b,z',y',x'] with z'=y, y'=x, x'=z
    T = lambda a: np.ascontiguousarray(np.transpose(a, (0, 2, 3, 1)))
    U = w["U"]; A = w["adm"]
    U2 = [T(U[0]), T(U[3]), T(U[1]), T(U[2]), T(U[4])]           # S'_x'=S_z, S'_y'=S_x, S'_z'=S_y
    # sym6 (xx,xy,xz,yy,yz,zz): new xx'=zz, x'y'=zx, x'z'=zy, y'y'=xx, y'z'=xy, z'z'=yy
    def sym(g):
        return [T(g[5]), T(g[2]), T(g[4]), T(g[0]), T(g[1]), T(g[3])]
    adm2 = sym(A[0:6]) + [T(A[6]), T(A[9]), T(A[7]), T(A[8])] + sym(A[10:16])
    bx = w["Bf"][0][..., :nt + 1]
    Bfx2 = np.zeros((1, nt, nt, nt + 4)); Bfx2[..., :nt + 1] = T(w["Bf"][2])    # B'^x' = B^z on z-faces
    Bf2 = [Bfx2, T(bx), T(w["Bf"][1])]
    return U2, Bf2, adm2


def test_T11_cyclic_axis_permutation():
    n = 6
    rng = np.random.default_rng(5)

    def metric(x, y, z):
        o = np.ones_like(x)
        g = [1.2 + 0.1 * np.sin(x + 2 * y), 0.05 * np.cos(z) * o, 0.03 * np.sin(y) * o,
             1.1 + 0.1 * np.cos(y - z), 0.04 * np.sin(x) * o, 1.3 + 0.1 * np.sin(z + x)]
        beta = [0.1 * np.sin(y), 0.05 * np.cos(z + x), -0.08 * np.sin(x)]
        K = [0.01 * np.sin(x) * o, 0.02 * o, -0.01 * np.cos(y) * o, 0.03 * np.sin(z) * o, 0.01 * o, -0.02 * np.cos(x) * o]
        return 0.8 + 0.1 * np.cos(x + y + z), beta, g, K

    def prim(x, y, z):
        rho = 1 + 0.3 * np.sin(1.3 * x) * np.cos(0.7 * y + z)
        low = np.sin(5 * x + 3 * y + 7 * z) > 0.9
        rho = np.where(low, 1e-5, rho)
        return rho, [0.3 * np.sin(y + z), -0.2 * np.cos(x), 0.25 * np.sin(2 * z - x)], np.where(low, 3e-9, 0.5 + 0.2 * np.cos(x - y))

    A = lambda c, x, y, z: [0.2 * np.sin(y + 0.5 * z), 0.15 * np.cos(z - x), 0.1 * np.sin(x * y)][c]
    w = sk.build_block(n, 0.2, (0.3, -0.4, 0.1), metric, prim, A_fn=A, gamma_ad=5.0 / 3)
    kw = dict(nmb=1, n=n, gamma_ad=5.0 / 3, rho_atm=1e-6, T_atm=1e-4, recon=2, riemann=1, fofc=1, dmp_M=1.2)
    par = po.make_params(**kw)
    r1 = po.rhs(par, w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], 0.35)
    U2, Bf2, adm2 = _cyc_inputs(w, n)
    r2 = po.rhs(par, w["dx"], U2, Bf2, adm2, 0.35)
    T = lambda a: np.transpose(a, (0, 2, 3, 1))
    assert (r1["flag"] > 0).sum() > 3
    assert np.array_equal(T(r1["flag"]), r2["flag"]) and np.array_equal(T(r1["status"]), r2["status"])
    pairs = [(0, 0), (3, 1), (1, 2), (2, 3), (4, 4)]
    for old, new in pairs:
        a, b = T(r1["dU"][old]), r2["dU"][new]
        assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    nt = n + 2 * NG
    # E'_x' = E_z, E'_y' = E_x, E'_z' = E_y (edge arrays transposed the same way)
    a = T(r1["E"][2][..., :nt + 1]); b = r2["E"][0]
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    a = T(r1["E"][0]); b = r2["E"][1][..., :nt + 1]
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    a = T(r1["E"][1][..., :nt + 1]); b = r2["E"][2][..., :nt + 1]
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()


# ---------------------------------------------------------------- T14
def test_T14_hydrostatic_test_fluid_converges_at_second_order():
    Mass, Kp, Gam, C = 1.0, 10.0, 2.0, 1.02

    def metric(x, y, z):
        r = np.sqrt(x * x + y * y + z * z)
        psi = 1 + Mass / (2 * r)
        o = np.ones_like(x); zr = np.zeros_like(x)
        p4 = psi ** 4
        return (1 - Mass / (2 * r)) / (1 + Mass / (2 * r)), [zr, zr, zr], [p4, zr, zr, p4, zr, p4], [zr] * 6

    def prim(x, y, z):
        alp = metric(x, y, z)[0]
        h = C / alp                                   # h alpha = const  (static, isentropic)
        rho = (h - 1) * (Gam - 1) / (Gam * Kp)        # h = 1 + Gamma K rho^(Gamma-1)/(Gamma-1), Gamma = 2
        return rho, [0 * x, 0 * x, 0 * x], Kp * rho ** Gam
    errs, other = [], []
    for n, d in ((8, 0.5), (16, 0.25)):
        w = sk.build_block(n, d, (8.0, 3.0, 2.0), metric, prim, gamma_ad=Gam)
        par = po.make_params(nmb=1, n=n, gamma_ad=Gam, rho_atm=1e-20, T_atm=1e-20, recon=2, riemann=1, fofc=1)
        r = po.rhs(par, w["dx"], [u.copy() for u in w["U"]], w["Bf"], w["adm"], 0.1 * d)
        assert not r["flag"].any()
        # v = 0: no advective mass/energy flux; what remains is the Riemann solver's diffusion on
        # the reconstructed jumps of sqrt(gamma) D, a truncation term that must also converge
        other.append(max(np.abs(sk.interior(r["dU"][c], n)).max() for c in (0, 4)))
        # force scale: sqrt(gamma) (rho h) d(alpha)/dx ~ E d_i alpha
        errs.append(max(np.abs(sk.interior(r["dU"][1 + c], n)).max() for c in range(3)))
        scale = np.abs(sk.interior(w["U"][4] + w["U"][0], n)).max() * Mass / 64.0
        assert errs[-1] < 0.05 * scale
    order = np.log2(errs[0] / errs[1])
    assert 1.8 <= order <= 2.3, (errs, order)
    assert other[1] <= other[0] / 3.5, other


# ---------------------------------------------------------------- generator invariants
@pytest.mark.parametrize("name,blocks", [("C0", None), ("C1", [0, 7]), ("C2", [21, 42]),
                                         ("C3", [0, 100, 213, 255]), ("C4", [0, 400])])
def test_generated_inputs_are_admissible(name, blocks):
    w = wl.make_blocks(name, blocks)
    n = w["params"]["n"]; nt = n + 2 * NG
    bx, by, bz = w["Bf"]
    for b in range(len(w["block_ids"])):
        d = w["dx"][b, 0]
        div = ((bx[b, :, :, 1:nt + 1] - bx[b, :, :, :nt]) + (by[b, :, 1:, :] - by[b, :, :-1, :]) +
               (bz[b, 1:] - bz[b, :-1])) / d
        bmax = max(np.abs(bx[b]).max(), np.abs(by[b]).max(), np.abs(bz[b]).max())
        assert np.abs(div).max() <= 2e-14 * max(bmax, 1e-300) / d * 40
    g = w["adm"][:6]
    det = (g[0] * (g[3] * g[5] - g[4] ** 2) - g[1] * (g[1] * g[5] - g[4] * g[2]) + g[2] * (g[1] * g[4] - g[3] * g[2]))
    assert np.all(g[0] > 0) and np.all(g[0] * g[3] - g[1] ** 2 > 0) and np.all(det > 0)
    assert np.all(w["adm"][6] > 0)
    for a in w["U"] + w["adm"] + w["Bf"]:
        assert np.all(np.isfinite(a)) and a.flags["C_CONTIGUOUS"] and a.dtype == np.float64
    assert np.all(w["U"][0] > 0)
    # same blocks regenerated alone are bit-identical (subset independence, used by the parity tests)
    w1 = wl.make_blocks(name, [int(w["block_ids"][-1])])
    assert np.array_equal(w1["U"][4][0], w["U"][4][-1]) and np.array_equal(w1["Bf"][0][0], w["Bf"][0][-1])
