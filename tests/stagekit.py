"""Small block builders for the stage-level oracle pins and the GPU parity tests (inputs only)."""
import numpy as np

from paper_2409_10384_b200 import workloads as wl

NG = 4


def grids(n, d=1.0, org=(0.0, 0.0, 0.0)):
    nt = n + 2 * NG
    cc = (np.arange(nt) - NG + 0.5) * d
    fc = (np.arange(nt + 1) - NG) * d
    return nt, cc, fc, org


def mesh(kk, jj, ii, org):
    Z, Y, X = np.meshgrid(kk + org[2], jj + org[1], ii + org[0], indexing="ij")
    return X, Y, Z


def build_block(n, d, org, metric_fn, prim_fn, A_fn=None, B_uniform=None, gamma_ad=2.0):
    """metric_fn(x,y,z) -> (alp, [beta^i], [g6], [K6]);  prim_fn(x,y,z) -> (rho, [u^i], P);
    B from a vector potential A_fn(comp,x,y,z) (B~ = curl A) or a uniform densitised B~."""
    nt, cc, fc, org = grids(n, d, org)
    px = nt + 4
    x, y, z = mesh(cc, cc, cc, org)
    one = np.ones_like(x)
    alp, beta, g6, K6 = metric_fn(x, y, z)
    rho, u, P = prim_fn(x, y, z)
    Bfx = np.zeros((1, nt, nt, px)); Bfy = np.zeros((1, nt, nt + 1, nt)); Bfz = np.zeros((1, nt + 1, nt, nt))
    if A_fn is not None:
        Ax = A_fn(0, *mesh(fc, fc, cc, org)); Ay = A_fn(1, *mesh(fc, cc, fc, org)); Az = A_fn(2, *mesh(cc, fc, fc, org))
        Bfx[0, :, :, :nt + 1] = ((Az[:, 1:, :] - Az[:, :-1, :]) - (Ay[1:, :, :] - Ay[:-1, :, :])) / d
        Bfy[0] = ((Ax[1:, :, :] - Ax[:-1, :, :]) - (Az[:, :, 1:] - Az[:, :, :-1])) / d
        Bfz[0] = ((Ay[:, :, 1:] - Ay[:, :, :-1]) - (Ax[:, 1:, :] - Ax[:, :-1, :])) / d
    if B_uniform is not None:
        Bfx[..., :nt + 1] += B_uniform[0]; Bfy += B_uniform[1]; Bfz += B_uniform[2]
    Bcc = [0.5 * (Bfx[0, :, :, :nt] + Bfx[0, :, :, 1:nt + 1]), 0.5 * (Bfy[0, :, :-1] + Bfy[0, :, 1:]),
           0.5 * (Bfz[0, :-1] + Bfz[0, 1:])]
    g = [np.ascontiguousarray(a * one) for a in g6]
    det = (g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) +
           g[2] * (g[1] * g[4] - g[3] * g[2]))
    sd = np.sqrt(det)
    u = [a * one for a in u]
    D, S, tau = wl._prim2cons_np(gamma_ad, g, rho * one, u, P * one, [b / sd for b in Bcc])
    c = lambda a: np.ascontiguousarray((a * one).reshape(1, nt, nt, nt))
    U = [c(sd * a) for a in (D, S[0], S[1], S[2], tau)]
    adm = [c(a) for a in g6] + [c(alp)] + [c(b) for b in beta] + [c(k) for k in K6]
    return dict(U=U, Bf=[Bfx, Bfy, Bfz], adm=adm, dx=np.full((1, 3), d),
                prim0=[c(rho), c(u[0]), c(u[1]), c(u[2]), c(P)], sdet=c(sd))


def flat_metric(x, y, z):
    o = np.ones_like(x); zr = np.zeros_like(x)
    return o, [zr, zr, zr], [o, zr, zr, o, zr, o], [zr] * 6


def interior(a, n):
    s = slice(NG, NG + n)
    return a[:, s, s, s]


def curlE_div(E, n, d):
    """-curl E at the faces of interior cells and its divergence per interior cell.
    E = [Ex, Ey, Ez] in boundary layouts (one or more blocks, uniform spacing d)."""
    s = slice(NG, NG + n); s1 = slice(NG, NG + n + 1)
    sp = slice(NG + 1, NG + n + 1)
    Ex, Ey, Ez = E
    # dBx/dt at x-faces (k in s, j in s, i in s1): -[(Ez(j+1)-Ez(j))/dy - (Ey(k+1)-Ey(k))/dz]
    dBx = -((Ez[:, s, sp, s1] - Ez[:, s, s, s1]) - (Ey[:, sp, s, s1] - Ey[:, s, s, s1])) / d
    dBy = -((Ex[:, sp, s1, s] - Ex[:, s, s1, s]) - (Ez[:, s, s1, sp] - Ez[:, s, s1, s])) / d
    dBz = -((Ey[:, s1, s, sp] - Ey[:, s1, s, s]) - (Ex[:, s1, sp, s] - Ex[:, s1, s, s])) / d
    div = ((dBx[..., 1:] - dBx[..., :-1]) + (dBy[:, :, 1:, :] - dBy[:, :, :-1, :]) +
           (dBz[:, 1:] - dBz[:, :-1])) / d
    return dBx, dBy, dBz, div


def loop_block(n):
    """Magnetic loop advection (Eq. 13): A_z = A0 max(R - r, 0), A0 = 1e-3, R = 0.3,
    rho = 1, P = 3, v = (1/1.2, 1/2.4, 0) on the periodic unit square, here one n^3 block (uniform
    in z).  The paper does not print Gamma for this test; 5/3 is used.  Returns (w, params, d)."""
    d = 1.0 / n
    v = np.array([1 / 1.2, 1 / 2.4, 0.0])
    lor = 1.0 / np.sqrt(1.0 - v @ v)

    def prim(x, y, z):
        o = np.ones_like(x)
        return o, [lor * v[0] * o, lor * v[1] * o, 0 * o], 3.0 * o

    def A(comp, x, y, z):
        if comp != 2:
            return 0 * x
        return 1e-3 * np.maximum(0.3 - np.sqrt(x * x + y * y), 0.0)
    w = build_block(n, d, (-0.5, -0.5, -0.5), flat_metric, prim, A_fn=A, gamma_ad=5.0 / 3.0)
    p = dict(nmb=1, n=n, gamma_ad=5.0 / 3.0, rho_atm=1e-10, T_atm=1e-8, recon=2, riemann=1, fofc=1)
    return w, p, d


def divB_rel(Bf, n, d, bmax):
    """max |div B~| dx / max|B~| over interior cells (the quantity of the paper's Figure 6, bottom)."""
    s = slice(NG, NG + n); s1 = slice(NG + 1, NG + n + 1)
    div = ((Bf[0][:, s, s, s1] - Bf[0][:, s, s, s]) + (Bf[1][:, s, s1, s] - Bf[1][:, s, s, s]) +
           (Bf[2][:, s1, s, s] - Bf[2][:, s, s, s]))
    return np.abs(div).max() / bmax


def loop_metrics(Bf, B0, n, shift_y):
    """correlation of the interior B~x with the initial loop displaced by shift_y cells in y, with the
    undisplaced one, and the ratio of sum B~x^2 to its initial value."""
    s = slice(NG, NG + n)
    bx = Bf[0][0, s, s, NG:NG + n]; b0 = B0[0][0, s, s, NG:NG + n]
    cor = lambda a, b: np.sum(a * b) / np.sqrt(np.sum(a * a) * np.sum(b * b))
    return cor(bx, np.roll(b0, shift_y, axis=1)), cor(bx, b0), np.sum(bx * bx) / np.sum(b0 * b0)
