"""TOV initial data for the paper's neutron-star test: a numpy TOV solver and the block
lattice built from it.  Test infrastructure only (no method arithmetic except the seeded generators'
prim->cons helper)."""
import numpy as np

from paper_2409_10384_b200 import workloads as wl

NG = 4

MSUN_S = 4.925491e-6            # G M_sun / c^3 in seconds


def tov_solve(rho_c=1.28e-3, K=100.0, gam=2.0, dr=1e-3, r_max=40.0):
    """Tolman-Oppenheimer-Volkoff equations in Schwarzschild coordinates for P = K rho^Gamma,
    classical RK4 in r.  Returns r, m(r), P(r), alpha(r) on a uniform radial grid, and M, R."""
    def rhs(r, y):
        m, P, phi = y
        if P <= 0.0:
            return np.array([0.0, 0.0, m / (r * (r - 2.0 * m))])
        rho = (P / K) ** (1.0 / gam)
        e = rho + P / (gam - 1.0)
        if r == 0.0:
            return np.zeros(3)
        s = (m + 4.0 * np.pi * r ** 3 * P) / (r * (r - 2.0 * m))
        return np.array([4.0 * np.pi * r * r * e, -(e + P) * s, s])
    nr = int(round(r_max / dr)) + 1
    r = np.arange(nr) * dr
    y = np.zeros((nr, 3))
    y[0] = [0.0, K * rho_c ** gam, 0.0]
    R = None
    for i in range(nr - 1):
        k1 = rhs(r[i], y[i]); k2 = rhs(r[i] + 0.5 * dr, y[i] + 0.5 * dr * k1)
        k3 = rhs(r[i] + 0.5 * dr, y[i] + 0.5 * dr * k2); k4 = rhs(r[i] + dr, y[i] + dr * k3)
        y[i + 1] = y[i] + dr / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
        if y[i + 1, 1] <= 0.0 and R is None:
            R = r[i] + dr * y[i, 1] / (y[i, 1] - y[i + 1, 1])           # linear zero of P
            y[i + 1, 1] = 0.0
        if R is not None:
            y[i + 1, 1] = 0.0
    M = y[-1, 0]
    phi = y[:, 2] + (0.5 * np.log(1.0 - 2.0 * M / r[-1]) - y[-1, 2])     # match alpha to Schwarzschild outside
    return r, y[:, 0], y[:, 1], np.exp(phi), M, R


def tov_lattice(sh, n, nb, half_width, amp=-0.024, K=100.0, gam=2.0, rho_atm=1e-10, T_atm=1e-8):
    """sh = shapes(nb^3, n) of the caller's library.  nb^3 blocks of n^3 covering [-half_width, half_width]^3, the star at the centre, in Cartesian
    coordinates built on the Schwarzschild radius: gamma_ij = delta_ij + (1/(1-2m/r) - 1) n_i n_j,
    beta = 0, K_ij = 0; radial velocity perturbation of Eq. 14 with amplitude `amp` at the surface."""
    r1, m1, P1, a1, M, R = tov_solve(K=K, gam=gam)
    nt = n + 2 * NG
    d = 2.0 * half_width / (n * nb)
    nmb = nb ** 3
    U = [np.zeros(sh["cell"]) for _ in range(5)]
    adm = [np.zeros(sh["cell"]) for _ in range(16)]
    for bz in range(nb):
        for by in range(nb):
            for bx in range(nb):
                mb = (bz * nb + by) * nb + bx
                c = [-half_width + (b * n + np.arange(nt) - NG + 0.5) * d for b in (bx, by, bz)]
                Z, Y, X = np.meshgrid(c[2], c[1], c[0], indexing="ij")
                r = np.sqrt(X * X + Y * Y + Z * Z)
                nrm = [X / r, Y / r, Z / r]
                m = np.interp(r, r1, m1); P = np.interp(r, r1, P1); alp = np.interp(r, r1, a1)
                A = 1.0 / (1.0 - 2.0 * m / r)
                g = [1.0 + (A - 1.0) * nrm[0] * nrm[0], (A - 1.0) * nrm[0] * nrm[1], (A - 1.0) * nrm[0] * nrm[2],
                     1.0 + (A - 1.0) * nrm[1] * nrm[1], (A - 1.0) * nrm[1] * nrm[2], 1.0 + (A - 1.0) * nrm[2] * nrm[2]]
                rho = (np.maximum(P, 0.0) / K) ** (1.0 / gam)
                inside = rho > 1.01 * rho_atm
                rho = np.where(inside, rho, rho_atm); P = np.where(inside, P, rho_atm * T_atm)
                x = np.minimum(r / R, 1.0)
                vr = np.where(inside, 0.5 * amp * (3.0 * x - x ** 3), 0.0)
                lor = 1.0 / np.sqrt(1.0 - A * vr * vr)
                u = [lor * vr * q for q in nrm]
                zr = np.zeros_like(r)
                D, S, tau = wl._prim2cons_np(gam, g, rho, u, P, [zr, zr, zr])
                sd = np.sqrt(A)                                            # det(delta + (A-1) n n) = A
                for dst, src in zip(U, (D, S[0], S[1], S[2], tau)):
                    dst[mb] = sd * src
                for q in range(6):
                    adm[q][mb] = g[q]
                adm[6][mb] = alp
    Bf = [np.zeros(sh[k]) for k in ("xf", "yf", "zf")]
    p = dict(nmb=nmb, n=n, gamma_ad=gam, rho_atm=rho_atm, T_atm=T_atm, f_thr=1.01, recon=1, riemann=1, fofc=1)
    return dict(U=U, Bf=Bf, adm=adm, dx=np.full((nmb, 3), d), params=p, dt_fofc=0.0), d, M, R
