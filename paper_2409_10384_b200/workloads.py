"""Seeded synthetic MeshBlock batches C0..C4 (BASELINE.json configs[0..4]); DESIGN.md §4.

These generators stand in for the paper's workloads (LORENE BNS data P:372, Fishbone-Moncrief
torus P:295, TOV solver output P:262 are not available): they take the shapes, sizes and
value ranges and are analytic formulas plus a counter-based integer hash.  The module serves
BOTH the CPU oracle and the CUDA library and therefore holds none of the method's arithmetic:
it only builds input arrays (including U~ = sqrt(gamma) * Eq. 6 of the initial primitives,
written here in vectorised numpy, independent of oracle/ and csrc/).  numpy only.

Layouts (include/ak.h): cell [nb,nt,nt,nt]; x-face [nb,nt,nt,nt+4]; y-face [nb,nt,nt+1,nt];
z-face [nb,nt+1,nt,nt]; i fastest; face i lies between cells i-1 and i; ghost cells are filled
by evaluating the same analytic fields.
"""
import numpy as np

NG = 4
SEED0 = 2409103840
CONFIG_NAMES = ("C0", "C1", "C2", "C3", "C4")


# ------------------------------------------------------------------ counter-based hash
def _mix(x):
    x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return x ^ (x >> np.uint64(31))


def hash_uniform(seed, block, field, idx):
    """uniform [0,1) from (seed, block, field, linear index); arrays broadcast."""
    with np.errstate(over="ignore"):
        s = np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15)
        b = np.asarray(block, dtype=np.uint64) * np.uint64(0xD1B54A32D192ED03)
        f = np.uint64(field) * np.uint64(0x8CB92BA72F3D8DD7)
        i = np.asarray(idx, dtype=np.uint64)
        h = _mix(_mix(_mix(s + b) + f) + i)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ------------------------------------------------------------------ config tables
def config_spec(name):
    """static description: params for ak_create / the oracle, block list, dt_fofc."""
    inf = float("inf")
    if name == "C0":
        p = dict(n=16, gamma_ad=2.0, rho_atm=1e-10, T_atm=1e-8, f_thr=1.0, mag_max=inf,
                 recon=1, riemann=1, fofc=1, fofc_riemann=0, dmp_M=0.0)
        org = np.zeros((1, 3)); dxs = np.full((1,), 1.0 / 16)
        return dict(name=name, params=p, origin=org, delta=dxs, dt_fofc=0.25 / 16, seed=SEED0)
    if name in ("C1", "C2", "C4"):
        # rho_atm = 1e-10 rho_c.  T_atm: see DESIGN.md §4 (half the atmosphere's
        # polytropic temperature K rho_atm so that a resting atmosphere is flag-free).
        p = dict(n=32, gamma_ad=2.0, rho_atm=1.28e-13, T_atm=0.64e-11, f_thr=0.1, mag_max=inf,
                 recon=1 if name == "C1" else 2, riemann=1, fofc=1, fofc_riemann=0,
                 dmp_M=0.0 if name == "C1" else 1.1)
        if name == "C1":
            nb3 = (2, 2, 2)
        elif name == "C2":
            nb3 = (4, 4, 4)
        else:
            nb3 = (8, 8, 12)
        bx, by, bz = np.meshgrid(np.arange(nb3[0]), np.arange(nb3[1]), np.arange(nb3[2]),
                                 indexing="ij")
        idx3 = np.stack([bx.ravel(), by.ravel(), bz.ravel()], axis=1).astype(np.float64)
        centre = 16.0 * (idx3 - (np.array(nb3) - 1) / 2.0)
        nb = centre.shape[0]
        seed = SEED0 + int(name[1])
        if name == "C4":
            u = hash_uniform(seed, np.arange(nb), 99, 0)
            fac = np.where(u < 0.25, 1.0, np.where(u < 0.5, 2.0, 4.0))
        else:
            fac = np.ones(nb)
        delta = 0.5 * fac
        org = centre - 16.0 * delta[:, None]
        return dict(name=name, params=p, origin=org, delta=delta, dt_fofc=0.125, seed=seed)
    if name == "C3":
        p = dict(n=16, gamma_ad=13.0 / 9.0, rho_atm=1e-10, T_atm=3.33e-13, f_thr=1.0,
                 mag_max=100.0, recon=1, riemann=1, fofc=1, fofc_riemann=0, dmp_M=0.0)
        orgs, dls = [], []
        for L in (40.0, 20.0, 10.0, 5.0):
            d = L / 32.0
            for a in range(4):
                for b in range(4):
                    for c in range(4):
                        orgs.append([-L + a * 16 * d, -L + b * 16 * d, -L + c * 16 * d])
                        dls.append(d)
        return dict(name=name, params=p, origin=np.array(orgs), delta=np.array(dls),
                    dt_fofc=0.25 * 5.0 / 32.0, seed=SEED0 + 3)
    raise ValueError(name)


def n_blocks(name):
    return config_spec(name)["origin"].shape[0]


# ------------------------------------------------------------------ analytic fields
M_STAR, SIG_STAR, RHO_C, K_POLY = 1.4, 4.0, 1.28e-3, 100.0
OMEGA = 0.02
KS_A, KS_RMIN = 0.9375, 1.2
C3_AB, C3_B0 = 1.0, 3.0e-4


def _stars(name):
    return [(0.0, 1)] if name == "C1" else [(8.0, 1), (-8.0, -1)]


def _metric(name, x, y, z):
    """returns dict alp, beta(3), g(6: xx,xy,xz,yy,yz,zz) at points (broadcast arrays)."""
    one = np.ones(np.broadcast(x, y, z).shape)
    if name == "C0":
        return dict(alp=one, beta=[0 * one, 0 * one, 0 * one],
                    g=[one, 0 * one, 0 * one, one, 0 * one, one])
    if name in ("C1", "C2", "C4"):
        sig = 0.0
        for xs, _ in _stars(name):
            sig = sig + M_STAR / (2.0 * np.sqrt((x - xs) ** 2 + y * y + z * z + SIG_STAR ** 2))
        psi = 1.0 + sig
        alp = (1.0 - sig) / (1.0 + sig)
        p4 = psi ** 4
        if name == "C1":
            beta = [0 * one, 0 * one, 0 * one]
        else:
            beta = [-OMEGA * y * one, OMEGA * x * one, 0 * one]
        return dict(alp=alp * one, beta=beta, g=[p4 * one, 0 * one, 0 * one, p4 * one, 0 * one, p4 * one],
                    psi=psi)
    if name == "C3":
        a = KS_A
        R2 = x * x + y * y + z * z
        r2 = 0.5 * ((R2 - a * a) + np.sqrt((R2 - a * a) ** 2 + 4.0 * a * a * z * z))
        r = np.maximum(np.sqrt(np.maximum(r2, 0.0)), KS_RMIN)
        f = 2.0 * r ** 3 / (r ** 4 + a * a * z * z)
        l = [(r * x + a * y) / (r * r + a * a), (r * y - a * x) / (r * r + a * a), z / r]
        g = [1.0 + f * l[0] * l[0], f * l[0] * l[1], f * l[0] * l[2],
             1.0 + f * l[1] * l[1], f * l[1] * l[2], 1.0 + f * l[2] * l[2]]
        alp = 1.0 / np.sqrt(1.0 + f)
        # beta^i = f l^i/(1+f) with l^i = l_i/(1 + f l.l) * ... ; for exact Kerr-Schild l.l = 1.
        # With the clamped radius l is no longer null, so raise with the true inverse metric:
        # gamma^{ij} = delta - f l l/(1 + f l.l);  beta_i = f l_i (the g_{0i} of KS)
        ll = l[0] ** 2 + l[1] ** 2 + l[2] ** 2
        beta = [f * l[i] / (1.0 + f * ll) for i in range(3)]
        return dict(alp=alp, beta=beta, g=g, r=r)
    raise ValueError(name)


def _extrinsic(name, x, y, z, h):
    """K_ij (6) of the stationary snapshot: K_ij = (D_i beta_j + D_j beta_i)/(2 alpha)."""
    m = _metric(name, x, y, z)
    zero = np.zeros_like(m["alp"])
    if name in ("C0", "C1"):
        return [zero] * 6
    if name in ("C2", "C4"):
        # gamma = psi^4 delta, beta a flat Killing vector: K_ij = 2 psi^3 (beta.grad psi) delta_ij/alpha
        gpx = gpy = gpz = 0.0
        for xs, _ in _stars(name):
            rt3 = ((x - xs) ** 2 + y * y + z * z + SIG_STAR ** 2) ** 1.5
            gpx = gpx - 0.5 * M_STAR * (x - xs) / rt3
            gpy = gpy - 0.5 * M_STAR * y / rt3
            gpz = gpz - 0.5 * M_STAR * z / rt3
        bg = m["beta"][0] * gpx + m["beta"][1] * gpy + m["beta"][2] * gpz
        kd = 2.0 * m["psi"] ** 3 * bg / m["alp"]
        return [kd, zero, zero, kd, zero, kd]
    # numeric: 4th-order centred differences of the analytic gamma_ij and beta_i
    idx = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (1, 1): 3, (1, 2): 4, (2, 2): 5}

    def gget(g, i, j):
        return g[idx[(min(i, j), max(i, j))]]

    def lowered(mm):
        return [sum(gget(mm["g"], i, j) * mm["beta"][j] for j in range(3)) for i in range(3)]

    dg = [[None] * 6 for _ in range(3)]   # dg[k][q] = d_k gamma_q
    db = [[None] * 3 for _ in range(3)]   # db[k][i] = d_k beta_i
    for k in range(3):
        acc_g = [0.0] * 6
        acc_b = [0.0] * 3
        for s, w in ((-2, 1.0 / 12), (-1, -8.0 / 12), (1, 8.0 / 12), (2, -1.0 / 12)):
            sh = [0.0, 0.0, 0.0]
            sh[k] = s * h
            mm = _metric(name, x + sh[0], y + sh[1], z + sh[2])
            bl = lowered(mm)
            for q in range(6):
                acc_g[q] = acc_g[q] + w * mm["g"][q]
            for i in range(3):
                acc_b[i] = acc_b[i] + w * bl[i]
        dg[k] = [a / h for a in acc_g]
        db[k] = [a / h for a in acc_b]
    K = []
    for (i, j) in ((0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)):
        # Gamma^k_ij beta_k = 1/2 beta^l (d_i g_lj + d_j g_li - d_l g_ij)
        chr_b = 0.0
        for l in range(3):
            chr_b = chr_b + 0.5 * m["beta"][l] * (
                gget(dg[i], l, j) + gget(dg[j], l, i) - gget(dg[l], i, j))
        K.append((db[i][j] + db[j][i] - 2.0 * chr_b) / (2.0 * m["alp"]))
    return K


def _fluid(name, spec, x, y, z, blk, lin):
    """primitives rho, v^i (Eulerian three-velocity), P at cell centres."""
    seed = spec["seed"]
    one = np.ones(np.broadcast(x, y, z).shape)
    if name == "C0":
        tp = 2.0 * np.pi
        rho = 1.0 + 0.1 * np.sin(tp * x) * np.sin(tp * y) * np.sin(tp * z)
        P = 0.5 + 0.05 * np.cos(tp * (x + y)) * one
        v = [(-0.3 + 0.6 * float(hash_uniform(seed, 0, 10 + c, 0))) * one for c in range(3)]
        return rho, v, P
    if name in ("C1", "C2", "C4"):
        rho_atm = spec["params"]["rho_atm"]
        parts = []
        for xs, sgn in _stars(name):
            parts.append((RHO_C * np.exp(-((x - xs) ** 2 + y * y + z * z) / (2 * SIG_STAR ** 2)), sgn))
        tot = sum(pp for pp, _ in parts)
        rho = np.maximum(tot, rho_atm)
        vy = 0 * one
        if name != "C1":
            xi = 2.0 * hash_uniform(seed, blk, 1, lin) - 1.0
            rho = rho * (1.0 + 1e-3 * xi)
            num = sum(0.15 * sgn * pp for pp, sgn in parts)
            vy = np.where(tot > 10 * rho_atm, num / np.maximum(tot, 1e-300), 0.0)
        P = K_POLY * rho * rho
        return rho, [0 * one, vy, 0 * one], P
    if name == "C3":
        m = _metric(name, x, y, z)
        w2 = x * x + y * y
        w = np.sqrt(w2)
        rho = np.maximum(1.0 - (w - 12.0) ** 2 / 36.0 - z * z / 16.0, 0.0) + 1e-8
        P = 0.01 * rho ** spec["params"]["gamma_ad"]
        vx = -y * w ** -1.5
        vy = x * w ** -1.5
        g = m["g"]
        v2 = g[0] * vx * vx + 2 * g[1] * vx * vy + g[3] * vy * vy
        sc = np.where(v2 > 0.81, np.sqrt(0.81 / np.maximum(v2, 1e-300)), 1.0)
        inside = m["r"] <= KS_RMIN
        vx = np.where(inside, 0.0, vx * sc)
        vy = np.where(inside, 0.0, vy * sc)
        rho = np.where(inside, 1e-8, rho)
        P = np.where(inside, 0.01 * 1e-8 ** spec["params"]["gamma_ad"], P)
        return rho, [vx, vy, 0 * one], P
    raise ValueError(name)


def _c0_modes(seed):
    modes = []
    for mI in range(4):
        k = [int(np.floor(5 * float(hash_uniform(seed, 0, 20 + mI, c)))) - 2 for c in range(3)]
        if k == [0, 0, 0]:
            k = [1, 0, 0]
        amp = 0.5 + float(hash_uniform(seed, 0, 20 + mI, 3))
        ph = 2 * np.pi * float(hash_uniform(seed, 0, 20 + mI, 4))
        comp = int(np.floor(3 * float(hash_uniform(seed, 0, 20 + mI, 5))))
        modes.append((k, amp, ph, comp))
    return modes


C0_BSCALE = {}  # per seed, filled lazily: rescales rms|B| to 0.1 (a function of the seed alone, not of call order)


def _vecpot(name, spec, comp, x, y, z):
    """component comp of the (densitised-B) vector potential A at points."""
    if name == "C0":
        tot = 0.0 * (x + y + z)
        for (k, amp, ph, c) in _c0_modes(spec["seed"]):
            if c == comp:
                tot = tot + amp * np.sin(2 * np.pi * (k[0] * x + k[1] * y + k[2] * z) + ph)
        return tot * _c0_scale(spec)
    if name in ("C1", "C2", "C4"):
        if comp == 2:
            return 0.0 * (x + y + z)
        Pmax = K_POLY * RHO_C ** 2
        tot = 0.0
        for xs, _ in _stars(name):
            rho = RHO_C * np.exp(-((x - xs) ** 2 + y * y + z * z) / (2 * SIG_STAR ** 2))
            A = np.maximum(K_POLY * rho * rho - 0.04 * Pmax, 0.0)
            tot = tot + (-(y) * A if comp == 0 else (x - xs) * A)
        # A_b from centre values: B~^z_c = 2 A_b 0.96 Pmax; B^2_c = psi_c^-8 (B~^z_c)^2 = 2e-3 Pmax
        psi_c = 1.0 + M_STAR / (2.0 * SIG_STAR)
        Ab = np.sqrt(2e-3 * Pmax) * psi_c ** 4 / (2 * 0.96 * Pmax)
        return Ab * tot
    if name == "C3":
        if comp == 2:
            return 0.0 * (x + y + z)
        w2 = x * x + y * y
        w = np.sqrt(w2)
        rho = np.maximum(1.0 - (w - 12.0) ** 2 / 36.0 - z * z / 16.0, 0.0) + 1e-8
        s = 0.0
        for mI in range(8):
            lam = 2.0 + 6.0 * float(hash_uniform(spec["seed"], 0, 40 + mI, 0))
            th = np.pi * float(hash_uniform(spec["seed"], 0, 40 + mI, 1))
            ph = 2 * np.pi * float(hash_uniform(spec["seed"], 0, 40 + mI, 2))
            pz = 2.0 * float(hash_uniform(spec["seed"], 0, 40 + mI, 3)) - 1.0
            kx, ky, kz = np.cos(th) * np.sqrt(1 - pz * pz), np.sin(th) * np.sqrt(1 - pz * pz), pz
            s = s + np.sin(2 * np.pi * (kx * x + ky * y + kz * z) / lam + ph) / np.sqrt(8.0)
        Aphi_t = C3_AB * np.maximum(rho / (1.0 + 1e-8) - 0.2, 0.0) * (1.0 + 0.02 * s)
        # A_x = -y A_phi / w^2, A_y = x A_phi / w^2 ; the uniform seed 1/2 B0 w^2 is regular
        over = np.where(w2 > 0, 1.0 / np.maximum(w2, 1e-300), 0.0)
        if comp == 0:
            return -y * (Aphi_t * over + 0.5 * C3_B0)
        return x * (Aphi_t * over + 0.5 * C3_B0)
    raise ValueError(name)


def _c0_scale(spec):
    seed = spec["seed"]
    if seed not in C0_BSCALE:
        C0_BSCALE[seed] = 1.0
        # rms |curl A| on a fixed 32^3 sample of [0,1]^3 (analytic derivative by differences)
        n = 32
        c = (np.arange(n) + 0.5) / n
        X, Y, Z = np.meshgrid(c, c, c, indexing="ij")
        h = 1e-5

        def A(comp, x, y, z):
            return _vecpot("C0", spec, comp, x, y, z)

        def d(comp, ax):
            sh = [0, 0, 0]; sh[ax] = h
            return (A(comp, X + sh[0], Y + sh[1], Z + sh[2]) - A(comp, X - sh[0], Y - sh[1], Z - sh[2])) / (2 * h)
        Bx = d(2, 1) - d(1, 2); By = d(0, 2) - d(2, 0); Bz = d(1, 0) - d(0, 1)
        rms = np.sqrt(np.mean(Bx * Bx + By * By + Bz * Bz))
        C0_BSCALE[seed] = 0.1 / rms
    return C0_BSCALE[seed]


# ------------------------------------------------------------------ Eq. 6 (generator's own)
def _prim2cons_np(gam, g, rho, u, P, B):
    gxx, gxy, gxz, gyy, gyz, gzz = g
    ul = [gxx * u[0] + gxy * u[1] + gxz * u[2], gxy * u[0] + gyy * u[1] + gyz * u[2],
          gxz * u[0] + gyz * u[1] + gzz * u[2]]
    Bl = [gxx * B[0] + gxy * B[1] + gxz * B[2], gxy * B[0] + gyy * B[1] + gyz * B[2],
          gxz * B[0] + gyz * B[1] + gzz * B[2]]
    usq = ul[0] * u[0] + ul[1] * u[1] + ul[2] * u[2]
    W = np.sqrt(1.0 + usq)
    vl = [a / W for a in ul]
    B2 = Bl[0] * B[0] + Bl[1] * B[1] + Bl[2] * B[2]
    Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2]
    hm1 = gam / (gam - 1.0) * P / rho
    D = rho * W
    wt = rho * (1.0 + hm1) * W * W + B2
    S = [wt * vl[i] - Bv * Bl[i] for i in range(3)]
    tau = D * (hm1 * W + usq / (1.0 + W)) + B2 - P - 0.5 * (Bv * Bv + B2 / (W * W))
    return D, S, tau


# ------------------------------------------------------------------ block batch builder
def make_blocks(name, blocks=None):
    """Build the input arrays of config `name` for the given block ids (default: all).

    Returns dict: params (with nmb = number of generated blocks), dx [nb,3], dt_fofc,
    U (5 arrays), Bf (3), adm (16: gxx,gxy,gxz,gyy,gyz,gzz,alp,betx,bety,betz,Kxx..Kzz),
    prim0 (the initial primitives rho,ux,uy,uz,P — for tests only), block_ids.
    """
    spec = config_spec(name)
    p = dict(spec["params"])
    n = p["n"]
    nt = n + 2 * NG
    px = nt + 4
    ids = np.arange(spec["origin"].shape[0]) if blocks is None else np.asarray(blocks, dtype=np.int64)
    nb = len(ids)
    org = spec["origin"][ids]
    dl = spec["delta"][ids]
    p["nmb"] = nb
    cc = (np.arange(nt) - NG + 0.5)          # cell-centre offsets in units of delta
    fc = (np.arange(nt + 1) - NG) * 1.0      # face offsets
    B4 = (nb, 1, 1, 1)
    d4 = dl.reshape(B4)
    ox, oy, oz = (org[:, c].reshape(B4) for c in range(3))

    def coords(kk, jj, ii):
        # kk, jj, ii: 1-D offset arrays along k, j, i
        return (ox + ii.reshape(1, 1, 1, -1) * d4, oy + jj.reshape(1, 1, -1, 1) * d4,
                oz + kk.reshape(1, -1, 1, 1) * d4)

    x, y, z = coords(cc, cc, cc)
    x, y, z = np.broadcast_arrays(x, y, z)
    blk = ids.reshape(B4).astype(np.uint64)
    lin = np.arange(nt ** 3, dtype=np.uint64).reshape(1, nt, nt, nt)
    m = _metric(name, x, y, z)
    g = [np.ascontiguousarray(a * np.ones(x.shape)) for a in m["g"]]
    alp = np.ascontiguousarray(m["alp"] * np.ones(x.shape))
    beta = [np.ascontiguousarray(b * np.ones(x.shape)) for b in m["beta"]]
    Kij = [np.ascontiguousarray(k * np.ones(x.shape)) for k in _extrinsic(name, x, y, z, 1e-3 * d4)]
    rho, v, P = _fluid(name, spec, x, y, z, blk, lin)
    vl2 = (g[0] * v[0] * v[0] + g[3] * v[1] * v[1] + g[5] * v[2] * v[2] +
           2 * (g[1] * v[0] * v[1] + g[2] * v[0] * v[2] + g[4] * v[1] * v[2]))
    Wl = 1.0 / np.sqrt(1.0 - vl2)
    u = [Wl * a for a in v]

    # face B~ = discrete curl of the edge-centred vector potential (divB~ = 0 to round-off)
    def A_at(comp, kk, jj, ii):
        xx, yy, zz = coords(kk, jj, ii)
        return _vecpot(name, spec, comp, *np.broadcast_arrays(xx, yy, zz))
    Ax = A_at(0, fc, fc, cc)   # x-edges: (k-1/2, j-1/2, i)    shape [nb, nt+1, nt+1, nt]
    Ay = A_at(1, fc, cc, fc)   # y-edges: (k-1/2, j, i-1/2)    [nb, nt+1, nt, nt+1]
    Az = A_at(2, cc, fc, fc)   # z-edges: (k, j-1/2, i-1/2)    [nb, nt, nt+1, nt+1]
    Bfx = np.zeros((nb, nt, nt, px))
    Bfx[..., :nt + 1] = ((Az[:, :, 1:, :] - Az[:, :, :-1, :]) - (Ay[:, 1:, :, :] - Ay[:, :-1, :, :])) / d4
    Bfy = ((Ax[:, 1:, :, :] - Ax[:, :-1, :, :]) - (Az[:, :, :, 1:] - Az[:, :, :, :-1])) / d4
    Bfz = ((Ay[:, :, :, 1:] - Ay[:, :, :, :-1]) - (Ax[:, :, 1:, :] - Ax[:, :, :-1, :])) / d4
    Bfy = np.ascontiguousarray(Bfy); Bfz = np.ascontiguousarray(Bfz)
    Bcc = [0.5 * (Bfx[..., :nt] + Bfx[..., 1:nt + 1]), 0.5 * (Bfy[:, :, :-1, :] + Bfy[:, :, 1:, :]),
           0.5 * (Bfz[:, :-1] + Bfz[:, 1:])]
    det = (g[0] * (g[3] * g[5] - g[4] * g[4]) - g[1] * (g[1] * g[5] - g[4] * g[2]) +
           g[2] * (g[1] * g[4] - g[3] * g[2]))
    sdet = np.sqrt(det)
    D, S, tau = _prim2cons_np(p["gamma_ad"], g, rho, u, P, [b / sdet for b in Bcc])
    U = [np.ascontiguousarray(sdet * a) for a in (D, S[0], S[1], S[2], tau)]
    adm = g + [alp] + beta + Kij
    prim0 = [np.ascontiguousarray(a * np.ones(x.shape)) for a in (rho, u[0], u[1], u[2], P)]
    dx = np.repeat(dl.reshape(nb, 1), 3, axis=1).copy()
    return dict(name=name, params=p, dx=dx, dt_fofc=spec["dt_fofc"], U=U,
                Bf=[np.ascontiguousarray(Bfx), Bfy, Bfz], adm=adm, prim0=prim0, block_ids=ids)


def make_test_noise_block(seed=7, n=8, frac=0.01):
    """C0n: tiny Minkowski block with per-cell hashed velocities and a
    fraction of cells whose rho and P are divided by 1e6 — exercises floors and FOFC.
    Not a reported config."""
    spec = dict(config_spec("C0"))
    spec["seed"] = seed
    nt = n + 2 * NG
    px = nt + 4
    p = dict(spec["params"]); p["n"] = n; p["nmb"] = 1
    d = 1.0 / n
    cc = (np.arange(nt) - NG + 0.5) * d
    fc = (np.arange(nt + 1) - NG) * d
    z, y, x = np.meshgrid(cc, cc, cc, indexing="ij")
    x, y, z = (a.reshape(1, nt, nt, nt) for a in (x, y, z))
    lin = np.arange(nt ** 3, dtype=np.uint64).reshape(1, nt, nt, nt)
    tp = 2 * np.pi
    rho = 1.0 + 0.1 * np.sin(tp * x) * np.sin(tp * y) * np.sin(tp * z)
    P = 0.5 + 0.05 * np.cos(tp * (x + y)) * np.ones_like(rho)
    low = hash_uniform(seed, 0, 3, lin) < frac
    rho = np.where(low, rho * 1e-6, rho); P = np.where(low, P * 1e-6, P)
    v = [-0.3 + 0.6 * hash_uniform(seed, 0, 4 + c, lin) for c in range(3)]
    Wl = 1.0 / np.sqrt(1.0 - (v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    u = [Wl * a for a in v]
    one = np.ones_like(rho)
    g = [one.copy(), 0 * one, 0 * one, one.copy(), 0 * one, one.copy()]

    def A(comp, zz, yy, xx):
        Z, Y, X = np.meshgrid(zz, yy, xx, indexing="ij")
        return _vecpot("C0", spec, comp, X, Y, Z)[None]
    Ax = A(0, fc, fc, cc); Ay = A(1, fc, cc, fc); Az = A(2, cc, fc, fc)
    Bfx = np.zeros((1, nt, nt, px))
    Bfx[..., :nt + 1] = ((Az[:, :, 1:, :] - Az[:, :, :-1, :]) - (Ay[:, 1:, :, :] - Ay[:, :-1, :, :])) / d
    Bfy = np.ascontiguousarray(((Ax[:, 1:] - Ax[:, :-1]) - (Az[:, :, :, 1:] - Az[:, :, :, :-1])) / d)
    Bfz = np.ascontiguousarray(((Ay[:, :, :, 1:] - Ay[:, :, :, :-1]) - (Ax[:, :, 1:, :] - Ax[:, :, :-1, :])) / d)
    Bcc = [0.5 * (Bfx[..., :nt] + Bfx[..., 1:nt + 1]), 0.5 * (Bfy[:, :, :-1] + Bfy[:, :, 1:]),
           0.5 * (Bfz[:, :-1] + Bfz[:, 1:])]
    D, S, tau = _prim2cons_np(p["gamma_ad"], g, rho, u, P, Bcc)
    U = [np.ascontiguousarray(a) for a in (D, S[0], S[1], S[2], tau)]
    adm = g + [one.copy(), 0 * one, 0 * one, 0 * one] + [0 * one for _ in range(6)]
    return dict(name="C0n", params=p, dx=np.full((1, 3), d), dt_fofc=0.4 * d, U=U,
                Bf=[Bfx, Bfy, Bfz], adm=adm, prim0=[rho, u[0], u[1], u[2], P],
                block_ids=np.zeros(1, dtype=np.int64))
