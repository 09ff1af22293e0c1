"""Pins of the oracle's same-level ghost exchange: the exchanged blocks must equal
slices of the padded global array (numpy wrap / edge), and a domain evolved as 2x2x2 blocks with
exchange must equal, bit for bit, the same domain evolved as one block."""
import numpy as np
import pytest

from oracle import pyoracle as orc

import stagekit as sk

NG = 4


def lattice_nbr(nb3, periodic):
    """neighbour table of an nb3 = (nbx, nby, nbz) lattice, block id = (bz*nby + by)*nbx + bx."""
    nbx, nby, nbz = nb3
    nbr = -np.ones((nbx * nby * nbz, 27), dtype=np.int32)
    for bz in range(nbz):
        for by in range(nby):
            for bx in range(nbx):
                m = (bz * nby + by) * nbx + bx
                for oz in (-1, 0, 1):
                    for oy in (-1, 0, 1):
                        for ox in (-1, 0, 1):
                            c = [bx + ox, by + oy, bz + oz]
                            ok = True
                            for d in range(3):
                                if c[d] < 0 or c[d] >= nb3[d]:
                                    if periodic[d]:
                                        c[d] %= nb3[d]
                                    else:
                                        ok = False
                            if ok and (ox, oy, oz) != (0, 0, 0):
                                nbr[m, (oz + 1) * 9 + (oy + 1) * 3 + (ox + 1)] = (c[2] * nby + c[1]) * nbx + c[0]
    return nbr


def split(G, nb3, n, pad_modes, face_dir=None):
    """blocks [nmb, ...] cut from the padded global array G[z, y, x] (face_dir: normal direction of a
    face field, whose global array has N (periodic) or N+1 (bounded) entries along that axis)."""
    nbx, nby, nbz = nb3
    a = G
    for ax, d in ((0, 2), (1, 1), (2, 0)):
        pw = [(0, 0)] * 3
        hi = NG
        if face_dir == d and pad_modes[d] == "wrap":
            hi = NG + 1
        pw[ax] = (NG, hi)
        a = np.pad(a, pw, mode=pad_modes[d])
    nt = n + 2 * NG
    out = []
    for bz in range(nbz):
        for by in range(nby):
            for bx in range(nbx):
                ext = [nt + (face_dir == 2), nt + (face_dir == 1), nt + (face_dir == 0)]
                out.append(a[bz * n: bz * n + ext[0], by * n: by * n + ext[1], bx * n: bx * n + ext[2]])
    return np.stack(out)


@pytest.mark.parametrize("periodic", [(True, True, True), (False, False, False), (True, False, False)])
def test_T26_exchange_equals_padded_global_array(periodic):
    n, nb3 = 6, (2, 2, 2)
    N = 2 * n
    rng = np.random.default_rng(5)
    modes = ["wrap" if p else "edge" for p in periodic]
    bc = [0 if p else 1 for p in periodic]
    nbr = lattice_nbr(nb3, periodic)
    nmb = 8
    par = orc.make_params(nmb=nmb, n=n)
    sh = orc.shapes(nmb, n)
    s = slice(NG, NG + n)
    # cells
    Gc = [rng.uniform(-1, 1, (N, N, N)) for _ in range(5)]
    expU = [split(g, nb3, n, modes) for g in Gc]
    U = [np.full(sh["cell"], np.nan) for _ in range(5)]
    for v in range(5):
        U[v][:, s, s, s] = expU[v][:, s, s, s]
    # faces: N entries along a periodic normal, N+1 along a bounded one
    Bf, expB = [], []
    for d, key in enumerate(("xf", "yf", "zf")):
        shp = [N, N, N]
        shp[2 - d] = N if periodic[d] else N + 1
        G = rng.uniform(-1, 1, shp)
        e = split(G, nb3, n, modes, face_dir=d)
        b = np.full(sh[key], np.nan)
        sl = [slice(None), s, s, s]
        sl[3 - d] = slice(NG, NG + n + 1)
        view = b[..., :n + 2 * NG + 1] if d == 0 else b
        view[tuple(sl)] = e[tuple(sl)]
        Bf.append(b); expB.append(e)
    orc.exchange_ghosts(par, nbr, bc, U, Bf)
    for v in range(5):
        assert np.array_equal(U[v], expU[v]), v
    nt = n + 2 * NG
    for d in range(3):
        got = Bf[d][..., :nt + 1] if d == 0 else Bf[d]
        assert np.array_equal(got, expB[d]), d


def test_T27_blocks_with_exchange_evolve_like_one_block():
    """[0,1]^3 periodic, flat space, magnetised smooth flow with a low-density patch (FOFC flags):
    one 12^3 block with its own periodic fill vs 2x2x2 blocks of 6^3 with exchange; RK3, 2 steps."""
    N, n = 12, 6
    d = 1.0 / N

    def prim(x, y, z):
        rho = 1.0 + 0.3 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) + 0.2 * np.sin(2 * np.pi * z)
        rho = np.where((abs(x - 0.3) < 0.1) & (abs(y - 0.6) < 0.1) & (abs(z - 0.5) < 0.1), 1e-3 * rho, rho)
        o = np.ones_like(x)
        return rho, [0.3 * np.sin(2 * np.pi * y) * o, -0.2 * o, 0.25 * np.cos(2 * np.pi * x) * o], 0.6 * o

    def A(comp, x, y, z):
        return 0.1 * np.sin(2 * np.pi * (x + 2 * y)) if comp == 2 else 0.05 * np.cos(2 * np.pi * z) * (comp == 0) + 0 * x
    p = dict(gamma_ad=5.0 / 3.0, rho_atm=1e-10, T_atm=1e-8, recon=2, riemann=1, fofc=1, dmp_M=1.2)
    one = sk.build_block(N, d, (0, 0, 0), sk.flat_metric, prim, A_fn=A, gamma_ad=5.0 / 3.0)
    par1 = orc.make_params(nmb=1, n=N, **p)
    U1 = [u.copy() for u in one["U"]]; B1 = [b.copy() for b in one["Bf"]]
    dt = 0.15 * d
    W1, f1 = orc.advance(par1, one["dx"], 3, 2, dt, (0, 0, 0), U1, B1, one["adm"], nthreads=4)
    assert np.count_nonzero(f1) > 0
    # the same data as 8 blocks: cut (with ghosts) out of the periodically filled single block, so
    # that both runs start from bit-identical numbers
    nb3 = (2, 2, 2)
    U0 = [u.copy() for u in one["U"]]; B0 = [b.copy() for b in one["Bf"]]
    orc.fill_ghosts(par1, (0, 0, 0), U0, B0)
    nts = n + 2 * NG

    def cut(a, face_dir=None):
        out = []
        for bz in range(2):
            for by in range(2):
                for bx in range(2):
                    ext = [nts + (face_dir == 2), nts + (face_dir == 1), nts + (face_dir == 0)]
                    out.append(a[0, bz * n: bz * n + ext[0], by * n: by * n + ext[1], bx * n: bx * n + ext[2]])
        return np.ascontiguousarray(np.stack(out))
    U8 = [cut(u) for u in U0]
    sh8 = orc.shapes(8, n)
    B8 = [np.zeros(sh8["xf"]), cut(B0[1], 1), cut(B0[2], 2)]
    B8[0][..., :nts + 1] = cut(B0[0][..., :N + 2 * NG + 1], 0)
    adm8 = [np.ascontiguousarray(np.broadcast_to(a[0, :1, :1, :1], sh8["cell"])) for a in one["adm"]]
    dx8 = np.full((8, 3), d)
    par8 = orc.make_params(nmb=8, n=n, **p)
    nbr = lattice_nbr(nb3, (True, True, True))
    W8, f8 = orc.advance_nbr(par8, dx8, 3, 2, dt, (0, 0, 0), nbr, U8, B8, adm8, nthreads=4)
    s1 = slice(NG, NG + N)
    for bz in range(2):
        for by in range(2):
            for bx in range(2):
                m = (bz * 2 + by) * 2 + bx
                sb = slice(NG, NG + n)
                gl = (0, slice(NG + bz * n, NG + bz * n + n), slice(NG + by * n, NG + by * n + n),
                      slice(NG + bx * n, NG + bx * n + n))
                for v in range(5):
                    assert np.array_equal(U8[v][m, sb, sb, sb], U1[v][gl]), (m, v)
                assert np.array_equal(f8[m, sb, sb, sb], f1[gl])
                # x-faces of the block, including the shared face ie+1
                glx = (0, gl[1], gl[2], slice(NG + bx * n, NG + bx * n + n + 1))
                assert np.array_equal(B8[0][m, sb, sb, NG:NG + n + 1], B1[0][glx])
