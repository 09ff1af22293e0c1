"""ctypes loader for the CPU ORACLE (test infrastructure only — see oracle/oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this module.  It never imports the CUDA binding.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = ["point.cpp", "stage.cpp", "driver.cpp"]


def build(force=False):
    """g++ -O2 -ffp-contract=off: no FMA contraction, IEEE fp64 in the written order."""
    srcs = [os.path.join(_HERE, s) for s in _SRC] + [os.path.join(_HERE, "oracle.h"), os.path.join(_HERE, "eos.h")]
    if not force and os.path.exists(_SO) and all(
            os.path.getmtime(_SO) >= os.path.getmtime(s) for s in srcs):
        return _SO
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c++17", "-o", _SO] + \
          [os.path.join(_HERE, s) for s in _SRC] + ["-lpthread"]
    subprocess.check_call(cmd)
    return _SO


class OrcParams(C.Structure):
    _fields_ = [("nmb", C.c_int), ("n", C.c_int), ("ng", C.c_int),
                ("gamma_ad", C.c_double), ("rho_atm", C.c_double), ("T_atm", C.c_double),
                ("f_thr", C.c_double), ("mag_max", C.c_double),
                ("recon", C.c_int), ("riemann", C.c_int), ("fofc", C.c_int),
                ("fofc_riemann", C.c_int), ("dmp_M", C.c_double),
                ("c2p_max_iter", C.c_int), ("c2p_tol", C.c_double),
                ("eos", C.c_int), ("pp_nseg", C.c_int), ("pp_K0", C.c_double),
                ("pp_gamma", C.c_double * 4), ("pp_rho", C.c_double * 3), ("gamma_th", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.orc_c2p_master.restype = C.c_double
        _lib.orc_c2p_master.argtypes = [C.c_double] * 6
        _lib.orc_con2prim_cell.restype = C.c_int
        _lib.orc_c2p_master_eos.restype = C.c_double
        _lib.orc_c2p_master_eos.argtypes = [C.c_void_p] + [C.c_double] * 6
    return _lib


def make_params(nmb=1, n=4, gamma_ad=2.0, rho_atm=1e-10, T_atm=1e-8, f_thr=1.0,
                mag_max=float("inf"), recon=1, riemann=1, fofc=1, fofc_riemann=0, dmp_M=0.0,
                c2p_max_iter=40, c2p_tol=1e-15, eos_hybrid=None, **_ignored):
    """eos_hybrid: None (ideal gas with gamma_ad) or dict(K0, gammas, rho_breaks, gamma_th)."""
    p = OrcParams(nmb, n, 4, gamma_ad, rho_atm, T_atm, f_thr, mag_max, recon, riemann,
                  fofc, fofc_riemann, dmp_M, c2p_max_iter, c2p_tol)
    if eos_hybrid is not None:
        gam, rb = list(eos_hybrid["gammas"]), list(eos_hybrid.get("rho_breaks", []))
        assert 1 <= len(gam) <= 4 and len(rb) == len(gam) - 1
        p.eos, p.pp_nseg, p.pp_K0, p.gamma_th = 1, len(gam), eos_hybrid["K0"], eos_hybrid["gamma_th"]
        for i, x in enumerate(gam):
            p.pp_gamma[i] = x
        for i, x in enumerate(rb):
            p.pp_rho[i] = x
    return p


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _ptrs(arrs, const=True):
    """array of double* from a list of contiguous float64 arrays (None -> NULL)."""
    P = (C.c_void_p * len(arrs))()
    for i, a in enumerate(arrs):
        if a is None:
            P[i] = None
        else:
            assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
            P[i] = a.ctypes.data
    return P


# ------------------------------------------------------------------ point level
def metric_inverse(g):
    g, gp = _d(g)
    det, sdet = C.c_double(), C.c_double()
    gi = np.zeros(6)
    lib().orc_metric_inverse(gp, C.byref(det), C.byref(sdet), gi.ctypes.data_as(_dp))
    return det.value, sdet.value, gi


def prim2cons(gamma_ad, g, prim, B):
    g, gp = _d(g); prim, pp = _d(prim); B, bp = _d(B)
    out = np.zeros(5)
    lib().orc_prim2cons(C.c_double(gamma_ad), gp, pp, bp, out.ctypes.data_as(_dp))
    return out


def con2prim_cell(par, g, Ut, Btcc, check_only=False):
    """returns (status, W[5], Ut_after[5], iters)"""
    g, gp = _d(g); Ut = np.array(Ut, dtype=np.float64); Bt, bp = _d(Btcc)
    W = np.zeros(5)
    it = C.c_int(0)
    st = lib().orc_con2prim_cell(C.byref(par), gp, Ut.ctypes.data_as(_dp), bp,
                                 W.ctypes.data_as(_dp), int(check_only), C.byref(it))
    return st, W, Ut, it.value


def prim2cons_eos(par, g, prim, B):
    g, gp = _d(g); prim, pp = _d(prim); B, bp = _d(B)
    out = np.zeros(5)
    lib().orc_prim2cons_eos(C.byref(par), gp, pp, bp, out.ctypes.data_as(_dp))
    return out


def eos_point(par, rho, eps):
    """{P(rho,eps), h-1, c_s^2, P_c, eps_c} of the EOS in par."""
    out = np.zeros(5)
    lib().orc_eos_point(C.byref(par), C.c_double(rho), C.c_double(eps), out.ctypes.data_as(_dp))
    return out


def c2p_master_eos(par, D, q, r2, bs2, rb2, mu):
    return lib().orc_c2p_master_eos(C.byref(par), D, q, r2, bs2, rb2, mu)


def c2p_master(gamma_ad, q, r2, bs2, rb2, mu):
    return lib().orc_c2p_master(gamma_ad, q, r2, bs2, rb2, mu)


def reconstruct(kind, q5):
    q5, qp_ = _d(q5)
    qm, qp = C.c_double(), C.c_double()
    lib().orc_reconstruct(int(kind), qp_, C.byref(qm), C.byref(qp))
    return qm.value, qp.value


def face_flux(par, d, riemann, gL, gR, WL, WR, Bfd, apply_floor=False, want_lam=False):
    gL, a = _d(gL); gR, b = _d(gR); WL, c = _d(WL); WR, e = _d(WR)
    F = np.zeros(7); lam = np.zeros(4)
    lib().orc_face_flux(C.byref(par), int(d), int(riemann), a, b, c, e, C.c_double(Bfd),
                        int(apply_floor), F.ctypes.data_as(_dp), lam.ctypes.data_as(_dp))
    return (F, lam) if want_lam else F


# ------------------------------------------------------------------ block level
def shapes(nmb, n, ng=4):
    nt = n + 2 * ng
    px = nt + 4
    return dict(cell=(nmb, nt, nt, nt), xf=(nmb, nt, nt, px), yf=(nmb, nt, nt + 1, nt),
                zf=(nmb, nt + 1, nt, nt), ex=(nmb, nt + 1, nt + 1, nt),
                ey=(nmb, nt + 1, nt, px), ez=(nmb, nt, nt + 1, px))


def con2prim(par, U, Bf, g, nthreads=1):
    """U: list of 5 cell arrays (modified in place), Bf: 3 face arrays, g: 6 cell arrays.
    returns W (8 arrays), status (u8)."""
    sh = shapes(par.nmb, par.n)
    W = [np.zeros(sh["cell"]) for _ in range(8)]
    st = np.zeros(sh["cell"], dtype=np.uint8)
    lib().orc_con2prim(C.byref(par), _ptrs(U), _ptrs(Bf), _ptrs(g), _ptrs(W),
                       st.ctypes.data_as(C.c_void_p), int(nthreads))
    return W, st


def rhs(par, dx, U, Bf, adm, dt_fofc, W=None, nthreads=1, want_flux=False):
    """One full stage.  U (5, modified in place where floored), Bf (3), adm (16): lists of
    float64 arrays in the boundary layouts.  Returns dict with W, dU, E, flag, status,
    and optionally flux (21 arrays) + refl (3 u8 arrays)."""
    sh = shapes(par.nmb, par.n)
    dx = np.ascontiguousarray(dx, dtype=np.float64).reshape(par.nmb, 3)
    w_valid = W is not None
    if W is None:
        W = [np.zeros(sh["cell"]) for _ in range(8)]
    dU = [np.zeros(sh["cell"]) for _ in range(5)]
    E = [np.zeros(sh["ex"]), np.zeros(sh["ey"]), np.zeros(sh["ez"])]
    flag = np.zeros(sh["cell"], dtype=np.uint8)
    status = np.zeros(sh["cell"], dtype=np.uint8)
    flux = refl = None
    fp = rp = None
    if want_flux:
        flux = [np.zeros(sh[k]) for k in ("xf", "yf", "zf") for _ in range(7)]
        refl = [np.zeros(sh[k], dtype=np.uint8) for k in ("xf", "yf", "zf")]
        fp = _ptrs(flux)
        rp = (C.c_void_p * 3)(*[r.ctypes.data for r in refl])
    lib().orc_rhs(C.byref(par), dx.ctypes.data_as(_dp), _ptrs(U), _ptrs(Bf), _ptrs(adm),
                  _ptrs(W), int(w_valid), C.c_double(dt_fofc), _ptrs(dU), _ptrs(E),
                  flag.ctypes.data_as(C.c_void_p), status.ctypes.data_as(C.c_void_p),
                  fp, rp, int(nthreads))
    return dict(W=W, dU=dU, E=E, flag=flag, status=status, flux=flux, refl=refl)


# ------------------------------------------------------------------ stage driver
def _ib(bc):
    return (C.c_int * 3)(*[int(b) for b in bc])


def fill_ghosts(par, bc, U, Bf):
    """in place.  bc[d]: 0 periodic, 1 outflow."""
    lib().orc_fill_ghosts(C.byref(par), _ib(bc), _ptrs(U), _ptrs(Bf))


def stage_update(par, dx, a, b, dt, U0, B0, U, Bf, dU, E):
    dx = np.ascontiguousarray(dx, dtype=np.float64).reshape(par.nmb, 3)
    lib().orc_stage_update(C.byref(par), dx.ctypes.data_as(_dp), C.c_double(a), C.c_double(b), C.c_double(dt),
                           _ptrs(U0), _ptrs(B0), _ptrs(U), _ptrs(Bf), _ptrs(dU), _ptrs(E))


def rhs_blend(par, dx, U, Bf, adm, dt_fofc, U0, fa, fb, nthreads=1):
    sh = shapes(par.nmb, par.n)
    dx = np.ascontiguousarray(dx, dtype=np.float64).reshape(par.nmb, 3)
    W = [np.zeros(sh["cell"]) for _ in range(8)]
    dU = [np.zeros(sh["cell"]) for _ in range(5)]
    E = [np.zeros(sh["ex"]), np.zeros(sh["ey"]), np.zeros(sh["ez"])]
    flag = np.zeros(sh["cell"], dtype=np.uint8)
    status = np.zeros(sh["cell"], dtype=np.uint8)
    lib().orc_rhs_blend(C.byref(par), dx.ctypes.data_as(_dp), _ptrs(U), _ptrs(Bf), _ptrs(adm), _ptrs(W), 0,
                        C.c_double(dt_fofc), _ptrs(U0) if U0 is not None else None, C.c_double(fa),
                        C.c_double(fb), _ptrs(dU), _ptrs(E), flag.ctypes.data_as(C.c_void_p),
                        status.ctypes.data_as(C.c_void_p), int(nthreads))
    return dict(W=W, dU=dU, E=E, flag=flag, status=status)


def advance(par, dx, integrator, nsteps, dt, bc, U, Bf, adm, nthreads=1):
    """nsteps of SSP-RK<integrator>; U, Bf advanced in place.  Returns (W, OR of FOFC flags)."""
    sh = shapes(par.nmb, par.n)
    dx = np.ascontiguousarray(dx, dtype=np.float64).reshape(par.nmb, 3)
    W = [np.zeros(sh["cell"]) for _ in range(8)]
    flag = np.zeros(sh["cell"], dtype=np.uint8)
    lib().orc_advance(C.byref(par), dx.ctypes.data_as(_dp), int(integrator), int(nsteps), C.c_double(dt),
                      _ib(bc), _ptrs(U), _ptrs(Bf), _ptrs(adm), _ptrs(W), flag.ctypes.data_as(C.c_void_p),
                      int(nthreads))
    return W, flag


def _nbr(nbr, nmb):
    a = np.ascontiguousarray(nbr, dtype=np.int32).reshape(nmb, 27)
    return a, a.ctypes.data_as(C.POINTER(C.c_int))


def exchange_ghosts(par, nbr, bc, U, Bf):
    a, ap = _nbr(nbr, par.nmb)
    lib().orc_exchange_ghosts(C.byref(par), ap, _ib(bc), _ptrs(U), _ptrs(Bf))


def advance_nbr(par, dx, integrator, nsteps, dt, bc, nbr, U, Bf, adm, nthreads=1):
    sh = shapes(par.nmb, par.n)
    dx = np.ascontiguousarray(dx, dtype=np.float64).reshape(par.nmb, 3)
    W = [np.zeros(sh["cell"]) for _ in range(8)]
    flag = np.zeros(sh["cell"], dtype=np.uint8)
    a, ap = _nbr(nbr, par.nmb)
    lib().orc_advance_nbr(C.byref(par), dx.ctypes.data_as(_dp), int(integrator), int(nsteps), C.c_double(dt),
                          _ib(bc), ap, _ptrs(U), _ptrs(Bf), _ptrs(adm), _ptrs(W),
                          flag.ctypes.data_as(C.c_void_p), int(nthreads))
    return W, flag


def advance_hooked(par, dx, integrator, nsteps, dt, bc, nbr, U, Bf, adm, refresh, nthreads=1):
    """advance_nbr with a Python callable run before every ghost fill; U, Bf may hold mirror blocks
    behind the par.nmb evolved ones (nbr = local table pointing at them)."""
    sh = shapes(par.nmb, par.n)
    dx = np.ascontiguousarray(dx, dtype=np.float64).reshape(par.nmb, 3)
    W = [np.zeros(sh["cell"]) for _ in range(8)]
    flag = np.zeros(sh["cell"], dtype=np.uint8)
    a, ap = _nbr(nbr, par.nmb)
    err = []

    def _cb(_user):
        try:
            refresh()
            return 0
        except BaseException as e:      # never unwind through C
            err.append(e)
            return 1
    cb = C.CFUNCTYPE(C.c_int, C.c_void_p)(_cb)
    lib().orc_advance_hooked.restype = C.c_int
    rc = lib().orc_advance_hooked(C.byref(par), dx.ctypes.data_as(_dp), int(integrator), int(nsteps), C.c_double(dt),
                                  _ib(bc), ap, _ptrs(U), _ptrs(Bf), _ptrs(adm), _ptrs(W),
                                  flag.ctypes.data_as(C.c_void_p), int(nthreads), cb, None)
    if err:
        raise err[0]
    assert rc == 0
    return W, flag


def matter_sources(par, W, g6):
    """E, S_i, S_ij (10 cell arrays, undensitised) from the primitives."""
    sh = shapes(par.nmb, par.n)
    out = [np.zeros(sh["cell"]) for _ in range(10)]
    lib().orc_matter_sources(C.byref(par), _ptrs(W), _ptrs(g6), _ptrs(out))
    return out
