"""Thin ctypes binding of include/ak.h — argument marshalling only.

Every step of the stage runs in the CUDA kernels of libak.so; this module converts torch
tensors (device memory, streams) to the plain pointers of the C-ABI and raises on any
non-zero return code.  There is no CPU path: if libak.so is missing or cannot be loaded the
import of the library fails loudly (build it with `python -m paper_2409_10384_b200.build`).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.environ.get("AK_LIBRARY") or os.path.join(_HERE, "libak.so")   # AK_LIBRARY: another build of the same library

AK_OK, AK_EINVAL, AK_ENOMEM, AK_ECUDA, AK_ESTATE, AK_EHOOK, AK_ETOOBIG = 0, -1, -2, -3, -4, -5, -6
STATIC_MAX_CELLS = 2097152      # AK_STATIC_MAX_CELLS of include/ak.h
RECON_DC, RECON_PPM4, RECON_WENOZ, RECON_PLM, RECON_PPMX = 0, 1, 2, 3, 4
RS_LLF, RS_HLLE = 0, 1
ST_DFLOOR, ST_TAUFLOOR, ST_MAGCAP, ST_RHOFLOOR, ST_TFLOOR, ST_FAIL, ST_DMP = 1, 2, 4, 8, 16, 32, 64
KERNEL_CLASSES = ("con2prim", "flux_x", "flux_y", "flux_z", "fofc_test", "fofc_fix", "ct", "div_src")
EXPORTS = ("ak_create", "ak_set_metric", "ak_con2prim", "ak_rhs", "ak_emf", "ak_get_stats",
           "ak_get_flux", "ak_rhs_host", "ak_timing", "ak_kernel_ms", "ak_probe_copy",
           "ak_probe_fp64", "ak_destroy", "ak_strerror", "ak_version",
           "ak_set_fofc_blend", "ak_fill_ghosts", "ak_stage_update", "ak_advance", "ak_set_neighbors",
           "ak_matter_sources", "ak_halo_slab_elems", "ak_halo_pack", "ak_halo_unpack",
           "ak_set_eos_hybrid", "ak_set_overlap", "ak_advance_hooked",
           "ak_set_exact_shortcuts", "ak_con2prim_static", "ak_set_graph", "ak_graph_replays")
BC_PERIODIC, BC_OUTFLOW = 0, 1

_dp = C.POINTER(C.c_double)


class AkParams(C.Structure):
    _fields_ = [("nmb", C.c_int), ("n", C.c_int), ("ng", C.c_int),
                ("gamma_ad", C.c_double), ("rho_atm", C.c_double), ("T_atm", C.c_double),
                ("f_thr", C.c_double), ("mag_max", C.c_double),
                ("recon", C.c_int), ("riemann", C.c_int), ("fofc", C.c_int), ("fofc_riemann", C.c_int),
                ("dmp_M", C.c_double), ("c2p_max_iter", C.c_int), ("c2p_tol", C.c_double),
                ("device", C.c_int), ("stream", C.c_void_p)]


class AkCons(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("D", "Sx", "Sy", "Sz", "tau")]


class AkFaceB(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("bx", "by", "bz")]


class AkPrim(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("rho", "ux", "uy", "uz", "p", "bccx", "bccy", "bccz")]


class AkAdm(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("gxx", "gxy", "gxz", "gyy", "gyz", "gzz", "alp", "betx", "bety",
                                          "betz", "Kxx", "Kxy", "Kxz", "Kyy", "Kyz", "Kzz")]


class AkRhsOut(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("dD", "dSx", "dSy", "dSz", "dtau", "Ex", "Ey", "Ez",
                                          "fofc_flag", "c2p_status", "matter")]


class AkMatter(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("E", "Sx", "Sy", "Sz", "Sxx", "Sxy", "Sxz", "Syy", "Syz", "Szz")]


class AkStats(C.Structure):
    _fields_ = [("n_c2p_fail", C.c_longlong), ("n_cons_floor", C.c_longlong),
                ("n_prim_floor", C.c_longlong), ("n_fofc_cells", C.c_longlong),
                ("n_dmp_cells", C.c_longlong), ("n_fofc_faces", C.c_longlong * 3)]


REFRESH_FN = C.CFUNCTYPE(C.c_int, C.c_void_p)      # ak_refresh_fn of include/ak.h


class AkError(RuntimeError):
    def __init__(self, code, what):
        super().__init__("%s failed: %d (%s)" % (what, code, strerror(code)))
        self.code = code


_lib = None


def lib():
    """Load libak.so.  Raises if it is missing: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise ImportError("libak.so not built: run `python -m paper_2409_10384_b200.build` "
                              "(nvcc, sm_100a); the library has no CPU fallback")
        L = C.CDLL(SO_PATH)
        L.ak_strerror.restype = C.c_char_p
        L.ak_strerror.argtypes = [C.c_int]
        L.ak_version.restype = C.c_char_p
        L.ak_create.argtypes = [C.POINTER(AkParams), _dp, C.POINTER(C.c_void_p)]
        L.ak_set_metric.argtypes = [C.c_void_p, C.POINTER(AkAdm)]
        L.ak_con2prim.argtypes = [C.c_void_p, C.POINTER(AkCons), C.POINTER(AkFaceB), C.POINTER(AkPrim), C.c_void_p]
        L.ak_rhs.argtypes = [C.c_void_p, C.POINTER(AkCons), C.POINTER(AkFaceB), C.POINTER(AkPrim), C.c_int,
                             C.c_double, C.POINTER(AkRhsOut)]
        L.ak_rhs_host.argtypes = [C.c_void_p, C.POINTER(AkCons), C.POINTER(AkFaceB), C.POINTER(AkPrim),
                                  C.c_double, C.POINTER(AkRhsOut)]
        L.ak_emf.argtypes = [C.c_void_p, C.POINTER(AkPrim), C.c_void_p, C.c_void_p, C.c_void_p]
        L.ak_get_stats.argtypes = [C.c_void_p, C.POINTER(AkStats)]
        L.ak_get_flux.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.ak_timing.argtypes = [C.c_void_p, C.c_int]
        L.ak_kernel_ms.argtypes = [C.c_void_p, _dp, C.POINTER(C.c_longlong)]
        L.ak_probe_copy.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong, C.c_int, _dp]
        L.ak_probe_fp64.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp]
        L.ak_destroy.argtypes = [C.c_void_p]
        L.ak_set_eos_hybrid.argtypes = [C.c_void_p, C.c_int, C.c_double, _dp, _dp, C.c_double]
        L.ak_halo_slab_elems.restype = C.c_longlong
        L.ak_halo_slab_elems.argtypes = [C.c_void_p, C.c_int]
        L.ak_halo_pack.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.POINTER(AkCons), C.POINTER(AkFaceB), C.c_void_p]
        L.ak_halo_unpack.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.POINTER(AkCons), C.POINTER(AkFaceB)]
        L.ak_set_fofc_blend.argtypes = [C.c_void_p, C.POINTER(AkCons), C.c_double, C.c_double]
        L.ak_fill_ghosts.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(AkCons), C.POINTER(AkFaceB)]
        L.ak_stage_update.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.POINTER(AkCons),
                                      C.POINTER(AkFaceB), C.POINTER(AkCons), C.POINTER(AkFaceB),
                                      C.POINTER(AkRhsOut)]
        L.ak_advance.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int), C.POINTER(AkCons),
                                 C.POINTER(AkFaceB), C.POINTER(AkPrim), C.c_void_p]
        L.ak_advance_hooked.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int), C.POINTER(AkCons),
                                        C.POINTER(AkFaceB), C.POINTER(AkPrim), C.c_void_p, REFRESH_FN, C.c_void_p]
        L.ak_matter_sources.argtypes = [C.c_void_p, C.POINTER(AkPrim), C.POINTER(AkMatter)]
        L.ak_set_neighbors.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.c_int]
        L.ak_set_overlap.argtypes = [C.c_void_p, C.c_int]
        L.ak_set_exact_shortcuts.argtypes = [C.c_void_p, C.c_int]
        L.ak_set_graph.argtypes = [C.c_void_p, C.c_int]
        L.ak_graph_replays.argtypes = [C.c_void_p]
        L.ak_graph_replays.restype = C.c_longlong
        L.ak_con2prim_static.argtypes = [C.POINTER(AkParams), C.POINTER(AkCons), C.POINTER(AkFaceB), C.POINTER(AkAdm),
                                         C.POINTER(AkPrim), C.c_void_p, C.POINTER(AkStats)]
        _lib = L
    return _lib


def use_library(path=None):
    """Switch the binding to another build of the same library (None: the default libak.so), e.g. the
    FMA-contracted libak_fma.so of build.py.  Contexts belong to the library that created them:
    destroy them before switching."""
    global _lib, SO_PATH
    SO_PATH = path or os.environ.get("AK_LIBRARY") or os.path.join(_HERE, "libak.so")
    _lib = None
    return lib()


def strerror(code):
    return lib().ak_strerror(int(code)).decode()


def version():
    return lib().ak_version().decode()


def _chk(code, what):
    if code != AK_OK:
        raise AkError(code, what)


def shapes(nmb, n):
    """array shapes of the boundary layouts (include/ak.h)."""
    nt = n + 8
    px = nt + 4
    return dict(cell=(nmb, nt, nt, nt), xf=(nmb, nt, nt, px), yf=(nmb, nt, nt + 1, nt), zf=(nmb, nt + 1, nt, nt),
                ex=(nmb, nt + 1, nt + 1, nt), ey=(nmb, nt + 1, nt, px), ez=(nmb, nt, nt + 1, px))


def _ptr(t):
    """data pointer of a torch tensor or numpy array (contiguity is the caller's contract)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _struct(cls, seq):
    seq = list(seq)
    assert len(seq) == len(cls._fields_), (cls.__name__, len(seq))
    return cls(*[_ptr(t) for t in seq])


def make_params(nmb, n, gamma_ad, rho_atm, T_atm, f_thr=1.0, mag_max=float("inf"), recon=RECON_PPM4,
                riemann=RS_HLLE, fofc=1, fofc_riemann=RS_LLF, dmp_M=0.0, c2p_max_iter=40, c2p_tol=1e-15,
                device=0, stream=0, ng=4, **_ignored):
    return AkParams(nmb, n, ng, gamma_ad, rho_atm, T_atm, f_thr, mag_max, recon, riemann, fofc, fofc_riemann,
                    dmp_M, c2p_max_iter, c2p_tol, device, stream)


# ---------------------------------------------------------------- the C-ABI, same names
def ak_create(params, dx3):
    dx3 = np.ascontiguousarray(dx3, dtype=np.float64)
    assert dx3.size == 3 * params.nmb
    h = C.c_void_p()
    _chk(lib().ak_create(C.byref(params), dx3.ctypes.data_as(_dp), C.byref(h)), "ak_create")
    return h


def ak_set_metric(ctx, adm):
    s = _struct(AkAdm, adm)
    _chk(lib().ak_set_metric(ctx, C.byref(s)), "ak_set_metric")


def ak_con2prim(ctx, U, Bf, W, status=None):
    u, b, w = _struct(AkCons, U), _struct(AkFaceB, Bf), _struct(AkPrim, W)
    _chk(lib().ak_con2prim(ctx, C.byref(u), C.byref(b), C.byref(w), _ptr(status)), "ak_con2prim")


def ak_rhs(ctx, U, Bf, W, w_is_valid, dt_fofc, dU, E, fofc_flag=None, c2p_status=None, matter=None):
    """matter: None or ten device cell fields E, S_i, S_ij written on interior cells by part (6)."""
    u, b, w = _struct(AkCons, U), _struct(AkFaceB, Bf), _struct(AkPrim, W)
    m = _struct(AkMatter, matter) if matter is not None else None
    o = _struct(AkRhsOut, list(dU) + list(E) + [fofc_flag, c2p_status, None])
    if m is not None:
        o.matter = C.cast(C.pointer(m), C.c_void_p)
    _chk(lib().ak_rhs(ctx, C.byref(u), C.byref(b), C.byref(w), int(w_is_valid), float(dt_fofc), C.byref(o)),
         "ak_rhs")


def ak_rhs_host(ctx, U, Bf, W, dt_fofc, dU, E, fofc_flag=None, c2p_status=None):
    """same stage with HOST buffers (numpy arrays or pinned CPU tensors); W = None: primitives not returned."""
    u, b = _struct(AkCons, U), _struct(AkFaceB, Bf)
    w = _struct(AkPrim, W) if W is not None else AkPrim()
    o = _struct(AkRhsOut, list(dU) + list(E) + [fofc_flag, c2p_status, None])
    _chk(lib().ak_rhs_host(ctx, C.byref(u), C.byref(b), C.byref(w), float(dt_fofc), C.byref(o)), "ak_rhs_host")


def ak_con2prim_static(params, U, Bf, adm, W, status=None, want_counts=False):
    """con2prim without a context and without any allocation (include/ak.h).  adm: the 16 ADM fields (only
    gamma_ij is read).  Returns the three con2prim counters when want_counts (synchronises), else None."""
    u, b, a, w = _struct(AkCons, U), _struct(AkFaceB, Bf), _struct(AkAdm, adm), _struct(AkPrim, W)
    s = AkStats()
    _chk(lib().ak_con2prim_static(C.byref(params), C.byref(u), C.byref(b), C.byref(a), C.byref(w), _ptr(status),
                                  C.byref(s) if want_counts else None), "ak_con2prim_static")
    if want_counts:
        return dict(n_c2p_fail=s.n_c2p_fail, n_cons_floor=s.n_cons_floor, n_prim_floor=s.n_prim_floor)
    return None


def ak_set_graph(ctx, on):
    """CUDA-graph replay of the serial stage (include/ak.h)."""
    _chk(lib().ak_set_graph(ctx, int(on)), "ak_set_graph")


def ak_graph_replays(ctx):
    return int(lib().ak_graph_replays(ctx))


def ak_set_exact_shortcuts(ctx, mask):
    """bit 0: skip the reconstruction of all-zero fields, bit 1: static-cell con2prim (include/ak.h)."""
    _chk(lib().ak_set_exact_shortcuts(ctx, int(mask)), "ak_set_exact_shortcuts")


def ak_set_overlap(ctx, nchunks):
    """schedule of ak_rhs: < 2 serial, else pipelined over nchunks groups of blocks (include/ak.h)."""
    _chk(lib().ak_set_overlap(ctx, int(nchunks)), "ak_set_overlap")


def ak_emf(ctx, W, Ex, Ey, Ez):
    w = _struct(AkPrim, W)
    _chk(lib().ak_emf(ctx, C.byref(w), _ptr(Ex), _ptr(Ey), _ptr(Ez)), "ak_emf")


def ak_get_stats(ctx):
    s = AkStats()
    _chk(lib().ak_get_stats(ctx, C.byref(s)), "ak_get_stats")
    return dict(n_c2p_fail=s.n_c2p_fail, n_cons_floor=s.n_cons_floor, n_prim_floor=s.n_prim_floor,
                n_fofc_cells=s.n_fofc_cells, n_dmp_cells=s.n_dmp_cells, n_fofc_faces=list(s.n_fofc_faces))


def ak_get_flux(ctx, d, comp, dst):
    _chk(lib().ak_get_flux(ctx, int(d), int(comp), _ptr(dst)), "ak_get_flux")


def ak_timing(ctx, enable):
    _chk(lib().ak_timing(ctx, int(enable)), "ak_timing")


def ak_kernel_ms(ctx):
    ms = (C.c_double * 8)()
    nl = (C.c_longlong * 8)()
    _chk(lib().ak_kernel_ms(ctx, ms, nl), "ak_kernel_ms")
    return dict(zip(KERNEL_CLASSES, list(ms))), dict(zip(KERNEL_CLASSES, list(nl)))


def ak_probe_copy(ctx, dst, src, n_doubles, reps=5):
    g = C.c_double()
    _chk(lib().ak_probe_copy(ctx, _ptr(dst), _ptr(src), int(n_doubles), int(reps), C.byref(g)), "ak_probe_copy")
    return g.value


def ak_probe_fp64(ctx, use_fma, reps=3):
    g = C.c_double()
    _chk(lib().ak_probe_fp64(ctx, int(use_fma), int(reps), C.byref(g)), "ak_probe_fp64")
    return g.value


def ak_destroy(ctx):
    _chk(lib().ak_destroy(ctx), "ak_destroy")


# ---------------------------------------------------------------- stage driver (same names)
def _bc(bc):
    return (C.c_int * 3)(*[int(b) for b in bc])


def ak_set_fofc_blend(ctx, U0, a=0.0, b=1.0):
    if U0 is None:
        _chk(lib().ak_set_fofc_blend(ctx, None, 0.0, 1.0), "ak_set_fofc_blend")
    else:
        u = _struct(AkCons, U0)
        _chk(lib().ak_set_fofc_blend(ctx, C.byref(u), float(a), float(b)), "ak_set_fofc_blend")


def ak_set_eos_hybrid(ctx, K0, gammas, rho_breaks=(), gamma_th=2.0):
    """Piecewise-polytropic hybrid EOS (include/ak.h); gammas = () returns to the ideal gas."""
    g = (C.c_double * max(len(gammas), 1))(*[float(x) for x in gammas])
    r = (C.c_double * max(len(rho_breaks), 1))(*[float(x) for x in rho_breaks])
    if len(gammas) > 0 and len(rho_breaks) != len(gammas) - 1:
        raise ValueError("rho_breaks must hold len(gammas) - 1 values")
    _chk(lib().ak_set_eos_hybrid(ctx, len(gammas), C.c_double(float(K0)), g, r, C.c_double(float(gamma_th))),
         "ak_set_eos_hybrid")


def ak_fill_ghosts(ctx, bc, U, Bf):
    u, b = _struct(AkCons, U), _struct(AkFaceB, Bf)
    _chk(lib().ak_fill_ghosts(ctx, _bc(bc), C.byref(u), C.byref(b)), "ak_fill_ghosts")


def ak_stage_update(ctx, a, b, dt, U0, B0, U, Bf, dU, E):
    u0, b0, u, bf = _struct(AkCons, U0), _struct(AkFaceB, B0), _struct(AkCons, U), _struct(AkFaceB, Bf)
    o = _struct(AkRhsOut, list(dU) + list(E) + [None, None, None])
    _chk(lib().ak_stage_update(ctx, float(a), float(b), float(dt), C.byref(u0), C.byref(b0), C.byref(u),
                               C.byref(bf), C.byref(o)), "ak_stage_update")


def ak_advance(ctx, integrator, nsteps, dt, bc, U, Bf, W, flag_or=None):
    u, bf, w = _struct(AkCons, U), _struct(AkFaceB, Bf), _struct(AkPrim, W)
    _chk(lib().ak_advance(ctx, int(integrator), int(nsteps), float(dt), _bc(bc), C.byref(u), C.byref(bf),
                          C.byref(w), _ptr(flag_or)), "ak_advance")


def ak_advance_hooked(ctx, integrator, nsteps, dt, bc, U, Bf, W, flag_or=None, refresh=None):
    """ak_advance with `refresh()` (a Python callable or None) run before every ghost fill."""
    u, bf, w = _struct(AkCons, U), _struct(AkFaceB, Bf), _struct(AkPrim, W)
    err = []

    def _cb(_user):
        try:
            refresh()
            return 0
        except BaseException as e:      # never unwind through C
            err.append(e)
            return 1
    cb = REFRESH_FN(_cb) if refresh is not None else C.cast(None, REFRESH_FN)
    code = lib().ak_advance_hooked(ctx, int(integrator), int(nsteps), float(dt), _bc(bc), C.byref(u), C.byref(bf),
                                   C.byref(w), _ptr(flag_or), cb, None)
    if err:
        raise err[0]
    _chk(code, "ak_advance_hooked")


def ak_set_neighbors(ctx, nbr, nmb_total=0):
    """nbr: int array [nmb][27] (host) or None; nmb_total: blocks in the arrays incl. read-only mirrors."""
    if nbr is None:
        _chk(lib().ak_set_neighbors(ctx, None, 0), "ak_set_neighbors")
        return
    a = np.ascontiguousarray(nbr, dtype=np.int32)
    _chk(lib().ak_set_neighbors(ctx, a.ctypes.data_as(C.POINTER(C.c_int)), int(nmb_total)), "ak_set_neighbors")


def ak_halo_slab_elems(ctx, code):
    """doubles in the ghost slab of neighbour code `code` (include/ak.h)."""
    v = int(lib().ak_halo_slab_elems(ctx, int(code)))
    if v < 0:
        raise ValueError("ak_halo_slab_elems: bad neighbour code %r" % (code,))
    return v


def ak_halo_pack(ctx, desc, U, Bf, buf):
    """desc: device int64 tensor [ndesc][3] = block, code, offset in buf; buf: device float64 tensor."""
    u, b = _struct(AkCons, U), _struct(AkFaceB, Bf)
    nd = 0 if desc is None else int(desc.shape[0])
    _chk(lib().ak_halo_pack(ctx, nd, _ptr(desc), C.byref(u), C.byref(b), _ptr(buf)),
         "ak_halo_pack")


def ak_halo_unpack(ctx, desc, buf, U, Bf):
    u, b = _struct(AkCons, U), _struct(AkFaceB, Bf)
    nd = 0 if desc is None else int(desc.shape[0])
    _chk(lib().ak_halo_unpack(ctx, nd, _ptr(desc), _ptr(buf), C.byref(u), C.byref(b)),
         "ak_halo_unpack")


def ak_matter_sources(ctx, W, out10):
    w, o = _struct(AkPrim, W), _struct(AkMatter, out10)
    _chk(lib().ak_matter_sources(ctx, C.byref(w), C.byref(o)), "ak_matter_sources")
