"""Helpers for the GPU parity tests: run a workload dict (numpy inputs in the boundary layouts)
through the C-ABI library via the ctypes binding, and compare with the oracle's outputs."""
import numpy as np

from paper_2409_10384_b200 import ak

RTOL = 1e-11          # BASELINE.json north_star: relative 1e-11 on dU/dt and EMFs ...
ATOL_FAC = 1e-14      # ... with an absolute floor of 1e-14 * max|U|


def to_dev(arrs, dev="cuda:0"):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in arrs]


class GpuStage:
    """Owns device tensors for one batch and a library context."""

    def __init__(self, w, dev="cuda:0", **override):
        import torch
        self.torch = torch
        p = dict(w["params"]); p.update(override)
        self.pd = p
        self.nmb, self.n = p["nmb"], p["n"]
        self.sh = ak.shapes(self.nmb, self.n)
        self.dev = dev
        self.U = to_dev(w["U"], dev); self.Bf = to_dev(w["Bf"], dev); self.adm = to_dev(w["adm"], dev)
        z = lambda k, dt=torch.float64: torch.zeros(self.sh[k], dtype=dt, device=dev)
        self.W = [z("cell") for _ in range(8)]
        self.dU = [z("cell") for _ in range(5)]
        self.E = [z("ex"), z("ey"), z("ez")]
        self.flag = z("cell", torch.uint8); self.status = z("cell", torch.uint8)
        self.dt_fofc = w["dt_fofc"]
        stream = torch.cuda.current_stream(dev).cuda_stream
        self.params = ak.make_params(device=torch.device(dev).index or 0, stream=stream, **p)
        self.ctx = ak.ak_create(self.params, w["dx"])
        ak.ak_set_metric(self.ctx, self.adm)
        hyb = p.get("eos_hybrid")
        if hyb is not None:
            ak.ak_set_eos_hybrid(self.ctx, hyb["K0"], hyb["gammas"], hyb.get("rho_breaks", ()), hyb["gamma_th"])

    def con2prim(self):
        ak.ak_con2prim(self.ctx, self.U, self.Bf, self.W, self.status)
        self.torch.cuda.synchronize()

    def rhs(self, w_is_valid=False, dt=None):
        ak.ak_rhs(self.ctx, self.U, self.Bf, self.W, int(w_is_valid), self.dt_fofc if dt is None else dt,
                  self.dU, self.E, self.flag, self.status)
        self.torch.cuda.synchronize()

    def flux(self):
        torch = self.torch
        out = []
        for d, k in enumerate(("xf", "yf", "zf")):
            for c in range(7):
                t = torch.zeros(self.sh[k], dtype=torch.float64, device=self.dev)
                ak.ak_get_flux(self.ctx, d, c, t)
                out.append(t)
        torch.cuda.synchronize()
        return [t.cpu().numpy() for t in out]

    def result(self):
        c = lambda ts: [t.cpu().numpy() for t in ts]
        return dict(W=c(self.W), dU=c(self.dU), E=c(self.E), flag=self.flag.cpu().numpy(),
                    status=self.status.cpu().numpy(), U=c(self.U))

    def stats(self):
        return ak.ak_get_stats(self.ctx)

    def close(self):
        if self.ctx is not None:
            ak.ak_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


def max_rel_dev(a, b, atol):
    """max over elements of |a-b| / (rtol-normalised bound); <= 1 passes.  Also returns max |a-b|."""
    d = np.abs(a - b)
    bound = atol + RTOL * np.abs(b)
    bad = ~(np.isfinite(a) & np.isfinite(b))
    same_nonfinite = bad & ((a == b) | (np.isnan(a) & np.isnan(b)))
    d = np.where(same_nonfinite, 0.0, d)
    if not d.size:
        return 0.0, 0.0
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(d == 0.0, 0.0, d / bound)     # identical values pass even when the bound is 0
    return float(np.max(ratio)), float(np.max(d))


def assert_parity(gpu, orc, U_in, label=""):
    """gpu, orc: dicts with W, dU, E, flag, status (+U after floors for gpu; orc's U list is the
    in-place-modified input).  U_in: the 5 input conserved arrays (for the absolute floor)."""
    umax = [float(np.max(np.abs(u))) for u in U_in]
    uall = max(umax)
    report = {}
    assert np.array_equal(gpu["status"], orc["status"]), label + ": con2prim status bytes differ at %d cells" % \
        int(np.count_nonzero(gpu["status"] != orc["status"]))
    assert np.array_equal(gpu["flag"], orc["flag"]), label + ": FOFC flag bytes differ at %d cells" % \
        int(np.count_nonzero(gpu["flag"] != orc["flag"]))
    for v in range(8):
        wmax = float(np.max(np.abs(orc["W"][v])))
        r, d = max_rel_dev(gpu["W"][v], orc["W"][v], ATOL_FAC * max(wmax, 1e-300))
        report["W%d" % v] = (r, d)
        assert r <= 1.0, "%s: W[%d] off by %.3g x tolerance (max abs %.3g)" % (label, v, r, d)
    for v in range(5):
        r, d = max_rel_dev(gpu["dU"][v], orc["dU"][v], ATOL_FAC * umax[v])
        report["dU%d" % v] = (r, d)
        assert r <= 1.0, "%s: dU[%d] off by %.3g x tolerance (max abs %.3g)" % (label, v, r, d)
    for v in range(3):
        r, d = max_rel_dev(gpu["E"][v], orc["E"][v], ATOL_FAC * uall)
        report["E%d" % v] = (r, d)
        assert r <= 1.0, "%s: E[%d] off by %.3g x tolerance (max abs %.3g)" % (label, v, r, d)
    if "U" in gpu and "U" in orc:
        for v in range(5):
            r, d = max_rel_dev(gpu["U"][v], orc["U"][v], ATOL_FAC * umax[v])
            assert r <= 1.0, "%s: floored U[%d] off by %.3g x tolerance" % (label, v, r)
    return report
