"""Thin ctypes binding over liblya.so (include/lya.h).  Argument marshalling only:
every step of the path runs in the library's CUDA kernels.  PyTorch is used for
device memory and streams.  There is NO CPU fallback: if the library has not been
built, or there is no CUDA device, this raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblya.so")

EXPORTS = ["lya_create", "lya_destroy", "lya_last_error", "lya_version", "lya_launch_count", "lya_set_option", "lya_neighbours",
           "lya_pairs_export", "lya_pairs_import", "lya_pairs_subsample", "lya_pairs_count", "lya_pairs_free",
           "lya_xi2pcf", "lya_xi2pcf_sub", "lya_xi2pcf_means", "lya_dmat", "lya_run_host", "lya_xi_normalise", "lya_dmat_normalise",
           "lya_plan_create", "lya_plan_free", "lya_xi2pcf_plan", "lya_xi2pcf_plan_noalloc", "lya_dmat_plan", "lya_tri_nbins", "lya_xi3pcf"]

STATUS = {0: "LYA_OK", 1: "LYA_ERR_INVALID_ARG", 2: "LYA_ERR_UNSORTED", 3: "LYA_ERR_DEGENERATE_FOREST",
          4: "LYA_ERR_CAPACITY", 5: "LYA_ERR_OOM", 6: "LYA_ERR_CUDA", 7: "LYA_ERR_UNIMPLEMENTED"}
OPTIONS = {"force_generic": 0, "generic_diagonals": 1, "check_holders": 2, "xi_merge_every": 3}


class LyaError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status
        self.name = STATUS.get(status, str(status))


class CForests(C.Structure):
    _fields_ = [("n_forest", C.c_int64), ("n_pix", C.c_int64),
                ("ra", C.c_void_p), ("dec", C.c_void_p),
                ("ux", C.c_void_p), ("uy", C.c_void_p), ("uz", C.c_void_p),
                ("pix_off", C.c_void_p),
                ("chi", C.c_void_p), ("w", C.c_void_p), ("delta", C.c_void_p), ("loglam", C.c_void_p)]


class CBinning(C.Structure):
    _fields_ = [("rpar_max", C.c_double), ("rperp_max", C.c_double), ("n_par", C.c_int32), ("n_perp", C.c_int32)]


class CTriBinning(C.Structure):
    _fields_ = [("r_max", C.c_double), ("n_r", C.c_int32), ("n_theta", C.c_int32), ("n_cosa", C.c_int32)]


class CStats(C.Structure):
    _fields_ = [("n_forest_pairs", C.c_uint64), ("n_visited", C.c_uint64), ("n_evaluated", C.c_uint64),
                ("n_binned", C.c_uint64), ("n_kept", C.c_uint64), ("n_scatter", C.c_uint64), ("ms_main", C.c_float), ("ms_total", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def load():
    """dlopen liblya.so; raises if it is missing (build with paper_2507_00129_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python -m paper_2507_00129_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.lya_last_error.restype = C.c_char_p
        lib.lya_last_error.argtypes = [C.c_void_p]
        lib.lya_version.restype = C.c_char_p
        lib.lya_launch_count.restype = C.c_uint64
        lib.lya_pairs_count.restype = C.c_int64
        lib.lya_pairs_count.argtypes = [C.c_void_p]
        lib.lya_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
        lib.lya_destroy.argtypes = [C.c_void_p]
        lib.lya_neighbours.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning),
                                       C.POINTER(C.c_void_p), C.POINTER(C.c_int64)]
        lib.lya_pairs_export.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.lya_pairs_import.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_void_p)]
        lib.lya_pairs_free.argtypes = [C.c_void_p, C.c_void_p]
        lib.lya_pairs_subsample.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_uint64,
                                            C.POINTER(C.c_void_p), C.POINTER(C.c_int64)]
        lib.lya_xi2pcf.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning), C.c_void_p,
                                   C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(CStats)]
        lib.lya_xi2pcf_sub.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning), C.c_void_p,
                                       C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(CStats)]
        lib.lya_xi2pcf_means.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning), C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.lya_dmat.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning), C.c_void_p,
                                 C.c_double, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(CStats)]
        lib.lya_run_host.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning), C.c_int, C.c_int,
                                     C.c_double, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.POINTER(C.c_int64), C.POINTER(CStats), C.POINTER(CStats)]
        lib.lya_tri_nbins.restype = C.c_int64
        lib.lya_tri_nbins.argtypes = [C.POINTER(CTriBinning)]
        lib.lya_xi3pcf.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CTriBinning), C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(CStats)]
        lib.lya_plan_create.argtypes = [C.c_void_p, C.POINTER(CForests), C.POINTER(CBinning), C.c_void_p, C.c_int, C.c_int,
                                        C.POINTER(C.c_void_p)]
        lib.lya_plan_free.argtypes = [C.c_void_p, C.c_void_p]
        lib.lya_plan_free.restype = None
        lib.lya_xi2pcf_plan.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(CStats)]
        lib.lya_xi2pcf_plan_noalloc.argtypes = lib.lya_xi2pcf_plan.argtypes
        lib.lya_dmat_plan.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.POINTER(CStats)]
        lib.lya_xi_normalise.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.lya_dmat_normalise.argtypes = [C.c_void_p, C.POINTER(CBinning), C.c_void_p, C.c_void_p, C.c_void_p]
        lib.lya_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int64]
        _lib = lib
    return _lib


def launch_count() -> int:
    """Kernels launched by liblya.so in this process so far."""
    return int(load().lya_launch_count())


def tri_binning(r_max=80.0, n_r=20, n_theta=10, n_cosa=20) -> CTriBinning:
    return CTriBinning(r_max, n_r, n_theta, n_cosa)


def binning(rpar_max=200.0, rperp_max=200.0, n_par=50, n_perp=50) -> CBinning:
    return CBinning(rpar_max, rperp_max, n_par, n_perp)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class DeviceForests:
    """A gen.Forests (or any object with the same arrays) resident in HBM."""

    def __init__(self, f, device="cuda:0", with_radec=False):
        import torch
        self.torch = torch
        dev = torch.device(device)
        up = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).to(dev)
        self.n_forest = int(len(f.ux))
        self.n_pix = int(len(f.chi))
        self.ux, self.uy, self.uz = (up(f.ux, np.float64), up(f.uy, np.float64), up(f.uz, np.float64))
        self.ra = up(f.ra, np.float64) if with_radec else None
        self.dec = up(f.dec, np.float64) if with_radec else None
        self.pix_off = up(f.pix_off, np.int64)
        self.chi, self.w = up(f.chi, np.float64), up(f.w, np.float64)
        self.delta, self.loglam = up(f.delta, np.float64), up(f.loglam, np.float64)

    def c(self, use_u=True) -> CForests:
        g = lambda t: (t.data_ptr() if t is not None else None)
        return CForests(self.n_forest, self.n_pix, g(self.ra), g(self.dec),
                        g(self.ux) if use_u else None, g(self.uy) if use_u else None, g(self.uz) if use_u else None,
                        g(self.pix_off), g(self.chi), g(self.w), g(self.delta), g(self.loglam))


class Pairs:
    def __init__(self, ctx, handle, n):
        self.ctx, self.handle, self.n = ctx, handle, int(n)

    def export(self):
        """int32 [n][2] torch tensor on the device."""
        torch = self.ctx.torch
        out = torch.empty((self.n, 2), dtype=torch.int32, device=self.ctx.device)
        self.ctx._check(load().lya_pairs_export(self.ctx.h, self.handle, _ptr(out) if self.n else None))
        self.ctx.sync()
        return out

    def free(self):
        if self.handle is not None:
            load().lya_pairs_free(self.ctx.h, self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Plan:
    """lya_plan handle (prepared catalogue + bucketed pair list); keeps the DeviceForests alive."""

    def __init__(self, ctx, handle, forests, b):
        self.ctx, self.handle, self.forests, self.b = ctx, handle, forests, b

    def free(self):
        if self.handle is not None:
            load().lya_plan_free(self.ctx.h, self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """lya_ctx bound to a torch device and torch's current stream on it."""

    def __init__(self, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: liblya has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        idx = self.device.index or 0
        torch.cuda.set_device(idx)
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        st = load().lya_create(C.byref(h), idx, C.c_void_p(self.stream.cuda_stream))
        if st:
            raise LyaError(st, "lya_create failed")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            load().lya_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sync(self):
        self.stream.synchronize()

    def sm_count(self) -> int:
        return int(self.torch.cuda.get_device_properties(self.device).multi_processor_count)

    def _check(self, st):
        if st:
            raise LyaError(st, load().lya_last_error(self.h).decode())

    # ---- lya_neighbours / pairs ----
    def lya_neighbours(self, forests: DeviceForests, b: CBinning, use_u=True) -> Pairs:
        h = C.c_void_p()
        n = C.c_int64()
        cf = forests.c(use_u)
        self._check(load().lya_neighbours(self.h, C.byref(cf), C.byref(b), C.byref(h), C.byref(n)))
        return Pairs(self, h, n.value)

    def lya_pairs_import(self, pq) -> Pairs:
        torch = self.torch
        if not torch.is_tensor(pq):
            pq = torch.from_numpy(np.ascontiguousarray(pq, dtype=np.int32).reshape(-1, 2))
        pq = pq.to(self.device, dtype=torch.int32).contiguous()
        h = C.c_void_p()
        self._check(load().lya_pairs_import(self.h, _ptr(pq) if len(pq) else None, len(pq), C.byref(h)))
        return Pairs(self, h, len(pq))

    def lya_pairs_subsample(self, pairs: Pairs, reject_fraction: float, seed: int) -> Pairs:
        h = C.c_void_p()
        n = C.c_int64()
        self._check(load().lya_pairs_subsample(self.h, pairs.handle, float(reject_fraction), C.c_uint64(seed),
                                               C.byref(h), C.byref(n)))
        return Pairs(self, h, n.value)

    # ---- plans ----
    def lya_plan_create(self, forests: DeviceForests, b: CBinning, pairs: Pairs, want_xi=True, want_dmat=True) -> Plan:
        h = C.c_void_p()
        cf = forests.c()
        self._check(load().lya_plan_create(self.h, C.byref(cf), C.byref(b), pairs.handle, int(want_xi), int(want_dmat),
                                           C.byref(h)))
        return Plan(self, h, forests, b)

    def lya_xi2pcf_plan(self, plan: Plan):
        torch = self.torch
        nb = plan.b.n_par * plan.b.n_perp
        S = torch.empty(nb, dtype=torch.float64, device=self.device)
        W = torch.empty_like(S); xi = torch.empty_like(S)
        N = torch.empty(nb, dtype=torch.int64, device=self.device)      # uint64 payload
        stats = CStats()
        self._check(load().lya_xi2pcf_plan(self.h, plan.handle, _ptr(S), _ptr(W), _ptr(N), _ptr(xi), C.byref(stats)))
        return dict(S=S, W=W, N=N, xi=xi, stats=stats.as_dict())

    def lya_xi2pcf_plan_noalloc(self, plan: Plan, out=None):
        """lya_xi2pcf_plan with the accumulators in the library's static device array (include/lya.h).  `out`: a dict
        of caller-owned S, W, N, xi tensors to write into (so that the call itself allocates nothing at all)."""
        torch = self.torch
        nb = plan.b.n_par * plan.b.n_perp
        if out is None:
            out = dict(S=torch.empty(nb, dtype=torch.float64, device=self.device),
                       W=torch.empty(nb, dtype=torch.float64, device=self.device),
                       N=torch.empty(nb, dtype=torch.int64, device=self.device),      # uint64 payload
                       xi=torch.empty(nb, dtype=torch.float64, device=self.device))
        stats = CStats()
        self._check(load().lya_xi2pcf_plan_noalloc(self.h, plan.handle, _ptr(out["S"]), _ptr(out["W"]), _ptr(out["N"]),
                                                   _ptr(out["xi"]), C.byref(stats)))
        return dict(S=out["S"], W=out["W"], N=out["N"], xi=out["xi"], stats=stats.as_dict())

    def lya_dmat_plan(self, plan: Plan, reject_fraction: float, seed: int, want_Dn=True, want_D=True):
        torch = self.torch
        nb = plan.b.n_par * plan.b.n_perp
        D = torch.empty((nb, nb), dtype=torch.float64, device=self.device) if want_D else None
        Dn = torch.empty((nb, nb), dtype=torch.float64, device=self.device) if want_Dn else None
        Wd = torch.empty(nb, dtype=torch.float64, device=self.device)
        stats = CStats()
        self._check(load().lya_dmat_plan(self.h, plan.handle, float(reject_fraction), C.c_uint64(seed),
                                         _ptr(D), _ptr(Dn), _ptr(Wd), C.byref(stats)))
        return dict(D=D, Dn=Dn, Wd=Wd, stats=stats.as_dict())

    # ---- lya_xi2pcf ----
    def lya_xi2pcf(self, forests: DeviceForests, b: CBinning, pairs: Pairs):
        torch = self.torch
        nb = b.n_par * b.n_perp
        S = torch.empty(nb, dtype=torch.float64, device=self.device)
        W = torch.empty_like(S); xi = torch.empty_like(S)
        N = torch.empty(nb, dtype=torch.int64, device=self.device)      # uint64 payload
        stats = CStats()
        cf = forests.c()
        self._check(load().lya_xi2pcf(self.h, C.byref(cf), C.byref(b), pairs.handle,
                                      _ptr(S), _ptr(W), _ptr(N), _ptr(xi), C.byref(stats)))
        return dict(S=S, W=W, N=N, xi=xi, stats=stats.as_dict())

    def lya_xi2pcf_sub(self, forests: DeviceForests, b: CBinning, pairs: Pairs, region, n_region: int):
        """region: int32 [n_forest] (numpy or torch).  Returns S, W [n_region][nb], N [n_region][nb]."""
        torch = self.torch
        if not torch.is_tensor(region):
            region = torch.from_numpy(np.ascontiguousarray(region, dtype=np.int32))
        region = region.to(self.device, dtype=torch.int32).contiguous()
        nb = b.n_par * b.n_perp
        S = torch.empty((n_region, nb), dtype=torch.float64, device=self.device)
        W = torch.empty_like(S)
        N = torch.empty((n_region, nb), dtype=torch.int64, device=self.device)      # uint64 payload
        stats = CStats()
        cf = forests.c()
        self._check(load().lya_xi2pcf_sub(self.h, C.byref(cf), C.byref(b), pairs.handle, _ptr(region), int(n_region),
                                          _ptr(S), _ptr(W), _ptr(N), C.byref(stats)))
        return dict(S=S, W=W, N=N, stats=stats.as_dict())

    def lya_xi2pcf_means(self, forests: DeviceForests, b: CBinning, pairs: Pairs, z):
        """z: per-pixel redshift (numpy or torch, [n_pix]).  Returns the SUMS Rpar, Rperp, Z and W."""
        torch = self.torch
        if not torch.is_tensor(z):
            z = torch.from_numpy(np.ascontiguousarray(z, dtype=np.float64))
        z = z.to(self.device, dtype=torch.float64).contiguous()
        nb = b.n_par * b.n_perp
        out = [torch.empty(nb, dtype=torch.float64, device=self.device) for _ in range(4)]
        cf = forests.c()
        self._check(load().lya_xi2pcf_means(self.h, C.byref(cf), C.byref(b), pairs.handle, _ptr(z), *[_ptr(o) for o in out]))
        return dict(Rpar=out[0], Rperp=out[1], Z=out[2], W=out[3])

    def lya_xi3pcf(self, forests: DeviceForests, tb: CTriBinning, cos_theta_edges, pairs: Pairs):
        """cos_theta_edges: cos(m pi / n_theta), m = 1..n_theta-1 (numpy or torch): an input, like chi."""
        torch = self.torch
        if not torch.is_tensor(cos_theta_edges):
            cos_theta_edges = torch.from_numpy(np.ascontiguousarray(cos_theta_edges, dtype=np.float64))
        ce = cos_theta_edges.to(self.device, dtype=torch.float64).contiguous()
        nb = int(load().lya_tri_nbins(C.byref(tb)))
        S3 = torch.empty(nb, dtype=torch.float64, device=self.device)
        W3 = torch.empty_like(S3); x3 = torch.empty_like(S3)
        N3 = torch.empty(nb, dtype=torch.int64, device=self.device)      # uint64 payload
        stats = CStats()
        cf = forests.c()
        self._check(load().lya_xi3pcf(self.h, C.byref(cf), C.byref(tb), _ptr(ce) if ce.numel() else None, pairs.handle,
                                      _ptr(S3), _ptr(W3), _ptr(N3), _ptr(x3), C.byref(stats)))
        return dict(S3=S3, W3=W3, N3=N3, xi3=x3, stats=stats.as_dict())

    # ---- lya_dmat ----
    def lya_dmat(self, forests: DeviceForests, b: CBinning, pairs: Pairs, reject_fraction: float, seed: int,
                 want_Dn=True, want_D=True):
        torch = self.torch
        nb = b.n_par * b.n_perp
        D = torch.empty((nb, nb), dtype=torch.float64, device=self.device) if want_D else None
        Dn = torch.empty((nb, nb), dtype=torch.float64, device=self.device) if want_Dn else None
        Wd = torch.empty(nb, dtype=torch.float64, device=self.device)
        stats = CStats()
        cf = forests.c()
        self._check(load().lya_dmat(self.h, C.byref(cf), C.byref(b), pairs.handle, float(reject_fraction),
                                    C.c_uint64(seed), _ptr(D), _ptr(Dn), _ptr(Wd), C.byref(stats)))
        return dict(D=D, Dn=Dn, Wd=Wd, stats=stats.as_dict())

    # ---- lya_run_host: host numpy in, host numpy out (uploads/downloads inside the call) ----
    def lya_run_host(self, f, b: CBinning, do_xi=True, do_dmat=False, reject_fraction=0.0, seed=0, out=None):
        nb = b.n_par * b.n_perp
        keep = [np.ascontiguousarray(a, dtype=dt) for a, dt in
                ((f.ux, np.float64), (f.uy, np.float64), (f.uz, np.float64), (f.pix_off, np.int64),
                 (f.chi, np.float64), (f.w, np.float64), (f.delta, np.float64), (f.loglam, np.float64))]
        cf = CForests(len(keep[0]), len(keep[4]), None, None, keep[0].ctypes.data, keep[1].ctypes.data,
                      keep[2].ctypes.data, keep[3].ctypes.data, keep[4].ctypes.data, keep[5].ctypes.data,
                      keep[6].ctypes.data, keep[7].ctypes.data)
        out = out if out is not None else {}
        if do_xi:
            for k in ("S", "W", "xi"):
                out.setdefault(k, np.empty(nb, np.float64))
            out.setdefault("N", np.empty(nb, np.uint64))
        if do_dmat:
            out.setdefault("D", np.empty((nb, nb), np.float64))
            out.setdefault("Wd", np.empty(nb, np.float64))
        p = lambda k: (C.c_void_p(out[k].ctypes.data) if k in out else None)
        n_pairs = C.c_int64()
        sx, sd = CStats(), CStats()
        self._check(load().lya_run_host(self.h, C.byref(cf), C.byref(b), int(do_xi), int(do_dmat),
                                        float(reject_fraction), C.c_uint64(seed),
                                        p("S"), p("W"), p("N"), p("xi"), p("D"), p("Wd"),
                                        C.byref(n_pairs), C.byref(sx), C.byref(sd)))
        out["n_pairs"] = n_pairs.value
        out["stats_xi"] = sx.as_dict()
        out["stats_dmat"] = sd.as_dict()
        return out

    def lya_xi_normalise(self, S, W):
        xi = self.torch.empty_like(S)
        self._check(load().lya_xi_normalise(self.h, S.numel(), _ptr(S), _ptr(W), _ptr(xi)))
        return xi

    def lya_dmat_normalise(self, b: CBinning, Dn, Wd):
        D = self.torch.empty_like(Dn)
        self._check(load().lya_dmat_normalise(self.h, C.byref(b), _ptr(Dn), _ptr(Wd), _ptr(D)))
        return D

    def lya_set_option(self, opt: str, value: int):
        self._check(load().lya_set_option(self.h, OPTIONS[opt], int(value)))
