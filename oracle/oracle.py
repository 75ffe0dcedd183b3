"""ctypes wrapper over oracle/lya_oracle.c -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  It never imports the CUDA package
(paper_2507_00129_b200.binding) and shares no code with it; the only common
module is the input generator paper_2507_00129_b200.gen (no method arithmetic).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lya_oracle.c")
_LIB = os.path.join(_HERE, "liblya_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc: -O2, no FMA contraction, no fast-math."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
                               "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Forests(C.Structure):
    _fields_ = [("n_forest", C.c_int64), ("n_pix", C.c_int64),
                ("ux", C.c_void_p), ("uy", C.c_void_p), ("uz", C.c_void_p),
                ("pix_off", C.c_void_p),
                ("chi", C.c_void_p), ("w", C.c_void_p), ("delta", C.c_void_p), ("loglam", C.c_void_p)]


class _Binning(C.Structure):
    _fields_ = [("rpar_max", C.c_double), ("rperp_max", C.c_double),
                ("n_par", C.c_int32), ("n_perp", C.c_int32)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_pairs_all.restype = C.c_int64
        _lib.orc_pairs_brute.restype = C.c_int64
        _lib.orc_pairs_window.restype = C.c_int64
        _lib.orc_mask_threshold.restype = C.c_uint64
        _lib.orc_mask_threshold.argtypes = [C.c_double]
        _lib.orc_keep.restype = C.c_int
        _lib.orc_keep.argtypes = [C.c_uint64, C.c_int64, C.c_int64, C.c_uint64]
        _lib.orc_pix_bin.restype = C.c_int32
        _lib.orc_pix_bin.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double]
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _c(a, dt):
    a = np.ascontiguousarray(a, dtype=dt)
    return a


class Catalogue:
    """Holds contiguous copies of a gen.Forests and the C struct over them."""

    def __init__(self, f):
        self.keep = [_c(f.ux, np.float64), _c(f.uy, np.float64), _c(f.uz, np.float64),
                     _c(f.pix_off, np.int64), _c(f.chi, np.float64), _c(f.w, np.float64),
                     _c(f.delta, np.float64), _c(f.loglam, np.float64)]
        k = self.keep
        self.n_forest = len(k[0])
        self.n_pix = len(k[4])
        self.c = _Forests(self.n_forest, self.n_pix, *[x.ctypes.data for x in k])


def binning(rpar_max=200.0, rperp_max=200.0, n_par=50, n_perp=50):
    return _Binning(rpar_max, rperp_max, n_par, n_perp)


def _pq(pairs):
    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    return pairs


def pair_sc(f, p, q):
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    s, c = C.c_double(), C.c_double()
    lib().orc_pair_sc(C.byref(cat.c), C.c_int64(p), C.c_int64(q), C.byref(s), C.byref(c))
    return s.value, c.value


def pix_bin(b, s, c, chi_i, chi_j):
    return int(lib().orc_pix_bin(C.byref(b), s, c, chi_i, chi_j))


def pairs_all(n_forest):
    n = n_forest * (n_forest - 1) // 2
    pq = np.empty((n, 2), np.int32)
    lib().orc_pairs_all(C.c_int64(n_forest), C.c_void_p(pq.ctypes.data))
    return pq


def pairs_brute(f, b=None):
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    b = b or binning()
    n = lib().orc_pairs_brute(C.byref(cat.c), C.byref(b), None)
    pq = np.empty((n, 2), np.int32)
    lib().orc_pairs_brute(C.byref(cat.c), C.byref(b), C.c_void_p(pq.ctypes.data))
    return pq


def pairs_window(f, b=None):
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    b = b or binning()
    n = lib().orc_pairs_window(C.byref(cat.c), C.byref(b), None, C.c_int64(0))
    pq = np.empty((n, 2), np.int32)
    m = lib().orc_pairs_window(C.byref(cat.c), C.byref(b), C.c_void_p(pq.ctypes.data), C.c_int64(n))
    assert m == n
    return pq


def xi(f, pairs, b=None):
    """eq. 2.4 over the listed forest pairs.  Returns a dict of arrays."""
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    b = b or binning()
    pq = _pq(pairs)
    nb = b.n_par * b.n_perp
    S = np.zeros(nb); W = np.zeros(nb); N = np.zeros(nb, np.uint64); x = np.zeros(nb)
    Sabs = np.zeros(nb); Q = np.zeros(nb); n_out = np.zeros(1, np.uint64)
    lib().orc_xi(C.byref(cat.c), C.byref(b), C.c_void_p(pq.ctypes.data), C.c_int64(len(pq)),
                 *[C.c_void_p(a.ctypes.data) for a in (S, W, N, x, Sabs, Q, n_out)])
    return dict(S=S, W=W, N=N, xi=x, Sabs=Sabs, Q=Q, n_out=int(n_out[0]))


def xi_means(f, pairs, z, b=None):
    """NEXT-1: per-bin weighted SUMS of r_par, r_perp, z (weights w_i w_j) and W; means = sums / W."""
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    b = b or binning()
    pq = _pq(pairs)
    z = _c(z, np.float64)
    nb = b.n_par * b.n_perp
    out = [np.zeros(nb) for _ in range(4)]
    lib().orc_xi_means(C.byref(cat.c), C.byref(b), C.c_void_p(pq.ctypes.data), C.c_int64(len(pq)),
                       C.c_void_p(z.ctypes.data), *[C.c_void_p(a.ctypes.data) for a in out])
    return dict(Rpar=out[0], Rperp=out[1], Z=out[2], W=out[3])


class _TriBinning(C.Structure):
    _fields_ = [("r_max", C.c_double), ("n_r", C.c_int32), ("n_theta", C.c_int32), ("n_cosa", C.c_int32)]


def tri_binning(r_max=80.0, n_r=20, n_theta=10, n_cosa=20):
    """Triangle bins of PAPER.md:225 (Fig. 5): r in [0, 80) Mpc/h x 20, theta in [0, pi] x 10, cos alpha x 20."""
    return _TriBinning(r_max, n_r, n_theta, n_cosa)


def xi3(f, pairs, tb=None, cosedge=None):
    """NEXT-4, eq. 2.8: brute-force anisotropic 3PCF over ordered triples (i; j, k) in three distinct forests
    (readings T1-T7 in lya_oracle.c).  cosedge: the cos(m pi / n_theta) table (input, m = 1..n_theta-1)."""
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    tb = tb or tri_binning()
    if cosedge is None:
        cosedge = np.cos(np.pi * np.arange(1, tb.n_theta) / tb.n_theta)
    cosedge = _c(cosedge, np.float64)
    pq = _pq(pairs)
    lib().orc_tri_nbins.restype = C.c_int64
    nb = int(lib().orc_tri_nbins(C.byref(tb)))
    S3 = np.zeros(nb); W3 = np.zeros(nb); N3 = np.zeros(nb, np.uint64)
    lib().orc_xi3(C.byref(cat.c), C.byref(tb), C.c_void_p(cosedge.ctypes.data), C.c_void_p(pq.ctypes.data),
                  C.c_int64(len(pq)), C.c_void_p(S3.ctypes.data), C.c_void_p(W3.ctypes.data), C.c_void_p(N3.ctypes.data))
    with np.errstate(divide="ignore", invalid="ignore"):
        x3 = np.where(W3 != 0.0, S3 / np.where(W3 == 0, 1.0, W3), 0.0)
    return dict(S3=S3, W3=W3, N3=N3, xi3=x3)


def eta(w, loglam):
    """eq. 2.7: explicit n x n eta of one forest (raises on a degenerate forest)."""
    w = _c(w, np.float64); ll = _c(loglam, np.float64)
    n = len(w)
    out = np.zeros((n, n))
    rc = lib().orc_eta(C.c_int64(n), C.c_void_p(w.ctypes.data), C.c_void_p(ll.ctypes.data),
                       C.c_void_p(out.ctypes.data))
    if rc:
        raise ValueError("degenerate forest (sum w == 0 or sum w (L-Lbar)^2 == 0)")
    return out


def mask_threshold(reject_fraction: float) -> int:
    return int(lib().orc_mask_threshold(float(reject_fraction)))


def keep(seed: int, a: int, b: int, threshold: int) -> bool:
    return bool(lib().orc_keep(C.c_uint64(seed), C.c_int64(a), C.c_int64(b), C.c_uint64(threshold)))


def dmat(f, pairs, reject_fraction=0.0, seed=0, b=None, want_D=True, collapsed=False):
    """eq. 2.6 by the naive quadruple sum (collapsed=True: the PD4 cross-check form)."""
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    b = b or binning()
    pq = _pq(pairs)
    nb = b.n_par * b.n_perp
    Dn = np.zeros((nb, nb)); Wd = np.zeros(nb); n_kept = np.zeros(1, np.uint64)
    if collapsed:
        rc = lib().orc_dmat_collapsed(C.byref(cat.c), C.byref(b), C.c_void_p(pq.ctypes.data),
                                      C.c_int64(len(pq)), C.c_double(reject_fraction), C.c_uint64(seed),
                                      C.c_void_p(Dn.ctypes.data), C.c_void_p(Wd.ctypes.data),
                                      C.c_void_p(n_kept.ctypes.data))
        Dover = None
    else:
        Dover = np.zeros(nb)
        rc = lib().orc_dmat(C.byref(cat.c), C.byref(b), C.c_void_p(pq.ctypes.data), C.c_int64(len(pq)),
                            C.c_double(reject_fraction), C.c_uint64(seed),
                            C.c_void_p(Dn.ctypes.data), C.c_void_p(Wd.ctypes.data),
                            C.c_void_p(Dover.ctypes.data), C.c_void_p(n_kept.ctypes.data), None)
    if rc:
        raise ValueError("degenerate forest in dmat (reading R-7)")
    out = dict(Dn=Dn, Wd=Wd, Dover=Dover, n_kept=int(n_kept[0]))
    if want_D:
        with np.errstate(divide="ignore", invalid="ignore"):
            out["D"] = np.where(Wd[:, None] != 0.0, Dn / np.where(Wd == 0, 1.0, Wd)[:, None], 0.0)
    return out


def subsample_forest_pairs(pairs, reject_fraction: float, seed: int):
    """The paper's forest-pair subsampling (DESIGN.md NEXT-2): keep (p, q) iff
    keep(seed, p, q) of the stage-4 integer mask with the forest indices as ids.  Order preserved."""
    pq = _pq(pairs)
    thr = mask_threshold(reject_fraction)
    sel = np.fromiter((keep(seed, int(p), int(q), thr) for p, q in pq), dtype=bool, count=len(pq))
    return pq[sel]


def xi_sub(f, pairs, region, n_region, b=None):
    """Per-sky-region sub-samples of eq. 2.4 (DESIGN.md NEXT-1): sub-sample r is
    eq. 2.4 over the forest pairs whose lower-index forest p lies in region r."""
    cat = f if isinstance(f, Catalogue) else Catalogue(f)
    pq = _pq(pairs)
    region = np.asarray(region)
    lo = np.minimum(pq[:, 0], pq[:, 1])
    return [xi(cat, pq[region[lo] == r], b) for r in range(n_region)]
