"""Seeded synthetic forest catalogues for BASELINE.json configs[0..4].

This module only *prepares inputs* (sky positions, pixel grids, comoving
distances, weights, deltas).  It holds none of the method's arithmetic (no
separations, no bins, no eta, no mask) and is the one module that both the
CUDA path's tests/bench and the CPU oracle's tests import.

Shapes follow PAPER.md:140-145 (Table 1: forest counts, areas) as scaled by
BASELINE.json configs[0..4]; the readings of the config text (R-9a..R-9f,
R-13 of SURVEY.md section 8(c)) are restated in DESIGN.md "Input recipe".
The data stand in for SDSS DR16 / DESI-Y5 mocks, which are not available.

Everything is NumPy on the host; unit vectors are computed here ONCE and
handed to both sides as inputs (reading G1), exactly like chi.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

LYA_REST = 1215.67          # Angstrom
LAM_REST_MIN = 1040.0       # rest-frame window of the forest (configs text)
LAM_REST_MAX = 1200.0
LAM_OBS_MIN = 3600.0
C_OVER_H0 = 2997.92458      # Mpc/h
OMEGA_M = 0.315             # configs[0]: flat LCDM, Om = 0.315
SEED_BASE = 250700129 * 10  # R-9f: seed = SEED_BASE + config index


# --------------------------------------------------------------------------
# cosmology: chi(z) for flat LCDM (input preparation only)
# --------------------------------------------------------------------------
def _inv_E(z):
    return 1.0 / np.sqrt(OMEGA_M * (1.0 + z) ** 3 + (1.0 - OMEGA_M))


class _ChiTable:
    """chi(z) = C_OVER_H0 * int_0^z dz'/E(z') [Mpc/h].

    Node values by 8-point Gauss-Legendre on each interval of a fine z grid
    (error far below 1e-12 relative), evaluated between nodes by cubic Hermite
    interpolation with the exact derivative C_OVER_H0/E(z).
    """

    def __init__(self, zmax: float = 4.6, n: int = 46001):
        self.z = np.linspace(0.0, zmax, n)
        h = self.z[1] - self.z[0]
        x, wq = np.polynomial.legendre.leggauss(8)
        mid = 0.5 * (self.z[:-1] + self.z[1:])
        seg = np.zeros(n - 1)
        for xi, wi in zip(x, wq):
            seg += wi * _inv_E(mid + 0.5 * h * xi)
        seg *= 0.5 * h * C_OVER_H0
        self.chi = np.concatenate([[0.0], np.cumsum(seg)])
        self.dchi = C_OVER_H0 * _inv_E(self.z)
        self.h = h

    def __call__(self, z):
        z = np.asarray(z, dtype=np.float64)
        k = np.clip((z / self.h).astype(np.int64), 0, len(self.z) - 2)
        t = (z - self.z[k]) / self.h
        h00 = (1 + 2 * t) * (1 - t) ** 2
        h10 = t * (1 - t) ** 2
        h01 = t * t * (3 - 2 * t)
        h11 = t * t * (t - 1)
        return (h00 * self.chi[k] + h10 * self.h * self.dchi[k]
                + h01 * self.chi[k + 1] + h11 * self.h * self.dchi[k + 1])


_CHI = None


def chi_of_z(z):
    global _CHI
    if _CHI is None:
        _CHI = _ChiTable()
    return _CHI(z)


# --------------------------------------------------------------------------
# catalogue container
# --------------------------------------------------------------------------
@dataclass
class Forests:
    """CSR catalogue: per-forest sky position, per-pixel chi/w/delta/loglam."""
    ra: np.ndarray          # [N] radians
    dec: np.ndarray         # [N] radians
    ux: np.ndarray          # [N] unit vector (computed once here, reading G1)
    uy: np.ndarray
    uz: np.ndarray
    zq: np.ndarray          # [N] quasar redshift (bookkeeping only)
    pix_off: np.ndarray     # [N+1] int64
    chi: np.ndarray         # [n_pix] Mpc/h, strictly increasing per forest
    w: np.ndarray           # [n_pix]
    delta: np.ndarray       # [n_pix]
    loglam: np.ndarray      # [n_pix] log10(lambda_obs / Angstrom)
    meta: dict = field(default_factory=dict)

    @property
    def n_forest(self) -> int:
        return int(self.ra.shape[0])

    @property
    def n_pix(self) -> int:
        return int(self.chi.shape[0])

    def subset(self, idx) -> "Forests":
        """Catalogue restricted to forests idx (order kept as given)."""
        idx = np.asarray(idx, dtype=np.int64)
        lens = (self.pix_off[1:] - self.pix_off[:-1])[idx]
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        take = np.concatenate(
            [np.arange(self.pix_off[i], self.pix_off[i + 1]) for i in idx]
        ).astype(np.int64) if len(idx) else np.zeros(0, np.int64)
        return Forests(self.ra[idx], self.dec[idx], self.ux[idx], self.uy[idx],
                       self.uz[idx], self.zq[idx], off, self.chi[take],
                       self.w[take], self.delta[take], self.loglam[take],
                       dict(self.meta, subset=len(idx)))


def unit_vectors(ra, dec):
    cd = np.cos(dec)
    return cd * np.cos(ra), cd * np.sin(ra), np.sin(dec)


def _trunc_normal(rng, mu, sigma, lo, hi, n):
    """Rejection sampling (R-9f)."""
    out = np.empty(n)
    filled = 0
    while filled < n:
        x = rng.normal(mu, sigma, size=max(1024, int(1.3 * (n - filled))))
        x = x[(x >= lo) & (x <= hi)]
        k = min(len(x), n - filled)
        out[filled:filled + k] = x[:k]
        filled += k
    return out


def _sky(rng, n, ra_width_deg, dec_lo_deg, dec_hi_deg):
    """Uniform on the sphere inside an RA/Dec box (R-9e)."""
    ra = rng.uniform(0.0, np.deg2rad(ra_width_deg), size=n)
    sd = rng.uniform(np.sin(np.deg2rad(dec_lo_deg)), np.sin(np.deg2rad(dec_hi_deg)), size=n)
    return ra, np.arcsin(sd)


def _ragged(counts):
    """(forest index, index within forest) for every pixel of a CSR layout."""
    counts = np.asarray(counts, dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    fid = np.repeat(np.arange(len(counts), dtype=np.int64), counts)
    k = np.arange(off[-1], dtype=np.int64) - off[fid]
    return off, fid, k


def _weights(rng, z_pix):
    s = rng.uniform(0.05, 0.5, size=z_pix.shape[0])      # R-9d: per pixel
    return ((1.0 + z_pix) / 3.25) ** 1.9 / (0.05 + s * s)


CONFIGS = {
    # name: (n_forest, ra_width_deg, dec_lo, dec_hi, zq law, grid, sigma_delta)
    0: dict(n=64, ra_w=4.0, dec=(-2.0, 2.0), zq=("uniform", 2.1, 3.0), grid="log24", sig=0.2),
    1: dict(n=20000, ra_w=10.0, dec=(-5.006, 5.006), zq=("tnorm", 2.5, 0.35, 2.1, 3.8),
            grid="logglobal", sig=0.2),
    2: dict(n=210000, ra_w=94.72, dec=(-60.0, 60.0), zq=("tnorm", 2.5, 0.35, 2.1, 3.8),
            grid="logglobal", sig=0.25),
    4: dict(n=900000, ra_w=141.07, dec=(-60.0, 60.0), zq=("tnorm", 2.45, 0.4, 2.1, 4.0),
            grid="lin2p4", sig=0.25),
}
CONFIGS[3] = CONFIGS[2]            # configs[3] = the same arrays as configs[2]


def make_config(cfg: int, n_forest: int | None = None, density_scale: float = 1.0,
                seed: int | None = None, fine: int = 1) -> Forests:
    """Catalogue for BASELINE.json configs[cfg].

    n_forest / density_scale give *shaped* sub-workloads for tests: fewer
    forests over a proportionally smaller RA width (same sky density, same
    pixel recipe) -- so the neighbour structure stays that of the config.
    fine = k divides the pixel step by k (k times more pixels per forest):
    native-resolution shapes of DESIGN.md NEXT-3 (fine=2 on configs[2] is the
    3.3 Mpc/h spacing of SDSS).  Throughput workloads only.
    """
    c = CONFIGS[cfg]
    fine = int(fine)
    seed_cfg = 2 if cfg == 3 else cfg
    rng = np.random.default_rng(SEED_BASE + seed_cfg if seed is None else seed)
    n = c["n"] if n_forest is None else int(n_forest)
    ra_w = c["ra_w"] * (n / c["n"]) / density_scale
    # draw order (R-9f): z_q, RA, Dec, then per-pixel delta, s
    if c["zq"][0] == "uniform":
        zq = rng.uniform(c["zq"][1], c["zq"][2], size=n)
    else:
        _, mu, sg, lo, hi = c["zq"]
        zq = _trunc_normal(rng, mu, sg, lo, hi, n)
    ra, dec = _sky(rng, n, ra_w, c["dec"][0], c["dec"][1])
    ux, uy, uz = unit_vectors(ra, dec)

    if c["grid"] == "log24":
        counts = np.full(n, 24 * fine, dtype=np.int64)
        off, fid, k = _ragged(counts)
        loglam = np.log10(LAM_REST_MIN * (1.0 + zq[fid])) + (1e-3 / fine) * k
        lam = 10.0 ** loglam
    elif c["grid"] == "logglobal":
        l0 = np.log10(LAM_OBS_MIN)
        # global grid index range per forest: 1040(1+zq) <= lam_k <= 1200(1+zq), lam_k >= 3600
        dl = 1e-3 / fine
        klo = np.ceil((np.log10(LAM_REST_MIN * (1 + zq)) - l0) / dl - 1e-9).astype(np.int64)
        khi = np.floor((np.log10(LAM_REST_MAX * (1 + zq)) - l0) / dl + 1e-9).astype(np.int64)
        klo = np.maximum(klo, 0)
        counts = np.maximum(khi - klo + 1, 0)
        off, fid, k = _ragged(counts)
        loglam = l0 + dl * (klo[fid] + k)
        lam = 10.0 ** loglam
    elif c["grid"] == "lin2p4":
        # R-9a: 2.4 A steps in the REST frame, k = 0..66
        st = 2.4 / fine
        kmin = np.ceil((LAM_OBS_MIN / (1 + zq) - LAM_REST_MIN) / st - 1e-9).astype(np.int64)
        kmin = np.maximum(kmin, 0)
        counts = np.maximum(int(np.floor(160.0 / st + 1e-9)) + 1 - kmin, 0)
        off, fid, k = _ragged(counts)
        lam = (LAM_REST_MIN + st * (kmin[fid] + k)) * (1 + zq[fid])
        loglam = np.log10(lam)
    else:
        raise ValueError(c["grid"])

    z_pix = lam / LYA_REST - 1.0
    chi = chi_of_z(z_pix)
    delta = rng.normal(0.0, c["sig"], size=off[-1])
    w = _weights(rng, z_pix)
    return Forests(ra, dec, ux, uy, uz, zq, off, chi, w, delta, loglam,
                   dict(cfg=cfg, n_forest=n, ra_width_deg=ra_w, seed=SEED_BASE + seed_cfg))


def mask_seed(cfg: int) -> int:
    """Seed of the pixel-pair keep mask for a config."""
    return SEED_BASE + cfg


def two_forests(chi_p, chi_q, ux_p, ux_q, w_p=None, w_q=None, d_p=None, d_q=None,
                ll_p=None, ll_q=None) -> Forests:
    """Hand-built two-forest catalogue (unit vectors given directly)."""
    chi_p = np.asarray(chi_p, float); chi_q = np.asarray(chi_q, float)
    def dflt(x, n, v):
        return np.full(n, v) if x is None else np.asarray(x, float)
    w = np.concatenate([dflt(w_p, len(chi_p), 1.0), dflt(w_q, len(chi_q), 1.0)])
    d = np.concatenate([dflt(d_p, len(chi_p), 1.0), dflt(d_q, len(chi_q), 1.0)])
    ll = np.concatenate([
        np.log10(3600.0) + 1e-3 * np.arange(len(chi_p)) if ll_p is None else np.asarray(ll_p, float),
        np.log10(3600.0) + 1e-3 * np.arange(len(chi_q)) if ll_q is None else np.asarray(ll_q, float)])
    u = np.array([ux_p, ux_q], dtype=float)
    ra = np.arctan2(u[:, 1], u[:, 0]); dec = np.arcsin(np.clip(u[:, 2], -1, 1))
    off = np.array([0, len(chi_p), len(chi_p) + len(chi_q)], dtype=np.int64)
    return Forests(ra, dec, u[:, 0].copy(), u[:, 1].copy(), u[:, 2].copy(), np.zeros(2), off,
                   np.concatenate([chi_p, chi_q]), w, d, ll, dict(cfg="hand"))
