"""Pins for the CPU oracle (oracle/lya_oracle.c): every check here compares the
oracle with something OTHER than itself -- hand-worked bins, closed forms,
invariants, textbook/library routines (numpy lstsq, histogram2d), or an
exhaustive numpy enumeration on tiny inputs.  Names P1..P8 / PD1..PD8 are the
pin ids of DESIGN.md ("Oracle pins").  CPU only.
"""
import os
from decimal import Decimal, getcontext

import numpy as np
import pytest

from paper_2507_00129_b200 import gen
from oracle import oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))


# ---------------------------------------------------------------- helpers
def np_brute_xi(f, pairs, nb=50, rmax=200.0):
    """Independent exhaustive enumeration with numpy broadcasting + histogram2d."""
    S = np.zeros((nb, nb)); W = np.zeros((nb, nb)); N = np.zeros((nb, nb), np.int64)
    n_out = 0
    edges = np.linspace(0.0, rmax, nb + 1)
    for p, q in pairs:
        chord = np.sqrt((f.ux[p] - f.ux[q]) ** 2 + (f.uy[p] - f.uy[q]) ** 2 + (f.uz[p] - f.uz[q]) ** 2)
        s = chord / 2.0
        c = np.sqrt(1.0 - s * s)
        a, b = f.pix_off[p], f.pix_off[p + 1]
        d, e = f.pix_off[q], f.pix_off[q + 1]
        ci = f.chi[a:b, None]; cj = f.chi[None, d:e]
        rpar = (np.abs(ci - cj) * c).ravel(); rperp = ((ci + cj) * s).ravel()
        ww = (f.w[a:b, None] * f.w[None, d:e]).ravel()
        dd = ((f.w[a:b] * f.delta[a:b])[:, None] * (f.w[d:e] * f.delta[d:e])[None, :]).ravel()
        ok = (rpar < rmax) & (rperp < rmax)
        n_out += int((~ok).sum())
        N += np.histogram2d(rpar[ok], rperp[ok], bins=[edges, edges])[0].astype(np.int64)
        W += np.histogram2d(rpar[ok], rperp[ok], bins=[edges, edges], weights=ww[ok])[0]
        S += np.histogram2d(rpar[ok], rperp[ok], bins=[edges, edges], weights=dd[ok])[0]
    return S.ravel(), W.ravel(), N.ravel(), n_out


@pytest.fixture(scope="module")
def xi0(cfg0):
    pq = orc.pairs_all(cfg0.n_forest)
    return pq, orc.xi(cfg0, pq)


# ---------------------------------------------------------------- P6
def test_P6_hand_built_bins():
    """tests/golden/p6_hand_cases.txt: bins derived by hand (R-1, R-2, R-3, R-5)."""
    getcontext().prec = 50
    rows = [l.split("#")[0].split() for l in open(os.path.join(HERE, "golden", "p6_hand_cases.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) >= 10
    b = orc.binning()
    for s_txt, ci, cj, ebpar, ebperp, eA in rows:
        s = float(s_txt)
        uq = (1.0 - 2.0 * s * s, 2.0 * s * float(Decimal(1 - Decimal(s_txt) ** 2).sqrt()), 0.0)
        f = gen.two_forests([float(ci)], [float(cj)], (1.0, 0.0, 0.0), uq)
        so, co = orc.pair_sc(f, 0, 1)
        assert abs(so - s) < 1e-15 and abs(co - float(Decimal(1 - Decimal(s_txt) ** 2).sqrt())) < 1e-15
        A = orc.pix_bin(b, so, co, float(ci), float(cj))
        assert A == int(eA), (s_txt, ci, cj, A, eA)
        r = orc.xi(f, [[0, 1]])
        if int(eA) >= 0:
            assert r["N"].sum() == 1 and r["N"][int(eA)] == 1 and r["n_out"] == 0
            assert int(eA) == 50 * int(ebpar) + int(ebperp)
        else:
            assert r["N"].sum() == 0 and r["n_out"] == 1


def test_P6_chord_is_sin_half_theta():
    """s from the chord equals sin(theta/2) computed from RA/Dec by the haversine formula."""
    f = gen.make_config(0)
    for p, q in [(0, 1), (3, 40), (10, 63)]:
        s, c = orc.pair_sc(f, p, q)
        hav = np.sin((f.dec[p] - f.dec[q]) / 2) ** 2 + np.cos(f.dec[p]) * np.cos(f.dec[q]) * np.sin((f.ra[p] - f.ra[q]) / 2) ** 2
        assert abs(s - np.sqrt(hav)) < 1e-14
        assert abs(s * s + c * c - 1.0) < 1e-15


# ---------------------------------------------------------------- P2
def test_P2_exhaustive_enumeration(cfg0, xi0):
    pq, r = xi0
    S, W, N, n_out = np_brute_xi(cfg0, pq)
    assert np.array_equal(r["N"].astype(np.int64), N)
    assert r["n_out"] == n_out
    n = np.diff(cfg0.pix_off)
    assert int(r["N"].sum()) + r["n_out"] == int(sum(n[p] * n[q] for p, q in pq))
    assert np.allclose(r["W"], W, rtol=1e-12, atol=0)
    assert np.all(np.abs(r["S"] - S) <= 1e-12 * r["Sabs"] + 1e-300)
    nz = r["W"] > 0
    assert np.allclose(r["xi"][nz], (S[nz] / W[nz]), rtol=0, atol=1e-12)
    assert np.all(r["xi"][~nz] == 0.0)


def test_P2_ragged_forests_and_generic_binning():
    """Ragged lengths (config-1 recipe) and a non-power-of-two bin width."""
    f = gen.make_config(1, n_forest=60)
    pq = orc.pairs_all(f.n_forest)
    b = orc.binning(150.0, 90.0, 30, 30)
    r = orc.xi(f, pq, b)
    # numpy enumeration with explicit (int)(r * (n/rmax)) binning
    N = np.zeros(900, np.int64)
    for p, q in pq:
        s, c = orc.pair_sc(f, p, q)
        ci = f.chi[f.pix_off[p]:f.pix_off[p + 1], None]; cj = f.chi[None, f.pix_off[q]:f.pix_off[q + 1]]
        rpar = np.abs(ci - cj) * c; rperp = (ci + cj) * s
        ok = (rpar < 150.0) & (rperp < 90.0)
        A = 30 * np.minimum((rpar * (30 / 150.0)).astype(np.int64), 29) + np.minimum((rperp * (30 / 90.0)).astype(np.int64), 29)
        N += np.bincount(A[ok], minlength=900)
    assert np.array_equal(r["N"].astype(np.int64), N)


# ---------------------------------------------------------------- P1
def test_P1_neighbour_list_equals_all_pairs(cfg0, xi0):
    pq_all, r_all = xi0
    pq_nb = orc.pairs_brute(cfg0)
    assert len(pq_nb) < len(pq_all)
    r_nb = orc.xi(cfg0, pq_nb)
    assert np.array_equal(r_all["N"], r_nb["N"])
    assert np.allclose(r_all["S"], r_nb["S"], rtol=0, atol=1e-12 * r_all["Sabs"].max())
    assert np.allclose(r_all["W"], r_nb["W"], rtol=1e-13)
    # a non-listed pair has no in-grid pixel pair (R-14)
    listed = set(map(tuple, pq_nb.tolist()))
    rest = np.array([x for x in pq_all.tolist() if tuple(x) not in listed], np.int32)
    assert orc.xi(cfg0, rest)["N"].sum() == 0


def test_P1_window_prefilter_equals_brute():
    f = gen.make_config(1, n_forest=1500)
    a = orc.pairs_brute(f); b = orc.pairs_window(f)
    assert np.array_equal(a, b)
    assert len(a) > 0 and np.all(a[:, 0] < a[:, 1])
    # criterion re-evaluated with numpy for every p<q
    s = 0.5 * np.sqrt((f.ux[:, None] - f.ux[None]) ** 2 + (f.uy[:, None] - f.uy[None]) ** 2 + (f.uz[:, None] - f.uz[None]) ** 2)
    cm = f.chi[f.pix_off[:-1]]
    listed = np.triu(((cm[:, None] + cm[None]) * s) < 200.0, 1)
    assert listed.sum() == len(a)
    assert listed[a[:, 0], a[:, 1]].all()


# ---------------------------------------------------------------- P3, P4
@pytest.mark.parametrize("k", [1.0, -0.5])
def test_P3_constant_delta(cfg0, k):
    f = gen.make_config(0); f.delta[:] = k
    r = orc.xi(f, orc.pairs_brute(f))
    nz = r["N"] > 0
    assert nz.sum() > 100
    assert np.allclose(r["xi"][nz], k * k, rtol=1e-13)
    assert np.allclose(r["S"][nz], k * k * r["W"][nz], rtol=1e-13)


def test_P4_unit_weights_W_equals_N(cfg0):
    f = gen.make_config(0); f.w[:] = 1.0
    r = orc.xi(f, orc.pairs_brute(f))
    assert np.array_equal(r["W"], r["N"].astype(np.float64))
    assert np.array_equal(r["Q"], r["N"].astype(np.float64))


# ---------------------------------------------------------------- P5
def test_P5_independent_gaussian_consistent_with_zero():
    """Var S_A = sigma^4 Q_A exactly for iid deltas: z_A = S_A/(sigma^2 sqrt Q_A) ~ N(0,1)."""
    f = gen.make_config(1, n_forest=600)
    r = orc.xi(f, orc.pairs_window(f))
    nz = r["N"] > 50
    assert nz.sum() > 2000
    z = r["S"][nz] / (0.2 ** 2 * np.sqrt(r["Q"][nz]))
    assert abs(z.mean()) < 3.0 / np.sqrt(nz.sum())
    assert abs((z ** 2).mean() - 1.0) < 0.1


# ---------------------------------------------------------------- P7, P8
def test_P7_order_independence(cfg0):
    pq = orc.pairs_brute(cfg0)
    r0 = orc.xi(cfg0, pq)
    rng = np.random.default_rng(5)
    r1 = orc.xi(cfg0, pq[rng.permutation(len(pq))])
    r2 = orc.xi(cfg0, pq[:, ::-1])                    # swap p <-> q
    perm = rng.permutation(cfg0.n_forest)            # relabel forests
    fp = cfg0.subset(perm)
    inv = np.empty_like(perm); inv[perm] = np.arange(len(perm))
    r3 = orc.xi(fp, inv[pq])
    for r in (r1, r2, r3):
        assert np.array_equal(r0["N"], r["N"])
        assert np.allclose(r0["W"], r["W"], rtol=1e-13)
        assert np.all(np.abs(r0["S"] - r["S"]) <= 1e-13 * r0["Sabs"])


def test_P8_degenerate_catalogues():
    f = gen.make_config(0)
    one = f.subset([3])
    assert len(orc.pairs_brute(one)) == 0 and len(orc.pairs_window(one)) == 0
    r = orc.xi(one, np.zeros((0, 2), np.int32))
    assert r["N"].sum() == 0 and r["S"].sum() == 0 and np.all(r["xi"] == 0)
    # two forests 90 degrees apart: not listed, and no pixel pair in the grid
    far = gen.two_forests(f.chi[:24], f.chi[24:48], (1, 0, 0), (0, 1, 0))
    assert len(orc.pairs_brute(far)) == 0
    assert orc.xi(far, [[0, 1]])["N"].sum() == 0


# ---------------------------------------------------------------- PD1, PD2
def _forest(cfg0, p):
    a, b = cfg0.pix_off[p], cfg0.pix_off[p + 1]
    return cfg0.w[a:b], cfg0.loglam[a:b]


def test_PD1_eta_is_wls_residual_maker(cfg0):
    """eq. 2.7 == I - X (X^T W X)^-1 X^T W, X = [1, log lambda] (PAPER.md:89 continuum model)."""
    rng = np.random.default_rng(1)
    for p in (0, 7, 31):
        w, ll = _forest(cfg0, p)
        eta = orc.eta(w, ll)
        y = rng.normal(size=len(w))
        X = np.stack([np.ones_like(ll), ll - ll.mean()], 1)     # centred for conditioning only
        sw = np.sqrt(w)
        coef = np.linalg.lstsq(X * sw[:, None], y * sw, rcond=None)[0]
        assert np.allclose(eta @ y, y - X @ coef, rtol=0, atol=1e-10)


def test_PD2_projector_identities(cfg0):
    f1 = gen.make_config(1, n_forest=40)
    for f, p in ((cfg0, 0), (cfg0, 50), (f1, 3), (f1, 17)):
        w, ll = _forest(f, p)
        n = len(w)
        eta = orc.eta(w, ll)
        lbar = (w * ll).sum() / w.sum()
        u = ll - lbar
        assert np.abs(eta @ np.ones(n)).max() < 1e-11          # annihilates constants
        assert np.abs(eta @ ll).max() < 1e-10                  # annihilates log-lambda-linear
        assert np.abs(w @ eta).max() < 1e-10                   # w^T eta = 0
        assert np.abs((w * u) @ eta).max() < 1e-10
        assert np.abs(eta @ eta - eta).max() < 1e-10           # idempotent
        assert abs(np.trace(eta) - (n - 2)) < 1e-10
        assert np.abs(eta.sum(1)).max() < 1e-11                # rows of the projector sum to zero


def test_PD2_degenerate_forest_rejected():
    with pytest.raises(ValueError):
        orc.eta(np.ones(3), np.full(3, 3.6))                   # a single distinct lambda: V = 0
    with pytest.raises(ValueError):
        orc.eta(np.zeros(3), np.array([3.6, 3.601, 3.602]))    # sum w = 0


# ---------------------------------------------------------------- PD3..PD8
@pytest.fixture(scope="module")
def d0(cfg0):
    pq = orc.pairs_brute(cfg0)
    return pq, orc.dmat(cfg0, pq, 0.0, gen.mask_seed(0))


def test_PD3_row_sums_with_overflow_bucket(d0):
    pq, d = d0
    scale = np.abs(d["Dn"]).sum(1) + np.abs(d["Dover"])
    assert np.all(np.abs(d["Dn"].sum(1) + d["Dover"]) <= 1e-11 * scale + 1e-300)


def test_PD4_collapsed_equals_naive(cfg0, d0):
    pq, d = d0
    dc = orc.dmat(cfg0, pq, 0.0, gen.mask_seed(0), collapsed=True)
    assert dc["n_kept"] == d["n_kept"]
    assert np.allclose(dc["Wd"], d["Wd"], rtol=1e-14)
    assert np.abs(dc["Dn"] - d["Dn"]).max() <= 1e-12 * np.abs(d["Dn"]).max()
    # and with a mask, on ragged forests
    f = gen.make_config(1, n_forest=80)
    pq1 = orc.pairs_window(f)
    a = orc.dmat(f, pq1, 0.9, 77); b = orc.dmat(f, pq1, 0.9, 77, collapsed=True)
    assert a["n_kept"] == b["n_kept"] and a["n_kept"] > 0
    assert np.abs(a["Dn"] - b["Dn"]).max() <= 1e-12 * np.abs(a["Dn"]).max()


def test_PD4_tiny_python_quadruple_sum():
    """Two forests of 5 and 6 pixels: D from a literal Python 4-fold loop with numpy-built eta."""
    f = gen.make_config(0).subset([0, 1])
    keep_p = np.r_[0:5]; keep_q = np.r_[24:30]
    f = gen.two_forests(f.chi[keep_p], f.chi[keep_q], (f.ux[0], f.uy[0], f.uz[0]), (f.ux[1], f.uy[1], f.uz[1]),
                        f.w[keep_p], f.w[keep_q], f.delta[keep_p], f.delta[keep_q], f.loglam[keep_p], f.loglam[keep_q])
    s, c = orc.pair_sc(f, 0, 1)
    b = orc.binning()

    def eta_np(w, ll):
        n = len(w); lbar = (w * ll).sum() / w.sum(); u = ll - lbar
        return np.eye(n) - np.outer(np.ones(n), w) / w.sum() - np.outer(u, w * u) / (w * u * u).sum()
    ep = eta_np(f.w[:5], f.loglam[:5]); eq = eta_np(f.w[5:], f.loglam[5:])
    Dn = np.zeros((2500, 2500)); Wd = np.zeros(2500)
    for i in range(5):
        for j in range(6):
            A = orc.pix_bin(b, s, c, f.chi[i], f.chi[5 + j])
            if A < 0:
                continue
            om = f.w[i] * f.w[5 + j]; Wd[A] += om
            for i2 in range(5):
                for j2 in range(6):
                    B = orc.pix_bin(b, s, c, f.chi[i2], f.chi[5 + j2])
                    if B >= 0:
                        Dn[A, B] += om * ep[i, i2] * eq[j, j2]
    d = orc.dmat(f, [[0, 1]], 0.0, 0)
    assert Wd.sum() > 0
    assert np.allclose(d["Wd"], Wd, rtol=1e-14)
    assert np.abs(d["Dn"] - Dn).max() <= 1e-12 * np.abs(Dn).max()


def test_PD5_two_pixel_forests_have_zero_eta():
    f = gen.make_config(0)
    idx = np.concatenate([np.arange(f.pix_off[p], f.pix_off[p] + 2) for p in range(f.n_forest)])
    g = gen.Forests(f.ra, f.dec, f.ux, f.uy, f.uz, f.zq, np.arange(0, 2 * f.n_forest + 1, 2, dtype=np.int64),
                    f.chi[idx], f.w[idx], f.delta[idx], f.loglam[idx])
    assert np.abs(orc.eta(g.w[:2], g.loglam[:2])).max() < 1e-12
    pq = orc.pairs_brute(g)
    d = orc.dmat(g, pq, 0.0, 0)
    x = orc.xi(g, pq)
    assert np.abs(d["Dn"]).max() <= 1e-9 * d["Wd"].max()
    assert np.allclose(d["Wd"], x["W"], rtol=1e-13)


def test_PD6_no_rejection_matches_xi(cfg0, d0, xi0):
    pq, d = d0
    x = orc.xi(cfg0, pq)
    assert d["n_kept"] == int(x["N"].sum())
    assert np.allclose(d["Wd"], x["W"], rtol=1e-12)


def test_PD7_mask_statistics_and_symmetry():
    thr = orc.mask_threshold(0.99)
    assert thr == round(0.99 * 2 ** 32)
    assert orc.mask_threshold(0.0) == 0 and orc.mask_threshold(1.0) == 2 ** 32
    n = 400
    kept = np.array([[orc.keep(12345, i, 1000 + j, thr) for j in range(n)] for i in range(n)])
    tot = n * n
    assert abs(kept.mean() - 0.01) < 4 * np.sqrt(0.01 * 0.99 / tot)
    assert orc.keep(12345, 5, 1007, thr) == orc.keep(12345, 1007, 5, thr)
    assert all(orc.keep(1, i, i + 1, 0) for i in range(50))                  # f = 0 keeps all
    assert not any(orc.keep(1, i, i + 1, 2 ** 32) for i in range(50))        # f = 1 keeps none
    # no visible structure: rows / columns / diagonals all at the nominal rate (f = 0.5 for power)
    thr5 = orc.mask_threshold(0.5)
    k5 = np.array([[orc.keep(999, i, 5000 + j, thr5) for j in range(n)] for i in range(n)], float)
    for v in (k5.mean(0), k5.mean(1)):
        chi2 = (((v - 0.5) ** 2) / (0.25 / n)).sum()
        assert abs(chi2 - n) < 5 * np.sqrt(2 * n)
    # 2x2 minors: keep(i,j) keep(i,j') keep(i',j) keep(i',j') independent -> product mean = 1/16
    m = (k5[:-1, :-1] * k5[:-1, 1:] * k5[1:, :-1] * k5[1:, 1:]).mean()
    assert abs(m - 1 / 16) < 5 * np.sqrt((1 / 16) * (15 / 16) / ((n - 1) ** 2)) * 2
    # a different seed gives a different, equally dense mask
    k6 = np.array([[orc.keep(1000, i, 5000 + j, thr5) for j in range(100)] for i in range(100)], float)
    assert abs((k6 == k5[:100, :100]).mean() - 0.5) < 0.03


def _mask_vectors():
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "mask_vectors.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    return [(int(r[0]), int(r[1]), int(r[2]), float(r[3]), int(r[4]), int(r[5]), int(r[6])) for r in rows]


def test_PD7_mask_known_answer_vectors():
    """DESIGN.md section 2.1 restated in Python big integers by tests/golden/make_mask_vectors.py
    (imports nothing from the repo): threshold and keep decision of every vector."""
    rows = _mask_vectors()
    assert len(rows) > 600 and 50 < sum(r[6] for r in rows) < len(rows) - 50
    for seed, a, b, f, thr, _, kp in rows:
        assert orc.mask_threshold(f) == thr
        assert int(orc.keep(seed, a, b, thr)) == kp, (seed, a, b, f)


def test_PD7_kept_fraction_in_dmat(cfg0):
    pq = orc.pairs_brute(cfg0)
    x = orc.xi(cfg0, pq)
    tot = int(x["N"].sum())
    d = orc.dmat(cfg0, pq, 0.9, gen.mask_seed(3))
    assert abs(d["n_kept"] / tot - 0.1) < 4 * np.sqrt(0.1 * 0.9 / tot)
    # kept fraction per bin shows no structure (chi^2 over well-filled bins)
    Nk = np.zeros(2500)
    thr = orc.mask_threshold(0.9)
    b = orc.binning()
    for p, q in pq[:300]:
        s, c = orc.pair_sc(cfg0, p, q)
        for i in range(cfg0.pix_off[p], cfg0.pix_off[p + 1]):
            for j in range(cfg0.pix_off[q], cfg0.pix_off[q + 1]):
                A = orc.pix_bin(b, s, c, cfg0.chi[i], cfg0.chi[j])
                if A >= 0 and orc.keep(gen.mask_seed(3), i, j, thr):
                    Nk[A] += 1
    x300 = orc.xi(cfg0, pq[:300])["N"].astype(float)
    sel = x300 >= 50
    chi2 = (((Nk[sel] - 0.1 * x300[sel]) ** 2) / (0.09 * x300[sel])).sum()
    assert abs(chi2 - sel.sum()) < 5 * np.sqrt(2 * sel.sum())


def test_PD8_normalisation_sanity(cfg0, d0):
    pq, d = d0
    D = d["D"]; nz = d["Wd"] > 0
    diag = np.diag(D)[nz]
    assert np.all(diag > 0.5) and np.all(diag < 1.0)             # 1 - O(1/n), n = 24
    off = D[nz][:, nz] - np.diag(diag)
    assert np.abs(off).max() < 0.5 and np.all(np.abs(off).max(1) < diag)   # diagonally dominant
    # large-grid variant: nothing is out of the grid, so rows of Dn sum to zero with no bucket
    big = orc.binning(8192.0, 8192.0, 16, 16)
    db = orc.dmat(cfg0, pq[:400], 0.0, 0, b=big)
    assert np.abs(db["Dover"]).max() == 0.0
    assert np.all(np.abs(db["Dn"].sum(1)) <= 1e-11 * np.abs(db["Dn"]).sum(1) + 1e-300)


# ---------------------------------------------------------------- NEXT-2: forest-pair subsampling
def test_forest_pair_subsample_statistics_and_linearity(cfg0):
    """The forest-pair subset is a deterministic ~(1-f) fraction of the list, keeps the order, and
    D of a union of disjoint forest-pair subsets is the Wd-weighted combination of their Dn
    (Dn and Wd are additive over forest pairs, eq. 2.6)."""
    pq = orc.pairs_all(cfg0.n_forest)
    sub = orc.subsample_forest_pairs(pq, 0.7, 77)
    n = len(pq)
    assert abs(len(sub) - 0.3 * n) < 4 * np.sqrt(0.21 * n)
    assert np.array_equal(sub, orc.subsample_forest_pairs(pq, 0.7, 77))
    idx = {(int(a), int(b)): k for k, (a, b) in enumerate(pq)}
    pos = [idx[(int(a), int(b))] for a, b in sub]
    assert pos == sorted(pos)
    assert len(orc.subsample_forest_pairs(pq, 0.0, 5)) == n and len(orc.subsample_forest_pairs(pq, 1.0, 5)) == 0
    keep_set = set(map(tuple, sub.tolist()))
    rest = np.array([e for e in pq.tolist() if tuple(e) not in keep_set], dtype=np.int32)
    some = sub[:60]; other = rest[:60]
    d1, d2 = orc.dmat(cfg0, some, 0.0, 0), orc.dmat(cfg0, other, 0.0, 0)
    d12 = orc.dmat(cfg0, np.concatenate([some, other]), 0.0, 0)
    assert np.allclose(d12["Dn"], d1["Dn"] + d2["Dn"], rtol=0, atol=1e-9 * np.abs(d12["Dn"]).max())
    assert np.allclose(d12["Wd"], d1["Wd"] + d2["Wd"], rtol=1e-12)


# ---------------------------------------------------------------- NEXT-1: per-region sub-samples
def test_region_subsamples_partition_the_full_result(cfg0, xi0):
    """Sub-samples partition the forest pairs by the region of the lower-index forest: their N add up
    to the full N exactly and S, W to rounding; a region without forests is empty."""
    pq, full = xi0
    region = (np.arange(cfg0.n_forest) * 7) % 3                       # regions 0, 1, 2 in use; 3 is empty
    subs = orc.xi_sub(cfg0, pq, region, 4)
    assert np.array_equal(sum(s["N"] for s in subs), full["N"])
    assert np.allclose(sum(s["W"] for s in subs), full["W"], rtol=1e-12)
    assert np.all(np.abs(sum(s["S"] for s in subs) - full["S"]) <= 1e-12 * full["Sabs"])
    assert subs[3]["N"].sum() == 0
    # forest 0 has the lowest index of all its pairs: moving it to its own region moves exactly its pairs
    region2 = region.copy(); region2[0] = 3
    subs2 = orc.xi_sub(cfg0, pq, region2, 4)
    only0 = orc.xi(cfg0, pq[pq[:, 0] == 0])
    assert np.array_equal(subs2[3]["N"], only0["N"])


# ---------------------------------------------------------------- NEXT-1: weighted mean r_par, r_perp, z per bin
def test_PM1_means_numpy_enumeration(cfg0):
    """Sums of om r_par, om r_perp, om z per bin against numpy's histogram2d with weights over every
    pixel pair of the neighbour list (an independent library routine, not the oracle's loop)."""
    pq = orc.pairs_brute(cfg0)
    z = 10.0 ** cfg0.loglam / 1215.67 - 1.0
    m = orc.xi_means(cfg0, pq, z)
    edges = np.linspace(0.0, 200.0, 51)
    R1 = np.zeros((50, 50)); R2 = np.zeros((50, 50)); Z = np.zeros((50, 50)); W = np.zeros((50, 50))
    f = cfg0
    for p, q in pq:
        s = 0.5 * np.sqrt((f.ux[p] - f.ux[q]) ** 2 + (f.uy[p] - f.uy[q]) ** 2 + (f.uz[p] - f.uz[q]) ** 2)
        c = np.sqrt(1.0 - s * s)
        a, b = f.pix_off[p], f.pix_off[p + 1]; d, e = f.pix_off[q], f.pix_off[q + 1]
        rpar = (np.abs(f.chi[a:b, None] - f.chi[None, d:e]) * c).ravel()
        rperp = ((f.chi[a:b, None] + f.chi[None, d:e]) * s).ravel()
        om = (f.w[a:b, None] * f.w[None, d:e]).ravel()
        zz = (0.5 * (z[a:b, None] + z[None, d:e])).ravel()
        ok = (rpar < 200.0) & (rperp < 200.0)
        for acc, wt in ((R1, om * rpar), (R2, om * rperp), (Z, om * zz), (W, om)):
            acc += np.histogram2d(rpar[ok], rperp[ok], bins=[edges, edges], weights=wt[ok])[0]
    for got, want in ((m["Rpar"], R1), (m["Rperp"], R2), (m["Z"], Z), (m["W"], W)):
        assert np.allclose(got, want.ravel(), rtol=1e-12, atol=0)


def test_PM2_means_lie_inside_their_bin_and_special_cases(cfg0):
    pq = orc.pairs_brute(cfg0)
    z = 10.0 ** cfg0.loglam / 1215.67 - 1.0
    m = orc.xi_means(cfg0, pq, z)
    x = orc.xi(cfg0, pq)
    assert np.allclose(m["W"], x["W"], rtol=1e-14)                       # the same denominator as eq. 2.4
    nz = m["W"] > 0
    A = np.arange(2500)[nz]
    rp, rt, zb = m["Rpar"][nz] / m["W"][nz], m["Rperp"][nz] / m["W"][nz], m["Z"][nz] / m["W"][nz]
    assert np.all((rp >= 4.0 * (A // 50)) & (rp < 4.0 * (A // 50) + 4.0))   # a weighted mean stays inside its bin
    assert np.all((rt >= 4.0 * (A % 50)) & (rt < 4.0 * (A % 50) + 4.0))
    assert np.all((zb > z.min()) & (zb < z.max()))
    # constant z: the mean redshift of every bin is that constant
    mc = orc.xi_means(cfg0, pq, np.full_like(z, 2.25))
    assert np.allclose(mc["Z"][nz] / mc["W"][nz], 2.25, rtol=1e-13)
    # one pixel pair: the sums are that pair's coordinates times its weight (50-digit arithmetic)
    from decimal import Decimal, getcontext
    getcontext().prec = 50
    s_txt = "0.0123"
    uq = (1.0 - 2.0 * float(s_txt) ** 2, 2.0 * float(s_txt) * float((1 - Decimal(s_txt) ** 2).sqrt()), 0.0)
    f2 = gen.two_forests([4000.0], [4070.5], (1.0, 0.0, 0.0), uq, w_p=[1.5], w_q=[0.25])
    s, c = orc.pair_sc(f2, 0, 1)
    m2 = orc.xi_means(f2, [[0, 1]], np.array([2.0, 3.0]))
    A2 = int(np.nonzero(m2["W"])[0][0])
    rpar = Decimal(70.5) * Decimal(c); rperp = Decimal(8070.5) * Decimal(s)
    assert A2 == 50 * int(rpar / 4) + int(rperp / 4)
    assert abs(m2["W"][A2] - 0.375) < 1e-15
    assert abs(Decimal(float(m2["Rpar"][A2])) / Decimal("0.375") - rpar) < Decimal("1e-11")
    assert abs(Decimal(float(m2["Rperp"][A2])) / Decimal("0.375") - rperp) < Decimal("1e-11")
    assert abs(m2["Z"][A2] / 0.375 - 2.5) < 1e-14


# ---------------------------------------------------------------- NEXT-4: anisotropic 3PCF (eq. 2.8)
def _np_xi3(f, r_max=80.0, n_r=20, n_t=10, n_a=20):
    """Independent numpy evaluation over ALL ordered forest triples: positions, norms, arccos for the two
    line-of-sight angles (the oracle uses cosine edges instead), plain floor for every bin."""
    X = f.chi[:, None] * np.repeat(np.stack([f.ux, f.uy, f.uz], 1), np.diff(f.pix_off), axis=0)
    fid = np.repeat(np.arange(f.n_forest), np.diff(f.pix_off))
    U = np.stack([f.ux, f.uy, f.uz], 1)[fid]
    a = f.w * f.delta
    nb = n_r * n_r * n_a * n_t * n_t
    S = np.zeros(nb); W = np.zeros(nb); N = np.zeros(nb, np.int64)
    for i in range(len(X)):
        d = X - X[i]
        r = np.sqrt((d * d).sum(1))
        ok = (fid != fid[i]) & (r > 0) & (r < r_max)
        idx = np.nonzero(ok)[0]
        if len(idx) < 2:
            continue
        dd, rr = d[idx], r[idx]
        br = np.minimum((rr * (n_r / r_max)).astype(np.int64), n_r - 1)
        th = np.arccos(np.clip((dd @ U[i]) / rr, -1, 1))
        bt = np.minimum((th / (np.pi / n_t)).astype(np.int64), n_t - 1)
        ca = (dd @ dd.T) / np.outer(rr, rr)
        ba = np.clip(((ca + 1.0) * (n_a / 2)).astype(np.int64), 0, n_a - 1)
        J, K = np.meshgrid(np.arange(len(idx)), np.arange(len(idx)), indexing="ij")
        m = fid[idx][J] != fid[idx][K]
        A = (((br[J] * n_r + br[K]) * n_a + ba) * n_t + bt[J]) * n_t + bt[K]
        np.add.at(N, A[m], 1)
        np.add.at(W, A[m], (f.w[i] * f.w[idx][J] * f.w[idx][K])[m])
        np.add.at(S, A[m], (a[i] * a[idx][J] * a[idx][K])[m])
    return S, W, N


@pytest.fixture(scope="module")
def tri_small():
    f = gen.make_config(0).subset(range(12))
    return f, orc.pairs_all(f.n_forest)


def test_PT1_xi3_numpy_brute_force(tri_small):
    f, pq = tri_small
    r = orc.xi3(f, pq)
    S, W, N = _np_xi3(f)
    assert N.sum() > 10000
    assert np.array_equal(r["N3"].astype(np.int64), N)
    assert np.allclose(r["W3"], W, rtol=1e-12) and np.allclose(r["S3"], S, rtol=0, atol=1e-12 * np.abs(S).max())


def test_PT2_xi3_constant_delta_unit_weights_and_swap_symmetry(tri_small):
    f, pq = tri_small
    import copy
    g = copy.deepcopy(f); g.delta[:] = -0.5
    r = orc.xi3(g, pq)
    nz = r["W3"] > 0
    assert np.allclose(r["xi3"][nz], -0.125, rtol=1e-12)                      # d = k  =>  xi3 = k^3
    h = copy.deepcopy(f); h.w[:] = 1.0
    r1 = orc.xi3(h, pq)
    assert np.array_equal(r1["W3"], r1["N3"].astype(float))                    # w = 1  =>  W3 = N3 exactly
    # both orders (j, k) and (k, j) are counted: swapping (r1, theta1) <-> (r2, theta2) is a symmetry
    r0 = orc.xi3(f, pq)
    for key in ("N3", "W3", "S3"):
        T = r0[key].reshape(20, 20, 20, 10, 10)
        assert np.allclose(T, T.transpose(1, 0, 2, 4, 3), rtol=1e-13, atol=1e-13 * np.abs(T).max())


def test_PT3_xi3_neighbour_list_is_enough_and_hand_built_triangle(cfg0):
    f = cfg0.subset(range(30))
    ra = orc.xi3(f, orc.pairs_all(f.n_forest))
    rb = orc.xi3(f, orc.pairs_brute(f, orc.binning(80.0, 80.0, 20, 20)))      # pairs with r_perp < r_max at their first pixels
    assert np.array_equal(ra["N3"], rb["N3"]) and np.allclose(ra["S3"], rb["S3"], rtol=0, atol=1e-13 * np.abs(ra["S3"]).max())
    # three one-pixel forests: vertex i on the x axis at chi = 4000; j 30 Mpc/h further along the line of sight
    # (theta1 = 0); k at 40 Mpc/h from i, 60 degrees off the line of sight, so cos alpha = cos theta2 = 0.5
    xk = np.array([4020.0, 40.0 * np.sqrt(0.75), 0.0])
    ck = float(np.linalg.norm(xk))
    t = gen.two_forests([4000.0], [4030.0], (1.0, 0.0, 0.0), (1.0, 0.0, 0.0), w_p=[2.0], w_q=[3.0], d_p=[0.5], d_q=[-1.0])
    f3 = gen.Forests(np.zeros(3), np.zeros(3), np.array([1.0, 1.0, xk[0] / ck]), np.array([0.0, 0.0, xk[1] / ck]), np.zeros(3),
                     np.zeros(3), np.array([0, 1, 2, 3], np.int64), np.array([4000.0, 4030.0, ck]), np.array([2.0, 3.0, 5.0]),
                     np.array([0.5, -1.0, 0.25]), np.full(3, 3.6))
    r3 = orc.xi3(f3, [[0, 1], [0, 2], [1, 2]])
    assert r3["N3"].sum() == 6                                                 # 3 vertices x 2 orders
    A_ijk = (((7 * 20 + 10) * 20 + 15) * 10 + 0) * 10 + 3                      # r1 = 30 -> 7, r2 = 40 -> 10, cos a = .5 -> 15, th 0 -> 0, 60 deg -> 3
    A_ikj = (((10 * 20 + 7) * 20 + 15) * 10 + 3) * 10 + 0
    assert r3["N3"][A_ijk] == 1 and r3["N3"][A_ikj] == 1
    assert abs(r3["W3"][A_ijk] - 30.0) < 1e-13 and abs(r3["S3"][A_ijk] - (1.0 * -3.0 * 1.25)) < 1e-13
    assert np.allclose(r3["xi3"][r3["N3"] > 0], 0.5 * -1.0 * 0.25)
