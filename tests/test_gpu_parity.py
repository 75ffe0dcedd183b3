"""GPU parity: the CUDA path (through the C-ABI, via the ctypes binding) against the
CPU oracle, element by element on the same seeded inputs.

Bars (BASELINE.json north_star; floors = reading R-16 of DESIGN.md):
  N, n_kept, pair lists : bit-exact / set-equal
  S : |dS_A| <= 1e-9 * max(|S_A|, 1e-4 * Sabs_A)      W : |dW_A| <= 1e-9 * W_A
  D : |dD_AB| <= 1e-7 * max(|D_AB|, 1e-6)
"""
import numpy as np
import pytest

from paper_2507_00129_b200 import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2507_00129_b200 import binding, build
    build.build()
    c = binding.Context("cuda:0")
    yield c
    c.close()


@pytest.fixture(scope="module")
def B():
    from paper_2507_00129_b200 import binding
    return binding


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle
    return oracle


def pair_set(pq):
    pq = np.asarray(pq, dtype=np.int64).reshape(-1, 2)
    return set((pq[:, 0] << 32 | pq[:, 1]).tolist())


def check_xi(g, o, label=""):
    N = g["N"].cpu().numpy().view(np.uint64)
    assert np.array_equal(N, o["N"]), f"{label}: pair counts differ in {(N != o['N']).sum()} bins"
    S = g["S"].cpu().numpy(); W = g["W"].cpu().numpy(); xi = g["xi"].cpu().numpy()
    tolS = 1e-9 * np.maximum(np.abs(o["S"]), 1e-4 * o["Sabs"])
    assert np.all(np.abs(S - o["S"]) <= tolS), f"{label}: S off by {np.max(np.abs(S - o['S']) / np.maximum(tolS, 1e-300))} tol"
    assert np.all(np.abs(W - o["W"]) <= 1e-9 * o["W"]), f"{label}: W"
    nz = o["W"] > 0
    assert np.all(np.abs(xi[nz] - o["xi"][nz]) <= 1e-9 * np.maximum(np.abs(o["xi"][nz]), 1e-4 * o["Sabs"][nz] / o["W"][nz]))
    assert np.all(xi[~nz] == 0.0)
    assert g["stats"]["n_binned"] == int(o["N"].sum())
    assert g["stats"]["n_visited"] == int(o["N"].sum()) + o["n_out"]


def check_dmat(g, o, label=""):
    assert g["stats"]["n_kept"] == o["n_kept"], f"{label}: n_kept {g['stats']['n_kept']} vs {o['n_kept']}"
    Wd = g["Wd"].cpu().numpy()
    assert np.all(np.abs(Wd - o["Wd"]) <= 1e-9 * o["Wd"]), f"{label}: Wd"
    D = g["D"].cpu().numpy()
    err = np.abs(D - o["D"]); tol = 1e-7 * np.maximum(np.abs(o["D"]), 1e-6)
    assert np.all(err <= tol), f"{label}: D worst {np.max(err / tol)} x tol at {np.unravel_index(np.argmax(err / tol), D.shape)}"
    if g["Dn"] is not None:
        Dn = g["Dn"].cpu().numpy()
        scale = np.maximum(o["Wd"], 1e-300)[:, None]
        assert np.all(np.abs(Dn - o["Dn"]) / scale <= tol), f"{label}: Dn"


# ------------------------------------------------------------------ configs[0]
def test_cfg0_neighbours_set_equal(ctx, B, orc, cfg0):
    d = B.DeviceForests(cfg0)
    pairs = ctx.lya_neighbours(d, B.binning())
    pq = pairs.export().cpu().numpy()
    ref = orc.pairs_brute(cfg0)
    assert pairs.n == len(ref)
    assert np.all(pq[:, 0] < pq[:, 1])
    assert len(pair_set(pq)) == len(pq)
    assert pair_set(pq) == pair_set(ref)


def test_cfg0_xi_all_pairs_and_neighbour_list(ctx, B, orc, cfg0):
    d = B.DeviceForests(cfg0)
    b = B.binning()
    pq_all = orc.pairs_all(cfg0.n_forest)
    o = orc.xi(cfg0, pq_all)
    g_all = ctx.lya_xi2pcf(d, b, ctx.lya_pairs_import(pq_all))
    check_xi(g_all, o, "cfg0 all pairs")
    g_nb = ctx.lya_xi2pcf(d, b, ctx.lya_neighbours(d, b))
    assert np.array_equal(g_nb["N"].cpu().numpy().view(np.uint64), o["N"])      # pin P1 on the GPU side


@pytest.mark.parametrize("variant", [1, 2, 4])
def test_cfg0_xi_kernel_variants(B, orc, cfg0, variant):
    c = B.Context("cuda:0")
    c.lya_set_option("force_generic", 1)
    c.lya_set_option("generic_diagonals", variant)
    d = B.DeviceForests(cfg0)
    pq = orc.pairs_brute(cfg0)
    check_xi(c.lya_xi2pcf(d, B.binning(), c.lya_pairs_import(pq)), orc.xi(cfg0, pq), f"variant {variant}")
    c.close()


def test_cfg0_dmat_no_rejection(ctx, B, orc, cfg0):
    d = B.DeviceForests(cfg0)
    pq = orc.pairs_brute(cfg0)
    o = orc.dmat(cfg0, pq, 0.0, gen.mask_seed(0))
    g = ctx.lya_dmat(d, B.binning(), ctx.lya_pairs_import(pq), 0.0, gen.mask_seed(0))
    check_dmat(g, o, "cfg0 f=0")
    # PD6 on the GPU: f = 0 => Wd == W of lya_xi2pcf, n_kept == sum N
    x = ctx.lya_xi2pcf(d, B.binning(), ctx.lya_pairs_import(pq))
    assert g["stats"]["n_kept"] == x["stats"]["n_binned"]
    assert np.allclose(g["Wd"].cpu().numpy(), x["W"].cpu().numpy(), rtol=1e-12)


@pytest.mark.parametrize("f", [0.5, 0.99, 1.0])
def test_cfg0_dmat_with_mask(ctx, B, orc, cfg0, f):
    d = B.DeviceForests(cfg0)
    pq = orc.pairs_brute(cfg0)
    o = orc.dmat(cfg0, pq, f, gen.mask_seed(3))
    g = ctx.lya_dmat(d, B.binning(), ctx.lya_pairs_import(pq), f, gen.mask_seed(3))
    check_dmat(g, o, f"cfg0 f={f}")
    if f == 1.0:
        assert g["stats"]["n_kept"] == 0 and float(g["D"].abs().max()) == 0.0


def test_hand_built_cases_P6(ctx, B, orc):
    import os
    from decimal import Decimal, getcontext
    getcontext().prec = 50
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "p6_hand_cases.txt")
    rows = [l.split("#")[0].split() for l in open(path) if l.strip() and not l.startswith("#")]
    for s_txt, ci, cj, _, _, eA in rows:
        s = float(s_txt)
        uq = (1.0 - 2.0 * s * s, 2.0 * s * float(Decimal(1 - Decimal(s_txt) ** 2).sqrt()), 0.0)
        f = gen.two_forests([float(ci)], [float(cj)], (1.0, 0.0, 0.0), uq)
        g = ctx.lya_xi2pcf(B.DeviceForests(f), B.binning(), ctx.lya_pairs_import([[0, 1]]))
        N = g["N"].cpu().numpy()
        if int(eA) >= 0:
            assert N.sum() == 1 and N[int(eA)] == 1, (s_txt, ci, cj)
        else:
            assert N.sum() == 0


# ------------------------------------------------------------------ shaped sub-workloads
@pytest.mark.parametrize("cfg,n", [(1, 1200), (4, 1500)])
def test_shaped_subpatch_neighbours_and_xi(ctx, B, orc, cfg, n):
    f = gen.make_config(cfg, n_forest=n)
    d = B.DeviceForests(f)
    b = B.binning()
    pairs = ctx.lya_neighbours(d, b)
    ref = orc.pairs_window(f)
    assert pairs.n == len(ref) and pair_set(pairs.export().cpu().numpy()) == pair_set(ref)
    check_xi(ctx.lya_xi2pcf(d, b, pairs), orc.xi(f, ref), f"cfg{cfg} n={n}")


@pytest.mark.parametrize("cfg,n,frac", [(1, 150, 0.9), (4, 200, 0.99), (4, 120, 0.0)])
def test_shaped_subpatch_dmat(ctx, B, orc, cfg, n, frac):
    f = gen.make_config(cfg, n_forest=n, density_scale=4.0)
    d = B.DeviceForests(f)
    pairs = ctx.lya_neighbours(d, B.binning())
    ref = orc.pairs_window(f)
    assert pairs.n == len(ref) and pairs.n > 100
    seed = gen.mask_seed(cfg)
    check_dmat(ctx.lya_dmat(d, B.binning(), pairs, frac, seed), orc.dmat(f, ref, frac, seed), f"cfg{cfg} f={frac}")


def test_generic_binning_non_power_of_two(ctx, B, orc):
    f = gen.make_config(1, n_forest=400)
    d = B.DeviceForests(f)
    b = B.binning(150.0, 90.0, 30, 40)
    ob = orc.binning(150.0, 90.0, 30, 40)
    pairs = ctx.lya_neighbours(d, b)
    ref = orc.pairs_window(f, ob)
    assert pair_set(pairs.export().cpu().numpy()) == pair_set(ref)
    check_xi(ctx.lya_xi2pcf(d, b, pairs), orc.xi(f, ref, ob), "generic bins")
    f2 = gen.make_config(1, n_forest=100, density_scale=4.0)
    ref2 = orc.pairs_window(f2, ob)
    g = ctx.lya_dmat(B.DeviceForests(f2), b, ctx.lya_pairs_import(ref2), 0.8, 5)
    check_dmat(g, orc.dmat(f2, ref2, 0.8, 5, b=ob), "generic bins D")


def test_long_and_ragged_forests_tiles(ctx, B, orc):
    """Forests longer than one staging tile (128 px), plus 1- and 2-pixel forests and an empty one."""
    rng = np.random.default_rng(3)
    lens = [300, 257, 1, 2, 0, 129, 128, 40]
    chis, ws, ds, lls = [], [], [], []
    for n in lens:
        c0 = rng.uniform(3600, 3700)
        chis.append(c0 + np.cumsum(rng.uniform(0.5, 2.5, n)))
        ws.append(rng.uniform(0.5, 2.0, n)); ds.append(rng.normal(0, 0.3, n))
        lls.append(3.55 + 1e-4 * np.arange(n) + rng.uniform(0, 1e-5, n))
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    ra = rng.uniform(0, 0.02, len(lens)); dec = rng.uniform(-0.01, 0.01, len(lens))
    ux, uy, uz = gen.unit_vectors(ra, dec)
    f = gen.Forests(ra, dec, ux, uy, uz, np.zeros(len(lens)), off, np.concatenate(chis), np.concatenate(ws),
                    np.concatenate(ds), np.concatenate(lls))
    d = B.DeviceForests(f)
    pairs = ctx.lya_neighbours(d, B.binning())
    ref = orc.pairs_brute(f)
    assert pair_set(pairs.export().cpu().numpy()) == pair_set(ref)
    check_xi(ctx.lya_xi2pcf(d, B.binning(), pairs), orc.xi(f, ref), "long forests")
    # the distortion matrix of forests longer than a tile (native-resolution shapes take the generic kernel)
    keep = [k for k, n in enumerate(lens) if n >= 2]
    f2 = f.subset(keep)
    ref2 = orc.pairs_brute(f2)
    g = ctx.lya_dmat(B.DeviceForests(f2), B.binning(), ctx.lya_pairs_import(ref2), 0.97, 9)
    check_dmat(g, orc.dmat(f2, ref2, 0.97, 9), "long forests D")


def test_window_search_edges(ctx, B, orc):
    """Forests at the size limits of the fast kernels (72 px for k_xi_fast / class 0 of k_dmat_fast, 144 px for class 1)
    and at the power-of-two lengths the branch-free window searches step through (31..33, 63..65, 127..129), with chi
    ranges that overlap fully, partly (windows that run off either end of q) and not at all."""
    rng = np.random.default_rng(17)
    for lens, (smin, smax), frac in (([72, 72, 71, 65, 64, 63, 33, 32, 31, 2], (4.8, 6.9), 0.9),
                                     ([144, 143, 129, 128, 127, 100, 65], (1.4, 2.6), 0.97)):
        chis, ws, ds, lls = [], [], [], []
        for k, n in enumerate(lens):
            c0 = 3600.0 + (0.0, 30.0, 150.0, 330.0)[k % 4] + rng.uniform(0, 5)       # same start, shifted, barely overlapping, beyond
            chis.append(c0 + np.cumsum(rng.uniform(smin, smax, n)))
            ws.append(rng.uniform(0.5, 2.0, n)); ds.append(rng.normal(0, 0.3, n))
            lls.append(3.55 + 1e-4 * np.arange(n) + rng.uniform(0, 1e-5, n))
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        ra = rng.uniform(0, 0.03, len(lens)); dec = rng.uniform(-0.015, 0.015, len(lens))
        ux, uy, uz = gen.unit_vectors(ra, dec)
        f = gen.Forests(ra, dec, ux, uy, uz, np.zeros(len(lens)), off, np.concatenate(chis), np.concatenate(ws),
                        np.concatenate(ds), np.concatenate(lls))
        d = B.DeviceForests(f)
        ref = orc.pairs_brute(f)
        pairs = ctx.lya_pairs_import(ref)
        check_xi(ctx.lya_xi2pcf(d, B.binning(), pairs), orc.xi(f, ref), f"window edges xi {lens[0]}")
        check_dmat(ctx.lya_dmat(d, B.binning(), pairs, frac, 5), orc.dmat(f, ref, frac, 5), f"window edges D {lens[0]}")


def test_kernel_routes_fast_and_generic(B, orc):
    """The same catalogue through (a) the fast kernels (bucketed list, warp-private tables), (b) the
    generic kernels forced for the whole list, (c) a grid whose 8 Mpc/h r_par bins exceed the pixel
    spacing, so that the bucketing pass itself routes every pair to the generic kernels, and (d) a grid
    with more r_par rows than a sub-histogram holds.  All match the oracle; (a) and (b) agree exactly
    on the integers."""
    f = gen.make_config(4, n_forest=400)
    pq = orc.pairs_window(f)
    pq_d = pq[:400]
    seed = gen.mask_seed(4)
    ox, od = orc.xi(f, pq), orc.dmat(f, pq_d, 0.9, seed)
    res = {}
    for variant in ("0", "9"):                                # "9": LYA_OPT_FORCE_GENERIC
        c = B.Context("cuda:0")
        c.lya_set_option("force_generic", 1 if variant == "9" else 0)
        d = B.DeviceForests(f)
        gx = c.lya_xi2pcf(d, B.binning(), c.lya_pairs_import(pq))
        gd = c.lya_dmat(d, B.binning(), c.lya_pairs_import(pq_d), 0.9, seed)
        check_xi(gx, ox, f"variant {variant}")
        check_dmat(gd, od, f"variant {variant} D")
        res[variant] = (gx["N"].cpu().numpy().copy(), gd["stats"]["n_kept"], gd["stats"]["n_binned"], gd["stats"]["n_scatter"])
        c.close()
    assert np.array_equal(res["0"][0], res["9"][0]) and res["0"][1:3] == res["9"][1:3]
    assert res["0"][3] > 0 and res["9"][3] == 0            # scatter-adds are counted by the fast kernel only
    with pytest.raises(B.LyaError):
        c.lya_set_option("generic_diagonals", 3)
    c = B.Context("cuda:0")
    d = B.DeviceForests(f)
    for (rp, rt, n_par, n_perp) in ((200.0, 200.0, 25, 25), (200.0, 200.0, 64, 50)):
        b, ob = B.binning(rp, rt, n_par, n_perp), orc.binning(rp, rt, n_par, n_perp)
        check_xi(c.lya_xi2pcf(d, b, c.lya_pairs_import(pq)), orc.xi(f, pq, ob), f"grid {n_par}x{n_perp}")
        check_dmat(c.lya_dmat(d, b, c.lya_pairs_import(pq_d), 0.9, seed), orc.dmat(f, pq_d, 0.9, seed, b=ob),
                   f"grid {n_par}x{n_perp} D")
    c.close()


def test_one_holder_invariant_debug_variant(B, orc):
    """LYA_OPT_CHECK_HOLDERS: the debug variant of the fast D kernel checks at every row step of pass A that no
    two lanes of a warp hold the same H-table entry (the invariant the atomic-free accumulation rests on).
    It must report no violation on a configs[4]-shaped sub-patch and give the same result."""
    f = gen.make_config(4, n_forest=300, density_scale=2.0)
    seed = gen.mask_seed(4)
    c = B.Context("cuda:0")
    c.lya_set_option("check_holders", 1)
    d = B.DeviceForests(f)
    pairs = c.lya_neighbours(d, B.binning())
    check_xi(c.lya_xi2pcf(d, B.binning(), pairs), orc.xi(f, orc.pairs_window(f)), "check_holders xi")   # same check in k_xi_fast
    g = c.lya_dmat(d, B.binning(), pairs, 0.9, seed)          # raises LYA_ERR_CUDA on a violation
    ref = orc.pairs_window(f)
    check_dmat(g, orc.dmat(f, ref, 0.9, seed), "check_holders")
    assert g["stats"]["n_scatter"] > 0                        # the fast kernel ran
    c.close()


def test_xi_merge_guard(B, orc):
    """The guard that merges a warp's sub-histogram before its 32-bit pair counters can overflow (default: every
    2^31 visited pairs, which no workload here reaches) is driven by lowering it: N stays bit-exact."""
    f = gen.make_config(4, n_forest=800)
    ref = orc.pairs_window(f)
    o = orc.xi(f, ref)
    for every in (1, 5000, 1 << 31):
        c = B.Context("cuda:0")
        c.lya_set_option("xi_merge_every", every)
        check_xi(c.lya_xi2pcf(B.DeviceForests(f), B.binning(), c.lya_pairs_import(ref)), o, f"merge every {every}")
        c.close()


@pytest.mark.parametrize("cfg,fine,n,frac", [(2, 2, 150, 0.97), (4, 2, 120, 0.99), (0, 4, 64, 0.9), (0, 6, 40, 0.5)])
def test_native_resolution_fast_class_next3(B, orc, cfg, fine, n, frac):
    """NEXT-3 shapes: pixel spacing BELOW the r_par bin width (3.3 Mpc/h at fine = 2, the SDSS spacing of
    PAPER.md:142; 1.6 / 1.1 Mpc/h at fine = 4 / 6) and forests of up to 144 pixels take the second size class of
    the fast D kernel (diagonal stride 2..4).  D and xi against the naive oracle; the debug variant also checks
    that no H-table entry ever has two holders."""
    f = gen.make_config(cfg, n_forest=n, density_scale=4.0, fine=fine)
    assert np.diff(f.pix_off).max() <= 144 and np.diff(f.chi)[np.diff(f.chi) > 0].min() < 4.0
    seed = gen.mask_seed(cfg)
    ref = orc.pairs_window(f)
    od, ox = orc.dmat(f, ref, frac, seed), orc.xi(f, ref)
    for check in (1, 0):
        c = B.Context("cuda:0")
        c.lya_set_option("check_holders", check)
        d = B.DeviceForests(f)
        pairs = c.lya_neighbours(d, B.binning())
        assert pairs.n == len(ref)
        g = c.lya_dmat(d, B.binning(), pairs, frac, seed)
        check_dmat(g, od, f"cfg{cfg} fine={fine} check={check}")
        assert g["stats"]["n_scatter"] > 0.5 * od["n_kept"]           # the fast kernel took (most of) the pairs
        check_xi(c.lya_xi2pcf(d, B.binning(), pairs), ox, f"cfg{cfg} fine={fine} xi")
        c.close()


@pytest.mark.parametrize("cfg,fine,n,frac", [(4, 5, 48, 0.99), (2, 4, 40, 0.9), (0, 12, 16, 0.98), (0, 8, 5, 0.0),
                                             (4, 10, 12, 0.995), (4, 16, 8, 0.995)])
def test_long_forest_kernel_next3(B, orc, cfg, fine, n, frac):
    """NEXT-3 shapes with LONG forests (observed-frame 2.4 A, SDSS 3e-4 log steps, DESI 0.8 A):
    145..1024 pixels, spacing down to 0.33 Mpc/h (diagonal stride up to 13 of the 16 allowed) take k_dmat_long, one
    CTA per forest pair (per-warp H tables summed, banded stage-4 scan and drain).  f = 0.9 and f = 0 need several
    bands per forest pair; the last case mixes in forests above 1024 pixels, which stay with the generic kernel.  D and xi against
    the naive oracle; the debug variant also checks that no H-table entry ever has two holders."""
    f = gen.make_config(cfg, n_forest=n, density_scale=4.0, fine=fine)
    assert np.diff(f.pix_off).max() > 144
    seed = gen.mask_seed(cfg)
    ref = orc.pairs_window(f)
    od, ox = orc.dmat(f, ref, frac, seed), orc.xi(f, ref)
    for check in (1, 0):
        c = B.Context("cuda:0")
        c.lya_set_option("check_holders", check)
        d = B.DeviceForests(f)
        pairs = c.lya_neighbours(d, B.binning())
        assert pairs.n == len(ref)
        g = c.lya_dmat(d, B.binning(), pairs, frac, seed)
        check_dmat(g, od, f"long cfg{cfg} fine={fine} check={check}")
        assert g["stats"]["n_scatter"] > 0.5 * od["n_kept"]           # k_dmat_long took (most of) the pairs
        check_xi(c.lya_xi2pcf(d, B.binning(), pairs), ox, f"long cfg{cfg} fine={fine} xi")
        c.close()


def test_forest_pair_subsampling_next2(ctx, B, orc):
    """D from a subset of FOREST pairs = lya_pairs_subsample + lya_dmat(f = 0)."""
    f = gen.make_config(1, n_forest=150, density_scale=4.0)
    d = B.DeviceForests(f)
    pairs = ctx.lya_neighbours(d, B.binning())
    pq = pairs.export().cpu().numpy()
    for frac, seed in ((0.9, 11), (0.5, 12)):
        sub = ctx.lya_pairs_subsample(pairs, frac, seed)
        want = orc.subsample_forest_pairs(pq, frac, seed)
        assert sub.n == len(want) and np.array_equal(sub.export().cpu().numpy(), want)      # same set, same order
        check_dmat(ctx.lya_dmat(d, B.binning(), sub, 0.0, 0), orc.dmat(f, want, 0.0, 0), f"forest-pair subset f={frac}")
    assert ctx.lya_pairs_subsample(pairs, 1.0, 3).n == 0 and ctx.lya_pairs_subsample(pairs, 0.0, 3).n == pairs.n


def test_mask_known_answer_vectors_gpu(ctx, B):
    """The CUDA keep mask against the big-integer vectors of tests/golden/mask_vectors.txt (the
    specification of DESIGN.md section 2.1, written by a script that imports nothing from the repo),
    through lya_pairs_subsample (forest indices as ids), one call per (seed, fraction) group."""
    import os
    from collections import defaultdict
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "mask_vectors.txt")
    groups = defaultdict(list)
    for l in open(path):
        if l.strip() and not l.startswith("#"):
            r = l.split()
            if int(r[1]) < 2 ** 31 and int(r[2]) < 2 ** 31:
                groups[(int(r[0]), r[3])].append((int(r[1]), int(r[2]), int(r[6])))
    n_checked = 0
    for (seed, f), rows in groups.items():
        pq = np.array([[a, b] for a, b, _ in rows], dtype=np.int32)
        sub = ctx.lya_pairs_subsample(ctx.lya_pairs_import(pq), float(f), seed)
        want = np.array([[min(a, b), max(a, b)] for a, b, k in rows if k], dtype=np.int32).reshape(-1, 2)
        assert sub.n == len(want) and np.array_equal(sub.export().cpu().numpy(), want), (seed, f)
        n_checked += len(rows)
    assert n_checked > 600


def test_region_subsamples_next1(ctx, B, orc):
    """lya_xi2pcf_sub against the oracle region by region: fast kernel (bucketed list) and, with a grid
    whose bins exceed the pixel spacing, the direct kernel; the regions add up to lya_xi2pcf."""
    f = gen.make_config(1, n_forest=600)
    d = B.DeviceForests(f)
    rng = np.random.default_rng(5)
    n_region = 5
    region = rng.integers(0, n_region - 1, f.n_forest).astype(np.int32)          # region 4 stays empty
    for grid in ((200.0, 200.0, 50, 50), (200.0, 200.0, 25, 25)):
        b, ob = B.binning(*grid), orc.binning(*grid)
        pairs = ctx.lya_neighbours(d, b)
        pq = pairs.export().cpu().numpy()
        g = ctx.lya_xi2pcf_sub(d, b, pairs, region, n_region)
        full = ctx.lya_xi2pcf(d, b, pairs)
        want = orc.xi_sub(f, pq, region, n_region, ob)
        N = g["N"].cpu().numpy().view(np.uint64); S = g["S"].cpu().numpy(); W = g["W"].cpu().numpy()
        for r in range(n_region):
            o = want[r]
            assert np.array_equal(N[r], o["N"]), f"region {r}"
            assert np.all(np.abs(W[r] - o["W"]) <= 1e-9 * o["W"])
            assert np.all(np.abs(S[r] - o["S"]) <= 1e-9 * np.maximum(np.abs(o["S"]), 1e-4 * o["Sabs"]))
        assert np.array_equal(N.sum(0), full["N"].cpu().numpy().view(np.uint64)) and N[4].sum() == 0
        assert g["stats"]["n_binned"] == full["stats"]["n_binned"]
    with pytest.raises(B.LyaError):
        ctx.lya_xi2pcf_sub(d, B.binning(), pairs, region + 3, n_region)


def test_region_subsamples_native_resolution(ctx, B, orc):
    """NEXT-1 on NEXT-3 shapes: per-region S, W, N of a fine-spacing catalogue (second size class of k_xi_fast, with the
    warp-private sub-histograms merged per region) against the oracle, and adding up to lya_xi2pcf."""
    f = gen.make_config(2, n_forest=160, fine=2)
    d = B.DeviceForests(f)
    rng = np.random.default_rng(6)
    n_region = 3
    region = rng.integers(0, n_region, f.n_forest).astype(np.int32)
    b, ob = B.binning(), orc.binning()
    pairs = ctx.lya_neighbours(d, b)
    pq = pairs.export().cpu().numpy()
    g = ctx.lya_xi2pcf_sub(d, b, pairs, region, n_region)
    full = ctx.lya_xi2pcf(d, b, pairs)
    want = orc.xi_sub(f, pq, region, n_region, ob)
    N = g["N"].cpu().numpy().view(np.uint64); S = g["S"].cpu().numpy(); W = g["W"].cpu().numpy()
    for r in range(n_region):
        o = want[r]
        assert np.array_equal(N[r], o["N"]), f"region {r}"
        assert np.all(np.abs(W[r] - o["W"]) <= 1e-9 * o["W"])
        assert np.all(np.abs(S[r] - o["S"]) <= 1e-9 * np.maximum(np.abs(o["S"]), 1e-4 * o["Sabs"]))
    assert np.array_equal(N.sum(0), full["N"].cpu().numpy().view(np.uint64))
    check_xi(full, orc.xi(f, pq), "fine-spacing xi")


def test_sharded_halves_sum_to_full(ctx, B, orc):
    """SURVEY 8(e) on one device: the two chunks of shard.split_pairs, run separately and summed,
    equal the un-split run (N, n_kept exactly) and, after lya_xi_normalise / lya_dmat_normalise,
    the oracle on the full list."""
    import torch
    from paper_2507_00129_b200 import shard
    f = gen.make_config(4, n_forest=500, density_scale=2.0)
    d = B.DeviceForests(f)
    b = B.binning()
    seed = gen.mask_seed(4)
    pairs = ctx.lya_neighbours(d, b)
    pq = pairs.export()
    lens = d.pix_off[1:] - d.pix_off[:-1]
    full_x = ctx.lya_xi2pcf(d, b, pairs)
    acc = None
    n_chunk = []
    for r in range(2):
        mine = shard.split_pairs(pq, lens, r, 2).contiguous()
        n_chunk.append(len(mine))
        pr = ctx.lya_pairs_import(mine)
        x = ctx.lya_xi2pcf(d, b, pr)
        dm = ctx.lya_dmat(d, b, pr, 0.9, seed, want_Dn=True, want_D=False)
        assert dm["D"] is None
        part = [x["S"], x["W"], x["N"], dm["Dn"], dm["Wd"], dm["stats"]["n_kept"]]
        acc = part if acc is None else [a + p for a, p in zip(acc, part)]
    assert sum(n_chunk) == pairs.n and min(n_chunk) > 0
    assert torch.equal(acc[2], full_x["N"])
    ref = orc.pairs_window(f)
    ox, od = orc.xi(f, ref), orc.dmat(f, ref, 0.9, seed)
    g = dict(S=acc[0], W=acc[1], N=acc[2], xi=ctx.lya_xi_normalise(acc[0], acc[1]), stats=full_x["stats"])
    check_xi(g, ox, "two chunks summed")
    gd = dict(D=ctx.lya_dmat_normalise(b, acc[3], acc[4]), Dn=acc[3], Wd=acc[4], stats=dict(n_kept=acc[5]))
    check_dmat(gd, od, "two chunks summed D")
    # the sharded step itself (world = 1: no group needed) equals the same oracle
    st = shard.sharded_step(ctx, d, b, 0.9, seed, 0, 1)
    check_xi(dict(S=st["S"], W=st["W"], N=st["N"], xi=st["xi"], stats=st["stats_xi"]), ox, "sharded_step")
    check_dmat(dict(D=st["D"], Dn=st["Dn"], Wd=st["Wd"], stats=st["stats_dmat"]), od, "sharded_step D")


def test_weighted_mean_coordinates_next1(ctx, B, orc):
    """lya_xi2pcf_means against the oracle: sums of om r_par, om r_perp, om z and W per bin to 1e-9, on a
    power-of-two and a generic grid; the means come out of lya_xi_normalise."""
    f = gen.make_config(1, n_forest=500)
    d = B.DeviceForests(f)
    z = 10.0 ** f.loglam / 1215.67 - 1.0
    for grid in ((200.0, 200.0, 50, 50), (150.0, 90.0, 30, 40)):
        b, ob = B.binning(*grid), orc.binning(*grid)
        pairs = ctx.lya_neighbours(d, b)
        pq = pairs.export().cpu().numpy()
        g = ctx.lya_xi2pcf_means(d, b, pairs, z)
        o = orc.xi_means(f, pq, z, ob)
        for k in ("Rpar", "Rperp", "Z", "W"):
            assert np.all(np.abs(g[k].cpu().numpy() - o[k]) <= 1e-9 * np.abs(o[k])), k
        nz = o["W"] > 0
        zbar = ctx.lya_xi_normalise(g["Z"], g["W"]).cpu().numpy()
        assert np.all(np.abs(zbar[nz] - o["Z"][nz] / o["W"][nz]) <= 1e-9) and np.all(zbar[~nz] == 0.0)
        x = ctx.lya_xi2pcf(d, b, pairs)
        assert np.allclose(g["W"].cpu().numpy(), x["W"].cpu().numpy(), rtol=1e-12)      # eq. 2.4's denominator


def test_anisotropic_3pcf_next4(ctx, B, orc):
    """lya_xi3pcf (eq. 2.8) against the brute-force oracle: ordered-triple counts per triangle bin bit-exact,
    S3 and W3 to 1e-9, on configs[0] with the paper's 20 x 20 x 20 x 10 x 10 bins up to 80 Mpc/h (Fig. 5) and on
    a denser configs[1]-shaped patch with the 40 Mpc/h of Tables 2-3 and a coarser grid."""
    for f, grid in ((gen.make_config(0), (80.0, 20, 10, 20)), (gen.make_config(1, n_forest=250, density_scale=6.0), (40.0, 8, 5, 6))):
        d = B.DeviceForests(f)
        tb, otb = B.tri_binning(*grid), orc.tri_binning(*grid)
        ce = np.cos(np.pi * np.arange(1, grid[2]) / grid[2])
        b2 = B.binning(grid[0], grid[0], 20, 20)
        pairs = ctx.lya_neighbours(d, b2)                                  # r_perp < r_max: a superset of what is needed
        g = ctx.lya_xi3pcf(d, tb, ce, pairs)
        o = orc.xi3(f, pairs.export().cpu().numpy(), otb, ce)
        N3 = g["N3"].cpu().numpy().view(np.uint64)
        assert int(o["N3"].sum()) > 100000
        assert np.array_equal(N3, o["N3"]), f"{(N3 != o['N3']).sum()} triangle bins differ"
        assert g["stats"]["n_binned"] == int(o["N3"].sum())
        assert np.all(np.abs(g["W3"].cpu().numpy() - o["W3"]) <= 1e-9 * o["W3"])
        S3 = g["S3"].cpu().numpy()
        assert np.all(np.abs(S3 - o["S3"]) <= 1e-9 * np.maximum(np.abs(o["S3"]), 1e-6 * np.abs(o["S3"]).max()))
        nz = o["W3"] > 0
        assert np.all(g["xi3"].cpu().numpy()[~nz] == 0.0)


# ------------------------------------------------------------------ invariances and edge cases
def test_P7_pair_order_and_swap(ctx, B, orc, cfg0):
    d = B.DeviceForests(cfg0)
    pq = orc.pairs_brute(cfg0)
    rng = np.random.default_rng(11)
    g0 = ctx.lya_xi2pcf(d, B.binning(), ctx.lya_pairs_import(pq))
    g1 = ctx.lya_xi2pcf(d, B.binning(), ctx.lya_pairs_import(pq[rng.permutation(len(pq))][:, ::-1].copy()))
    assert np.array_equal(g0["N"].cpu().numpy(), g1["N"].cpu().numpy())
    assert np.allclose(g0["W"].cpu().numpy(), g1["W"].cpu().numpy(), rtol=1e-12)
    a = ctx.lya_dmat(d, B.binning(), ctx.lya_pairs_import(pq), 0.9, 9)
    b = ctx.lya_dmat(d, B.binning(), ctx.lya_pairs_import(pq[rng.permutation(len(pq))]), 0.9, 9)
    assert a["stats"]["n_kept"] == b["stats"]["n_kept"]
    assert np.allclose(a["Dn"].cpu().numpy(), b["Dn"].cpu().numpy(), rtol=0, atol=1e-10 * float(a["Wd"].max()))


def test_P8_degenerate_catalogues(ctx, B, cfg0):
    one = cfg0.subset([5])
    d = B.DeviceForests(one)
    pairs = ctx.lya_neighbours(d, B.binning())
    assert pairs.n == 0
    g = ctx.lya_xi2pcf(d, B.binning(), pairs)
    assert int(g["N"].sum()) == 0 and float(g["S"].abs().sum()) == 0 and float(g["xi"].abs().sum()) == 0
    far = gen.two_forests(cfg0.chi[:24], cfg0.chi[24:48], (1, 0, 0), (0, 1, 0))
    assert ctx.lya_neighbours(B.DeviceForests(far), B.binning()).n == 0


def test_P9_rotations_wrap_and_pole(ctx, B, orc, cfg0):
    """Rigid rotations (across RA = 0 and over a pole): the cell grid must list the same set;
    N equal except for pairs the rounding of the rotated unit vectors moves across an edge."""
    d0 = B.DeviceForests(cfg0)
    N0 = ctx.lya_xi2pcf(d0, B.binning(), ctx.lya_neighbours(d0, B.binning()))["N"].cpu().numpy()
    for ang_y, ang_z in [(0.0, -0.03), (np.pi / 2 - 0.01, 0.3), (np.pi / 2, 0.0), (-np.pi / 2 + 0.02, 3.1)]:
        cy, sy, cz, sz = np.cos(ang_y), np.sin(ang_y), np.cos(ang_z), np.sin(ang_z)
        Ry = np.array([[cy, 0, -sy], [0, 1, 0], [sy, 0, cy]]); Rz = np.array([[cz, -sz, 0], [sz, cz, 0], [0, 0, 1]])
        u = (Rz @ Ry @ np.stack([cfg0.ux, cfg0.uy, cfg0.uz]))
        f = gen.Forests(np.arctan2(u[1], u[0]), np.arcsin(np.clip(u[2], -1, 1)), u[0].copy(), u[1].copy(), u[2].copy(),
                        cfg0.zq, cfg0.pix_off, cfg0.chi, cfg0.w, cfg0.delta, cfg0.loglam)
        d = B.DeviceForests(f, with_radec=True)
        pairs = ctx.lya_neighbours(d, B.binning())
        assert pair_set(pairs.export().cpu().numpy()) == pair_set(orc.pairs_brute(f))
        g = ctx.lya_xi2pcf(d, B.binning(), pairs)
        check_xi(g, orc.xi(f, orc.pairs_brute(f)), "rotated")
        assert np.abs(g["N"].cpu().numpy() - N0).sum() <= 8          # edge-straddling pairs only
        # device-derived unit vectors (ra/dec only): same list up to edge-ambiguous pairs
        p2 = ctx.lya_neighbours(d, B.binning(), use_u=False)
        assert abs(p2.n - pairs.n) <= 2


def test_error_statuses(ctx, B, cfg0):
    bad = gen.make_config(0)
    bad.chi[5], bad.chi[6] = bad.chi[6], bad.chi[5]
    d = B.DeviceForests(bad)
    with pytest.raises(B.LyaError) as e:
        ctx.lya_neighbours(d, B.binning())
    assert e.value.name == "LYA_ERR_UNSORTED"
    nanf = gen.make_config(0); nanf.w[100] = np.nan
    with pytest.raises(B.LyaError) as e:
        ctx.lya_neighbours(B.DeviceForests(nanf), B.binning())
    assert e.value.name == "LYA_ERR_INVALID_ARG"
    with pytest.raises(B.LyaError) as e:
        ctx.lya_neighbours(B.DeviceForests(cfg0), B.binning(200.0, 200.0, 100, 100))
    assert e.value.name == "LYA_ERR_CAPACITY"
    deg = gen.make_config(0); deg.loglam[:24] = 3.6                    # forest 0: a single lambda -> V = 0
    dd = B.DeviceForests(deg)
    with pytest.raises(B.LyaError) as e:
        ctx.lya_dmat(dd, B.binning(), ctx.lya_pairs_import([[0, 1]]), 0.0, 1)
    assert e.value.name == "LYA_ERR_DEGENERATE_FOREST"
    with pytest.raises(B.LyaError) as e:
        ctx.lya_xi2pcf(B.DeviceForests(cfg0), B.binning(), ctx.lya_pairs_import([[0, 99]]))
    assert e.value.name == "LYA_ERR_INVALID_ARG"
    with pytest.raises(B.LyaError):
        ctx.lya_pairs_import([[3, 3]])
    with pytest.raises(B.LyaError) as e:                               # sentinel pixels must stay outside any grid
        ctx.lya_neighbours(B.DeviceForests(cfg0), B.binning(2.0e5, 200.0, 50, 50))
    assert e.value.name == "LYA_ERR_CAPACITY"
    notunit = gen.make_config(0); notunit.ux[3] *= 1.001
    with pytest.raises(B.LyaError) as e:
        ctx.lya_neighbours(B.DeviceForests(notunit), B.binning())
    assert e.value.name == "LYA_ERR_INVALID_ARG"
    # the degenerate-forest rule (reading R-7) is the same on the generic route: all L equal up to rounding
    deg2 = gen.make_config(0); deg2.loglam[:24] = 3.6 + 4.5e-16 * np.arange(24)
    cg = B.Context("cuda:0")
    cg.lya_set_option("force_generic", 1)
    with pytest.raises(B.LyaError) as e:
        cg.lya_dmat(B.DeviceForests(deg2), B.binning(), cg.lya_pairs_import([[0, 1]]), 0.0, 1)
    assert e.value.name == "LYA_ERR_DEGENERATE_FOREST"
    cg.close()


def test_zero_weights_count_geometrically(ctx, B, orc):
    f = gen.make_config(0); f.w[::3] = 0.0                              # reading R-7
    pq = orc.pairs_brute(f)
    check_xi(ctx.lya_xi2pcf(B.DeviceForests(f), B.binning(), ctx.lya_pairs_import(pq)), orc.xi(f, pq), "w=0")


def test_run_host_end_to_end(ctx, B, orc, cfg0):
    out = ctx.lya_run_host(cfg0, B.binning(), do_xi=True, do_dmat=True, reject_fraction=0.5, seed=42)
    pq = orc.pairs_brute(cfg0)
    o = orc.xi(cfg0, pq)
    assert out["n_pairs"] == len(pq)
    assert np.array_equal(out["N"], o["N"])
    assert np.all(np.abs(out["W"] - o["W"]) <= 1e-9 * o["W"])
    od = orc.dmat(cfg0, pq, 0.5, 42)
    assert out["stats_dmat"]["n_kept"] == od["n_kept"]
    assert np.all(np.abs(out["D"] - od["D"]) <= 1e-7 * np.maximum(np.abs(od["D"]), 1e-6))


# ------------------------------------------------------------------ full-size configs, bench launch configuration
@pytest.mark.parametrize("cfg", [1, 2, 4])
def test_full_size_properties_and_sampled_parity(ctx, B, orc, cfg):
    """At BASELINE.json's full sizes the oracle cannot run everything: check the neighbour list
    on sampled forests against a numpy brute force over ALL forests, the exact bookkeeping
    identities, and element-by-element parity on a random sample of the listed forest pairs."""
    import torch
    f = gen.make_config(cfg)
    d = B.DeviceForests(f)
    b = B.binning()
    pairs = ctx.lya_neighbours(d, b)
    pq = pairs.export()
    assert bool((pq[:, 0] < pq[:, 1]).all())
    # (1) neighbour sets of sampled forests vs numpy over all N
    rng = np.random.default_rng(cfg)
    cm = f.chi[f.pix_off[:-1]]
    for p in rng.choice(f.n_forest, 40, replace=False):
        s = 0.5 * np.sqrt((f.ux - f.ux[p]) ** 2 + (f.uy - f.uy[p]) ** 2 + (f.uz - f.uz[p]) ** 2)
        want = set(np.nonzero(((cm + cm[p]) * s < 200.0) & (np.arange(f.n_forest) != p))[0].tolist())
        got = set(pq[pq[:, 0] == p][:, 1].cpu().tolist()) | set(pq[pq[:, 1] == p][:, 0].cpu().tolist())
        assert got == want
    # (2) exact bookkeeping at full size
    g = ctx.lya_xi2pcf(d, b, pairs)
    lens = torch.from_numpy(np.diff(f.pix_off)).to(pq.device)
    visited = int((lens[pq[:, 0].long()] * lens[pq[:, 1].long()]).sum())
    assert g["stats"]["n_visited"] == visited
    assert int(g["N"].sum()) == g["stats"]["n_binned"] <= visited
    assert float(g["W"].min()) > 0
    # (3) sampled forest pairs: full parity
    sel = torch.from_numpy(rng.choice(pairs.n, 20000, replace=False)).to(pq.device)
    sub = pq[sel].cpu().numpy()
    check_xi(ctx.lya_xi2pcf(d, b, ctx.lya_pairs_import(sub)), orc.xi(f, sub), f"cfg{cfg} sampled pairs")
    subd = sub[:5000]
    seed = gen.mask_seed(3 if cfg == 2 else cfg)
    check_dmat(ctx.lya_dmat(d, b, ctx.lya_pairs_import(subd), 0.99, seed), orc.dmat(f, subd, 0.99, seed),
               f"cfg{cfg} sampled pairs D")
