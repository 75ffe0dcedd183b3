"""lya_xi2pcf_plan_noalloc (include/lya.h): stage 2 with its accumulators in the library's static device array.

Collected last on purpose (the suite runs with `pytest -x`).  Runs alone in a fresh process or after the rest of
the suite: it makes its own context and catalogues and depends on no state left by other tests.
"""
import numpy as np
import pytest

from paper_2507_00129_b200 import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_00129_b200 import binding
    return binding


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle
    return oracle


def same_as(g, ref, o, label):
    """The no-alloc result g against the existing path's ref: pair counts bit-exact, S / W / xi within the suite's
    1e-9 (floors from the oracle's sum of |terms|, as check_xi in test_gpu_parity.py)."""
    Ng, Nr = g["N"].cpu().numpy().view(np.uint64), ref["N"].cpu().numpy().view(np.uint64)
    assert np.array_equal(Ng, Nr), f"{label}: pair counts differ in {(Ng != Nr).sum()} bins"
    assert np.array_equal(Ng, o["N"]), f"{label}: pair counts differ from the oracle"
    S, Sr = g["S"].cpu().numpy(), ref["S"].cpu().numpy()
    W, Wr = g["W"].cpu().numpy(), ref["W"].cpu().numpy()
    xi, xir = g["xi"].cpu().numpy(), ref["xi"].cpu().numpy()
    tolS = 1e-9 * np.maximum(np.abs(Sr), 1e-4 * o["Sabs"])
    assert np.all(np.abs(S - Sr) <= tolS), f"{label}: S"
    assert np.all(np.abs(S - o["S"]) <= tolS), f"{label}: S against the oracle"
    assert np.all(np.abs(W - Wr) <= 1e-9 * Wr), f"{label}: W"
    assert np.all(np.abs(W - o["W"]) <= 1e-9 * o["W"]), f"{label}: W against the oracle"
    nz = Wr > 0
    assert np.all(np.abs(xi[nz] - xir[nz]) <= 1e-9 * np.maximum(np.abs(xir[nz]), 1e-4 * o["Sabs"][nz] / o["W"][nz])), f"{label}: xi"
    assert np.all(xi[~nz] == 0.0)
    assert g["stats"]["n_binned"] == ref["stats"]["n_binned"] == int(o["N"].sum())
    assert g["stats"]["n_visited"] == ref["stats"]["n_visited"]


def test_xi_noalloc_matches_existing_path_on_calls_in_a_row(B, orc):
    import torch
    c = B.Context("cuda:0")
    b = B.binning()
    # two different catalogues: the static array must not carry sums from one call into the next.  The second has
    # native-resolution forests, which the bucketing pass sends to the generic xi kernel.
    cases = []
    for cfg, kw in ((4, dict(n_forest=800)), (2, dict(n_forest=150, density_scale=4.0, fine=2))):
        f = gen.make_config(cfg, **kw)
        ref_pairs = orc.pairs_window(f)
        d = B.DeviceForests(f)
        pairs = c.lya_neighbours(d, b)
        assert pairs.n == len(ref_pairs)
        plan = c.lya_plan_create(d, b, pairs, True, False)
        cases.append((plan, c.lya_xi2pcf_plan(plan), orc.xi(f, ref_pairs), d, pairs))
    nb = b.n_par * b.n_perp
    out = dict(S=torch.empty(nb, dtype=torch.float64, device="cuda:0"), W=torch.empty(nb, dtype=torch.float64, device="cuda:0"),
               N=torch.empty(nb, dtype=torch.int64, device="cuda:0"), xi=torch.empty(nb, dtype=torch.float64, device="cuda:0"))
    for rep, k in enumerate((0, 0, 1, 0, 1, 1)):                    # calls in a row, same plan and alternating plans
        plan, ref, o, _, _ = cases[k]
        for t in out.values():
            t.fill_(-7)                                             # outputs are overwritten, never accumulated into
        g = c.lya_xi2pcf_plan_noalloc(plan, out)
        same_as(g, ref, o, f"call {rep} (catalogue {k})")
    # free device memory does not move over further calls (every kernel involved has been launched by now: the first
    # launch of a kernel may load its module, which takes device memory in any path)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for k in (0, 1, 1, 0):
        c.lya_xi2pcf_plan_noalloc(cases[k][0], out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "device memory was allocated by lya_xi2pcf_plan_noalloc"
    same_as(dict(out, stats=cases[0][1]["stats"]), cases[0][1], cases[0][2], "after the back-to-back calls")
    # a second context on the same device shares the array (one address per device); used one after the other it is fine
    c2 = B.Context("cuda:0")
    plan2 = c2.lya_plan_create(cases[0][3], b, c2.lya_pairs_import(cases[0][4].export().cpu().numpy()), True, False)
    same_as(c2.lya_xi2pcf_plan_noalloc(plan2), cases[0][1], cases[0][2], "second context")
    same_as(c.lya_xi2pcf_plan_noalloc(cases[1][0]), cases[1][1], cases[1][2], "first context again")
    c2.close()
    c.close()


def test_xi_noalloc_rejects_what_it_cannot_hold(B):
    c = B.Context("cuda:0")
    f = gen.make_config(0)
    d = B.DeviceForests(f)
    big = B.binning(208.0, 208.0, 52, 52)                            # 2704 bins > LYA_XI_NOALLOC_MAX_BINS = 2560
    pairs = c.lya_neighbours(d, big)
    plan = c.lya_plan_create(d, big, pairs, True, False)
    ref = c.lya_xi2pcf_plan(plan)                                    # the allocating path takes it
    assert int(ref["N"].cpu().numpy().view(np.uint64).sum()) > 0
    n0 = B.launch_count()
    with pytest.raises(B.LyaError) as ei:
        c.lya_xi2pcf_plan_noalloc(plan)
    assert ei.value.name == "LYA_ERR_CAPACITY" and "2560" in str(ei.value)
    assert B.launch_count() == n0                                    # nothing was launched
    plan_d = c.lya_plan_create(d, B.binning(), c.lya_neighbours(d, B.binning()), False, True)
    with pytest.raises(B.LyaError) as ei:
        c.lya_xi2pcf_plan_noalloc(plan_d)                            # a plan without the xi arrays
    assert ei.value.name == "LYA_ERR_INVALID_ARG"
    c.close()
