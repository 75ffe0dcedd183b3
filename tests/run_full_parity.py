#!/usr/bin/env python
"""Full-size parity, run by hand on a GPU box (too slow for the pytest suite: the oracle needs minutes):

    python tests/run_full_parity.py [cfg] [--dmat] [--no-xi] [--dmat-frac F] [--dmat-skip F0]

configs[cfg] (default 2) in full: lya_neighbours -> lya_xi2pcf against the CPU oracle over EVERY listed
forest pair (N bit-exact, S/W to 1e-9), and with --dmat lya_dmat (f = 0.99, the config's mask seed)
against the naive quadruple sum (n_kept exact, D to 1e-7 per entry); --dmat-frac F restricts the D check
to the first fraction F of the forest-pair list (the naive oracle of configs[4] needs ~75 min for all of
it).  Prints one summary line per check.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import oracle as orc                      # noqa: E402
from paper_2507_00129_b200 import binding as B, gen   # noqa: E402


def xi_check(ctx, d, b, pairs, cat, pq, cfg):
    g = ctx.lya_xi2pcf(d, b, pairs)
    t0 = time.time()
    o = orc.xi(cat, pq)
    N = g["N"].cpu().numpy().view(np.uint64)
    S, W = g["S"].cpu().numpy(), g["W"].cpu().numpy()
    errS = np.max(np.abs(S - o["S"]) / np.maximum(np.abs(o["S"]), 1e-4 * o["Sabs"]))
    errW = np.max(np.abs(W - o["W"]) / o["W"])
    print(f"cfg{cfg} xi: {len(pq)} forest pairs, {int(o['N'].sum())} binned pixel pairs; N mismatching bins "
          f"{int((N != o['N']).sum())}; max rel err S {errS:.2e} W {errW:.2e}; GPU {g['stats']['ms_main']:.0f} ms, "
          f"oracle {time.time() - t0:.0f} s on {orc.num_threads()} threads", flush=True)
    assert np.array_equal(N, o["N"]) and errS <= 1e-9 and errW <= 1e-9


def main():
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 and sys.argv[1].isdigit() else 2
    do_d = "--dmat" in sys.argv
    do_xi = "--no-xi" not in sys.argv
    f = gen.make_config(cfg)
    ctx = B.Context("cuda:0")
    d = B.DeviceForests(f)
    b = B.binning()
    pairs = ctx.lya_neighbours(d, b)
    pq = pairs.export().cpu().numpy()
    cat = orc.Catalogue(f)
    if do_xi:
        xi_check(ctx, d, b, pairs, cat, pq, cfg)
    if do_d:
        seed = gen.mask_seed(3 if cfg == 2 else cfg)
        frac = float(sys.argv[sys.argv.index("--dmat-frac") + 1]) if "--dmat-frac" in sys.argv else 1.0
        skip = float(sys.argv[sys.argv.index("--dmat-skip") + 1]) if "--dmat-skip" in sys.argv else 0.0
        if frac < 1.0 or skip > 0.0:                   # forest pairs [skip, skip + frac) of the list
            pq = pq[int(len(pq) * skip): int(len(pq) * min(skip + frac, 1.0))]
            pairs = ctx.lya_pairs_import(pq)
        gd = ctx.lya_dmat(d, b, pairs, 0.99, seed, want_Dn=False)
        t0 = time.time()
        od = orc.dmat(cat, pq, 0.99, seed)
        D = gd["D"].cpu().numpy()
        err = np.max(np.abs(D - od["D"]) / np.maximum(np.abs(od["D"]), 1e-6))
        errWd = np.max(np.abs(gd["Wd"].cpu().numpy() - od["Wd"]) / np.maximum(od["Wd"], 1e-300))
        print(f"cfg{cfg} D (f=0.99, {len(pq)} forest pairs): n_kept GPU {gd['stats']['n_kept']} oracle {od['n_kept']}; max err D / max(|D|,1e-6) "
              f"{err:.2e}; Wd {errWd:.2e}; GPU {gd['stats']['ms_main']:.0f} ms, oracle {time.time() - t0:.0f} s", flush=True)
        assert gd["stats"]["n_kept"] == od["n_kept"] and err <= 1e-7 and errWd <= 1e-9
    print("full parity ok")


if __name__ == "__main__":
    main()
