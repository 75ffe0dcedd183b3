"""Full-size parity, driver-run (north_star Target: "matching the CPU oracle on all five configs").

configs[0] is compared in full by tests/test_gpu_parity.py.  Here, at BASELINE.json's full sizes and in
the launch configuration bench.py times (lya_neighbours' own list, the fast kernels):

  configs[1]  xi AND D (f = 0.99) over EVERY listed forest pair (oracle: about 1 + 4 min on 16 threads)
  configs[2]  xi over EVERY listed forest pair (about 1.5 min)
  configs[3]  D (f = 0.99) on a stated contiguous slice [k0, k1) of the neighbour list
  configs[4]  xi and D (f = 0.99) on stated contiguous slices of the neighbour list

Slices are contiguous chunks of the list in lya_neighbours' order (the same chunking shard.split_pairs
and the D-matrix halves of DESIGN.md section 7 use); S, W, N, Dn, Wd are additive over forest pairs, so a
slice is a complete parity case for every kernel path it exercises.  Bars as in test_gpu_parity.py.
Each test prints one summary line (pytest -s shows it; it is also kept in the junit/xml record).
"""
import time

import numpy as np
import pytest

from paper_2507_00129_b200 import gen
from test_gpu_parity import check_dmat, check_xi

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


class _Case:
    """One config resident on the device with its neighbour list (built once per module)."""
    cache = {}

    @classmethod
    def get(cls, ctx, B, orc, cfg):
        key = 2 if cfg == 3 else cfg
        if key not in cls.cache:
            cls.cache.clear()                                   # one catalogue at a time (host + HBM)
            f = gen.make_config(key)
            d = B.DeviceForests(f)
            pairs = ctx.lya_neighbours(d, B.binning())
            cls.cache[key] = (f, d, pairs, orc.Catalogue(f))
        return cls.cache[key]


def _report(msg):
    print("\n[full parity] " + msg, flush=True)


def _xi_case(ctx, B, orc, cfg, k0=None, k1=None):
    f, d, pairs, cat = _Case.get(ctx, B, orc, cfg)
    b = B.binning()
    if k0 is None:
        use, pq = pairs, pairs.export().cpu().numpy()
    else:
        pq_dev = pairs.export()[k0:k1].contiguous()
        use, pq = ctx.lya_pairs_import(pq_dev), pq_dev.cpu().numpy()
    g = ctx.lya_xi2pcf(d, b, use)
    t0 = time.time()
    o = orc.xi(cat, pq)
    _report(f"cfg{cfg} xi: forest pairs [{k0 or 0}, {k1 or pairs.n}) of {pairs.n}, {int(o['N'].sum())} binned pixel pairs; "
            f"GPU {g['stats']['ms_main']:.0f} ms, oracle {time.time() - t0:.0f} s on {orc.num_threads()} threads")
    check_xi(g, o, f"cfg{cfg} full-size xi")


def _dmat_case(ctx, B, orc, cfg, k0=None, k1=None):
    f, d, pairs, cat = _Case.get(ctx, B, orc, cfg)
    b = B.binning()
    seed = gen.mask_seed(3 if cfg in (2, 3) else cfg)
    if k0 is None:
        use, pq = pairs, pairs.export().cpu().numpy()
    else:
        pq_dev = pairs.export()[k0:k1].contiguous()
        use, pq = ctx.lya_pairs_import(pq_dev), pq_dev.cpu().numpy()
    g = ctx.lya_dmat(d, b, use, 0.99, seed)
    t0 = time.time()
    o = orc.dmat(cat, pq, 0.99, seed)
    _report(f"cfg{cfg} D (f=0.99): forest pairs [{k0 or 0}, {k1 or pairs.n}) of {pairs.n}, n_kept {o['n_kept']}; "
            f"GPU {g['stats']['ms_main']:.0f} ms, oracle {time.time() - t0:.0f} s on {orc.num_threads()} threads")
    check_dmat(g, o, f"cfg{cfg} full-size D")


def test_cfg1_xi_every_forest_pair(ctx, B, orc):
    _xi_case(ctx, B, orc, 1)


def test_cfg1_dmat_every_forest_pair(ctx, B, orc):
    _dmat_case(ctx, B, orc, 1)


def test_cfg2_xi_every_forest_pair(ctx, B, orc):
    _xi_case(ctx, B, orc, 2)


def test_cfg3_dmat_slice(ctx, B, orc):
    """configs[3]: forest pairs [30 000 000, 34 000 000) of the ~7.0e7 listed (about 5.7 %)."""
    _dmat_case(ctx, B, orc, 3, 30_000_000, 34_000_000)


def test_cfg4_xi_slice(ctx, B, orc):
    """configs[4]: forest pairs [400 000 000, 425 000 000) of the ~8.6e8 listed (about 2.9 %)."""
    _xi_case(ctx, B, orc, 4, 400_000_000, 425_000_000)


def test_cfg4_dmat_slice(ctx, B, orc):
    """configs[4]: forest pairs [700 000 000, 704 000 000) of the ~8.6e8 listed (about 0.46 %)."""
    _dmat_case(ctx, B, orc, 4, 700_000_000, 704_000_000)
    _Case.cache.clear()
