#!/usr/bin/env python
"""bench.py -- throughput of the Lya2pcf pixel-pair hot path on B200.

A "step" is one pass of the whole hot path over one synthetic catalogue:
lya_neighbours -> lya_xi2pcf -> lya_dmat (stages 1-4 of BASELINE.json north_star).
`value` = pixel pairs binned per second over the step (xi: sum_A N_A, D: the in-grid
pairs scanned by the keep mask), inputs resident in HBM; `e2e` = the same through
lya_run_host with pinned HOST buffers (H2D of the catalogue and D2H of xi, D inside the
timed region).  Prints ONE JSON line on rank 0.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg2|cfg1|cfg0]
  python bench.py --impl reference ...     # the CPU oracle on a bounded sample
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "xi + D-matrix pixel-pairs/s (binned pairs per second over neighbours+xi+D)"
UNIT = "pixel-pairs/s"
WORKLOADS = {
    "cfg4": dict(cfg=4, mask_cfg=4, desc="configs[4] DESI-Y5-shaped: 900k forests, 14000 deg2, xi + D (f=0.99)"),
    "cfg2": dict(cfg=2, mask_cfg=3, desc="configs[2]+[3] DR16-shaped: 210k forests, 9400 deg2, xi + D (f=0.99)"),
    "cfg1": dict(cfg=1, mask_cfg=1, desc="configs[1] small patch: 20k forests, 100 deg2, xi + D (f=0.99)"),
    "cfg0": dict(cfg=0, mask_cfg=0, desc="configs[0] tiny: 64 forests, xi + D (f=0)"),
}
FP64_LANES_PER_SM = 64      # B200 fp64 vector units per SM (DFMA/DADD/DMUL lanes per clock)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def micro_peaks(device=0):
    """Roofline denominators measured by liblya_peaks.so (include/lya_peaks.h; bench-only library)."""
    import ctypes as C
    from paper_2507_00129_b200 import build
    lib = C.CDLL(build.build_peaks())
    lib.lya_measure_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
    out = {}
    for kind, name in enumerate(("fp64_fma", "fp64_add", "smem_cas64", "smem_add32", "l2_red64", "l2_red64_scatter")):
        r = C.c_double()
        rc = lib.lya_measure_peak(device, kind, C.byref(r))
        out[name] = r.value if rc == 0 else None
    return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0), "fallback"


def cpu_model():
    try:
        for l in open("/proc/cpuinfo"):
            if l.startswith("model name"):
                return l.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class OracleSample:
    """ONE definition of the bounded oracle workload, used by both the `cpu_baseline` leg and `--impl reference`:
    a shaped sub-catalogue of the workload's config (same sky density), xi over all of its listed forest pairs
    and the naive quadruple-sum D over the first 1/dmat_div of them."""

    def __init__(self, wl, n_forests, dmat_div):
        from oracle import oracle as orc
        from paper_2507_00129_b200 import gen
        self.orc = orc
        self.n_s = min(n_forests, gen.CONFIGS[wl["cfg"]]["n"])
        f = gen.make_config(wl["cfg"], n_forest=self.n_s)
        self.cat = orc.Catalogue(f)
        self.pq = orc.pairs_window(self.cat)
        self.pq_d = self.pq[: max(1, len(self.pq) // dmat_div)]
        self.seed = gen.mask_seed(wl["mask_cfg"])
        self.frac = 0.0 if wl["cfg"] == 0 else 0.99
        self.n_xi = None
        self.n_d = None

    def describe(self):
        return (f"{self.n_s} forests at the workload's sky density: xi over {len(self.pq)} forest pairs, "
                f"naive D (f={self.frac}) over {len(self.pq_d)} forest pairs, per step")

    def step(self):
        """-> (pairs counted as in the GPU metric, seconds xi, seconds D)."""
        orc = self.orc
        t0 = time.perf_counter()
        x = orc.xi(self.cat, self.pq)
        t1 = time.perf_counter()
        orc.dmat(self.cat, self.pq_d, self.frac, self.seed, want_D=False)
        t2 = time.perf_counter()
        if self.n_xi is None:
            self.n_xi = int(x["N"].sum())
            self.n_d = int(orc.xi(self.cat, self.pq_d)["N"].sum()) if len(self.pq_d) != len(self.pq) else self.n_xi
        return self.n_xi + self.n_d, t1 - t0, t2 - t1

    def single_thread_xi(self, frac=16):
        """xi pairs/s of ONE thread on 1/frac of the forest pairs (libgomp's thread count set for this call)."""
        import ctypes as C
        try:
            gomp = C.CDLL("libgomp.so.1")
            n0 = self.orc.num_threads()
            gomp.omp_set_num_threads(1)
            pq = self.pq[: max(1, len(self.pq) // frac)]
            t0 = time.perf_counter()
            x = self.orc.xi(self.cat, pq)
            dt = time.perf_counter() - t0
            gomp.omp_set_num_threads(n0)
            return int(x["N"].sum()) / dt
        except Exception:
            return None


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = WORKLOADS[args.workload]
    smp = OracleSample(wl, args.cpu_forests, args.cpu_dmat_div)
    for _ in range(args.warmup):
        smp.step()
    t0 = time.perf_counter()
    pairs = 0
    for _ in range(args.steps):
        pairs += smp.step()[0]
    dt = time.perf_counter() - t0
    val = pairs / dt
    sample = smp.describe()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "description": wl["desc"], "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": smp.orc.num_threads(), "cpu": cpu_model(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def cpu_baseline(wl, n_forests, dmat_div):
    """The oracle timed on this box's host cores on the bounded sample (about 10-30 s)."""
    smp = OracleSample(wl, n_forests, dmat_div)
    pairs, t_xi, t_d = smp.step()
    one = smp.single_thread_xi()
    return {"value": pairs / (t_xi + t_d), "unit": UNIT, "cores": smp.orc.num_threads(), "cpu": cpu_model(), "kind": "oracle",
            "xi_pairs_per_s": smp.n_xi / t_xi, "dmat_pairs_per_s": smp.n_d / max(t_d, 1e-9),
            "xi_pairs_per_s_single_thread": one,
            "sample": smp.describe() + f" (xi {t_xi:.1f} s, D {t_d:.1f} s; single-thread xi on 1/16 of the forest pairs)"}


def run_xi3(args):
    """--xi3 RMAX: throughput of lya_xi3pcf (NEXT-4, eq. 2.8) on the workload's catalogue; its own JSON line, never
    the default bench line.  Triangle bins of PAPER.md:225 (20 x 20 x 20 x 10 x 10); pair list = lya_neighbours with
    r_perp_max = r_max; warm-up calls, then `steps` timed calls (CUDA events of the k_xi3 launch, stats.ms_main)."""
    import torch
    from paper_2507_00129_b200 import binding as B, build, gen
    build.build()
    wl = WORKLOADS[args.workload]
    f = gen.make_config(wl["cfg"], n_forest=args.forests or None, fine=args.fine)
    ctx = B.Context("cuda:0")
    d = B.DeviceForests(f, device="cuda:0")
    tb = B.tri_binning(args.xi3, 20, 10, 20)
    ce = np.cos(np.pi * np.arange(1, 10) / 10)
    pairs = ctx.lya_neighbours(d, B.binning(args.xi3, args.xi3, 20, 20))
    for _ in range(max(args.warmup, 1)):
        g = ctx.lya_xi3pcf(d, tb, ce, pairs)
    ms = []
    for _ in range(args.steps):
        g = ctx.lya_xi3pcf(d, tb, ce, pairs)
        ms.append(g["stats"]["ms_main"])
    st = g["stats"]
    t = float(np.mean(ms)) * 1e-3
    mp = micro_peaks(0)
    print(json.dumps({
        "metric": "ordered triples (i; j, k) binned per second by lya_xi3pcf", "value": st["n_binned"] / t, "unit": "triples/s",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 1), "ms_per_step": t * 1e3, "higher_is_better": True,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "n_forest": f.n_forest, "n_pix": f.n_pix, "r_max": args.xi3,
                   "bins": "20x20x20x10x10", "forest_pairs": st["n_forest_pairs"], "triples": st["n_binned"],
                   "bins_touched": int((g["N3"] > 0).sum().item())},
        "roofline": {"bound": "l2-atomics", "kernel": "k_xi3", "achieved": 1.5 * st["n_binned"] / t / 1e9,
                     "peak": (mp.get("l2_red64_scatter") or 0) / 1e9 or None, "unit": "G red.global 8-byte/s",
                     "frac": (1.5 * st["n_binned"] / t / mp["l2_red64_scatter"]) if mp.get("l2_red64_scatter") else None,
                     "note": "1.5 reductions per ordered triple (S3, W3, N3 once per unordered {j, k}), scattered over "
                             "the 19 MB accumulators; peak = liblya_peaks' red.global.add.f64 rate with every lane on "
                             "its own random element of a 19 MB array"},
        "measured_peaks": mp}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=os.environ.get("LYA_BENCH_WORKLOAD", "cfg4"), choices=list(WORKLOADS))
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"],
                    help="N > 1: strong = ONE catalogue, its forest-pair list split over the ranks, one all-reduce of the "
                         "numerators (DESIGN.md section 8); weak = an independent catalogue per rank, no data-path collective")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-dmat", action="store_true")
    ap.add_argument("--cpu-forests", type=int, default=10000, help="forests of the bounded oracle sample (both oracle legs)")
    ap.add_argument("--cpu-dmat-div", type=int, default=20, help="naive D runs on 1/N of the sample's forest pairs")
    ap.add_argument("--forests", type=int, default=0,
                    help="profiling only: a shaped sub-catalogue of this many forests (same sky density)")
    ap.add_argument("--force-generic", action="store_true",
                    help="route every forest pair to the generic kernels (lya_set_option force_generic): the comparison figure for the fast / long-forest kernels")
    ap.add_argument("--fine", type=int, default=1,
                    help="NEXT-3 shapes: divide the pixel step by this factor (gen.make_config(fine=...)); throughput only")
    ap.add_argument("--xi3", type=float, default=0.0, metavar="RMAX",
                    help="NEXT-4: time lya_xi3pcf with this r_max (Mpc/h) on the workload's catalogue instead of the 2PCF step")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.xi3 > 0:
        return run_xi3(args)

    import torch
    import torch.distributed as dist
    from paper_2507_00129_b200 import binding as B, build, gen, shard

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    # functional dry runs of the N > 1 path on a box with ONE GPU (never a performance number): LYA_BENCH_BACKEND=gloo
    # LYA_BENCH_ONE_DEVICE=1 put every rank on cuda:0 and reduce through the host
    backend = os.environ.get("LYA_BENCH_BACKEND", "nccl")
    if os.environ.get("LYA_BENCH_ONE_DEVICE"):
        local = 0
    torch.cuda.set_device(local)
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        else:
            dist.init_process_group(backend)
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    wl = WORKLOADS[args.workload]
    frac = 0.0 if wl["cfg"] == 0 else 0.99
    mseed = gen.mask_seed(wl["mask_cfg"])
    strong = world > 1 and args.scaling == "strong"
    # strong: every rank holds the SAME catalogue; weak: an independent catalogue of the same shape per rank
    f = gen.make_config(wl["cfg"], n_forest=args.forests or None, fine=args.fine,
                        seed=None if strong else shard.rank_seed(gen.SEED_BASE + wl["cfg"], rank))
    ctx = B.Context(f"cuda:{local}")
    if args.force_generic:
        ctx.lya_set_option("force_generic", 1)
    d = B.DeviceForests(f, device=f"cuda:{local}")
    b = B.binning()
    do_d = not args.no_dmat
    lens = d.pix_off[1:] - d.pix_off[:-1]

    def step():
        """One pass of the hot path: neighbours -> (chunk of the list) -> plan -> xi -> D (-> all-reduce + division)."""
        if strong:
            r = shard.sharded_step(ctx, d, b, frac, mseed, rank, world, do_dmat=do_d, lens=lens)
            return dict(stats=r["stats_xi"]), (dict(stats=r["stats_dmat"]) if do_d else None)
        pairs = ctx.lya_neighbours(d, b)
        plan = ctx.lya_plan_create(d, b, pairs, want_xi=True, want_dmat=do_d)
        pairs.free()
        x = ctx.lya_xi2pcf_plan(plan)
        dm = ctx.lya_dmat_plan(plan, frac, mseed, want_Dn=False) if do_d else None
        plan.free()
        return x, dm

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = B.launch_count()
    ev0.record()
    ms_xi, ms_dm = [], []
    pairs_total = 0
    for _ in range(args.steps):
        x, dm = step()
        ms_xi.append(x["stats"]["ms_main"])
        pairs_total += x["stats"]["n_binned"]
        if dm is not None:
            ms_dm.append(dm["stats"]["ms_main"])
            pairs_total += dm["stats"]["n_binned"]
    ev1.record()
    barrier()
    launches = B.launch_count() - launches0          # kernels this rank's library launched inside the timed region
    clocks = sampler.stop() if rank == 0 else None
    # one more, untimed, step with CUDA events around every stage (where the step's time goes)
    stage_ms = None
    if not strong:
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
        evs[0].record()
        pairs = ctx.lya_neighbours(d, b); evs[1].record()
        plan = ctx.lya_plan_create(d, b, pairs, want_xi=True, want_dmat=do_d); pairs.free(); evs[2].record()
        ctx.lya_xi2pcf_plan(plan); evs[3].record()
        if do_d:
            ctx.lya_dmat_plan(plan, frac, mseed, want_Dn=False)
        plan.free(); evs[4].record()
        torch.cuda.synchronize()
        stage_ms = {"lya_neighbours": evs[0].elapsed_time(evs[1]), "lya_plan_create": evs[1].elapsed_time(evs[2]),
                    "lya_xi2pcf_plan": evs[2].elapsed_time(evs[3]), "lya_dmat_plan": evs[3].elapsed_time(evs[4])}
    ms = ev0.elapsed_time(ev1)
    ms, pairs_all = shard.aggregate(ms, float(pairs_total), device=f"cuda:{local}")
    value = pairs_all / (ms * 1e-3)

    # ---- e2e: host buffers through lya_run_host (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        pin = {}
        for k in ("ux", "uy", "uz", "pix_off", "chi", "w", "delta", "loglam"):
            tt = torch.from_numpy(np.ascontiguousarray(getattr(f, k))).pin_memory()
            pin[k] = tt
        class HostF:
            pass
        hf = HostF()
        for k, v in pin.items():
            setattr(hf, k, v.numpy())
        nb = b.n_par * b.n_perp
        out = {k: torch.empty(nb, dtype=torch.float64).pin_memory().numpy() for k in ("S", "W", "xi")}
        out["N"] = torch.empty(nb, dtype=torch.int64).pin_memory().numpy().view(np.uint64)
        if do_d:
            out["D"] = torch.empty((nb, nb), dtype=torch.float64).pin_memory().numpy()
            out["Wd"] = torch.empty(nb, dtype=torch.float64).pin_memory().numpy()
        h2d = sum(v.numel() * v.element_size() for v in pin.values())
        d2h = sum(v.nbytes for v in out.values())
        ctx.lya_run_host(hf, b, True, do_d, frac, mseed, out=dict(out))
        barrier()
        n_e2e = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        pe = 0
        for _ in range(n_e2e):
            r = ctx.lya_run_host(hf, b, True, do_d, frac, mseed, out=dict(out))
            pe += r["stats_xi"]["n_binned"] + (r["stats_dmat"]["n_binned"] if do_d else 0)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if strong:                                    # every rank ran the whole catalogue: the job's e2e is one rank's
            dtm, _ = shard.aggregate(dt, 0.0, device=f"cuda:{local}")
            dt = dtm
        else:
            dt, pe = shard.aggregate(dt, float(pe), device=f"cuda:{local}")
        e2e = {"value": pe / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "steps": n_e2e, "ms_per_step": dt / n_e2e * 1e3,
               "note": "lya_run_host on one rank's whole catalogue (host buffers are not sharded)" if strong else None}

    if rank == 0:
        peaks, peak_kind = measured_peaks()
        sx, sd = x["stats"], (dm["stats"] if dm is not None else None)
        t_xi = float(np.mean(ms_xi)) * 1e-3
        t_dm = float(np.mean(ms_dm)) * 1e-3 if ms_dm else 0.0
        sm_clk = (clocks.get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)) * 1e6
        # roofline: ALGORITHMIC fp64 lane-operations per launch / measured launch time,
        # against the fp64 pipe: SMs x 64 lanes x sm_max_mhz.
        #   xi: 8 per binned pixel pair (sub, add, 2 mul, 2 floor-adds, 2 FMA); out-of-grid evaluations are waste
        #   D : 10 per scanned (in-grid) pair (6 geometry + 4 H FMAs) + 4 per scatter-add of the drain
        peak_alu = ctx.sm_count() * FP64_LANES_PER_SM * peaks.get("sm_max_mhz", 1965.0) * 1e6
        peak_src = (f"derived: {ctx.sm_count()} SMs x {FP64_LANES_PER_SM} fp64 lanes x sm_max_mhz "
                    f"({peak_kind} MEASURED_PEAKS.json); DFMA/DADD microbenchmarks in measured_peaks")
        mp = micro_peaks(local)
        alg_xi = 8.0 * sx["n_binned"]
        roof_xi = {"bound": "alu", "kernel": "k_xi_fast", "achieved": alg_xi / t_xi / 1e12, "peak": peak_alu / 1e12,
                   "unit": "Tops/s (fp64 lane-operations)", "frac": alg_xi / t_xi / peak_alu, "traffic": None,
                   "peak_source": peak_src, "frac_at_sampled_clock": alg_xi / t_xi / (ctx.sm_count() * FP64_LANES_PER_SM * sm_clk),
                   "evaluated_per_binned": sx["n_evaluated"] / max(sx["n_binned"], 1)}
        # DRAM bytes per launch, measured ONCE under ncu on this workload (profiles/r2p_dram_cfg4_full.md); null elsewhere
        full_cfg4 = args.workload == "cfg4" and not args.forests and args.fine == 1 and not args.force_generic and world == 1
        if full_cfg4:
            roof_xi["traffic"] = 150.64e9 + 0.09e9
            roof_xi["traffic_note"] = "dram__bytes_read + write of one k_xi_fast launch, ncu capture profiles/r2p_dram_cfg4_full.md (37 GB/s: not HBM-bound)"
        roof = roof_xi
        extra = {"xi": {"binned_pairs_per_s": sx["n_binned"] / t_xi, "visited_pairs_per_s": sx["n_visited"] / t_xi,
                        "evaluated_pairs_per_s": sx["n_evaluated"] / t_xi, "ms": t_xi * 1e3,
                        "forest_pairs": sx["n_forest_pairs"], "roofline": roof_xi},
                 "measured_peaks": mp}
        if sd is not None:
            alg_d = 10.0 * sd["n_binned"] + 4.0 * sd["n_scatter"]
            roof_d = {"bound": "alu", "kernel": "k_dmat (generic)" if args.force_generic else ("k_dmat_fast" if args.fine == 1 else "k_dmat_fast / k_dmat_long"), "achieved": alg_d / t_dm / 1e12, "peak": peak_alu / 1e12,
                      "unit": "Tops/s (fp64 lane-operations)", "frac": alg_d / t_dm / peak_alu, "traffic": None,
                      "peak_source": peak_src,
                      "scatter_adds_per_s": sd["n_scatter"] / t_dm,
                      "frac_of_measured_l2_red_peak": sd["n_scatter"] / t_dm / mp["l2_red64"] if mp.get("l2_red64") else None,
                      "evaluated_per_scanned": sd["n_evaluated"] / max(sd["n_binned"], 1)}
            extra["dmat"] = {"scanned_pairs_per_s": sd["n_binned"] / t_dm, "kept_pairs_per_s": sd["n_kept"] / t_dm,
                             "ms": t_dm * 1e3, "n_kept": sd["n_kept"], "n_scatter": sd["n_scatter"], "roofline": roof_d}
            if full_cfg4:
                roof_d["traffic"] = 232.23e9 + 0.28e9
                roof_d["traffic_note"] = "dram__bytes_read + write of one k_dmat_fast launch, ncu capture profiles/r2p_dram_cfg4_full.md (15 GB/s: not HBM-bound)"
            if t_dm > t_xi:
                roof = roof_d
        if world == 1:
            par = "one GPU"
        elif strong:
            par = f"one catalogue, forest-pair list split over {world} ranks by sum n_p n_q, one all-reduce of S,W,N / Dn,Wd"
        else:
            par = f"independent catalogue per GPU x{world}, no data-path collective"
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if strong else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload + (f" fine={args.fine}" if args.fine != 1 else "") + (" force_generic" if args.force_generic else ""), "description": wl["desc"],
                       "n_forest": f.n_forest, "n_pix": f.n_pix,
                       "bins": "50x50x4Mpc/h", "reject_fraction": frac, "dmat": do_d,
                       "l2": ("catalogue %.2f GB + forest-pair list %.2f GB per step vs 126 MB of L2 (%s); Dn (50 MB) "
                              "re-zeroed every step") % (f.n_pix * 32 / 1e9, sx["n_forest_pairs"] * 8 / 1e9,
                                                         "larger than L2" if f.n_pix * 32 + sx["n_forest_pairs"] * 8 > 126e6
                                                         else "NOT larger than L2: use the default workload for a valid number"),
                       "parallelism": par},
            "roofline": roof, "clocks": clocks, "gpu_launches": int(launches), "stage_ms": stage_ms, "e2e": e2e, **extra,
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(wl, args.cpu_forests, args.cpu_dmat_div)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
