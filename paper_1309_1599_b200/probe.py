"""Kernel probe: runs / times one piece of the hot path on a BASELINE.json workload under a chosen kernel, for A/B
measurements and as the short command line `ncu` wraps (profiles/*.md name these commands).

    python -m paper_1309_1599_b200.probe sweep --cfg 4 --impl fused --sweeps 32        # us per OR sweep, CUDA events
    python -m paper_1309_1599_b200.probe sweep --cfg 4 --impl zmarch --samples 2 --reps 1 --sweeps 6   # a short run for ncu
    python -m paper_1309_1599_b200.probe units --cfg 1 --graph 1                       # us per MCS through sg_run_units
    python -m paper_1309_1599_b200.probe exercise --shape 8,2,2,6 --impl zmarch        # every entry point once (compute-sanitizer)
    python -m paper_1309_1599_b200.probe sustained --cfg 4 --impl zmarch               # us per OR half-sweep over 6 x 1024 sweeps (power-capped)

Prints one JSON line per measurement.  Timing is on the device (CUDA events on the context's stream), best and median
of `--reps` repetitions after a warm-up; nothing here is a bench value (bench.py is)."""
import argparse
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

IMPLS = {"auto": 0, "tiled": 1, "zmarch": 2, "resident": 3, "fused": 4, "cluster": 5}


def _context(sg, W, args, stream=None):
    cfg = W.CONFIGS[args.cfg]
    S = args.samples or cfg.n_samples
    g = sg.SpinGlass(cfg.L, S, cfg.n_replicas, cfg.n_temps, cfg.betas, seed=1, stream=stream, fused_buffer=(args.impl == "fused"))
    g.tune(sg.TUNE_SWEEP_IMPL, IMPLS[args.impl])
    if args.zchunk:
        g.tune(sg.TUNE_ZCHUNK, args.zchunk)
    if args.cluster_ctas:
        g.tune(sg.TUNE_CLUSTER_CTAS, args.cluster_ctas)
    for s in range(S):
        g.init_sample(s, sg.GEN_OFFDIAG_SYM, cfg.sigma_D)
    return cfg, S, g


def sweep(args):
    import torch
    import paper_1309_1599_b200 as sg
    import sg_workloads as W
    cfg, S, g = _context(sg, W, args)
    kind = g.sweep_hb if args.kind == "hb" else g.sweep_or
    kind(2)
    g.sync()
    times = []
    for _ in range(args.reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        kind(args.sweeps)
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1) * 1e3 / args.sweeps)
    updates = S * cfg.n_copies * cfg.n_sites
    out = dict(probe="sweep", cfg=cfg.name, kind=args.kind, impl=args.impl, zchunk=args.zchunk, cluster_ctas=args.cluster_ctas, samples=S, sweeps=args.sweeps,
               us_per_sweep_best=min(times), us_per_sweep_median=float(np.median(times)),
               ps_per_update_best=min(times) * 1e6 / updates, updates_per_sweep=updates,
               energy_sum=float(g.get_energies().sum()))
    g.close()
    print(json.dumps(out), flush=True)


def units(args):
    import time
    import torch
    import paper_1309_1599_b200 as sg
    import sg_workloads as W
    cfg, S, g = _context(sg, W, args, stream=torch.cuda.Stream())
    g.tune(sg.TUNE_GRAPH, args.graph)
    n = args.units or max(20, min(2000, int(2e9 / cfg.updates_per_unit)))
    g.run_units(max(8, n // 4), cfg.n_or)
    g.sync()
    times = []
    for _ in range(args.reps):
        t0 = time.perf_counter()
        g.run_units(n, cfg.n_or)
        g.sync()
        times.append((time.perf_counter() - t0) / n)
    upd = cfg.updates_per_unit * S / cfg.n_samples
    out = dict(probe="units", cfg=cfg.name, impl=args.impl, graph=args.graph, samples=S, units=n, us_per_unit_best=min(times) * 1e6,
               us_per_unit_median=float(np.median(times)) * 1e6, updates_per_s=upd / min(times))
    g.close()
    print(json.dumps(out), flush=True)


def sustained(args):
    """us per OR half-sweep in back-to-back segments of 1024 sweeps: what the kernel holds under the power cap."""
    import torch
    import paper_1309_1599_b200 as sg
    import sg_workloads as W
    cfg, S, g = _context(sg, W, args)
    g.sweep_or(8)
    g.sync()
    res = []
    for _ in range(6):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.sweep_or(1024)
        e1.record()
        torch.cuda.synchronize()
        res.append(round(e0.elapsed_time(e1) * 1e3 / 2048, 1))
    g.close()
    print(json.dumps(dict(probe="sustained", cfg=cfg.name, impl=args.impl, lib=os.environ.get("SG_B200_LIB", "libsg_b200.so"),
                          us_per_halfsweep=res)), flush=True)


def exercise(args):
    """Every kernel family once on a small shape: what compute-sanitizer (memcheck / racecheck) is pointed at."""
    import paper_1309_1599_b200 as sg
    L, S, R, T = [int(v) for v in args.shape.split(",")]
    betas = np.linspace(0.5, 1.8, T)
    g = sg.SpinGlass(L, S, R, T, betas, seed=7, fused_buffer=(args.impl == "fused"))
    g.tune(sg.TUNE_SWEEP_IMPL, IMPLS[args.impl])
    for s in range(S):
        g.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
    g.run_units(9, 2)
    g.unit(1)
    g.halfsweep(sg.KIND_OR, 0); g.halfsweep(sg.KIND_HB, 1)
    e, q0, qk = g.measure()
    out = dict(probe="exercise", shape=[L, S, R, T], impl=args.impl, e_mean=float(e.mean()), launches=0)
    if R > 1:
        g.measure_chiral(); g.accumulate(True); g.get_logbins()
        buf = g.export_replica(1)
        q0x, _ = g.measure_cross(0, buf)
        out["cross_minus_measure"] = float(np.abs(q0x - q0[:, 0]).max())
    g.schwinger_dyson(); g.pt_walk(); g.pt_visits(); g.pt_stats()
    spins = g.get_spins(0)
    out["norm_err"] = float(np.abs(np.sqrt((spins.astype(np.float64) ** 2).sum(axis=1)) - 1.0).max())
    out["launches"] = g.kernel_launches()
    g.close()
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("what", choices=["sweep", "units", "exercise", "sustained"])
    ap.add_argument("--shape", default="8,2,2,6", help="exercise: L,S,R,T")
    ap.add_argument("--cfg", type=int, default=4, help="index into BASELINE.json configs (sg_workloads.CONFIGS)")
    ap.add_argument("--impl", choices=sorted(IMPLS), default="auto", help="SG_TUNE_SWEEP_IMPL")
    ap.add_argument("--kind", choices=["or", "hb"], default="or")
    ap.add_argument("--zchunk", type=int, default=0, help="SG_TUNE_ZCHUNK (0 = automatic)")
    ap.add_argument("--cluster-ctas", type=int, default=0, help="SG_TUNE_CLUSTER_CTAS (0 = the library's default)")
    ap.add_argument("--samples", type=int, default=0, help="samples in the context (0 = the config's)")
    ap.add_argument("--sweeps", type=int, default=32)
    ap.add_argument("--units", type=int, default=0)
    ap.add_argument("--graph", type=int, default=1, help="SG_TUNE_GRAPH")
    ap.add_argument("--reps", type=int, default=5)
    args = ap.parse_args()
    {"sweep": sweep, "units": units, "exercise": exercise, "sustained": sustained}[args.what](args)


if __name__ == "__main__":
    main()
