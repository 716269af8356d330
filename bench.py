"""bench.py -- throughput of the hot path on the BASELINE.json headline workload (cfg 4: L=64, 4 samples,
4 replicas x 48 temperatures, 1 HB + 32 OR sweeps per PT swap, measurement every 10 units).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4]

A step is one unit (MCS): sg_sweep_hb(1); sg_sweep_or(n_or); sg_pt_swap(); and sg_measure
after every `measure_every`-th unit.  `value` = HB + OR single-spin updates per second over the whole job
(all ranks), state resident in HBM, timed with CUDA events on the launching stream, max over ranks.
`e2e` = the same unit through the C ABI with host buffers: every step uploads the spin state of every
sample from pinned host memory (sg_set_spins), runs the unit and reads the measurement back (sg_measure);
the samples are independent chains, each driven through its own context / stream / host thread.
`roofline` = the OR half-sweep kernel against the measured HBM copy bandwidth;
`sustained` / `roofline.sustained_frac` = the same loop over >= 3 back-to-back segments of >= 50 units (about 10 s),
median: what the box holds under its power cap, next to the burst the --steps loop times.
`cpu_baseline` / `--impl reference` = the fp64 oracle (oracle/), as it stands, on the host cores.
Prints ONE JSON line on rank 0.
"""
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

import sg_workloads as W
from paper_1309_1599_b200 import multi

METRIC = "spin updates/s (ps/spin-update) at L=64 PT; fraction of HBM/FP32 roofline"
UNIT = "spin updates/s"
ALG_BYTES_FIXED = 36.0      # B per update: 12 read own + 12 read as neighbour (amortised) + 12 write
ALG_BYTES_COUPLINGS = 216.0  # B per site: six 3x3 fp32 matrices, shared by the C copies of a sample


def algorithmic_bytes_per_update(C):
    """SURVEY.md section 8(d) / DESIGN.md section 10: 36 + 216/C bytes per single-spin update."""
    return ALG_BYTES_FIXED + ALG_BYTES_COUPLINGS / C


def measured_hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons of one GPU, sampled every 200 ms while the timed region runs."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.QUERY,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for ts, line in self.rows:
            if ts < t0 or ts > t1 + 0.2:
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_unit_rate(cfg, n_or_timed):
    """The oracle, as it stands, on one L = cfg.L sample: `cores` copies (one per OpenMP thread), one HB
    sweep and n_or_timed OR sweeps, timed separately and combined in the unit's mix 1 HB : cfg.n_or OR.
    Returns (updates/s, cores, description, seconds spent, split) -- split: ns per update of OR, HB and the
    unit mix, with all cores and per core."""
    from oracle import sg_oracle as oracle
    oracle.build()
    cores = oracle.num_threads()
    L, N = cfg.L, cfg.n_sites
    M = oracle.gen_couplings(L, cfg.seed, 0, oracle.OFFDIAG_SYM, cfg.sigma_D)
    spins = np.stack([oracle.gen_spins(L, cfg.seed, c) for c in range(cores)])
    betas = np.resize(cfg.betas, cores)
    t0 = time.perf_counter()
    oracle.sweep_copies(L, M, spins, oracle.KIND_HB, 1, beta_of_copy=betas, seed=cfg.seed, g0=0, hb_counter0=0,
                        store_fp32=True)
    t1 = time.perf_counter()
    oracle.sweep_copies(L, M, spins, oracle.KIND_OR, n_or_timed, store_fp32=True)
    t2 = time.perf_counter()
    t_hb, t_or = t1 - t0, (t2 - t1) / n_or_timed
    rate = (1 + cfg.n_or) * cores * N / (t_hb + cfg.n_or * t_or)
    what = ("1 sample of L=%d, %d copies (one per thread): 1 HB sweep + %d OR sweeps timed, combined in the "
            "unit mix 1 HB : %d OR" % (L, cores, n_or_timed, cfg.n_or))
    per = 1e9 / (cores * N)          # seconds per sweep of `cores` copies -> ns per update with all cores
    split = {"or_ns_per_update": t_or * per, "hb_ns_per_update": t_hb * per, "unit_ns_per_update": 1e9 / rate,
             "or_ns_per_update_per_core": t_or * per * cores, "hb_ns_per_update_per_core": t_hb * per * cores,
             "unit_ns_per_update_per_core": 1e9 / rate * cores}
    return rate, cores, what, t2 - t0, split


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank, _, world = multi.env_rank()
    if rank != 0:
        return
    # size the per-step sample so that (warmup + steps) steps end within a few minutes
    from oracle import sg_oracle as oracle
    oracle.build()
    probe_rate, cores, _, _, _ = oracle_unit_rate(cfg, 1)
    per_sweep = cores * cfg.n_sites / probe_rate
    budget = 150.0 / max(1, args.steps + args.warmup)
    n_or_timed = int(max(1, min(cfg.n_or, budget / per_sweep - 1)))
    rates, secs = [], []
    for k in range(args.warmup + args.steps):
        r, cores, what, dt, split = oracle_unit_rate(cfg, n_or_timed)
        if k >= args.warmup:
            rates.append(r); secs.append(dt)
    value = float(len(rates) / np.sum(1.0 / np.asarray(rates)))      # steps / total normalised time
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(secs) * 1e3),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "ps_per_update": 1e12 / value,
        "config": workload_config(cfg, args.gpus, "host cores only"),
        "cpu_baseline": dict({"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what}, **split),
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def workload_config(cfg, n_gpus, flush):
    return {"workload": "%s: L=%d, %d samples per GPU, %d replicas x %d temperatures (beta %.1f..%.1f), "
                        "1 HB + %d OR sweeps per PT swap, measure every %d units"
                        % (cfg.name, cfg.L, cfg.n_samples, cfg.n_replicas, cfg.n_temps, cfg.beta_min, cfg.beta_max,
                           cfg.n_or, cfg.measure_every),
            "L": cfg.L, "samples_per_gpu": cfg.n_samples, "replicas": cfg.n_replicas, "temps": cfg.n_temps,
            "n_or": cfg.n_or, "updates_per_step_per_gpu": cfg.updates_per_unit,
            "parallelism": "samples sharded over %d GPU(s), no collective" % n_gpus, "l2": flush}


def run_ours(args, cfg):
    import torch
    import paper_1309_1599_b200 as sg

    rank, local_rank, world = multi.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    multi.init_process_group("nccl", world)

    S, R, T, L, N, C = cfg.n_samples, cfg.n_replicas, cfg.n_temps, cfg.L, cfg.n_sites, cfg.n_copies
    gpu = sg.SpinGlass(L, S, R, T, cfg.betas, seed=cfg.seed, first_sample=multi.first_sample_of_rank(rank, S))
    gpu.tune(sg.TUNE_SWEEP_IMPL, {"auto": sg.SWEEP_AUTO, "tiled": sg.SWEEP_TILED, "zmarch": sg.SWEEP_ZMARCH, "resident": sg.SWEEP_RESIDENT}[args.sweep_impl])
    if args.zchunk:
        gpu.tune(sg.TUNE_ZCHUNK, args.zchunk)
    for s in range(S):
        gpu.init_sample(s, sg.GEN_OFFDIAG_SYM, cfg.sigma_D)
    state_bytes = S * C * N * 12

    ev = lambda: torch.cuda.Event(enable_timing=True)
    or_pairs, hb_pairs = [], []

    def unit(k, timed):
        """one MCS; with `timed`, CUDA events bracket the HB and the OR calls on the launching stream"""
        if timed:
            a, b, c = ev(), ev(), ev()
            a.record(); gpu.sweep_hb(1); b.record(); gpu.sweep_or(cfg.n_or); c.record()
            hb_pairs.append((a, b)); or_pairs.append((b, c))
        else:
            gpu.sweep_hb(1); gpu.sweep_or(cfg.n_or)
        gpu.pt_swap()
        if (k + 1) % cfg.measure_every == 0:
            return gpu.measure()
        return None

    # ---- device-resident throughput ----
    for k in range(args.warmup):
        unit(k, False)
    gpu.sync()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    multi.barrier(); torch.cuda.synchronize()
    launches0 = gpu.kernel_launches()
    t_wall0 = time.time()
    start, stop = ev(), ev()
    # per-call events sit inside the timed region (the roofline's launch time is measured live there) unless a unit is so
    # short (configs 0-1: tens of microseconds) that recording them would be what is timed: then a separate pass follows
    events_inside = cfg.updates_per_unit >= 10 ** 8
    start.record()
    for k in range(args.steps):
        unit(k, events_inside)
    stop.record()
    torch.cuda.synchronize(); multi.barrier()
    t_wall1 = time.time()
    launches = gpu.kernel_launches() - launches0
    if not events_inside:
        for k in range(min(args.steps, 10)):
            unit(k, True)
        torch.cuda.synchronize()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    seconds = start.elapsed_time(stop) * 1e-3
    value, total_updates, slowest = multi.whole_job_rate(args.steps * cfg.updates_per_unit, seconds, device)

    # dominant kernel: the OR half-sweep (2*n_or launches per sg_sweep_or call, plus one tiny reduction)
    or_ms = float(np.mean([a.elapsed_time(b) for a, b in or_pairs]))
    hb_ms = float(np.mean([a.elapsed_time(b) for a, b in hb_pairs]))
    # small lattices (8 copies fit in shared memory): one launch of the resident kernel runs all n_or sweeps of the call and
    # moves every spin across HBM once per call (12 B read + 12 B written per site and copy, couplings of both colours once per group)
    resident = args.sweep_impl == "resident" or (args.sweep_impl == "auto" and N * 96 <= 200 * 1024)
    if resident:
        or_launch_s = or_ms * 1e-3
        updates_per_launch = S * C * N * cfg.n_or
        alg_bytes = S * C * N * 24.0 + S * ((C + 31) // 32) * N * 216.0
        kernel_name = "k_sweep_res<OR>: %d OR sweeps per launch, lattice resident in shared memory" % cfg.n_or
    else:
        or_launch_s = or_ms * 1e-3 / (2 * cfg.n_or)
        updates_per_launch = S * C * N // 2
        alg_bytes = algorithmic_bytes_per_update(C) * updates_per_launch
        kernel_name = "OR half-sweep (k_sweep_zm<OR> for L %% 8 == 0, else k_sweep<OR>), sweep_impl=%s zchunk=%d" % (args.sweep_impl, args.zchunk)
    peak, peak_src = measured_hbm_peak()
    achieved = alg_bytes / or_launch_s / 1e9

    # ---- sustained leg: >= 3 timed segments of >= 50 units, median; what the box holds once the
    # power cap has settled (the --steps loop above is a burst of about a second at cfg 4) ----
    sustained = None
    if args.sustain_segments > 0:
        unit_s = seconds / args.steps
        seg_units = max(50, int(np.ceil(args.sustain_seconds / args.sustain_segments / unit_s)))
        every = 1 if events_inside else 64                      # short units: per-call events only on every 64th unit
        sampler2 = ClockSampler(local_rank) if rank == 0 else None
        multi.barrier(); torch.cuda.synchronize()
        t_s0 = time.time()
        seg_rates, seg_or_us = [], []
        for seg in range(args.sustain_segments):
            del or_pairs[:], hb_pairs[:]
            a, b = ev(), ev()
            a.record()
            for k in range(seg_units):
                unit(k, k % every == 0)
            b.record()
            torch.cuda.synchronize()
            sec = multi.max_over_ranks(a.elapsed_time(b) * 1e-3, device)
            seg_rates.append(multi.sum_over_ranks(seg_units * cfg.updates_per_unit, device) / sec)
            seg_or_us.append(float(np.mean([x.elapsed_time(y) for x, y in or_pairs])) * 1e3)
        t_s1 = time.time()
        clocks2 = sampler2.stop(t_s0, t_s1) if sampler2 else None
        sustained = {"segments": args.sustain_segments, "units_per_segment": seg_units, "seconds": t_s1 - t_s0,
                     "value": float(np.median(seg_rates)), "values": [float(v) for v in seg_rates],
                     "or_call_us": float(np.median(seg_or_us)), "clocks": clocks2}

    # ---- end to end through the C ABI with host buffers ----
    host = [torch.empty((C, 3, N), dtype=torch.float32).pin_memory() for _ in range(S)]
    for s in range(S):
        host[s].numpy()[...] = gpu.get_spins(s)
    e2e_steps = max(1, min(args.steps, 20))     # the chains pipeline uploads against sweeps: enough steps to amortise the fill and the drain

    # One single-sample context per sample, each on its own stream and host thread (ctypes releases the GIL):
    # the samples are independent chains, and `first_sample` gives every context the Philox
    # streams it has inside the S-sample context, so the upload of one sample overlaps the sweeps of the others.
    first = multi.first_sample_of_rank(rank, S)
    gpu.close(); del gpu
    import concurrent.futures as cf
    ctxs = []
    for s in range(S):
        c = sg.SpinGlass(L, 1, R, T, cfg.betas, seed=cfg.seed, first_sample=first + s, stream=torch.cuda.Stream(device))
        c.init_sample(0, sg.GEN_OFFDIAG_SYM, cfg.sigma_D)
        # a single-sample context alone would want short chunks (many CTAs); here the other samples' kernels fill the device,
        # so the long chunks of the S-sample context are the better shape (1.28e11 -> 1.32e11 updates/s end to end)
        e2e_zc = args.e2e_zchunk if args.e2e_zchunk else (32 if L % 32 == 0 else 0)
        if e2e_zc:
            c.tune(sg.TUNE_ZCHUNK, e2e_zc)
        ctxs.append(c)

    upload = threading.Lock()       # one upload at a time: the samples take turns on the PCIe link instead of sharing it

    def e2e_chain(s, n_steps):
        torch.cuda.set_device(local_rank)
        c, nbytes = ctxs[s], 0
        for k in range(n_steps):
            with upload:
                c.set_spins(0, host[s].numpy())
            c.sweep_hb(1); c.sweep_or(cfg.n_or); c.pt_swap()
            nbytes = sum(a.nbytes for a in c.measure())
        return nbytes

    with cf.ThreadPoolExecutor(max_workers=S) as pool:
        list(pool.map(lambda s: e2e_chain(s, 1), range(S)))          # warm-up step
        multi.barrier(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        d2h = sum(pool.map(lambda s: e2e_chain(s, e2e_steps), range(S)))
        torch.cuda.synchronize()
        e2e_seconds = time.perf_counter() - t0
    multi.barrier()
    e2e_value, _, _ = multi.whole_job_rate(e2e_steps * cfg.updates_per_unit, e2e_seconds, device)

    if rank != 0:
        return
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": slowest * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "ps_per_update": 1e12 / value,
        "config": workload_config(cfg, world, "state %.2f GB per GPU >> 126 MB L2: every sweep streams from HBM, no flush needed"
                                  % (state_bytes / 1e9)),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps, "what": "per step and sample: sg_set_spins from pinned host memory, one unit, sg_measure to "
                                            "host; one single-sample context, stream and host thread per sample (independent "
                                            "chains), so uploads overlap sweeps; wall clock over all samples and steps; every "
                                            "step uploads the same host state (a fresh start of the chain) and reads back the "
                                            "measurement only: no device-to-host copy of the spins is included"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": kernel_name,
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "peak_source": peak_src, "alg_bytes_per_update": alg_bytes / updates_per_launch,
                     "updates_per_launch": updates_per_launch, "launch_us": or_launch_s * 1e6,
                     "ps_per_update_or": or_launch_s / updates_per_launch * 1e12,
                     "hb_sweep_ms": hb_ms, "or_call_ms": or_ms},
    }
    if sustained is not None:
        # the same kernel, the same algorithmic bytes, over the median OR call of the sustained segments
        sus_launch_s = sustained["or_call_us"] * 1e-6 / (1 if resident else 2 * cfg.n_or)
        out["roofline"]["sustained_launch_us"] = sus_launch_s * 1e6
        out["roofline"]["sustained_frac"] = alg_bytes / sus_launch_s / 1e9 / peak
        out["sustained"] = dict(sustained, unit=UNIT, ps_per_update=1e12 / sustained["value"],
                                what="median over %d back-to-back segments of %d units each, same loop as the timed steps"
                                     % (sustained["segments"], sustained["units_per_segment"]))
    if world == 1 and not args.no_cpu_baseline:
        rate, cores, what, _, split = oracle_unit_rate(cfg, cfg.n_or if cfg.L >= 32 else 4 * cfg.n_or)
        out["cpu_baseline"] = dict({"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what}, **split)
    traffic_path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_path):     # DRAM bytes per launch of the dominant kernel, from the committed ncu capture
        try:
            with open(traffic_path) as f:
                tr = json.load(f)
            if tr.get("workload") == cfg.name:
                out["roofline"]["traffic"] = tr["dram_bytes_per_launch"]
        except Exception:
            pass
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default: the headline cfg 4)")
    ap.add_argument("--sweep-impl", default="auto", choices=["auto", "tiled", "zmarch", "resident"],
                    help="sg_tune(SG_TUNE_SWEEP_IMPL): which half-sweep kernel serves the sweeps (default: the library's choice)")
    ap.add_argument("--zchunk", type=int, default=0, help="sg_tune(SG_TUNE_ZCHUNK): planes per CTA of the z-marching kernel")
    ap.add_argument("--e2e-zchunk", type=int, default=0, help="sg_tune(SG_TUNE_ZCHUNK) of the single-sample contexts of the e2e leg (0: 32 planes when L is a multiple of 32)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing (profiling runs)")
    ap.add_argument("--sustain-segments", type=int, default=4, help="segments of the sustained leg (0: skip it)")
    ap.add_argument("--sustain-seconds", type=float, default=10.0, help="target duration of the whole sustained leg (each segment is at least 50 units)")
    args = ap.parse_args()
    if args.impl == "ours":
        args.warmup = max(args.warmup, 3)      # timing rule: at least 3 untimed warm-up steps
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
