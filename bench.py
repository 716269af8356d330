"""bench.py -- throughput of the hot path on the BASELINE.json headline workload (cfg 4: L=64, 4 samples,
4 replicas x 48 temperatures, 1 HB + 32 OR sweeps per PT swap, measurement every 10 units).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4]
    python bench.py --kernel sweep|units|sustained|exercise ...     (kernel-level timings for profiles/, see below; not the bench line)

--gpus N > 1 without a torchrun environment starts the N ranks itself (re-runs this command under torch.distributed.run, one rank per
GPU, NCCL; fails if fewer than N devices are visible); under torchrun it joins the ranks it finds.  --shard samples (default): every
rank holds the config's samples, no data-path collective, weak scaling.  --shard slots: the paper's layout -- ONE sample, its
temperature slots over the ranks, one all-gather of the energies per PT step, strong scaling.  --check-launch: rendezvous only.

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
# FP32 work of one overrelaxation update (Eq. (A2) on the field of footnote 64): six 3x3 matrix-vector products = 54 multiply-adds,
# s.h and h.h 3 each, s' = (2 s.h / h.h) h - s another 3: 63 FMA-pipe operations (plus one reciprocal and one multiply, not counted).
# The "alu" peak they are held against is SMs x 128 FP32 lanes x the SM clock sampled during the run.
FMA_PER_OR_UPDATE = 63
N_SMS, FP32_LANES_PER_SM = 148, 128


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
    gpu = sg.SpinGlass(L, S, R, T, cfg.betas, seed=cfg.seed, first_sample=multi.first_sample_of_rank(rank, S),
                       fused_buffer=args.sweep_impl == "fused")
    gpu.tune(sg.TUNE_SWEEP_IMPL, {"auto": sg.SWEEP_AUTO, "tiled": sg.SWEEP_TILED, "zmarch": sg.SWEEP_ZMARCH, "resident": sg.SWEEP_RESIDENT,
                                  "cluster": sg.SWEEP_CLUSTER, "fused": sg.SWEEP_FUSED}[args.sweep_impl])
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
    # Which kernel served sg_sweep_or is the LIBRARY's answer (sg_sweep_impl_used), not a guess from the shape.
    # On-chip kernels (resident: L <= 12, lattice in one CTA's shared memory; cluster: L = 16, lattice in a cluster's): one launch
    # runs all n_or sweeps of the call and moves every spin across HBM once per call (12 B read + 12 B written per site and copy,
    # the couplings of both colours once per copy group), so HBM is not what bounds them: their roofline is the FP32 pipe.
    served, cluster_fallback = gpu.sweep_impl_used(sg.KIND_OR)
    served_name = {sg.SWEEP_TILED: "tiled", sg.SWEEP_ZMARCH: "zmarch", sg.SWEEP_RESIDENT: "resident", sg.SWEEP_FUSED: "fused",
                   sg.SWEEP_CLUSTER: "cluster"}[served]
    on_chip = served in (sg.SWEEP_RESIDENT, sg.SWEEP_CLUSTER)
    peak, peak_src = measured_hbm_peak()
    if on_chip:
        or_launch_s = or_ms * 1e-3
        launches_per_call = 1
        updates_per_launch = S * C * N * cfg.n_or
        alg_bytes = S * C * N * 24.0 + S * ((C + 31) // 32) * N * 216.0
        kernel_name = ("k_sweep_res<OR>: %d OR sweeps per launch, lattice resident in shared memory" if served == sg.SWEEP_RESIDENT else
                       "k_sweep_cres<OR>: %d OR sweeps per launch, lattice resident in the shared memory of thread-block clusters") % cfg.n_or
    elif served == sg.SWEEP_FUSED:
        or_launch_s = or_ms * 1e-3 / cfg.n_or
        launches_per_call = cfg.n_or
        updates_per_launch = S * C * N
        alg_bytes = (24.0 + ALG_BYTES_COUPLINGS / C) * updates_per_launch      # every spin read once and written once per sweep
        kernel_name = "k_sweep_fz: both colours of an OR sweep in one out-of-place pass, zchunk=%d" % args.zchunk
    else:
        or_launch_s = or_ms * 1e-3 / (2 * cfg.n_or)
        launches_per_call = 2 * cfg.n_or
        updates_per_launch = S * C * N // 2
        alg_bytes = algorithmic_bytes_per_update(C) * updates_per_launch
        kernel_name = "OR half-sweep (%s), sweep_impl=%s zchunk=%d" % ("k_sweep_zm<OR>" if served == sg.SWEEP_ZMARCH else "k_sweep<OR>", args.sweep_impl, args.zchunk)
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
        "roofline": {"bound": "hbm", "kernel": kernel_name, "served_by": served_name, "cluster_fallback_cuda_error": cluster_fallback,
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "peak_source": peak_src, "alg_bytes_per_update": alg_bytes / updates_per_launch,
                     "updates_per_launch": updates_per_launch, "launch_us": or_launch_s * 1e6,
                     "ps_per_update_or": or_launch_s / updates_per_launch * 1e12,
                     "hb_sweep_ms": hb_ms, "or_call_ms": or_ms},
    }
    # the FP32 floor of the same launch, for every kernel; for the on-chip kernels it IS the roofline (the HBM figures stay as
    # "hbm_*": what the launch moves across HBM by construction, far from the peak because the launch is not bound by it)
    sm_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz")
    if sm_mhz:
        alu_peak = N_SMS * FP32_LANES_PER_SM * sm_mhz * 1e6 * 2 / 1e12           # TFLOP/s at the clock the run held
        alu_achieved = 2.0 * FMA_PER_OR_UPDATE * updates_per_launch / or_launch_s / 1e12
        alu = {"achieved": alu_achieved, "peak": alu_peak, "unit": "TFLOP/s", "frac": alu_achieved / alu_peak,
               "fma_per_update": FMA_PER_OR_UPDATE, "sm_mhz": sm_mhz,
               "peak_source": "%d SMs x %d FP32 lanes x 2 flop x the median SM clock sampled during the timed loop" % (N_SMS, FP32_LANES_PER_SM)}
        if on_chip:
            r = out["roofline"]
            r.update({"hbm_achieved": r["achieved"], "hbm_peak": r["peak"], "hbm_frac": r["frac"], "hbm_peak_source": r["peak_source"]})
            r.update({"bound": "alu", "achieved": alu["achieved"], "peak": alu["peak"], "unit": "TFLOP/s", "frac": alu["frac"],
                      "peak_source": alu["peak_source"], "fma_per_update": FMA_PER_OR_UPDATE, "sm_mhz": sm_mhz})
        else:
            out["roofline"]["alu"] = alu
    if sustained is not None:
        # the same kernel, the same algorithmic bytes, over the median OR call of the sustained segments
        sus_launch_s = sustained["or_call_us"] * 1e-6 / launches_per_call
        out["roofline"]["sustained_launch_us"] = sus_launch_s * 1e6
        if out["roofline"]["bound"] == "alu":
            out["roofline"]["sustained_frac"] = out["roofline"]["frac"] * or_launch_s / sus_launch_s     # at the burst loop's clock
        else:
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
            if tr.get("workload") == cfg.name and tr.get("served_by", "zmarch") == served_name:
                out["roofline"]["traffic"] = tr["dram_bytes_per_launch"]
                out["roofline"]["traffic_source"] = ("NOT measured by this run: dram__bytes_read.sum + dram__bytes_write.sum of one launch from the "
                                                     "committed ncu capture profiles/traffic.json (%s)" % tr.get("source", "see profiles/"))
        except Exception:
            pass
    print(json.dumps(out), flush=True)


def run_slots(args, cfg):
    """--shard slots: the paper's own multi-GPU layout (App. A.3: "each GPU updates only 2 lattices ... N_GPU =
    N_T").  ONE disorder sample of the workload; the T temperature slots of its R chains are split over the ranks (a rank holds
    R x T/N lattices), the sweeps touch only a rank's own lattices, and the PT step is one all-gather of the R*T energies (NCCL)
    followed by the same swap kernel on every rank (multi.pt_step_sharded).  Every `measure_every` units: energies per
    temperature from the gathered vector and the overlaps of all replica pairs across the shards (multi.overlaps_sharded).
    Total work is fixed as N grows ("scaling": "strong").  Same JSON line as the default mode."""
    import torch
    import paper_1309_1599_b200 as sg
    rank, local_rank, world = multi.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    multi.init_process_group("nccl", world)
    L, R, T, N = cfg.L, cfg.n_replicas, cfg.n_temps, cfg.n_sites
    first_slot, n_t = multi.slot_window_of_rank(rank, world, T)
    gpu = sg.SpinGlass(L, 1, R, n_t, cfg.betas, seed=cfg.seed, first_slot=first_slot, n_temps_total=T)
    gpu.init_sample(0, sg.GEN_OFFDIAG_SYM, cfg.sigma_D)
    C_loc = R * n_t
    updates_rank = (1 + cfg.n_or) * C_loc * N
    state_bytes = C_loc * N * 12
    ev = lambda: torch.cuda.Event(enable_timing=True)
    or_pairs, box = [], {"gathered": None}

    def unit(k, timed):
        gpu.sweep_hb(1)
        if timed:
            a, b = ev(), ev()
            a.record(); gpu.sweep_or(cfg.n_or); b.record()
            or_pairs.append((a, b))
        else:
            gpu.sweep_or(cfg.n_or)
        box["gathered"] = multi.pt_step_sharded(gpu, world, box["gathered"])
        if (k + 1) % cfg.measure_every == 0:
            return (gpu.energy_by_temp(box["gathered"]),) + tuple(multi.overlaps_sharded(gpu, world))
        return None

    for k in range(args.warmup):
        unit(k, False)
    gpu.sync()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    multi.barrier(); torch.cuda.synchronize()
    launches0, t_wall0 = gpu.kernel_launches(), time.time()
    start, stop = ev(), ev()
    start.record()
    for k in range(args.steps):
        unit(k, True)
    stop.record()
    torch.cuda.synchronize(); multi.barrier()
    t_wall1 = time.time()
    launches = gpu.kernel_launches() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    seconds = start.elapsed_time(stop) * 1e-3
    value, _, slowest = multi.whole_job_rate(args.steps * updates_rank, seconds, device)
    or_ms = float(np.mean([a.elapsed_time(b) for a, b in or_pairs]))
    served, _ = gpu.sweep_impl_used(sg.KIND_OR)
    on_chip = served in (sg.SWEEP_RESIDENT, sg.SWEEP_CLUSTER)
    or_launch_s = or_ms * 1e-3 / (1 if on_chip else 2 * cfg.n_or)
    updates_per_launch = C_loc * N * cfg.n_or if on_chip else C_loc * N // 2
    alg_bytes = (C_loc * N * 24.0 + ((C_loc + 31) // 32) * N * 216.0) if on_chip else algorithmic_bytes_per_update(C_loc) * updates_per_launch
    peak, peak_src = measured_hbm_peak()
    # end to end: upload of the rank's lattices from pinned host memory, one unit, energies and overlaps back, every step
    host = torch.empty((C_loc, 3, N), dtype=torch.float32).pin_memory()
    host.numpy()[...] = gpu.get_spins(0)
    e2e_steps = max(1, min(args.steps, 10))
    multi.barrier(); torch.cuda.synchronize()
    t0, d2h = time.perf_counter(), 0
    for k in range(e2e_steps):
        gpu.set_spins(0, host.numpy())
        gpu.sweep_hb(1); gpu.sweep_or(cfg.n_or)
        box["gathered"] = multi.pt_step_sharded(gpu, world, box["gathered"])
        res = (gpu.energy_by_temp(box["gathered"]),) + tuple(multi.overlaps_sharded(gpu, world))
        d2h = sum(a.nbytes for a in res)
    torch.cuda.synchronize()
    e2e_value, _, _ = multi.whole_job_rate(e2e_steps * updates_rank, time.perf_counter() - t0, device)
    if rank != 0:
        return
    conf = workload_config(cfg, world, "state %.2f GB per GPU: every sweep streams from HBM" % (state_bytes / 1e9))
    conf.update({"samples_per_gpu": 1.0 / world, "updates_per_step_per_gpu": updates_rank,
                 "parallelism": "ONE sample; the %d temperature slots of its %d chains over %d GPU(s) (%d slots x %d replicas per GPU); per PT step "
                                "one all-gather of %d doubles (NCCL), overlaps across shards by all-reduce at measurement time" % (T, R, world, n_t, R, R * T)})
    achieved = alg_bytes / or_launch_s / 1e9
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": slowest * 1e3 / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "ps_per_update": 1e12 / value, "config": conf, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                "what": "per step and rank: sg_set_spins of the rank's lattices from pinned host memory, one slot-sharded unit, energies "
                        "and overlaps of all pairs to the host"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu" if on_chip else "hbm", "kernel": "OR sweeps of a rank's %d lattices, served_by=%d" % (C_loc, served),
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                     "alg_bytes_per_update": alg_bytes / updates_per_launch, "updates_per_launch": updates_per_launch,
                     "launch_us": or_launch_s * 1e6, "or_call_ms": or_ms},
    }), flush=True)


# ---- starting the ranks (`--gpus N` outside torchrun) ----
def spawn_command(n, argv, port):
    """The command the round driver itself uses for N > 1 (one rank per GPU, rendezvous on 127.0.0.1)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def free_port():
    import socket
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        return sock.getsockname()[1]


def spawn_ranks_if_needed(args, argv):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: re-run this command under torch.distributed.run with N
    ranks and return its exit code (rank 0 of that job prints the ONE line); None when nothing is to be spawned.  Refuses to
    run fewer ranks than asked for."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ or args.impl == "reference" or args.kernel:
        return None
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus and not (args.check_launch and have == 0):
        raise SystemExit("bench.py: --gpus %d needs %d CUDA devices, %d visible; refusing to run fewer ranks than asked for" % (args.gpus, args.gpus, have))
    return subprocess.call(spawn_command(args.gpus, argv, free_port()))


def check_launch(args):
    """--check-launch: every rank joins the process group (nccl with a GPU each, gloo on a CPU-only box), all-reduces its rank
    number, and rank 0 prints one JSON line -- the rendezvous and the one-line contract, without the workload."""
    import torch
    import torch.distributed as dist
    rank, local_rank, world = multi.env_rank()
    cuda = torch.cuda.is_available()
    if cuda:
        torch.cuda.set_device(local_rank)
    multi.init_process_group("nccl" if cuda else "gloo", world)
    t = torch.tensor([float(rank)], dtype=torch.float64, device="cuda" if cuda else "cpu")
    if world > 1:
        dist.all_reduce(t)
    multi.barrier()
    if rank == 0:
        print(json.dumps({"check_launch": True, "n_gpus": world, "asked": args.gpus, "backend": "nccl" if cuda else "gloo",
                          "rank_sum": float(t.item()), "rank_sum_expected": world * (world - 1) / 2.0}), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---- kernel-level timings (`--kernel ...`): one piece of the hot path on a BASELINE.json workload under a chosen kernel, for A/B
# measurements and as the short command line ncu wraps; the commands profiles/*.md name.  One JSON line per measurement, device
# timing (CUDA events on the context's stream), best and median of --reps repetitions after a warm-up.  NOT the bench line.
SWEEP_IMPLS = {"auto": 0, "tiled": 1, "zmarch": 2, "resident": 3, "fused": 4, "cluster": 5}


def kernel_context(sg, args, stream=None):
    cfg = W.CONFIGS[args.config]
    S = args.samples or cfg.n_samples
    g = sg.SpinGlass(cfg.L, S, cfg.n_replicas, cfg.n_temps, cfg.betas, seed=1, stream=stream, fused_buffer=(args.sweep_impl == "fused"))
    g.tune(sg.TUNE_SWEEP_IMPL, SWEEP_IMPLS[args.sweep_impl])
    if args.zchunk:
        g.tune(sg.TUNE_ZCHUNK, args.zchunk)
    if args.cluster_ctas:
        g.tune(sg.TUNE_CLUSTER_CTAS, args.cluster_ctas)
    for s in range(S):
        g.init_sample(s, sg.GEN_OFFDIAG_SYM, cfg.sigma_D)
    return cfg, S, g


def kernel_sweep(sg, torch, args):
    """us per sweep of --sweeps OR (or --kind hb) sweeps per call."""
    cfg, S, g = kernel_context(sg, args)
    call = g.sweep_hb if args.kind == "hb" else g.sweep_or
    call(2)
    g.sync()
    times = []
    for _ in range(args.reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); call(args.sweeps); e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1) * 1e3 / args.sweeps)
    updates = S * cfg.n_copies * cfg.n_sites
    served = g.sweep_impl_used(sg.KIND_HB if args.kind == "hb" else sg.KIND_OR)[0]
    out = dict(kernel="sweep", cfg=cfg.name, kind=args.kind, sweep_impl=args.sweep_impl, served_by=served, zchunk=args.zchunk,
               cluster_ctas=args.cluster_ctas, samples=S, sweeps=args.sweeps, us_per_sweep_best=min(times),
               us_per_sweep_median=float(np.median(times)), ps_per_update_best=min(times) * 1e6 / updates, updates_per_sweep=updates,
               energy_sum=float(g.get_energies().sum()))
    g.close()
    return out


def kernel_units(sg, torch, args):
    """us per MCS through sg_run_units (wall clock around a synchronised call of --units units)."""
    cfg, S, g = kernel_context(sg, args, stream=torch.cuda.Stream())
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
    out = dict(kernel="units", cfg=cfg.name, sweep_impl=args.sweep_impl, graph=args.graph, graph_replays=g.graph_replays(), samples=S, units=n,
               us_per_unit_best=min(times) * 1e6, us_per_unit_median=float(np.median(times)) * 1e6, updates_per_s=upd / min(times))
    g.close()
    return out


def kernel_sustained(sg, torch, args):
    """us per OR half-sweep in six back-to-back segments of 1024 sweeps: what the kernel holds under the power cap."""
    cfg, S, g = kernel_context(sg, args)
    g.sweep_or(8)
    g.sync()
    res = []
    for _ in range(6):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); g.sweep_or(1024); e1.record()
        torch.cuda.synchronize()
        res.append(round(e0.elapsed_time(e1) * 1e3 / 2048, 1))
    g.close()
    return dict(kernel="sustained", cfg=cfg.name, sweep_impl=args.sweep_impl, us_per_halfsweep=res)


def kernel_exercise(sg, torch, args):
    """Every kernel family once on a small --shape L,S,R,T: what compute-sanitizer (memcheck / racecheck) is pointed at."""
    L, S, R, T = [int(v) for v in args.shape.split(",")]
    g = sg.SpinGlass(L, S, R, T, np.linspace(0.5, 1.8, T), seed=7, fused_buffer=(args.sweep_impl == "fused"))
    g.tune(sg.TUNE_SWEEP_IMPL, SWEEP_IMPLS[args.sweep_impl])
    for s in range(S):
        g.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
    g.run_units(9, 2)
    g.unit(1)
    g.halfsweep(sg.KIND_OR, 0); g.halfsweep(sg.KIND_HB, 1)
    e, q0, qk = g.measure()
    out = dict(kernel="exercise", shape=[L, S, R, T], sweep_impl=args.sweep_impl, e_mean=float(e.mean()))
    if R > 1:
        g.measure_chiral(); g.accumulate(True); g.get_logbins()
        q0x, _ = g.measure_cross(0, g.export_replica(1))
        out["cross_minus_measure"] = float(np.abs(q0x - q0[:, 0]).max())
        za, zb = g.export_chirality(0), g.export_chirality(1)
        if S <= 3:
            a, _ = sg.chiral_cross_static(L, S, T, za, zb)
            out["static_minus_ctx"] = float(np.abs(a.cpu().numpy() - g.chiral_cross(za, zb)[0]).max())
    g.schwinger_dyson(); g.pt_walk(); g.pt_visits(); g.pt_stats()
    spins = g.get_spins(0)
    out["norm_err"] = float(np.abs(np.sqrt((spins.astype(np.float64) ** 2).sum(axis=1)) - 1.0).max())
    out["launches"] = g.kernel_launches()
    g.close()
    return out


def run_kernel_mode(args):
    import torch
    import paper_1309_1599_b200 as sg
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --kernel: no CUDA device (the product has no CPU path)")
    fn = {"sweep": kernel_sweep, "units": kernel_units, "sustained": kernel_sustained, "exercise": kernel_exercise}[args.kernel]
    print(json.dumps(fn(sg, torch, args)), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default: the headline cfg 4)")
    ap.add_argument("--sweep-impl", default="auto", choices=["auto", "tiled", "zmarch", "resident", "cluster", "fused"],
                    help="sg_tune(SG_TUNE_SWEEP_IMPL): which half-sweep kernel serves the sweeps (default: the library's choice)")
    ap.add_argument("--zchunk", type=int, default=0, help="sg_tune(SG_TUNE_ZCHUNK): planes per CTA of the z-marching kernel")
    ap.add_argument("--e2e-zchunk", type=int, default=0, help="sg_tune(SG_TUNE_ZCHUNK) of the single-sample contexts of the e2e leg (0: 32 planes when L is a multiple of 32)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing (profiling runs)")
    ap.add_argument("--sustain-segments", type=int, default=4, help="segments of the sustained leg (0: skip it)")
    ap.add_argument("--sustain-seconds", type=float, default=10.0, help="target duration of the whole sustained leg (each segment is at least 50 units)")
    ap.add_argument("--kernel", choices=["sweep", "units", "sustained", "exercise"], default=None,
                    help="kernel-level timing instead of the bench line (uses --config, --sweep-impl, --zchunk and the flags below)")
    ap.add_argument("--kind", choices=["or", "hb"], default="or", help="--kernel sweep: which sweep")
    ap.add_argument("--sweeps", type=int, default=32, help="--kernel sweep: sweeps per timed call")
    ap.add_argument("--samples", type=int, default=0, help="--kernel: samples in the context (0 = the config's)")
    ap.add_argument("--cluster-ctas", type=int, default=0, help="--kernel: sg_tune(SG_TUNE_CLUSTER_CTAS) (0 = the library's default)")
    ap.add_argument("--units", type=int, default=0, help="--kernel units: units per timed call (0 = about 2e9 updates' worth)")
    ap.add_argument("--graph", type=int, default=1, help="--kernel units: sg_tune(SG_TUNE_GRAPH)")
    ap.add_argument("--reps", type=int, default=5, help="--kernel: repetitions")
    ap.add_argument("--shape", default="8,2,2,6", help="--kernel exercise: L,S,R,T")
    ap.add_argument("--shard", choices=["samples", "slots"], default="samples",
                    help="samples (default): every GPU holds the config's samples, no collective; slots: ONE sample, its temperature slots "
                         "over the GPUs with an all-gather per PT step (the paper's layout, PAPER.md:358-364)")
    ap.add_argument("--check-launch", action="store_true", help="start the ranks, all-reduce the rank numbers, print one line; no workload")
    args = ap.parse_args()
    if args.kernel:
        return run_kernel_mode(args)
    rc = spawn_ranks_if_needed(args, sys.argv[1:])
    if rc is not None:
        sys.exit(rc)
    if args.check_launch:
        return check_launch(args)
    world = multi.env_rank()[2]
    if world != args.gpus and multi.env_rank()[0] == 0:
        print("bench.py: --gpus %d but the launcher started %d rank(s); reporting n_gpus = %d" % (args.gpus, world, world), file=sys.stderr)
    if args.impl == "ours":
        args.warmup = max(args.warmup, 3)      # timing rule: at least 3 untimed warm-up steps
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.shard == "slots":
        run_slots(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
