"""Multi-process plumbing: one process per GPU.  Disorder samples sharded across ranks need no
data-path collective (samples are independent); one sample can be sharded by replica (whole PT chains per
rank, no exchange inside the Monte Carlo) or by temperature slot (the paper's mode: one all-gather of
the energies per PT step).  Orchestration only: every number is computed by the library's kernels; the functions work with
any torch.distributed backend (nccl on the GPU box, gloo in the CPU tests)."""
import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) outside torchrun."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def first_sample_of_rank(rank, samples_per_rank):
    """Global number of the first sample rank `rank` owns: ranks hold [r*n, (r+1)*n).  The number enters
    every Philox counter (sg_shape.first_sample), so a rank draws exactly the numbers a single process
    holding all samples would draw for them."""
    if rank < 0 or samples_per_rank <= 0:
        raise ValueError("rank >= 0 and samples_per_rank > 0 required")
    return rank * samples_per_rank


def replica_window_of_rank(rank, world_size, n_replicas_total, min_replicas=2):
    """(first_replica, n_replicas) of rank `rank` when the replicas of every sample are sharded over the ranks
    (sg_shape.first_replica / n_replicas_total): the PT chains of a sample are per replica, so whole
    chains live on one GPU and the Monte Carlo needs no exchange; a rank keeps at least `min_replicas` replicas so
    that it can measure overlaps among its own (the paper uses two replicas per sample).  Contiguous,
    disjoint windows that cover [0, n_replicas_total); world_size must divide n_replicas_total."""
    if world_size <= 0 or not 0 <= rank < world_size:
        raise ValueError("0 <= rank < world_size required")
    if n_replicas_total % world_size != 0 or n_replicas_total // world_size < min_replicas:
        raise ValueError("world_size must divide n_replicas_total and leave at least min_replicas replicas per rank")
    n = n_replicas_total // world_size
    return rank * n, n


def gather_overlaps(local, world_size, device="cpu"):
    """All ranks' arrays of per-pair overlaps, concatenated along the pair axis in rank order: local is a float64
    array [S][P_local][...]; returns [S][world_size * P_local][...] on every rank (the only data-path collective of
    the replica-sharded run: a few KB per measurement)."""
    import numpy as np
    import torch
    import torch.distributed as dist
    local = np.ascontiguousarray(local, dtype=np.float64)
    if world_size == 1 or not (dist.is_available() and dist.is_initialized()):
        return local
    t = torch.from_numpy(local).to(device)
    parts = [torch.empty_like(t) for _ in range(world_size)]
    dist.all_gather(parts, t)
    return np.concatenate([x.cpu().numpy() for x in parts], axis=1)


def _pairs_from_blocks(local_blocks, rank, world_size, n_local, export, cross, alloc=None, stream=None):
    """Shared orchestration of measure_all_pairs: `local_blocks` are the per-pair arrays [S][P_local]... of the pairs inside
    this rank; a pair across ranks is computed by the rank that holds a, from what b's rank exports and sends to every
    rank below it (one buffer alive at a time; ranks above the source neither export nor receive).  `alloc()` returns an
    uninitialised receive buffer of export()'s shape (default: export(0), which costs a kernel).  `stream`: the CUDA
    stream the context's kernels run on -- export, the transfers and cross are issued with it as torch's current stream,
    because torch.distributed orders its NCCL work against the current stream only.
    Returns the arrays stacked over all pairs in the global order, on every rank."""
    import contextlib
    import numpy as np
    import torch
    import torch.distributed as dist
    mine = {}
    k = 0
    for a in range(n_local):
        for b in range(a + 1, n_local):
            mine[(rank * n_local + a, rank * n_local + b)] = tuple(blk[:, k] for blk in local_blocks)
            k += 1
    if world_size > 1:
        on_stream = torch.cuda.stream(stream) if isinstance(stream, torch.cuda.Stream) else contextlib.nullcontext()
        with on_stream:
            for src in range(1, world_size):                     # rank 0 never sends: nobody holds smaller replicas
                for r in range(n_local):
                    if rank == src:
                        buf = export(r)
                        for dst in range(src):
                            dist.send(buf, dst=dst)
                    elif rank < src:
                        buf = alloc() if alloc is not None else export(0)
                        dist.recv(buf, src=src)
                        for a in range(n_local):
                            mine[(rank * n_local + a, src * n_local + r)] = tuple(cross(a, buf))
        parts = [None] * world_size
        dist.all_gather_object(parts, mine)
        mine = {key: val for part in parts for key, val in part.items()}
    R = world_size * n_local
    pairs = [(a, b) for a in range(R) for b in range(a + 1, R)]
    return tuple(np.stack([mine[pr][j] for pr in pairs], axis=1) for j in range(len(local_blocks)))


def measure_all_pairs(gpu, rank, world_size, n_local, chirality=False):
    """Overlaps of ALL replica pairs a < b of the replica-sharded run (ranks hold n_local consecutive replicas each):
    pairs inside a rank by sg_measure; a pair across ranks by the rank that holds a, from the configurations of b
    (ordered by temperature, sg_export_replica) that b's rank broadcasts: one lattice set per (rank, replica) crosses
    NVLink per measurement, one buffer alive at a time.  `gpu` needs measure(), export_replica(r), measure_cross(r, buf)
    (and, with `chirality`, measure_chiral(), export_chirality(r), chiral_cross(za, zb)).
    Returns (q0 [S][P][T], qk [S][P][T][3][2]) -- with `chirality` also (qc0 [S][P][T][3], qck [S][P][T][3][3][2]) -- on
    every rank, pairs in the order (0,1),(0,2),...,(R-2,R-1) of the GLOBAL replica numbers, R = world_size * n_local."""
    _, q0_loc, qk_loc = gpu.measure()
    alloc, stream = getattr(gpu, "export_buffer", None), getattr(gpu, "stream", None)
    out = _pairs_from_blocks((q0_loc, qk_loc), rank, world_size, n_local, gpu.export_replica, gpu.measure_cross, alloc, stream)
    if chirality:
        local_z = {}

        def cross(a, zb):
            if a not in local_z:
                local_z[a] = gpu.export_chirality(a)
            return gpu.chiral_cross(local_z[a], zb)

        out = out + _pairs_from_blocks(tuple(gpu.measure_chiral()), rank, world_size, n_local, gpu.export_chirality, cross, alloc, stream)
    return out


def slot_window_of_rank(rank, world_size, n_temps_total):
    """(first_slot, n_temps) of rank `rank` when the configurations (slots) of every PT chain are sharded over the ranks
    (sg_shape.first_slot / n_temps_total; the paper's multi-GPU mode, where N_GPU = N_T and a GPU holds
    the two replicas of one slot).  Contiguous, disjoint windows of equal length; world_size must divide n_temps_total."""
    if world_size <= 0 or not 0 <= rank < world_size:
        raise ValueError("0 <= rank < world_size required")
    if n_temps_total % world_size != 0:
        raise ValueError("world_size must divide n_temps_total")
    n = n_temps_total // world_size
    return rank * n, n


def _on_stream(gpu):
    import contextlib
    import torch
    stream = getattr(gpu, "stream", None)
    return torch.cuda.stream(stream) if isinstance(stream, torch.cuda.Stream) else contextlib.nullcontext()


def pt_step_sharded(gpu, world_size, gathered=None):
    """The PT sweep of slot-sharded chains: every rank publishes the energies of its slots (S*R*n_temps doubles, a device
    buffer), ONE all-gather carries them to all ranks (the paper's "exchange with the master of a double precision
    number"; 8*C bytes per sample in all), and every rank runs the same swap kernel on the gathered vector:
    identical Philox counters, identical decisions, so the temperature assignment stays replicated with no second
    exchange.  `gathered`: reusable device tensor [world_size][S][R][n_temps] float64.  Returns it."""
    import torch
    import torch.distributed as dist
    with _on_stream(gpu):
        mine = gpu.pt_publish()
        if gathered is None:
            gathered = torch.empty((world_size,) + tuple(mine.shape), dtype=mine.dtype, device=mine.device)
        if world_size > 1:
            dist.all_gather(list(gathered.unbind(0)), mine)
        else:
            gathered[0].copy_(mine)
        gpu.pt_swap_gathered(gathered)
    return gathered


def unit_sharded(gpu, n_or, world_size, gathered=None):
    """One MCS of slot-sharded chains: the sweeps touch only the rank's own lattices, the PT step is pt_step_sharded."""
    gpu.sweep_hb(1)
    gpu.sweep_or(n_or)
    return pt_step_sharded(gpu, world_size, gathered)


def overlaps_sharded(gpu, world_size, pairs=None, chirality=False):
    """Overlaps of slot-sharded chains.  The two configurations at temperature t of a replica pair (a, b) may live on
    different ranks.  Per replica b: every rank exports the temperatures whose configuration it holds (zeros elsewhere,
    sg_export_replica), an all-reduce (sum) assembles the replica ordered by temperature on every rank, every rank forms the
    overlap with its part of replica a (sg_measure_cross: zero where it does not hold the configuration), and a last
    all-reduce (sum) of the few numbers completes every temperature.  Returns (q0 [S][P][T], qk [S][P][T][3][2]) on every
    rank, pairs a < b in the order of sg_measure (or the given list).  At measurement time only.
    chirality=True: the chiral-glass overlaps instead, (qc0 [S][P][T][3], qck [S][P][T][3][3][2]) (Eq. (2); the
    paper measured them on the runs it sharded by temperature): sg_export_chirality in place of sg_export_replica
    (zeta of the temperatures a rank holds, zeros elsewhere), sg_chiral_cross between the rank's own zero-padded export of
    replica a and the all-reduced buffer of replica b, and the same final all-reduce."""
    import numpy as np
    import torch
    import torch.distributed as dist
    R = gpu.R
    if pairs is None:
        pairs = [(a, b) for a in range(R) for b in range(a + 1, R)]
    q0s, qks = {}, {}
    with _on_stream(gpu):
        own = {}
        for b in sorted({b for _, b in pairs}):
            full = gpu.export_chirality(b) if chirality else gpu.export_replica(b)
            if world_size > 1:
                dist.all_reduce(full, op=dist.ReduceOp.SUM)
            for a in [a for a, bb in pairs if bb == b]:
                if chirality:
                    if a not in own:
                        own[a] = gpu.export_chirality(a)
                    q0s[(a, b)], qks[(a, b)] = gpu.chiral_cross(own[a], full)
                else:
                    q0s[(a, b)], qks[(a, b)] = gpu.measure_cross(a, full)
    q0 = np.stack([q0s[pr] for pr in pairs], axis=1)
    qk = np.stack([qks[pr] for pr in pairs], axis=1)
    if world_size > 1:
        t0, tk = torch.from_numpy(q0), torch.from_numpy(qk)
        dev = getattr(gpu, "device", "cpu") if dist.get_backend() == "nccl" else "cpu"
        t0, tk = t0.to(dev), tk.to(dev)
        dist.all_reduce(t0, op=dist.ReduceOp.SUM)
        dist.all_reduce(tk, op=dist.ReduceOp.SUM)
        q0, qk = t0.cpu().numpy(), tk.cpu().numpy()
    return q0, qk


def schwinger_dyson_sharded(gpu, world_size):
    """Schwinger-Dyson monitor (Eq. (A6)) of slot-sharded chains: every rank reduces the two site averages of
    the configurations it holds (sg_schwinger_dyson: indexed by temperature, exact zeros elsewhere) and one all-reduce (sum) of
    S*R*T*2 doubles completes every temperature on every rank.  Returns sd [S][R][T][2]."""
    import torch
    import torch.distributed as dist
    sd = gpu.schwinger_dyson()
    if world_size > 1:
        dev = getattr(gpu, "device", "cpu") if dist.get_backend() == "nccl" else "cpu"
        t = torch.from_numpy(sd).to(dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        sd = t.cpu().numpy()
    return sd


def init_process_group(backend, world_size):
    """Joins the torchrun rendezvous (MASTER_ADDR / MASTER_PORT from the environment) when world_size > 1."""
    import torch.distributed as dist
    if world_size > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)
    return dist.is_initialized()


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _reduce(value, op_name, device):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(value, device="cpu"):
    """Max of a host scalar over all ranks (device-timed durations: the job ends with its slowest rank)."""
    return _reduce(value, "MAX", device)


def sum_over_ranks(value, device="cpu"):
    """Sum of a host scalar over all ranks (units of work processed)."""
    return _reduce(value, "SUM", device)


def whole_job_rate(units_this_rank, seconds_this_rank, device="cpu"):
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    total = sum_over_ranks(units_this_rank, device)
    slowest = max_over_ranks(seconds_this_rank, device)
    return total / slowest, total, slowest
