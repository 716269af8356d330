"""Multi-process plumbing of the weak-scaling run: one process per GPU, disorder
samples sharded across ranks, no data-path collective (samples are independent).
torch.distributed carries only the barrier and the max / sum of a few host scalars; the functions
work with any backend (nccl on the GPU box, gloo in the CPU tests)."""
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
