"""Host logic of the weak-scaling run (paper_1309_1599_b200/multi.py) with two gloo processes on CPU:
sample sharding, the barrier, max-over-ranks timing and the whole-job rate.  No GPU, no oracle."""
import os
import socket

import pytest
import torch.multiprocessing as mp

from paper_1309_1599_b200 import multi


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


import numpy as np


class _FakeShard:
    """Stands in for a replica-sharded SpinGlass in the orchestration test: 'configurations' are tensors filled with the
    global replica number, an 'overlap' of replicas a, b is 10 a + b (so who was paired with whom is visible)."""
    S, T = 2, 3

    def __init__(self, rank, n_local):
        self.rank, self.n = rank, n_local

    def measure(self):
        import numpy as np
        pairs = [(a, b) for a in range(self.n) for b in range(a + 1, self.n)]
        v = np.array([10.0 * (self.rank * self.n + a) + (self.rank * self.n + b) for a, b in pairs])
        q0 = np.broadcast_to(v[None, :, None], (self.S, len(pairs), self.T)).copy()
        return None, q0, np.broadcast_to(q0[..., None, None], q0.shape + (3, 2)).copy()

    def export_replica(self, r):
        import torch
        return torch.full((self.S, 3, 4, self.T), float(self.rank * self.n + r))

    def measure_chiral(self):
        _, q0, _ = self.measure()
        return -q0[..., None] * np.ones(3), -q0[..., None, None, None] * np.ones((3, 3, 2))

    def export_chirality(self, r):
        return -self.export_replica(r)

    def chiral_cross(self, za, zb):
        v = -(10.0 * float(-za[0, 0, 0, 0]) + float(-zb[0, 0, 0, 0]))
        return np.full((self.S, self.T, 3), v), np.full((self.S, self.T, 3, 3, 2), v)

    def measure_cross(self, a, buf):
        import numpy as np
        v = 10.0 * (self.rank * self.n + a) + float(buf[0, 0, 0, 0])
        return np.full((self.S, self.T), v), np.full((self.S, self.T, 3, 2), v)


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    assert multi.env_rank() == (rank, rank, world)
    assert multi.init_process_group("gloo", world)
    multi.barrier()
    first = multi.first_sample_of_rank(rank, 4)
    seconds = 1.0 + rank                       # rank 1 is the slow one
    rate, total, slowest = multi.whole_job_rate(100.0 * (rank + 1), seconds)
    import numpy as np
    window = multi.replica_window_of_rank(rank, world, 4)
    q = multi.gather_overlaps(np.full((3, 1, 5), float(rank)), world)       # [S][P_local][T] of this rank's one pair
    q0_all, qk_all, qc0_all, qck_all = multi.measure_all_pairs(_FakeShard(rank, 2), rank, world, 2, chirality=True)
    assert qc0_all[0, :, 0, 0].tolist() == [-v for v in q0_all[0, :, 0].tolist()] and qck_all.shape == (2, 6, 3, 3, 3, 2)
    out.put((rank, first, multi.max_over_ranks(seconds), multi.sum_over_ranks(first), rate, total, slowest, window,
             q.shape, q[:, :, 0].tolist(), q0_all[0, :, 0].tolist(), qk_all.shape))
    multi.barrier()
    import torch.distributed as dist
    dist.destroy_process_group()


def test_two_rank_gloo_sharding_and_reduction():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [0, 4]                       # disjoint, contiguous sample ranges
    for g in got:
        assert g[2] == 2.0 and g[3] == 4.0                     # max / sum agree on every rank
        assert g[5] == 300.0 and g[6] == 2.0 and g[4] == 150.0  # all units / slowest rank
        assert g[8] == (3, 2, 5) and g[9] == [[0.0, 1.0]] * 3   # every rank sees both ranks' pairs, in rank order
        # all six pairs of the four replicas, in the global order, each formed from the right two replicas, on every rank
        assert g[10] == [1.0, 2.0, 3.0, 12.0, 13.0, 23.0] and g[11] == (2, 6, 3, 3, 2)
    assert [g[7] for g in got] == [(0, 2), (2, 2)]             # replica windows: disjoint, contiguous, two replicas each


def test_single_process_passthrough():
    assert multi.max_over_ranks(3.5) == 3.5 and multi.sum_over_ranks(2.0) == 2.0
    assert multi.whole_job_rate(10.0, 2.0) == (5.0, 10.0, 2.0)
    assert multi.first_sample_of_rank(3, 4) == 12
    with pytest.raises(ValueError):
        multi.first_sample_of_rank(-1, 4)
    q0_one, _ = multi.measure_all_pairs(_FakeShard(0, 3), 0, 1, 3)
    assert q0_one[0, :, 0].tolist() == [1.0, 2.0, 12.0]
    assert multi.replica_window_of_rank(0, 1, 4) == (0, 4) and multi.replica_window_of_rank(1, 2, 4) == (2, 2)
    assert multi.replica_window_of_rank(2, 4, 4, min_replicas=1) == (2, 1)
    for bad in ((0, 4, 4), (0, 3, 4), (2, 2, 4)):               # one replica per rank, not a divisor, rank out of range
        with pytest.raises(ValueError):
            multi.replica_window_of_rank(*bad)


class _FakeSlotShard:
    """Stands in for a slot-sharded SpinGlass (no GPU): it 'holds' n_temps slots of every chain, its energies are
    100 * rank + slot, its exported replica carries the rank in the columns it owns, a cross overlap counts what it saw."""
    S, R, N = 2, 2, 4

    def __init__(self, rank, world, n_temps_total):
        self.rank, self.W, self.Tt = rank, world, n_temps_total
        self.first_slot, self.T = multi.slot_window_of_rank(rank, world, n_temps_total)
        self.swapped_with = None
        self.calls = []

    def sweep_hb(self, n):
        self.calls.append("hb")

    def sweep_or(self, n):
        self.calls.append("or%d" % n)

    def pt_publish(self):
        import torch
        self.calls.append("publish")
        return torch.full((self.S, self.R, self.T), 100.0 * self.rank, dtype=torch.float64) + torch.arange(self.T, dtype=torch.float64)

    def pt_swap_gathered(self, gathered):
        self.calls.append("swap")
        self.swapped_with = gathered.clone()

    def export_replica(self, b):
        import torch
        out = torch.zeros((self.S, 3, self.N, self.Tt))
        out[..., self.first_slot:self.first_slot + self.T] = 1.0 + b          # the temperatures this shard holds (identity assignment)
        return out

    def measure_cross(self, a, full):
        q0 = np.zeros((self.S, self.Tt)); qk = np.zeros((self.S, self.Tt, 3, 2))
        own = slice(self.first_slot, self.first_slot + self.T)
        q0[:, own] = 10.0 * a + full[0, 0, 0, own].numpy()                    # 10 a + (1 + b) where the whole replica b arrived
        qk[:, own] = q0[:, own, None, None]
        return q0, qk

    def schwinger_dyson(self):
        sd = np.zeros((self.S, self.R, self.Tt, 2))
        sd[:, :, self.first_slot:self.first_slot + self.T] = 1.0 + self.rank      # the temperatures held, zeros elsewhere
        return sd

    def export_chirality(self, r):
        return 100.0 * self.export_replica(r)                                 # 100 (1 + r) at the temperatures held, zeros elsewhere

    def chiral_cross(self, za, zb):
        # product of the two buffers at one site: non-zero only where this shard's own export is (its temperatures)
        prod = (za[:, :, 0, :] * zb[:, :, 0, :]).numpy()                       # [S][3][Tt]
        qc0 = np.moveaxis(prod, 1, 2).copy()                                  # [S][Tt][3]
        return qc0, np.zeros((self.S, self.Tt, 3, 3, 2))


def _slot_worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    assert multi.init_process_group("gloo", world)
    shard = _FakeSlotShard(rank, world, 6)
    gathered = multi.unit_sharded(shard, 3, world)
    q0, qk = multi.overlaps_sharded(shard, world)
    qc0, qck = multi.overlaps_sharded(shard, world, chirality=True)
    sd = multi.schwinger_dyson_sharded(shard, world)
    out.put((rank, shard.calls, gathered.tolist(), shard.swapped_with.tolist(), q0.tolist(), qk.shape, qc0.tolist(), qck.shape, sd[0, 0, :, 0].tolist()))
    multi.barrier()
    import torch.distributed as dist
    dist.destroy_process_group()


def test_two_rank_gloo_temperature_slot_sharding():
    """The PT step of slot-sharded chains: sweeps, publish, ONE all-gather, the same swap call on every
    rank with the same gathered energies in rank order; overlaps: export, sum, cross, sum -- every temperature complete on
    every rank."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_slot_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    expect = [[[[100.0 * w + t for t in range(3)]] * 2] * 2 for w in range(2)]        # [W][S][R][Tl]
    for g in got:
        assert g[1] == ["hb", "or3", "publish", "swap"]
        assert g[2] == expect and g[3] == expect                 # identical gathered energies on both ranks
        assert g[4] == [[[0.0 + 2.0] * 6]] * 2 and g[5] == (2, 1, 6, 3, 2)   # pair (0, 1): 10*0 + (1 + 1) at all six temperatures
        # chirality: own zero-padded export of replica 0 (100) x the summed export of replica 1 (200), complete at every temperature
        assert g[6] == [[[[20000.0] * 3] * 6]] * 2 and g[7] == (2, 1, 6, 3, 3, 2)
        assert g[8] == [1.0, 1.0, 1.0, 2.0, 2.0, 2.0]              # Schwinger-Dyson: every temperature from the rank that holds it
    assert multi.slot_window_of_rank(1, 3, 12) == (4, 4)
    with pytest.raises(ValueError):
        multi.slot_window_of_rank(0, 4, 6)


def test_bench_gpus_n_starts_n_ranks_and_prints_one_line():
    """`python bench.py --gpus 2` outside torchrun must start two ranks itself (the command the round driver
    runs for the scaling record): --check-launch drives exactly that path -- re-exec under torch.distributed.run, rendezvous on
    127.0.0.1, an all-reduce over the ranks (gloo here, nccl on a GPU box), ONE JSON line from rank 0 -- without the workload.
    Without the devices the workload itself must refuse to start rather than run fewer ranks than asked for."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env["CUDA_VISIBLE_DEVICES"] = ""                       # gloo ranks also on a box that has GPUs
    run = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--check-launch"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert run.returncode == 0, run.stderr[-2000:]
    lines = [l for l in run.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, run.stdout
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["asked"] == 2 and out["backend"] == "gloo" and out["rank_sum"] == out["rank_sum_expected"] == 1.0
    run = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert run.returncode != 0 and "refusing to run fewer ranks" in run.stderr and not run.stdout.strip()
    sys.path.insert(0, root)
    import bench
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "3"], 29512)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node" in cmd and cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[-4:] == ["--gpus", "4", "--steps", "3"]
