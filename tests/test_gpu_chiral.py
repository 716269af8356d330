"""GPU parity of sg_measure_chiral (Eq. (2)) against the oracle on the same seeded inputs,
element by element; tolerance 1e-6 absolute on every q^_CG (fp32 triple products of unit vectors, fp64 sums:
the same bar as the overlap q^ of sg_measure)."""
import numpy as np
import pytest

import sg_workloads as W
from tests.util import make_pair

pytestmark = pytest.mark.gpu

TOL = 1e-6


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_1599_b200 import build
    build.build()
    import paper_1309_1599_b200 as mod
    return mod


SHAPES = [
    dict(L=4, S=1, R=2, T=4),          # cfg 0
    dict(L=2, S=2, R=2, T=3),          # x+e = x-e: every zeta vanishes
    dict(L=6, S=2, R=4, T=10),         # non power of two, padded copy group
    dict(L=10, S=1, R=3, T=11),        # ragged site chunks
    dict(L=8, S=3, R=4, T=16),         # cfg 1 shape
    dict(L=16, S=1, R=4, T=24),        # cfg 2 shape (one sample)
]


@pytest.mark.parametrize("sh", SHAPES)
def test_measure_chiral_matches_oracle(sg, oracle, sh):
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, np.linspace(0.5, 2.0, T), seed=17)
    rng = np.random.default_rng(3)
    for s in range(S):                                   # a non-trivial temperature permutation per chain
        tos = np.stack([rng.permutation(T) for _ in range(R)]).astype(np.int32)
        gpu.set_perm(s, tos)
        sim.temp_of_slot[s] = tos
        for r in range(R):
            sim.slot_of_temp[s, r, tos[r]] = np.arange(T)
    qc0, qck = gpu.measure_chiral()
    r0, rk = sim.measure_chiral()
    assert np.abs(qc0 - r0).max() <= TOL and np.abs(qck - rk).max() <= TOL
    if L == 2:
        assert np.abs(qc0).max() < 1e-12 and np.abs(qck).max() < 1e-12
    else:
        assert np.abs(r0).max() > 1e-4                   # the comparison is not vacuous


def test_measure_chiral_closed_form_on_gpu(sg):
    """Conical spiral along x1 in both replicas (tests/test_oracle_chiral.py): q^_CG^0(0) = zeta^2 with
    zeta = cos a sin^2 a (sin 2 theta - 2 sin theta), everything else 0; opposite handedness flips the sign."""
    L, R, T, a = 8, 2, 2, 0.7
    th = 2 * np.pi / L
    x1 = np.arange(L ** 3) % L
    s = np.stack([np.sin(a) * np.cos(th * x1), np.sin(a) * np.sin(th * x1), np.cos(a) * np.ones(L ** 3)])
    sm = s.copy(); sm[1] = -sm[1]
    gpu = sg.SpinGlass(L, 1, R, T, [0.5, 1.0])
    gpu.init_sample(0, spins=np.stack([s, s, s, sm]).astype(np.float32))   # copies: (r0,t0) (r0,t1) (r1,t0) (r1,t1)
    qc0, qck = gpu.measure_chiral()
    z2 = (np.cos(a) * np.sin(a) ** 2 * (np.sin(2 * th) - 2 * np.sin(th))) ** 2
    assert np.abs(qc0[0, 0, 0] - [z2, 0, 0]).max() < 1e-6 and np.abs(qc0[0, 0, 1] - [-z2, 0, 0]).max() < 1e-6
    assert np.abs(qck).max() < 1e-6


def test_measure_chiral_at_full_size(sg, oracle):
    """cfg 4 shape for one sample (L = 64, 4 x 48 copies), in the launch configuration of the product call:
    sampled (pair, temperature) entries against the oracle; spins drawn by the oracle's generator."""
    cfg = W.CONFIGS[4]
    L, R, T = cfg.L, cfg.n_replicas, cfg.n_temps
    C = R * T
    X = np.empty((C, 3, L ** 3), dtype=np.float32)
    for c in range(C):
        X[c] = oracle.gen_spins(L, cfg.seed, c)
    gpu = sg.SpinGlass(L, 1, R, T, cfg.betas, seed=cfg.seed)
    gpu.init_sample(0, spins=X)
    qc0, qck = gpu.measure_chiral()
    pairs = oracle.replica_pairs(R)
    for p, t in [(0, 0), (5, 47), (2, 13), (3, 31)]:
        a, b = pairs[p]
        r0, rk = oracle.chiral_overlap(L, X[a * T + t].astype(np.float64), X[b * T + t].astype(np.float64))
        assert np.abs(qc0[0, p, t] - r0).max() <= TOL and np.abs(qck[0, p, t] - rk).max() <= TOL


def test_correlation_length_matches_eq4(sg, oracle):
    for L, c0, ck in [(8, 2.0, 1.0), (64, 10.0, 0.3), (16, 1.5, 1.4)]:
        assert abs(sg.correlation_length(L, c0, ck) - oracle.xi(L, c0, ck)) <= 1e-12 * oracle.xi(L, c0, ck)
