"""GPU parity of the widened observables: sg_schwinger_dyson (Eq. (A6); end of file) and sg_measure_chiral (Eq. (2)) against the oracle on the same seeded inputs,
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


# ---------------------------------------------------------------------------------------------
# Schwinger-Dyson monitor (Eq. (A6))
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sh", SHAPES)
def test_schwinger_dyson_terms_match_oracle(sg, oracle, sh):
    """Element by element on the same seeded configuration, through a non-trivial permutation.  Tolerance: the
    north star's energy bar, 1e-6 relative to max(1, |value|) (fp32 fields, fp64 sums)."""
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, np.linspace(0.5, 2.0, T), seed=23, gen_mode=2)
    rng = np.random.default_rng(4)
    for s in range(S):
        tos = np.stack([rng.permutation(T) for _ in range(R)]).astype(np.int32)
        gpu.set_perm(s, tos)
        sim.temp_of_slot[s] = tos
        for r in range(R):
            sim.slot_of_temp[s, r, tos[r]] = np.arange(T)
    got, want = gpu.schwinger_dyson(), sim.schwinger_dyson()
    assert np.all(np.abs(got - want) <= 1e-6 * np.maximum(1.0, np.abs(want))), np.abs(got - want).max()


def test_schwinger_dyson_identity_holds_in_equilibrium_on_gpu(sg, oracle):
    """cfg 0 chain on the GPU (HB + OR + PT): the time average of 2 T s.h - (h^2 - (s.h)^2) vanishes within errors at
    every temperature, and does not when the temperature is misassigned by 10 % (power check)."""
    cfg = W.CONFIGS[0]
    K, n_units = 4, 3000
    L, R, T = cfg.L, cfg.n_replicas, cfg.n_temps
    gpu = sg.SpinGlass(L, K, R, T, cfg.betas, seed=5)
    M = oracle.gen_couplings(L, cfg.seed, 0, oracle.OFFDIAG_SYM, cfg.sigma_D).astype(np.float32)
    for k in range(K):
        gpu.init_sample(k, couplings=M)
    rows = []
    for u in range(n_units):
        gpu.unit(cfg.n_or)
        if u >= n_units // 3:
            rows.append(gpu.schwinger_dyson())
    sd = np.array(rows)                                              # [n][K][R][T][2]
    Tt = 1.0 / cfg.betas
    for scale, must_hold in ((1.0, True), (1.1, False)):
        v = 2 * scale * Tt * sd[..., 0] - sd[..., 1]                 # [n][K][R][T]
        nb = 10
        n = (v.shape[0] // nb) * nb
        b = v[:n].reshape(nb, n // nb, K, R, T).mean(axis=1).reshape(nb * K * R, T)
        z = b.mean(axis=0) / (b.std(axis=0, ddof=1) / np.sqrt(b.shape[0]))
        assert (np.abs(z).max() < 4.5) == must_hold, (scale, z)


def test_schwinger_dyson_at_full_size(sg, oracle):
    cfg = W.CONFIGS[4]
    L, R, T = cfg.L, cfg.n_replicas, cfg.n_temps
    C = R * T
    M = oracle.gen_couplings(L, cfg.seed, 0, oracle.OFFDIAG_SYM, cfg.sigma_D)
    X = np.empty((C, 3, L ** 3), dtype=np.float32)
    for c in range(C):
        X[c] = oracle.gen_spins(L, cfg.seed, c)
    gpu = sg.SpinGlass(L, 1, R, T, cfg.betas, seed=cfg.seed)
    gpu.init_sample(0, couplings=M.astype(np.float32), spins=X)
    got = gpu.schwinger_dyson()
    for r, t in [(0, 0), (3, 47), (1, 16), (2, 31)]:
        want = oracle.sd_terms(L, M, X[r * T + t].astype(np.float64))
        assert np.all(np.abs(got[0, r, t] - want) <= 1e-6 * np.maximum(1.0, np.abs(want)))


# ---------------------------------------------------------------------------------------------
# sg_accumulate / sg_get_logbins: logarithmic data binning on the device (Sect. III)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sh", [SHAPES[0], SHAPES[2], dict(L=4, S=2, R=1, T=3)])
def test_logbins_match_oracle(sg, oracle, sh):
    """11 measurements of an evolving chain: the oracle advances (HB + OR + PT), its state is copied to the device
    before every measurement (inputs flow oracle -> CUDA), both sides bin.  Bins 0..3 hold 1, 2, 4, 4 measurements."""
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, np.linspace(0.5, 2.0, T), seed=23)
    for n in range(11):
        sim.unit(1)
        for s in range(S):
            gpu.set_spins(s, sim.spins[s].astype(np.float32))
            gpu.set_perm(s, sim.temp_of_slot[s])
        gpu.accumulate(with_chirality=(n % 2 == 0))         # chirality on every other call: its own count per bin
        sim.accumulate(with_chirality=(n % 2 == 0))
    sums, counts, counts_cg = gpu.get_logbins()
    assert list(counts[:5]) == [1, 2, 4, 4, 0] and np.array_equal(counts, sim.logbin_counts)
    assert list(counts_cg[:5]) == [1, 1, 2, 2, 0] and np.array_equal(counts_cg, sim.logbin_counts_cg)
    scale = np.maximum(1.0, np.abs(sim.logbin_sums))
    assert (np.abs(sums - sim.logbin_sums) <= 4 * TOL * scale).all()          # <= 4 measurements of 1e-6 each per bin
    assert not sums[4:].any()
    if R > 1:
        assert (sums[:4, :, :, 1:4] > 0).all()                               # the comparison is not vacuous
        if L > 2:
            assert (sums[:4, :, :, 4:] > 0).all()
    else:
        assert not sums[..., 1:].any()
    e, _, _ = gpu.measure()                                                    # sg_measure still serves after sg_accumulate
    assert np.abs(e - sim.measure()[0]).max() <= TOL * max(1.0, np.abs(e).max())


# ---------------------------------------------------------------------------------------------
# sg_export_replica / sg_measure_cross: overlaps between replicas held by different contexts (replica sharding)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,S,T", [(4, 1, 4), (6, 2, 10), (8, 2, 16), (10, 1, 37)])
def test_cross_context_overlaps(sg, oracle, L, S, T):
    """Two contexts with replicas (0, 1) and (2, 3) of the same samples, evolved for three units (non-trivial temperature
    permutations): the exported configurations are the spins reordered by temperature, bit for bit; the cross overlaps of
    every pair (a local, b remote) equal the oracle's overlap of the two configurations at that temperature (<= 1e-6) and
    what a single context holding all four replicas measures for the pair (summation order only)."""
    betas = np.linspace(0.5, 2.0, T)
    N = L ** 3
    def make(R, first, total):
        g = sg.SpinGlass(L, S, R, T, betas, seed=31, first_replica=first, n_replicas_total=total)
        for s in range(S):
            g.init_sample(s)
        for _ in range(3):
            g.unit(2)
        return g
    lo, hi, whole = make(2, 0, 4), make(2, 2, 4), make(4, 0, 0)
    _, q0_r, qk_r = whole.measure()                                             # streaming row kernel: fp32 row sums
    whole.tune(sg.TUNE_MEASURE_IMPL, sg.MEASURE_STAGED)
    _, q0_w, qk_w = whole.measure()                                             # staged kernel: fp64 sums of the same products
    assert np.abs(q0_r - q0_w).max() <= 2e-7 and np.abs(qk_r - qk_w).max() <= 2e-7
    pair_index = {(a, b): k for k, (a, b) in enumerate(oracle.replica_pairs(4))}
    spins = {g: [g.get_spins(s).reshape(2, T, 3, N) for s in range(S)] for g in (lo, hi)}
    perms = {g: [g.get_perm(s)[1] for s in range(S)] for g in (lo, hi)}           # slot_of_temp [R][T]
    assert any((perms[g][s] != np.arange(T)).any() for g in (lo, hi) for s in range(S))
    for b in range(2):
        buf = hi.export_replica(b)
        host = buf.cpu().numpy()                                                   # [S][3][N][T]
        for s in range(S):
            want = spins[hi][s][b][perms[hi][s][b]]                                # [T][3][N] by temperature
            assert np.array_equal(host[s], want.transpose(1, 2, 0))
        for a in range(2):
            q0, qk = lo.measure_cross(a, buf)
            k = pair_index[(a, b + 2)]
            assert np.abs(q0 - q0_w[:, k]).max() <= 1e-12 and np.abs(qk - qk_w[:, k]).max() <= 1e-12
            for s in range(S):
                for t in range(0, T, max(1, T // 5)):
                    o = oracle.overlap(L, spins[lo][s][a][perms[lo][s][a][t]].astype(np.float64),
                                       spins[hi][s][b][perms[hi][s][b][t]].astype(np.float64))
                    assert abs(o[0] - q0[s, t]) <= TOL and np.abs(o[1:].reshape(3, 2) - qk[s, t]).max() <= TOL
    for g in (lo, hi, whole):
        g.close()


@pytest.mark.parametrize("L,S,T", [(4, 1, 4), (6, 2, 10), (8, 1, 16)])
def test_cross_context_chiral_overlaps(sg, oracle, L, S, T):
    """sg_export_chirality / sg_chiral_cross between two replica shards against a single four-replica context's
    sg_measure_chiral for the same pair (summation order only) and against the oracle's chiral overlap (<= 1e-6)."""
    betas = np.linspace(0.5, 2.0, T)
    N = L ** 3
    def make(R, first, total):
        g = sg.SpinGlass(L, S, R, T, betas, seed=41, first_replica=first, n_replicas_total=total)
        for s in range(S):
            g.init_sample(s)
        for _ in range(3):
            g.unit(2)
        return g
    lo, hi, whole = make(2, 0, 4), make(2, 2, 4), make(4, 0, 0)
    qc0_w, qck_w = whole.measure_chiral()
    pair_index = {(a, b): k for k, (a, b) in enumerate(oracle.replica_pairs(4))}
    spins = {g: [g.get_spins(s).reshape(2, T, 3, N).astype(np.float64) for s in range(S)] for g in (lo, hi)}
    perms = {g: [g.get_perm(s)[1] for s in range(S)] for g in (lo, hi)}
    for a in range(2):
        za = lo.export_chirality(a)
        for b in range(2):
            zb = hi.export_chirality(b)
            qc0, qck = lo.chiral_cross(za, zb)
            k = pair_index[(a, b + 2)]
            assert np.abs(qc0 - qc0_w[:, k]).max() <= 1e-12 and np.abs(qck - qck_w[:, k]).max() <= 1e-12
            for s in range(S):
                for t in range(0, T, max(1, T // 4)):
                    r0, rk = oracle.chiral_overlap(L, spins[lo][s][a][perms[lo][s][a][t]], spins[hi][s][b][perms[hi][s][b][t]])
                    assert np.abs(r0 - qc0[s, t]).max() <= TOL and np.abs(rk - qck[s, t]).max() <= TOL
    assert np.abs(qc0_w).max() > 1e-4
    for g in (lo, hi, whole):
        g.close()
