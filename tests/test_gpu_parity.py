"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are the north star's: spins after one sweep <= 1e-5 absolute per
component (ill-conditioned sites excluded by the oracle's flags), energy per
spin within 1e-6*max(1,|e|), identical PT decisions on identical energies."""
import numpy as np
import pytest

import sg_workloads as W
from tests.util import gpu_spins, make_pair, neighbour_dilate, oracle_spins

pytestmark = pytest.mark.gpu

SPIN_TOL = 1e-5
MAX_FLAG_FRACTION = 1e-4


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_1599_b200 import build
    build.build()
    import paper_1309_1599_b200 as mod
    return mod


# shapes: cfg 0; the generic (non power-of-two) path with a ragged tile and a padded copy group; L = 2;
# several tiles with a ragged tail (L = 10: 500 sites per colour = 3 tiles of 128 + 116); cfg-1-like
SHAPES = [
    dict(L=4, S=1, R=2, T=4, b=(0.6, 1.6)),
    dict(L=2, S=2, R=2, T=3, b=(0.5, 1.5)),
    dict(L=6, S=2, R=4, T=10, b=(0.5, 2.0)),
    dict(L=10, S=1, R=3, T=11, b=(0.4, 2.4)),
    dict(L=8, S=3, R=4, T=16, b=(0.5, 2.0)),
    dict(L=16, S=1, R=2, T=20, b=(0.5, 2.2)),
    # the same two shapes through the tiled kernel (L = 8, 16 go to the z-marching kernel by default), and the
    # z-marching kernel with several chunks per column, one chunk of all planes, and 3 x 3 tiles (L = 24)
    dict(L=8, S=3, R=4, T=16, b=(0.5, 2.0), tune=((0, 1),)),
    dict(L=16, S=1, R=2, T=20, b=(0.5, 2.2), tune=((0, 1),)),
    dict(L=16, S=2, R=2, T=17, b=(0.5, 2.2), tune=((0, 2), (1, 4))),
    dict(L=16, S=1, R=2, T=17, b=(0.5, 2.2), tune=((0, 2), (1, 16))),
    dict(L=24, S=1, R=2, T=5, b=(0.5, 2.2), tune=((0, 2), (1, 6))),
    # L <= 8 defaults to the shared-memory-resident multi-sweep kernel for the sweep calls: keep the tiled and the
    # z-marching kernels covered there too, and name the resident kernel explicitly once
    dict(L=4, S=1, R=2, T=4, b=(0.6, 1.6), tune=((0, 1),)),
    dict(L=6, S=2, R=4, T=10, b=(0.5, 2.0), tune=((0, 1),)),
    dict(L=8, S=3, R=4, T=16, b=(0.5, 2.0), tune=((0, 2),)),
    dict(L=8, S=3, R=4, T=16, b=(0.5, 2.0), tune=((0, 3),)),
]


def betas_of(sh):
    return np.linspace(sh["b"][0], sh["b"][1], sh["T"])


def colour_mask(L):
    idx = np.arange(L ** 3)
    return (idx % L + (idx // L) % L + idx // (L * L)) % 2


def assert_spins_close(got, want, exclude, what):
    """got, want [S][C][3][N]; exclude [S][C][N] bool."""
    frac = exclude.mean()
    assert frac <= max(MAX_FLAG_FRACTION * 6, 2.0 / exclude.size), (what, "flagged fraction", frac)
    err = np.abs(got - want).max(axis=2)
    err = np.where(exclude, 0.0, err)
    assert err.max() <= SPIN_TOL, (what, err.max(), np.unravel_index(err.argmax(), err.shape))


# ---------------------------------------------------------------------------------------------
# S0
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode,sigma", [(0, 1.0), (0, 2 ** 0.5), (1, 0.5), (2, 1.0), (3, 0.5), (4, 0.0)])
def test_coupling_generator_matches_oracle(sg, oracle, mode, sigma):
    L, S = 6, 2
    gpu = sg.SpinGlass(L, S, 2, 3, [0.5, 1.0, 1.5], seed=12345678901234, first_sample=7)
    for s in range(S):
        gpu.init_sample(s, mode, sigma)
        want = oracle.gen_couplings(L, 12345678901234, 7 + s, mode, sigma)
        got = gpu.get_couplings(s).astype(np.float64)
        # same Philox words, same fp64 formulae, rounded to fp32 on both sides: bit-exact up to the
        # last fp32 bit of libm's last-ulp freedom
        assert np.abs(got - want).max() <= 1.2e-7 * max(1.0, np.abs(want).max())
        assert (got != want).mean() < 1e-3


@pytest.mark.parametrize("sh", SHAPES[:4])
def test_initial_spins_match_oracle(sg, oracle, sh):
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    gpu = sg.SpinGlass(L, S, R, T, betas_of(sh), seed=99, first_sample=3)
    for s in range(S):
        gpu.init_sample(s)
        got = gpu.get_spins(s).astype(np.float64)
        want = np.stack([oracle.gen_spins(L, 99, (3 + s) * R * T + c) for c in range(R * T)])
        assert np.abs(got - want).max() <= 5e-7
        tos, sot = gpu.get_perm(s)
        assert np.array_equal(tos, np.tile(np.arange(T), (R, 1))) and np.array_equal(sot, tos)


@pytest.mark.parametrize("sh", SHAPES)
def test_set_get_spins_roundtrip(sg, sh):
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    rng = np.random.default_rng(L)
    gpu = sg.SpinGlass(L, S, R, T, betas_of(sh))
    data = [W.random_spins(rng, R * T, L ** 3).astype(np.float32) for _ in range(S)]
    for s in range(S):
        gpu.init_sample(s, spins=data[s])
    for s in range(S):
        assert np.array_equal(gpu.get_spins(s), data[s])
    gpu.set_spins(0, data[-1])
    assert np.array_equal(gpu.get_spins(0), data[-1])


# ---------------------------------------------------------------------------------------------
# S1, S2: half-sweeps and sweeps, element by element
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sh", SHAPES)
@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("gen_mode", [0, 2])
def test_half_sweeps_match_oracle(sg, oracle, sh, kind, gen_mode):
    """Each colour separately, each compared from the oracle's state (no error propagation)."""
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=5, gen_mode=gen_mode, tune=sh.get("tune"))
    sim.hb_counter = 17
    gpu.set_counters(17, 0)
    col = colour_mask(L)
    for colour in (0, 1):
        before = oracle_spins(sim)
        for s in range(S):
            gpu.set_spins(s, sim.spins[s].astype(np.float32))      # restart from the oracle's state
        flags = sim.halfsweep(kind, colour, want_flags=True)
        gpu.halfsweep(kind, colour)
        got, want = gpu_spins(gpu), oracle_spins(sim)
        assert_spins_close(got, want, flags != 0, ("half", kind, colour))
        other = col != colour
        assert np.array_equal(got[..., other], before[..., other])       # the other colour is untouched
        assert np.abs(want[..., ~other] - before[..., ~other]).max() > 0.1
    assert gpu.get_counters() == (17, 0)


def sweep_both(sim, gpu, kind, L):
    """One full sweep (the product's sg_sweep_* call) on both sides from identical states, checked twice
    (DESIGN.md section 6).

    (a) Composition, no error propagation: the colour-0 sites of the GPU result are the output of its
        first half-sweep (the second one does not touch them) and are compared with the oracle's first
        half-sweep; the oracle's second half-sweep is then run *from the GPU's colour-0 values* and
        compared on the colour-1 sites.  Both at SPIN_TOL with the oracle's ill-conditioning flags.
    (b) Directly against the oracle's own full sweep.  The second colour inherits the first colour's
        fp32 rounding, amplified by 2|A|/|h|: every site must lie within SPIN_TOL plus the propagated
        term, which the oracle itself supplies (its second half-sweep from the two first-colour states),
        and all but a fraction <= 5e-4 of the unflagged sites within the plain SPIN_TOL.
    Leaves sim at the oracle's own full-sweep result."""
    S = sim.S
    col = colour_mask(L)
    start = [sim.spins[s].copy() for s in range(S)]
    if kind == 1:
        gpu.sweep_hb(1)
    else:
        gpu.sweep_or(1)
    got = gpu_spins(gpu)
    # (a) first colour
    f0 = sim.halfsweep(kind, 0, want_flags=True)
    want0 = oracle_spins(sim)
    assert_spins_close(got[..., col == 0], want0[..., col == 0], (f0 != 0)[..., col == 0], ("compose", kind, 0))
    # (a) second colour, from the GPU's first-colour output
    for s in range(S):
        sim.spins[s] = np.where(col == 0, got[s], start[s])
    fa = sim.halfsweep(kind, 1, want_flags=True)
    wanta = oracle_spins(sim)
    assert np.array_equal(wanta[..., col == 0], got[..., col == 0])
    assert_spins_close(got[..., col == 1], wanta[..., col == 1], (fa != 0)[..., col == 1], ("compose", kind, 1))
    # (b) the oracle's own sweep
    for s in range(S):
        sim.spins[s] = want0[s].copy()
    f1 = sim.halfsweep(kind, 1, want_flags=True)
    if kind == 1:
        sim.hb_counter += 1
    want = oracle_spins(sim)
    exclude = (f0 != 0) | (f1 != 0) | (fa != 0) | neighbour_dilate(f0 != 0, L)
    assert exclude.mean() <= max(1e-3, 2.0 / exclude.size), ("excluded fraction", exclude.mean())
    err = np.where(exclude, 0.0, np.abs(got - want).max(axis=2))
    propagated = np.abs(wanta - want).max(axis=2)
    assert np.all(err <= SPIN_TOL + 1.01 * propagated), ("sweep", kind, (err - propagated).max())
    assert np.mean(err > SPIN_TOL) <= max(5e-4, 2.0 / err.size), ("sweep", kind, np.mean(err > SPIN_TOL))
    assert np.median(np.abs(got - want)) <= 5e-7 and err.max() <= 1e-3, ("sweep", kind, err.max())


@pytest.mark.parametrize("sh", SHAPES)
@pytest.mark.parametrize("kind", [0, 1])
def test_full_sweep_matches_oracle(sg, oracle, sh, kind):
    """north_star: spins after one sweep within 1e-5 absolute per component; energy per spin within 1e-6."""
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    N = L ** 3
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=6, tune=sh.get("tune"))
    sweep_both(sim, gpu, kind, L)
    # fused energy of the sweep's last half-sweep against Eq. (1) on the oracle's spins
    e_gpu, e_ref = gpu.get_energies() / N, sim.energies() / N
    assert np.all(np.abs(e_gpu - e_ref) <= 1e-6 * np.maximum(1.0, np.abs(e_ref)))
    assert gpu.get_counters()[0] == (1 if kind == 1 else 0)


def test_or_conserves_energy_and_norm_on_gpu(sg, oracle):
    sh = SHAPES[4]
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    N = L ** 3
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=8, tune=sh.get("tune"))
    e0 = gpu.get_energies() / N                   # standalone energy kernel
    assert np.all(np.abs(e0 - sim.energies() / N) <= 1e-6 * np.maximum(1.0, np.abs(e0)))
    gpu.sweep_or(8)
    e1 = gpu.get_energies() / N                   # fused into the last half-sweep
    assert np.abs(e1 - e0).max() < 2e-5           # fp32 reflections: drift ~ sqrt(sweeps) * 1e-7 * |h|
    s = gpu_spins(gpu)
    assert np.abs(np.sum(s * s, axis=2) - 1.0).max() < 2e-5
    for smp in range(S):                          # fused vs standalone reduction on the same state
        gpu.set_spins(smp, gpu.get_spins(smp))
    e2 = gpu.get_energies() / N
    assert np.abs(e2 - e1).max() < 1e-6


def test_time_reversal_and_involution_on_gpu(sg, oracle):
    sh = SHAPES[2]
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=9, gen_mode=2, tune=sh.get("tune"))
    s0 = gpu_spins(gpu)
    gpu.halfsweep(0, 0)
    s1 = gpu_spins(gpu)
    gpu.halfsweep(0, 0)
    assert np.abs(gpu_spins(gpu) - s0).max() < 5e-5       # reflection twice = identity (up to fp32; small |h| sites)
    for s in range(S):
        gpu.set_spins(s, (-s0[s]).astype(np.float32))
    gpu.halfsweep(0, 0)
    assert np.array_equal(gpu_spins(gpu), -s1)            # OR(-s) = -OR(s) exactly


# ---------------------------------------------------------------------------------------------
# S3, S5: energies and overlaps
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sh", SHAPES)
@pytest.mark.parametrize("staged", [False, True])
def test_measure_matches_oracle(sg, oracle, sh, staged):
    """Both overlap kernels: the streaming row kernel (default for R <= 4) and the staged one (any R)."""
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=10, tune=sh.get("tune"))
    gpu.tune(sg.TUNE_MEASURE_IMPL, sg.MEASURE_STAGED if staged else sg.MEASURE_AUTO)
    rng = np.random.default_rng(3)
    for s in range(S):                                    # a non-trivial temperature assignment
        tos = np.stack([rng.permutation(T) for _ in range(R)]).astype(np.int32)
        gpu.set_perm(s, tos)
        sim.temp_of_slot[s] = tos
        sim.slot_of_temp[s] = np.argsort(tos, axis=1).astype(np.int32)
        got_tos, got_sot = gpu.get_perm(s)
        assert np.array_equal(got_tos, tos) and np.array_equal(got_sot, sim.slot_of_temp[s])
    e, q0, qk = gpu.measure()
    e_ref, q0_ref, qk_ref = sim.measure()
    assert np.all(np.abs(e - e_ref) <= 1e-6 * np.maximum(1.0, np.abs(e_ref)))
    assert np.abs(q0 - q0_ref).max() <= 1e-6 and np.abs(qk - qk_ref).max() <= 1e-6


def test_measure_five_replicas_and_many_temperatures(sg, oracle):
    """R = 5 (ten pairs: the staged kernel serves R > 4) and T = 300 > 256 (the row kernel tiles the temperatures)."""
    for L, S, R, T in ((4, 1, 5, 3), (4, 1, 2, 300)):
        betas = np.linspace(0.5, 1.5, T)
        sim, gpu = make_pair(oracle, sg, L, S, R, T, betas, seed=14)
        rng = np.random.default_rng(8)
        tos = np.stack([rng.permutation(T) for _ in range(R)]).astype(np.int32)
        gpu.set_perm(0, tos)
        sim.temp_of_slot[0] = tos
        sim.slot_of_temp[0] = np.argsort(tos, axis=1).astype(np.int32)
        e, q0, qk = gpu.measure()
        e_ref, q0_ref, qk_ref = sim.measure()
        assert np.all(np.abs(e - e_ref) <= 1e-6 * np.maximum(1.0, np.abs(e_ref)))
        assert np.abs(q0 - q0_ref).max() <= 1e-6 and np.abs(qk - qk_ref).max() <= 1e-6


def test_measure_closed_forms_on_gpu(sg):
    """Identical replicas: q(0) = 1, q(k) = 0; a cosine modulation along x_mu: q(k_mu) = 1/2."""
    L, R, T = 8, 2, 2
    N = L ** 3
    rng = np.random.default_rng(4)
    gpu = sg.SpinGlass(L, 1, R, T, [0.5, 1.0])
    idx = np.arange(N)
    coords = [idx % L, (idx // L) % L, idx // (L * L)]
    base = W.random_spins(rng, 1, N)[0]
    spins = np.zeros((R * T, 3, N))
    spins[0] = base; spins[2] = base                       # replica 0 and 1 at temperature 0: identical
    spins[1, 2] = 1.0                                      # temperature 1: z^ against a modulation along x2
    th = 2 * np.pi * coords[1] / L
    spins[3, 0] = np.sin(th); spins[3, 2] = np.cos(th)
    gpu.init_sample(0, couplings=np.zeros((3, N, 3, 3)), spins=spins)
    e, q0, qk = gpu.measure()
    assert np.all(e == 0)
    assert abs(q0[0, 0, 0] - 1) < 1e-6 and np.abs(qk[0, 0, 0]).max() < 1e-6
    want = np.zeros((3, 2)); want[1, 0] = 0.5
    assert abs(q0[0, 0, 1]) < 1e-6 and np.abs(qk[0, 0, 1] - want).max() < 1e-6


def test_ferromagnet_energy_on_gpu(sg):
    """The paper's own cross-check: ferromagnetic couplings, exact energies."""
    L = 8
    N = L ** 3
    gpu = sg.SpinGlass(L, 1, 1, 2, [0.5, 1.0])
    spins = np.zeros((2, 3, N))
    spins[0, 1] = 1.0
    idx = np.arange(N)
    spins[1, 2] = 1.0 - 2.0 * ((idx % L + (idx // L) % L + idx // (L * L)) % 2)
    gpu.init_sample(0, sg.GEN_FERRO, 0.0, spins=spins)
    E = gpu.get_energies()[0] / N
    assert E[0] == -3.0 and E[1] == 3.0


# ---------------------------------------------------------------------------------------------
# S4: parallel tempering
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sh", [SHAPES[0], SHAPES[2], SHAPES[4]])
def test_pt_decisions_identical_on_identical_energies(sg, oracle, sh):
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=11, first_sample=2, tune=sh.get("tune"))
    rng = np.random.default_rng(5)
    for k in range(40):
        # energies spaced so that acceptance is neither 0 nor 1
        E = rng.normal(0.0, 3.0 / (betas_of(sh)[1] - betas_of(sh)[0]) / 4, size=(S, R * T))
        gpu.set_energies(E)
        gpu.pt_swap()
        sim.pt_swap(energies=E)
        for s in range(S):
            tos, sot = gpu.get_perm(s)
            assert np.array_equal(tos, sim.temp_of_slot[s]) and np.array_equal(sot, sim.slot_of_temp[s]), k
    att, acc = gpu.pt_stats()
    assert np.array_equal(att, sim.attempts) and np.array_equal(acc, sim.accepts)
    assert 0 < acc.sum() < att.sum()
    assert gpu.get_counters() == (0, 40)


@pytest.mark.parametrize("sh", [SHAPES[0], SHAPES[2]])
def test_pt_random_walk_in_temperature_bit_exact(sg, oracle, sh):
    """Round-trip bookkeeping of the walk in temperature against the oracle, sweep by sweep: integer work."""
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=13, first_sample=1, tune=sh.get("tune"))
    rng = np.random.default_rng(6)
    trips0, lab0 = gpu.pt_walk()
    assert trips0.sum() == 0 and not lab0.any()
    for k in range(60 * T):
        E = rng.normal(0.0, 0.5 / abs(betas_of(sh)[1] - betas_of(sh)[0]), size=(S, R * T))   # acceptance well above 1/2
        gpu.set_energies(E); gpu.pt_swap(); sim.pt_swap(energies=E)
        if k % 37 == 0 or k == 60 * T - 1:
            trips, lab = gpu.pt_walk()
            assert np.array_equal(trips, sim.round_trips[..., 0]) and np.array_equal(lab, sim.walk_label), k
    assert trips.sum() > 0 and set(np.unique(lab)) <= {0, 1, 2}


def test_pt_moves_temperatures_not_spins_and_hb_follows(sg, oracle):
    """After PT the heat bath must use each slot's *new* temperature (beta by slot follows the swap)."""
    sh = SHAPES[0]
    L, S, R, T = sh["L"], sh["S"], sh["R"], sh["T"]
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas_of(sh), seed=12, tune=sh.get("tune"))
    before = gpu_spins(gpu)
    E = np.array([[0.0, -50.0, -20.0, -90.0, 5.0, 1.0, -3.0, 2.0]])     # forces some swaps
    gpu.set_energies(E); gpu.pt_swap(); sim.pt_swap(energies=E)
    assert np.array_equal(gpu_spins(gpu), before)
    tos, _ = gpu.get_perm(0)
    assert np.array_equal(tos, sim.temp_of_slot[0]) and not np.array_equal(tos, np.tile(np.arange(T), (R, 1)))
    f0 = sim.halfsweep(1, 0, want_flags=True)
    gpu.halfsweep(1, 0)
    assert_spins_close(gpu_spins(gpu), oracle_spins(sim), f0 != 0, "hb after pt")


def test_unit_sequence_with_resync(sg, oracle):
    """Three units of cfg 0 (1 HB + 4 OR + PT): every sweep is compared from the oracle's state, PT is
    compared on the GPU's own energies (decisions may differ only at a near-tie)."""
    cfg = W.CONFIGS[0]
    L, S, R, T = cfg.L, cfg.n_samples, cfg.n_replicas, cfg.n_temps
    sim, gpu = make_pair(oracle, sg, L, S, R, T, cfg.betas, seed=cfg.seed)
    N = L ** 3
    for unit in range(3):
        for kind, n in ((1, 1), (0, cfg.n_or)):
            for _ in range(n):
                for s in range(S):
                    gpu.set_spins(s, sim.spins[s].astype(np.float32))
                sweep_both(sim, gpu, kind, L)
        E_gpu, E_ref = gpu.get_energies(), sim.energies()
        assert np.all(np.abs(E_gpu - E_ref) / N <= 1e-6 * np.maximum(1.0, np.abs(E_ref) / N))
        gpu.pt_swap()
        sim.pt_swap(energies=E_gpu)              # same energies -> the decisions must be identical
        tos, sot = gpu.get_perm(0)
        assert np.array_equal(tos, sim.temp_of_slot[0])
        assert gpu.get_counters() == (sim.hb_counter, sim.pt_counter)


def test_sharded_samples_draw_the_single_process_numbers(sg, oracle):
    """first_sample shifts every Philox counter: a context holding samples [2,4) reproduces samples 2, 3 of
    a context holding [0,4) (weak-scaling shard by sample)."""
    L, R, T = 4, 2, 4
    betas = np.linspace(0.6, 1.6, T)
    full = sg.SpinGlass(L, 4, R, T, betas, seed=21)
    part = sg.SpinGlass(L, 2, R, T, betas, seed=21, first_sample=2)
    for s in range(4):
        full.init_sample(s)
    for s in range(2):
        part.init_sample(s)
    for g in (full, part):
        g.unit(3); g.unit(3)
    for s in range(2):
        assert np.array_equal(part.get_couplings(s), full.get_couplings(2 + s))
        assert np.array_equal(part.get_spins(s), full.get_spins(2 + s))
        assert np.array_equal(part.get_perm(s)[0], full.get_perm(2 + s)[0])
    assert np.array_equal(part.get_energies(), full.get_energies()[2:])


def test_errors_on_gpu(sg):
    gpu = sg.SpinGlass(4, 2, 2, 4, np.linspace(0.6, 1.6, 4))
    gpu.init_sample(0)
    with pytest.raises(sg.SgError) as ei:
        gpu.sweep_or(1)                          # sample 1 not initialised
    assert ei.value.code == -2
    with pytest.raises(sg.SgError):
        gpu.init_sample(5)
    with pytest.raises(sg.SgError):
        gpu.set_perm(0, np.zeros((2, 4), dtype=np.int32))
    gpu.init_sample(1)
    n0 = gpu.kernel_launches()
    gpu.sweep_or(2)
    assert gpu.kernel_launches() == n0 + 1       # L = 4: the resident kernel runs both sweeps and the energies in one launch
    gpu.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_TILED)
    gpu.sweep_or(2)
    assert gpu.kernel_launches() == n0 + 6       # 4 half-sweeps + 1 energy reduction
    with pytest.raises(sg.SgError):
        sg.SpinGlass(32, 1, 2, 4, np.linspace(0.6, 1.6, 4)).tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_RESIDENT)   # 1.5 MB for 4 copies


@pytest.mark.parametrize("L,S,R,T", [(2, 2, 2, 3), (4, 1, 2, 4), (6, 2, 4, 10), (8, 3, 4, 16), (8, 8, 4, 16), (10, 1, 3, 11), (16, 1, 2, 20)])
def test_resident_kernel_is_bit_identical_to_the_per_half_sweep_kernels(sg, L, S, R, T):
    """Same seeded start, one unit sequence (2 HB sweeps, 5 OR sweeps) through the resident multi-sweep kernel and
    through the tiled kernel (and the z-marching kernel for L = 8): the spins must agree bit for bit (same arithmetic,
    same order), the fused energies to summation-order rounding, the HB counter must advance alike."""
    betas = np.linspace(0.5, 2.0, T)
    # (kernel, copies per CTA of the resident kernel): every CTA shape of the resident kernel against the other two
    impls = [(sg.SWEEP_TILED, 0), (sg.SWEEP_RESIDENT, 0)] + ([(sg.SWEEP_ZMARCH, 0)] if L % 8 == 0 else []) + \
            [(sg.SWEEP_RESIDENT, c) for c in (4, 8, 16, 32) if L ** 3 * 12 * c <= 200 * 1024]
    out = []
    for impl, cpc in impls:
        gpu = sg.SpinGlass(L, S, R, T, betas, seed=11)
        gpu.tune(sg.TUNE_SWEEP_IMPL, impl)
        if cpc:
            gpu.tune(sg.TUNE_RES_COPIES, cpc)
        for s in range(S):
            gpu.init_sample(s, sg.GEN_GENERAL9, 1.0)
        gpu.sweep_hb(2); gpu.sweep_or(5)
        E = gpu.get_energies()
        gpu.pt_swap(); gpu.sweep_hb(1); gpu.sweep_or(1)          # beta follows the permutation in the next call
        out.append((np.stack([gpu.get_spins(s) for s in range(S)]), E, gpu.get_counters(), gpu.get_energies()))
        gpu.close()
    for spins, E, ctr, E2 in out[1:]:
        assert ctr == out[0][2]
        assert np.abs(E - out[0][1]).max() <= 1e-6 * max(1.0, np.abs(E).max())
        # identical energies up to rounding may still flip a PT decision at a near-tie; compare the pre-PT part strictly
        if np.array_equal(spins, out[0][0]):
            assert np.abs(E2 - out[0][3]).max() <= 1e-6 * max(1.0, np.abs(E2).max())
    # the strict part: state before the PT step
    ref = None
    for impl, cpc in impls:
        gpu = sg.SpinGlass(L, S, R, T, betas, seed=11)
        gpu.tune(sg.TUNE_SWEEP_IMPL, impl)
        if cpc:
            gpu.tune(sg.TUNE_RES_COPIES, cpc)
        for s in range(S):
            gpu.init_sample(s, sg.GEN_GENERAL9, 1.0)
        gpu.sweep_hb(2); gpu.sweep_or(5)
        spins = np.stack([gpu.get_spins(s) for s in range(S)])
        gpu.close()
        if ref is None:
            ref = spins
        else:
            assert np.array_equal(spins, ref), (impl, cpc)


@pytest.mark.parametrize("L,S,R,T,n_units,own_stream", [(6, 2, 2, 6, 7, False), (6, 2, 2, 6, 25, False), (8, 3, 4, 16, 30, True), (4, 1, 2, 4, 40, True),
                                                    (16, 1, 2, 8, 12, True)])
def test_run_units_equals_the_three_calls(sg, L, S, R, T, n_units, own_stream):
    """sg_run_units(n, n_or) = n x (sg_sweep_hb(1); sg_sweep_or(n_or); sg_pt_swap()), bit for bit -- issued one by one
    (n < 8, L = 16, SG_TUNE_GRAPH = 0) or as replays of one captured unit with patched sweep counters (CUDA graph; on the
    caller's stream, or on the library's own when the caller's is the legacy default stream)."""
    import torch
    betas = np.linspace(0.5, 1.8, T)
    stream = torch.cuda.Stream() if own_stream else None
    a = sg.SpinGlass(L, S, R, T, betas, seed=4, stream=stream); b = sg.SpinGlass(L, S, R, T, betas, seed=4, stream=stream)
    c = sg.SpinGlass(L, S, R, T, betas, seed=4, stream=stream)
    c.tune(sg.TUNE_GRAPH, 0)
    for g in (a, b, c):
        for s in range(S):
            g.init_sample(s)
    for _ in range(n_units):
        a.unit(3)
    b.run_units(n_units, 3)
    c.run_units(n_units, 3)
    b.run_units(9, 0); c.run_units(9, 0)          # a second capture on the same context, n_or = 0
    for _ in range(9):
        a.unit(0)
    assert b.kernel_launches() == c.kernel_launches()      # replays count the launches of the captured unit
    for g in (b, c):
        for s in range(S):
            assert np.array_equal(a.get_spins(s), g.get_spins(s))
            assert np.array_equal(a.get_perm(s)[0], g.get_perm(s)[0])
        assert np.array_equal(a.get_energies(), g.get_energies()) and a.get_counters() == g.get_counters() == (n_units + 9, n_units + 9)
        assert np.array_equal(a.pt_stats()[1], g.pt_stats()[1]) and np.array_equal(a.pt_visits(), g.pt_visits())


@pytest.mark.parametrize("L,S,T,impl", [(8, 2, 5, 2), (6, 1, 7, 1), (4, 2, 4, 0), (16, 1, 20, 0)])
def test_replica_shards_draw_the_single_context_numbers(sg, L, S, T, impl):
    """sg_shape.first_replica / n_replicas_total: two contexts holding replicas (0, 1) and (2, 3) of every sample against
    one context holding all four: initial spins, three units (HB draws by global copy id, PT by global chain id), spins,
    permutations, energies and PT statistics of every replica identical bit for bit; overlaps of the local pairs too."""
    betas = np.linspace(0.5, 2.0, T)
    def run(R, first_replica, total):
        gpu = sg.SpinGlass(L, S, R, T, betas, seed=77, first_sample=3, first_replica=first_replica, n_replicas_total=total)
        gpu.tune(sg.TUNE_SWEEP_IMPL, impl)
        for s in range(S):
            gpu.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
        start = np.stack([gpu.get_spins(s) for s in range(S)])
        for _ in range(3):
            gpu.unit(2)
        e, q0, qk = gpu.measure()
        out = dict(start=start.reshape(S, R, T, 3, -1), spins=np.stack([gpu.get_spins(s) for s in range(S)]).reshape(S, R, T, 3, -1),
                   perm=np.stack([gpu.get_perm(s)[0] for s in range(S)]), E=gpu.get_energies().reshape(S, R, T),
                   acc=gpu.pt_stats()[1], e=e, q0=q0)
        gpu.close()
        return out
    whole = run(4, 0, 0)
    lo, hi = run(2, 0, 4), run(2, 2, 4)
    for key in ("start", "spins", "perm", "E", "acc", "e"):
        assert np.array_equal(whole[key][:, 0:2], lo[key]), key
        assert np.array_equal(whole[key][:, 2:4], hi[key]), key
    # pairs in the order (0,1),(0,2),(0,3),(1,2),(1,3),(2,3): the shards hold the first and the last
    assert np.array_equal(whole["q0"][:, 0], lo["q0"][:, 0]) and np.array_equal(whole["q0"][:, 5], hi["q0"][:, 0])
    assert whole["acc"].sum() > 0


@pytest.mark.parametrize("L,S,R,T,impl", [(8, 2, 2, 6, 2), (6, 2, 3, 5, 1), (4, 1, 2, 4, 0)])
def test_checkpoint_resume_is_bit_exact(sg, L, S, R, T, impl):
    """Philox is counter-based, so the chain's state is (couplings, spins, temperature permutation, HB and PT counters):
    a second context restored from those through the state hooks continues exactly as the first one does."""
    betas = np.linspace(0.5, 2.0, T)
    a = sg.SpinGlass(L, S, R, T, betas, seed=5, first_sample=2)
    a.tune(sg.TUNE_SWEEP_IMPL, impl)
    for s in range(S):
        a.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
    for _ in range(3):
        a.unit(3)
    snap = dict(M=[a.get_couplings(s) for s in range(S)], spins=[a.get_spins(s) for s in range(S)],
                perm=[a.get_perm(s)[0] for s in range(S)], ctr=a.get_counters())
    assert snap["ctr"] == (3, 3)
    for _ in range(3):
        a.unit(3)
    b = sg.SpinGlass(L, S, R, T, betas, seed=5, first_sample=2)
    b.tune(sg.TUNE_SWEEP_IMPL, impl)
    for s in range(S):
        b.init_sample(s, couplings=snap["M"][s], spins=snap["spins"][s])
        b.set_perm(s, snap["perm"][s])
    b.set_counters(*snap["ctr"])
    for _ in range(3):
        b.unit(3)
    assert a.get_counters() == b.get_counters() == (6, 6)
    for s in range(S):
        assert np.array_equal(a.get_spins(s), b.get_spins(s))
        assert np.array_equal(a.get_perm(s)[0], b.get_perm(s)[0]) and np.array_equal(a.get_perm(s)[1], b.get_perm(s)[1])
    assert np.array_equal(a.get_energies(), b.get_energies())


@pytest.mark.parametrize("L,S,R,T,W,impl", [(8, 2, 2, 8, 2, 2), (6, 1, 3, 6, 3, 1), (4, 2, 2, 4, 4, 0), (8, 1, 4, 12, 2, 0)])
def test_temperature_slot_shards_reproduce_the_single_context(sg, L, S, R, T, W, impl):
    """sg_shape.first_slot / n_temps_total (the paper's multi-GPU mode): W contexts on one GPU, each
    holding T/W consecutive slots of every chain, against one context holding whole chains, over 50 units: initial spins,
    spins, the whole temperature assignment, energies, PT statistics, round trips and the visit histogram identical bit for
    bit (heat bath keyed by global copy id; the PT kernel runs on the all-gathered energies with the same counters on every
    shard), and the overlaps assembled across the shards equal the single context's sg_measure."""
    import torch
    from paper_1309_1599_b200 import multi
    betas = np.linspace(0.5, 1.6, T)
    Tl, n_or, units = T // W, 2, 50
    whole = sg.SpinGlass(L, S, R, T, betas, seed=91, first_sample=2)
    shards = [sg.SpinGlass(L, S, R, Tl, betas, seed=91, first_sample=2, first_slot=w * Tl, n_temps_total=T) for w in range(W)]
    for g in [whole] + shards:
        g.tune(sg.TUNE_SWEEP_IMPL, impl)
        for s in range(S):
            g.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
    def shard_spins(s):
        parts = [g.get_spins(s).reshape(R, Tl, 3, -1) for g in shards]
        return np.concatenate(parts, axis=1).reshape(R * T, 3, -1)
    for s in range(S):
        assert np.array_equal(whole.get_spins(s), shard_spins(s)), "initial spins"
    gathered = torch.empty((W, S, R, Tl), dtype=torch.float64, device="cuda")
    for u in range(units):
        whole.unit(n_or)
        for w, g in enumerate(shards):
            g.sweep_hb(1); g.sweep_or(n_or)
            g.pt_publish(out=gathered[w])
        torch.cuda.synchronize()
        for g in shards:
            g.pt_swap_gathered(gathered)
    E = whole.get_energies().reshape(S, R, T)
    for s in range(S):
        assert np.array_equal(whole.get_spins(s), shard_spins(s)), "spins"
        for g in shards:
            assert np.array_equal(whole.get_perm(s)[0], g.get_perm(s)[0]) and np.array_equal(whole.get_perm(s)[1], g.get_perm(s)[1])
    for w, g in enumerate(shards):
        assert np.array_equal(E[:, :, w * Tl:(w + 1) * Tl], g.get_energies().reshape(S, R, Tl))
        assert np.array_equal(whole.pt_stats()[0], g.pt_stats()[0]) and np.array_equal(whole.pt_stats()[1], g.pt_stats()[1])
        assert np.array_equal(whole.pt_walk()[0], g.pt_walk()[0]) and np.array_equal(whole.pt_walk()[1], g.pt_walk()[1])
        assert np.array_equal(whole.pt_visits(), g.pt_visits())
        with pytest.raises(sg.SgError):
            g.pt_swap()
        with pytest.raises(sg.SgError):
            g.measure()
    assert whole.pt_stats()[1].sum() > 0 and whole.pt_visits().sum() == S * R * T * units
    # measurement across the shards: e by temperature from the gathered energies, overlaps by export / sum / cross / sum
    whole.tune(sg.TUNE_MEASURE_IMPL, sg.MEASURE_STAGED)      # fp64 sums per site, as sg_measure_cross forms them
    e, q0, qk = whole.measure()
    for w, g in enumerate(shards):
        g.pt_publish(out=gathered[w])
    torch.cuda.synchronize()
    assert np.array_equal(shards[0].energy_by_temp(gathered), e)
    pairs = [(a, b) for a in range(R) for b in range(a + 1, R)]
    for p, (a, b) in enumerate(pairs):
        full = sum(g.export_replica(b) for g in shards)
        parts = [g.measure_cross(a, full) for g in shards]
        q0_x = sum(pp[0] for pp in parts); qk_x = sum(pp[1] for pp in parts)
        assert np.abs(q0_x - q0[:, p]).max() <= 1e-12 and np.abs(qk_x - qk[:, p]).max() <= 1e-12
        # every temperature is held by exactly one shard: the other shards contribute exact zeros
        assert all(((pp[0] == 0) | (pp[0] == q0_x)).all() for pp in parts)
    # the chiral-glass overlaps across the shards the same way (Eq. (2); measured by the paper on the runs it sharded by
    # temperature): zero-padded zeta exports, their sum, each shard's own export against it, sum of the shards' results
    qc0, qck = whole.measure_chiral()
    for p, (a, b) in enumerate(pairs):
        full = sum(g.export_chirality(b) for g in shards)
        parts = [g.chiral_cross(g.export_chirality(a), full) for g in shards]
        qc0_x = sum(pp[0] for pp in parts); qck_x = sum(pp[1] for pp in parts)
        assert qc0_x.shape == qc0[:, p].shape
        assert np.abs(qc0_x - qc0[:, p]).max() <= 1e-12 and np.abs(qck_x - qck[:, p]).max() <= 1e-12
        assert all(((pp[0] == 0) | (pp[0] == qc0_x)).all() for pp in parts)
    if L > 2:
        assert np.abs(qc0).max() > 1e-5
    # Schwinger-Dyson monitor (Eq. (A6)): each shard reports the temperatures it holds, zeros elsewhere; their sum is the whole chain's
    sd_w = whole.schwinger_dyson()
    sd_parts = [g.schwinger_dyson() for g in shards]
    assert sd_parts[0].shape == sd_w.shape and np.abs(sum(sd_parts) - sd_w).max() <= 1e-12
    assert all(((pp == 0) | (pp == sd_w)).all() for pp in sd_parts) and np.abs(sd_w).min() > 0
    # one shard alone through the orchestration (world size 1 path of multi.pt_step_sharded on a whole-chain context)
    solo = sg.SpinGlass(L, S, R, T, betas, seed=91, first_sample=2)
    solo.tune(sg.TUNE_SWEEP_IMPL, impl)
    ref = sg.SpinGlass(L, S, R, T, betas, seed=91, first_sample=2)
    ref.tune(sg.TUNE_SWEEP_IMPL, impl)
    for g in (solo, ref):
        for s in range(S):
            g.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
    for _ in range(3):
        multi.unit_sharded(solo, n_or, 1)
        ref.unit(n_or)
    for s in range(S):
        assert np.array_equal(solo.get_spins(s), ref.get_spins(s)) and np.array_equal(solo.get_perm(s)[0], ref.get_perm(s)[0])
    for g in [whole, solo, ref] + shards:
        g.close()


def test_pt_visit_histogram_and_tau_int_match_oracle(sg, oracle):
    """sg_pt_visits is the oracle's visit histogram bit for bit (fed the oracle's energies), and sg_walk_tau_int of a
    recorded walk in temperature equals the oracle's estimator."""
    L, S, R, T = 4, 2, 2, 6
    betas = np.linspace(0.4, 1.2, T)
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas, seed=12)
    series = []
    for _ in range(300):
        sim.sweep_hb(1)
        E = sim.energies()
        gpu.set_energies(E)
        sim.pt_swap(energies=E)
        gpu.pt_swap()
        series.append(gpu.get_perm(0)[0][0, 0])
    assert np.array_equal(gpu.pt_visits(), sim.visits) and sim.visits.sum() == S * R * T * 300
    assert np.array_equal(gpu.pt_walk()[0], sim.round_trips[..., 0])
    for c in (6.0, 3.0):
        assert sg.walk_tau_int(series, c) == pytest.approx(oracle.walk_tau_int(series, c), rel=1e-12)
    assert len(set(series)) > 2


@pytest.mark.parametrize("L,S,R,T,zc", [(8, 2, 2, 5, 0), (8, 1, 1, 3, 4), (16, 2, 4, 12, 0), (16, 1, 2, 20, 8), (24, 1, 2, 16, 0), (24, 1, 1, 7, 6),
                                        (32, 1, 2, 24, 0), (32, 1, 1, 32, 32), (40, 1, 1, 8, 0)])
def test_fused_sweep_is_bit_identical_to_two_half_sweeps(sg, L, S, R, T, zc):
    """SG_SWEEP_FUSED: the colour-fused, out-of-place overrelaxation sweep (colour 0 of plane k and
    colour 1 of plane k-1 in one pass, ring values recomputed) gives the spins of the two half-sweeps of the z-marching
    kernel bit for bit -- for every chunk length, tiles that wrap in x1 / x2 (L = 8), several groups, padded groups, odd
    numbers of sweeps (the state ends in the second buffer) -- and the same energies; heat bath, PT and measurement
    run unchanged on whichever buffer holds the state."""
    betas = np.linspace(0.5, 1.9, T)
    a = sg.SpinGlass(L, S, R, T, betas, seed=23); b = sg.SpinGlass(L, S, R, T, betas, seed=23, fused_buffer=True)
    with pytest.raises(sg.SgError):
        a.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_FUSED)            # no second state buffer in this context's workspace
    a.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_ZMARCH); b.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_FUSED)
    if zc:
        b.tune(sg.TUNE_ZCHUNK, zc)
    for g in (a, b):
        for s in range(S):
            g.init_sample(s, sg.GEN_GENERAL9 if s % 2 else sg.GEN_OFFDIAG_SYM, 1.0)
    for n_or in (1, 2, 3):
        for g in (a, b):
            g.sweep_or(n_or)
        for s in range(S):
            assert np.array_equal(a.get_spins(s), b.get_spins(s)), (n_or, s)
        Ea, Eb = a.get_energies(), b.get_energies()
        assert np.abs(Ea - Eb).max() <= 1e-7 * L ** 3          # fp32 partial sums per thread over a chunk: the chunkings differ
    for g in (a, b):
        g.sweep_hb(1); g.sweep_or(3); g.pt_swap(); g.sweep_or(1)
    for s in range(S):
        assert np.array_equal(a.get_spins(s), b.get_spins(s)) and np.array_equal(a.get_perm(s)[0], b.get_perm(s)[0])
    if R > 1:
        assert np.abs(a.measure()[1] - b.measure()[1]).max() <= 1e-12
    a.close(); b.close()


@pytest.mark.parametrize("ctas", [4, 8])
@pytest.mark.parametrize("S,R,T", [(1, 1, 5), (2, 2, 16), (3, 4, 24), (1, 2, 40)])
def test_cluster_resident_kernel_is_bit_identical_at_L16(sg, S, R, T, ctas):
    """SG_SWEEP_CLUSTER: the L = 16 lattice of a copy group in the shared memory of a cluster of
    8 CTAs, all sweeps of a call in one launch, x3 neighbours across the cuts through distributed shared memory -- spins and
    temperature assignment bit-identical to the z-marching kernel for OR and heat bath, one or several sweeps per call,
    one to three (padded) copy groups; energies to summation order; also through sg_run_units."""
    L = 16
    betas = np.linspace(0.5, 2.2, T)
    a = sg.SpinGlass(L, S, R, T, betas, seed=31, first_sample=1); b = sg.SpinGlass(L, S, R, T, betas, seed=31, first_sample=1)
    a.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_ZMARCH); b.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_CLUSTER); b.tune(sg.TUNE_CLUSTER_CTAS, ctas)
    for g in (a, b):
        for s in range(S):
            g.init_sample(s, sg.GEN_GENERAL9 if s % 2 else sg.GEN_OFFDIAG_SYM, 1.0)
    for n in (1, 2, 3):
        for g in (a, b):
            g.sweep_or(n)
        for s in range(S):
            assert np.array_equal(a.get_spins(s), b.get_spins(s)), ("or", n, s)
        assert np.abs(a.get_energies() - b.get_energies()).max() <= 1e-7 * L ** 3
        for g in (a, b):
            g.sweep_hb(n)
        for s in range(S):
            assert np.array_equal(a.get_spins(s), b.get_spins(s)), ("hb", n, s)
        assert np.abs(a.get_energies() - b.get_energies()).max() <= 1e-7 * L ** 3
    E = a.get_energies()
    for g in (a, b):
        g.set_energies(E)                         # identical energies: identical PT decisions
        g.pt_swap()
        g.sweep_hb(1); g.sweep_or(4)
    for s in range(S):
        assert np.array_equal(a.get_spins(s), b.get_spins(s)) and np.array_equal(a.get_perm(s)[0], b.get_perm(s)[0])
    assert a.get_counters() == b.get_counters()
    with pytest.raises(sg.SgError):
        sg.SpinGlass(8, 1, 1, 2, [0.5, 1.0]).tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_CLUSTER)
    a.close(); b.close()



def test_replica_and_slot_sharding_combine(sg):
    """Four contexts -- replicas (0, 1) / (2, 3) times slots [0, 3) / [3, 6) of every chain -- against one context holding
    the four replicas and six temperatures of every sample: the global copy id and the global chain id are what key the
    heat bath and the PT stream, so spins, assignments and PT statistics agree bit for bit after 20 units."""
    import torch
    L, S, R, T = 6, 2, 4, 6
    betas = np.linspace(0.5, 1.5, T)
    whole = sg.SpinGlass(L, S, R, T, betas, seed=13, first_sample=1)
    shards = {(rw, sw): sg.SpinGlass(L, S, 2, 3, betas, seed=13, first_sample=1, first_replica=2 * rw, n_replicas_total=4,
                                     first_slot=3 * sw, n_temps_total=T) for rw in range(2) for sw in range(2)}
    for g in [whole] + list(shards.values()):
        for s in range(S):
            g.init_sample(s, sg.GEN_OFFDIAG_SYM, 1.0)
    gathered = {rw: torch.empty((2, S, 2, 3), dtype=torch.float64, device="cuda") for rw in range(2)}
    for _ in range(20):
        whole.unit(2)
        for (rw, sw), g in shards.items():
            g.sweep_hb(1); g.sweep_or(2)
            g.pt_publish(out=gathered[rw][sw])
        torch.cuda.synchronize()
        for (rw, sw), g in shards.items():
            g.pt_swap_gathered(gathered[rw])
    for s in range(S):
        ref = whole.get_spins(s).reshape(R, T, 3, -1)
        tos = whole.get_perm(s)[0]
        for (rw, sw), g in shards.items():
            assert np.array_equal(ref[2 * rw:2 * rw + 2, 3 * sw:3 * sw + 3], g.get_spins(s).reshape(2, 3, 3, -1)), (s, rw, sw)
            assert np.array_equal(tos[2 * rw:2 * rw + 2], g.get_perm(s)[0])
    acc = whole.pt_stats()[1]
    for (rw, sw), g in shards.items():
        assert np.array_equal(acc[:, 2 * rw:2 * rw + 2], g.pt_stats()[1])
    assert acc.sum() > 0
    for g in [whole] + list(shards.values()):
        g.close()


@pytest.mark.parametrize("T", [853, 1000])
def test_pt_long_chains_warp_and_serial_kernels_match_oracle(sg, oracle, T):
    """A chain of 853 temperatures is the longest the warp-per-chain kernel stages in shared memory, 1000 falls back to
    k_pt_swap_serial: decisions, statistics, walk labels and round trips identical to the oracle (fed identical energies)."""
    L, S, R = 2, 1, 2
    betas = np.linspace(0.2, 3.0, T)
    sim, gpu = make_pair(oracle, sg, L, S, R, T, betas, seed=17)
    rng = np.random.default_rng(9)
    for k in range(6):
        E = rng.normal(0.0, 0.7 / (betas[1] - betas[0]), size=(S, R * T))
        gpu.set_energies(E)
        gpu.pt_swap()
        sim.pt_swap(energies=E)
    tos, sot = gpu.get_perm(0)
    assert np.array_equal(tos, sim.temp_of_slot[0]) and np.array_equal(sot, sim.slot_of_temp[0])
    att, acc = gpu.pt_stats()
    assert np.array_equal(att, sim.attempts) and np.array_equal(acc, sim.accepts) and 0 < acc.sum() < att.sum()
    trips, lab = gpu.pt_walk()
    assert np.array_equal(lab, sim.walk_label) and np.array_equal(trips, sim.round_trips[..., 0])
    assert np.array_equal(gpu.pt_visits(), sim.visits)
    gpu.close()
