"""GPU parity of the paper's packed bimodal couplings: one byte per link,
decoded by the producer warp of the z-marching sweep (opt-in: SG_TUNE_PACKED).  Byte work is compared bit for bit (the decoded matrices, the packed sweep
against the fp32-matrix sweep); the sweeps themselves against the oracle within the north star's tolerances."""
import numpy as np
import pytest

from tests.util import gpu_spins, oracle_spins

pytestmark = pytest.mark.gpu

SPIN_TOL = 1e-5


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_1599_b200 import build
    build.build()
    import paper_1309_1599_b200 as mod
    return mod


def random_links(rng, N):
    return rng.integers(0, 128, size=(3, N), dtype=np.uint8)


def make_bimodal_pair(oracle, sg, L, S, R, T, D, seed, links=None, tune=()):
    """Oracle chain on the decoded matrices and CUDA context on the bytes; spins flow oracle -> CUDA."""
    betas = np.linspace(0.5, 2.0, T)
    sim = oracle.OracleSim(L, S, R, T, betas, seed, store_fp32=True)
    gpu = sg.SpinGlass(L, S, R, T, betas, seed=seed)
    for knob, value in tune:
        gpu.tune(knob, value)
    for s in range(S):
        b = oracle.bimodal_links(L, seed, s) if links is None else links[s]
        sim.init_sample(s, couplings=oracle.bimodal_couplings(L, b, D))
        gpu.init_sample_bimodal(s, D, links=None if links is None else links[s], spins=sim.spins[s].astype(np.float32))
    return sim, gpu


@pytest.mark.parametrize("L,D", [(8, 0.5), (6, 1.0), (16, 0.3)])
def test_decoded_matrices_are_the_oracles_bit_for_bit(sg, oracle, L, D):
    """sg_get_couplings after sg_init_sample_bimodal: caller's bytes, and the generator's bytes (links = NULL)."""
    rng = np.random.default_rng(L)
    S = 2
    links = [random_links(rng, L ** 3) for _ in range(S)]
    gpu = sg.SpinGlass(L, S, 2, 2, [0.5, 1.0], seed=99, first_sample=3)
    for s in range(S):
        gpu.init_sample_bimodal(s, D, links=links[s])
        assert np.array_equal(gpu.get_couplings(s).astype(np.float64), oracle.bimodal_couplings(L, links[s], D))
    for s in range(S):
        gpu.init_sample_bimodal(s, D)
        assert np.array_equal(gpu.get_couplings(s).astype(np.float64), oracle.gen_couplings(L, 99, 3 + s, oracle.BIMODAL, D))


def test_bad_bytes_and_bad_D_are_rejected(sg):
    gpu = sg.SpinGlass(8, 1, 2, 2, [0.5, 1.0], seed=1)
    bad = np.zeros((3, 512), dtype=np.uint8); bad[1, 7] = 0x80
    with pytest.raises(Exception):
        gpu.init_sample_bimodal(0, 0.5, links=bad)
    with pytest.raises(Exception):
        gpu.init_sample_bimodal(0, -1.0)
    with pytest.raises(Exception):
        gpu.init_sample_bimodal(0, float("nan"))


@pytest.mark.parametrize("sh", [dict(L=8, S=2, R=2, T=5, D=0.5, zc=0), dict(L=16, S=1, R=2, T=17, D=1.0, zc=4),
                                dict(L=24, S=1, R=1, T=3, D=0.7, zc=0)])
def test_packed_sweep_is_bit_identical_to_the_matrix_sweep(sg, oracle, sh):
    """The packed z-marching kernel decodes the very fp32 operands the unpacked one loads: OR and HB sweeps, fused and
    stand-alone energies identical bit for bit.  (L = 8 goes to the resident kernel by default, so the z-marching
    kernel is asked for.)"""
    L, S, R, T, D = sh["L"], sh["S"], sh["R"], sh["T"], sh["D"]
    rng = np.random.default_rng(7)
    links = [random_links(rng, L ** 3) for _ in range(S)]
    out = []
    for packed in (1, 0):
        tune = [(sg.TUNE_SWEEP_IMPL, sg.SWEEP_ZMARCH), (sg.TUNE_PACKED, packed)]
        if sh["zc"]:
            tune.append((sg.TUNE_ZCHUNK, sh["zc"]))
        sim, gpu = make_bimodal_pair(oracle, sg, L, S, R, T, D, seed=5, links=links, tune=tune)
        n0 = gpu.kernel_launches()
        gpu.sweep_hb(1); gpu.sweep_or(3)
        E_fused = gpu.get_energies()
        gpu.halfsweep(sg.KIND_HB, 1); gpu.halfsweep(sg.KIND_OR, 0)
        out.append((gpu_spins(gpu), E_fused, gpu.get_energies(), gpu.kernel_launches() - n0))
    assert np.array_equal(out[0][0], out[1][0])
    assert np.array_equal(out[0][1], out[1][1]) and np.array_equal(out[0][2], out[1][2])
    assert out[0][3] == out[1][3] > 0


@pytest.mark.parametrize("sh", [dict(L=8, S=2, R=2, T=5, D=0.5), dict(L=16, S=1, R=2, T=6, D=1.0)])
def test_packed_sweeps_match_oracle(sg, oracle, sh):
    """Half-sweep by half-sweep from the oracle's state (no propagation): OR and HB, then energies."""
    L, S, R, T, D = sh["L"], sh["S"], sh["R"], sh["T"], sh["D"]
    sim, gpu = make_bimodal_pair(oracle, sg, L, S, R, T, D, seed=31, tune=[(sg.TUNE_SWEEP_IMPL, sg.SWEEP_ZMARCH), (sg.TUNE_PACKED, 1)])
    for kind in (sg.KIND_OR, sg.KIND_HB):
        for colour in (0, 1):
            for s in range(S):
                gpu.set_spins(s, sim.spins[s].astype(np.float32))
            flags = sim.halfsweep(kind, colour, want_flags=True)
            gpu.halfsweep(kind, colour)
            err = np.abs(gpu_spins(gpu) - oracle_spins(sim)).max(axis=2)
            bad = flags != 0
            assert bad.mean() <= 1e-3
            assert np.where(bad, 0.0, err).max() <= SPIN_TOL, (kind, colour)
    for s in range(S):
        gpu.set_spins(s, sim.spins[s].astype(np.float32))
    e_gpu = gpu.get_energies() / L ** 3
    e_ref = sim.energies() / L ** 3
    assert (np.abs(e_gpu - e_ref) <= 1e-6 * np.maximum(1.0, np.abs(e_ref))).all()


def test_mixed_contexts_fall_back_to_the_matrices(sg, oracle):
    """One sample packed, one not (or two different D): the sweep must read the fp32 arrays, same results as the oracle's."""
    L, R, T = 8, 2, 3
    betas = np.linspace(0.5, 1.5, T)
    for second in ("gauss", "otherD"):
        sim = oracle.OracleSim(L, 2, R, T, betas, 4, store_fp32=True)
        gpu = sg.SpinGlass(L, 2, R, T, betas, seed=4)
        gpu.tune(sg.TUNE_SWEEP_IMPL, sg.SWEEP_ZMARCH); gpu.tune(sg.TUNE_PACKED, 1)
        b0 = oracle.bimodal_links(L, 4, 0)
        sim.init_sample(0, couplings=oracle.bimodal_couplings(L, b0, 0.5))
        gpu.init_sample_bimodal(0, 0.5, spins=sim.spins[0].astype(np.float32))
        if second == "gauss":
            sim.init_sample(1)
            gpu.init_sample(1, couplings=sim.M[1].astype(np.float32), spins=sim.spins[1].astype(np.float32))
        else:
            sim.init_sample(1, couplings=oracle.bimodal_couplings(L, oracle.bimodal_links(L, 4, 1), 0.25))
            gpu.init_sample_bimodal(1, 0.25, spins=sim.spins[1].astype(np.float32))
        flags = sim.halfsweep(sg.KIND_OR, 0, want_flags=True)
        gpu.halfsweep(sg.KIND_OR, 0)
        err = np.abs(gpu_spins(gpu) - oracle_spins(sim)).max(axis=2)
        assert np.where(flags != 0, 0.0, err).max() <= SPIN_TOL, second


def test_packed_sweep_full_size_lattice(sg):
    """L = 64 (the headline lattice), 32 copies, the launch shape the bench uses (automatic chunking): packed against
    matrix sweeps bit for bit, and against the properties that hold at any size (|s| = 1 after HB, OR conserves the energy)."""
    L, S, R, T, D = 64, 1, 1, 32, 0.5
    betas = np.linspace(0.5, 2.6, T)
    out = []
    for packed in (1, 0):
        gpu = sg.SpinGlass(L, S, R, T, betas, seed=9)
        gpu.tune(sg.TUNE_PACKED, packed)
        gpu.init_sample_bimodal(0, D)
        gpu.sweep_hb(1)
        s1 = gpu.get_spins(0)
        E1 = gpu.get_energies()
        gpu.sweep_or(2)
        out.append((s1, E1, gpu.get_spins(0), gpu.get_energies()))
        gpu.close()
    for k in range(4):
        assert np.array_equal(out[0][k], out[1][k]), k
    s1, E1, s2, E2 = out[0]
    assert np.abs(np.linalg.norm(s1.astype(np.float64), axis=1) - 1.0).max() < 1e-6
    assert np.abs(E2 - E1).max() <= 2e-6 * np.abs(E1).max()          # OR keeps H (fp32 rounding of 2 sweeps)
