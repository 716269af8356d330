"""GPU parity at the shapes of BASELINE.json configs 1-3 (cfg 0 and cfg 4 have their own files: test_gpu_parity.py,
test_gpu_fullsize.py), through the library's default kernel choice -- the launch configuration bench.py --config k times --
and the north star's covariance checks (3) and (4) on the CUDA path itself:

    cfg 1  L =  8, 8 samples, 4 x 16 copies (C =  64, 2 copy groups)                  resident multi-sweep kernel
           + its isotropic rerun (sigma_D = 0): global O(3) covariance of the OR sweep, invariance of e and q
    cfg 2  L = 16, 32 samples, 4 x 24 copies (C =  96, 3 copy groups)                 OR sweeps: cluster-resident kernel (the full-
           sweep pass holds 5 samples = 15 copy groups, the least the automatic choice takes it for); heat bath and
           sg_halfsweep: z-marching kernel, 2 chunks
    cfg 3  L = 32, 16 samples, 4 x 32 copies (C = 128, 4 copy groups), sigma_D = sqrt 2  z-marching kernel

Element by element against the oracle on the same seeded inputs (oracle -> CUDA only), tolerances of the north star
(DESIGN.md section 6).  cfg 3 at its full 16 samples is compared on sampled whole copies plus size-independent
properties, as cfg 4 is."""
import numpy as np
import pytest

import sg_workloads as W
from tests.test_gpu_parity import assert_spins_close, colour_mask, sweep_both
from tests.test_oracle_model import gauge_transform
from tests.util import gpu_spins, make_pair, oracle_spins

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


# (config index, samples used for the element-by-element pass, samples for the full-sweep pass)
CASES = [(1, 8, 8), (2, 32, 5), (3, 2, 1)]
# the kernel the library's automatic choice must have taken for the sweep call, per (config, kind): asserted, so that a change
# of the dispatch cannot silently move a configuration's oracle comparison onto another kernel
SERVED_BY = {(1, 0): "SWEEP_RESIDENT", (1, 1): "SWEEP_RESIDENT", (2, 0): "SWEEP_CLUSTER", (2, 1): "SWEEP_ZMARCH",
             (3, 0): "SWEEP_ZMARCH", (3, 1): "SWEEP_ZMARCH"}


@pytest.mark.parametrize("k,S,S_sweep", CASES)
@pytest.mark.parametrize("kind", [0, 1])
def test_half_sweeps_at_config_shape(sg, oracle, k, S, S_sweep, kind):
    cfg = W.CONFIGS[k]
    L, R, T = cfg.L, cfg.n_replicas, cfg.n_temps
    sim, gpu = make_pair(oracle, sg, L, S, R, T, cfg.betas, seed=cfg.seed, sigma_D=cfg.sigma_D)
    sim.hb_counter = 3
    gpu.set_counters(3, 0)
    col = colour_mask(L)
    for colour in (0, 1):
        before = oracle_spins(sim)
        for s in range(S):
            gpu.set_spins(s, sim.spins[s].astype(np.float32))
        flags = sim.halfsweep(kind, colour, want_flags=True)
        gpu.halfsweep(kind, colour)
        got, want = gpu_spins(gpu), oracle_spins(sim)
        assert_spins_close(got, want, flags != 0, ("cfg", k, kind, colour))
        assert np.array_equal(got[..., col != colour], before[..., col != colour])


@pytest.mark.parametrize("k,S,S_sweep", CASES)
@pytest.mark.parametrize("kind", [0, 1])
def test_full_sweep_energy_and_measure_at_config_shape(sg, oracle, k, S, S_sweep, kind):
    """The product's sweep call through the automatic kernel choice (cfg 1: the resident kernel; cfg 2: the cluster-resident
    kernel for OR, two z-marching launches for the heat bath; cfg 3: z-marching; energies fused), then the measurement through
    a random temperature assignment."""
    cfg = W.CONFIGS[k]
    L, R, T, N = cfg.L, cfg.n_replicas, cfg.n_temps, cfg.n_sites
    sim, gpu = make_pair(oracle, sg, L, S_sweep, R, T, cfg.betas, seed=cfg.seed, sigma_D=cfg.sigma_D, first_sample=1)
    sweep_both(sim, gpu, kind, L)
    assert gpu.sweep_impl_used(kind) == (getattr(sg, SERVED_BY[(k, kind)]), 0)
    e_gpu, e_ref = gpu.get_energies() / N, sim.energies() / N
    assert np.all(np.abs(e_gpu - e_ref) <= 1e-6 * np.maximum(1.0, np.abs(e_ref)))
    rng = np.random.default_rng(40 + k)
    for s in range(S_sweep):
        sim.spins[s] = gpu.get_spins(s).astype(np.float64)        # measure the same state on both sides
        tos = np.stack([rng.permutation(T) for _ in range(R)]).astype(np.int32)
        gpu.set_perm(s, tos)
        sim.temp_of_slot[s] = tos
        sim.slot_of_temp[s] = np.argsort(tos, axis=1).astype(np.int32)
    e, q0, qk = gpu.measure()
    e_ref, q0_ref, qk_ref = sim.measure()
    assert np.all(np.abs(e - e_ref) <= 1e-6 * np.maximum(1.0, np.abs(e_ref)))
    assert np.abs(q0 - q0_ref).max() <= 1e-6 and np.abs(qk - qk_ref).max() <= 1e-6


def test_cfg3_full_size_sampled_copies(sg, oracle):
    """cfg 3 at its own size (16 samples x 128 copies of 32^3, sigma_D = sqrt 2) in the default launch configuration:
    sampled whole copies element by element, every copy by properties."""
    cfg = W.CONFIGS[3]
    L, S, R, T, C, N = cfg.L, cfg.n_samples, cfg.n_replicas, cfg.n_temps, cfg.n_copies, cfg.n_sites
    gpu = sg.SpinGlass(L, S, R, T, cfg.betas, seed=cfg.seed)
    for s in range(S):
        gpu.init_sample(s, sg.GEN_OFFDIAG_SYM, cfg.sigma_D)       # the library's own generators (checked against the oracle's below)
    sampled = [(0, 0), (0, 127), (3, 31), (3, 32), (7, 64), (9, 95), (15, 96), (15, 127)]
    M = {s: oracle.gen_couplings(L, cfg.seed, s, oracle.OFFDIAG_SYM, cfg.sigma_D) for s in {s for s, _ in sampled}}
    for s in M:
        assert np.array_equal(gpu.get_couplings(s), M[s].astype(np.float32))
    X = {s: gpu.get_spins(s) for s in M}
    for s, c in sampled:
        assert np.abs(X[s][c].astype(np.float64) - oracle.gen_spins(L, cfg.seed, s * C + c)).max() <= 5e-7
    E0 = gpu.get_energies()
    for s, c in sampled:
        e_ref = oracle.energy(L, M[s], np.ascontiguousarray(X[s][c], dtype=np.float64)) / N
        assert abs(E0[s, c] / N - e_ref) <= 1e-6 * max(1.0, abs(e_ref))
    gpu.set_counters(2, 0)
    for kind in (1, 0):
        for colour in (0, 1):
            mask = colour_mask(L) == colour
            for s in M:
                gpu.set_spins(s, X[s])
            gpu.halfsweep(kind, colour)
            for s in M:
                got = gpu.get_spins(s)
                assert np.array_equal(got[:, :, ~mask], X[s][:, :, ~mask])
                assert np.abs(np.sqrt((got.astype(np.float64) ** 2).sum(axis=1)) - 1).max() <= 5e-6
                for c in [c for s2, c in sampled if s2 == s]:
                    ref = X[s][c].astype(np.float64)
                    flags, _ = oracle.halfsweep(L, M[s], ref, kind, colour, beta=cfg.betas[c % T], seed=cfg.seed, g=s * C + c,
                                                hb_counter=2, store_fp32=True, want_flags=True)
                    err = np.abs(got[c].astype(np.float64) - ref).max(axis=0)
                    err[flags != 0] = 0.0
                    assert err.max() <= SPIN_TOL, (kind, colour, s, c, err.max())
                    assert (flags != 0).sum() <= 1e-3 * mask.sum()
    E0 = gpu.get_energies()                                        # of the state the half-sweeps above left (stand-alone pass)
    gpu.sweep_or(1)                                                # OR conserves every copy's energy (fused reduction)
    E1 = gpu.get_energies()
    assert np.all(np.abs(E1 - E0) / N <= 1e-6 * np.maximum(1.0, np.abs(E0) / N))


# ---------------------------------------------------------------------------------------------
# north star checks (3) and (4) on the CUDA path
# ---------------------------------------------------------------------------------------------
def test_gauge_covariance_of_the_or_sweep_on_gpu(sg, oracle):
    """s_x -> R_x s_x, M_{x,mu} -> R_x M_{x,mu} R_{x+mu}^T: the energy is invariant and an OR sweep commutes with the
    transform (h_x -> R_x h_x).  Both sides of the identity are computed by the CUDA kernels (fp32; the transformed
    inputs are rounded to fp32, which moves a field by ~1e-7 |h|); the oracle only supplies the ill-conditioning flags."""
    L, R, T = 8, 2, 4
    N, C = L ** 3, R * T
    rng = np.random.default_rng(77)
    M = W.random_couplings(rng, N, "offdiag_sym")
    s = W.random_spins(rng, C, N)
    M2 = None
    s2 = np.empty_like(s)
    Rx = W.random_rotations(rng, N)
    for c in range(C):
        M2, s2[c] = gauge_transform(L, M, s[c], Rx)
    M2 = M2.astype(np.float32).astype(np.float64)
    s2 = s2.astype(np.float32).astype(np.float64)
    betas = np.linspace(0.5, 1.5, T)
    sim, a = make_pair(oracle, sg, L, 1, R, T, betas, couplings=[M], spins=[s], tune=((0, 2),))
    _, b = make_pair(oracle, sg, L, 1, R, T, betas, couplings=[M2], spins=[s2], tune=((0, 2),))
    Ea, Eb = a.get_energies() / N, b.get_energies() / N
    assert np.abs(Ea - Eb).max() <= 2e-6 * max(1.0, np.abs(Ea).max())
    exclude = np.zeros((1, C, N), dtype=bool)
    for colour in (0, 1):
        exclude |= sim.halfsweep(0, colour, want_flags=True) != 0
        a.halfsweep(0, colour); b.halfsweep(0, colour)
    sa, sb = gpu_spins(a)[0], gpu_spins(b)[0]
    rot = np.einsum("nab,cbn->can", Rx, sa)
    err = np.where(exclude[0], 0.0, np.abs(rot - sb).max(axis=1))
    assert np.mean(err > SPIN_TOL) <= 1e-3 and err.max() <= 1e-3 and np.median(err) <= 1e-6, (err.max(), np.mean(err > SPIN_TOL))
    assert np.abs(sa - s).max() > 0.5                              # the sweep did move the spins


def test_isotropic_rerun_of_cfg1_global_rotation_on_gpu(sg, oracle):
    """cfg 1 'rerun with D = 0': with isotropic couplings a global O(3) rotation (here an improper one) of every spin
    commutes with an OR sweep and leaves e, q^(0), q^(k) unchanged -- asserted on the CUDA path (fp32 tolerances)."""
    cfg = W.CONFIGS[1]
    L, S, R, T, N = cfg.L, 2, cfg.n_replicas, cfg.n_temps, cfg.n_sites
    rng = np.random.default_rng(78)
    Q = W.random_rotations(rng, 1, proper=False)[0]
    Q[:, 0] *= -np.sign(np.linalg.det(Q))                          # det = -1: O(3), not only SO(3)
    sim, a = make_pair(oracle, sg, L, S, R, T, cfg.betas, seed=cfg.seed, sigma_D=0.0)
    rotated = [np.einsum("ab,cbn->can", Q, sim.spins[s]).astype(np.float32).astype(np.float64) for s in range(S)]
    _, b = make_pair(oracle, sg, L, S, R, T, cfg.betas, seed=cfg.seed, sigma_D=0.0, spins=rotated)
    ea, q0a, qka = a.measure()
    eb, q0b, qkb = b.measure()
    assert np.abs(ea - eb).max() <= 2e-6 and np.abs(q0a - q0b).max() <= 2e-6 and np.abs(qka - qkb).max() <= 2e-6
    exclude = np.zeros((S, R * T, N), dtype=bool)
    for colour in (0, 1):
        exclude |= sim.halfsweep(0, colour, want_flags=True) != 0
    a.sweep_or(1); b.sweep_or(1)
    sa, sb = gpu_spins(a), gpu_spins(b)
    err = np.where(exclude, 0.0, np.abs(np.einsum("ab,scbn->scan", Q, sa) - sb).max(axis=2))
    assert np.mean(err > SPIN_TOL) <= 1e-3 and err.max() <= 1e-3 and np.median(err) <= 1e-6, (err.max(), np.mean(err > SPIN_TOL))
    # with anisotropy the same rotation does NOT commute (the check has power)
    sim2, c = make_pair(oracle, sg, L, 1, R, T, cfg.betas, seed=cfg.seed, sigma_D=1.0)
    _, d = make_pair(oracle, sg, L, 1, R, T, cfg.betas, seed=cfg.seed, sigma_D=1.0,
                     spins=[np.einsum("ab,cbn->can", Q, sim2.spins[0]).astype(np.float32).astype(np.float64)])
    c.sweep_or(1); d.sweep_or(1)
    assert np.abs(np.einsum("ab,scbn->scan", Q, gpu_spins(c)) - gpu_spins(d)).max() > 0.1


# ---------------------------------------------------------------------------------------------
# automatic chunking of the z-marching kernel for L = 8 * odd with few CTAs (one sample, one copy group)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [24, 40, 56])
def test_zmarch_auto_chunk_is_valid_for_L_eight_times_odd(sg, L):
    """The automatic chunk length must be even and divide L (the kernel steps through a chunk in pairs of planes): the
    z-marching kernel with its automatic chunking against the tiled kernel, bit for bit, spins and HB draws."""
    R, T = 1, 5
    betas = np.linspace(0.5, 1.5, T)
    out = []
    for impl in (sg.SWEEP_TILED, sg.SWEEP_ZMARCH):
        gpu = sg.SpinGlass(L, 1, R, T, betas, seed=7)
        gpu.tune(sg.TUNE_SWEEP_IMPL, impl)
        gpu.init_sample(0, sg.GEN_GENERAL9, 1.0)
        gpu.sweep_hb(1); gpu.sweep_or(2)
        out.append((gpu.get_spins(0), gpu.get_energies()))
        gpu.close()
    assert np.array_equal(out[0][0], out[1][0])
    assert np.abs(out[0][1] - out[1][1]).max() <= 1e-6 * L ** 3
