"""Long runs: thermal averages of the CUDA chain against the oracle's own chain (north star: energy and q^2
within 3 statistical sigma).  Both sides run the same disorder sample, the same temperature ladder and the
same unit (1 HB + n_or OR + PT).  K independent chains of that one disorder sample are run side by side by
giving every "sample" of the context the same couplings (their Philox streams differ through the global copy
id), so the error bars need no autocorrelation model: each chain's second half
(thermalisation) is cut into a few long bins and the K x bins bin means are the sample.
The oracle and CUDA trajectories separate after a few sweeps (fp32 vs fp64 rounding amplified by the
chaotic dynamics), so the two sides' errors are independent.  The bar is the SURVEY's (section 8(c)): every
comparison within max |z| < 4 and chi^2/n consistent with 1 (n = 12 comparisons for cfg 0, 32 for cfg 1; the
north star's 3 sigma is a per-comparison statement, P(|z| > 3) = 2.7e-3, so over n comparisons the family-wise
bar at the same confidence is |z| < 4).  The observed max |z| and chi^2/n are printed (pytest -s / -rP shows them)
and recorded in DESIGN.md section 6.  Seeds are fixed, both chains are deterministic."""
import warnings

import numpy as np
import pytest

import sg_workloads as W

pytestmark = pytest.mark.gpu

FAMILY = {}        # test name -> z values of its comparisons (the family-wise bar is taken over all of them, last test of the file)


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_1599_b200 import build
    build.build()
    import paper_1309_1599_b200 as mod
    return mod


def bin_mean_err(x, n_bins):
    """x [n_meas][K chains][...] -> (mean, standard error) from the K*n_bins bin means of the second half."""
    x = x[x.shape[0] // 2:]
    n = (x.shape[0] // n_bins) * n_bins
    b = x[:n].reshape((n_bins, n // n_bins) + x.shape[1:]).mean(axis=1)       # [n_bins][K][...]
    b = b.reshape((-1,) + b.shape[2:])
    return b.mean(axis=0), b.std(axis=0, ddof=1) / np.sqrt(b.shape[0])


def observables(e, q0, qk):
    """per measurement: e averaged over replicas [K][T]; q0^2 and |q(k_min)|^2 averaged over pairs (and axes)."""
    return e.mean(axis=1), (q0 ** 2).mean(axis=1), (qk ** 2).sum(axis=-1).mean(axis=(1, 3))


def run_chain(chain, n_units, n_or, measure_every=1):
    out = [[], [], []]
    for u in range(n_units):
        chain.unit(n_or)
        if (u + 1) % measure_every == 0:
            for acc, v in zip(out, observables(*chain.measure())):
                acc.append(v)
    return [np.array(a) for a in out]


def compare(obs_gpu, obs_ref, names, n_bins, family_key):
    zs = []
    for g, r, name in zip(obs_gpu, obs_ref, names):
        mg, sg_ = bin_mean_err(g, n_bins)
        mr, sr = bin_mean_err(r, n_bins)
        z = (mg - mr) / np.sqrt(sg_ ** 2 + sr ** 2)
        assert np.all(np.isfinite(z)), name
        zs.append(z.reshape(-1))
    z = np.concatenate(zs)
    chi2 = float((z ** 2).mean())
    msg = ("STATS-MARGIN %s %s: n = %d comparisons, max |z| = %.3f (bar 4), chi^2/n = %.3f (bar %.3f), fraction |z| > 3: %.3f"
           % (family_key, "+".join(names), z.size, np.abs(z).max(), chi2, 1.1 + 4.0 * np.sqrt(2.0 / z.size), np.mean(np.abs(z) > 3)))
    print(msg)
    warnings.warn(msg)          # pytest's warnings summary keeps the line in a plain `pytest -q` log (DESIGN.md section 6 quotes it)
    FAMILY[family_key] = z
    assert np.abs(z).max() < 4.0, ("max |z|", np.abs(z).max(), "chi2/n", chi2, z)
    assert chi2 < 1.1 + 4.0 * np.sqrt(2.0 / z.size), ("chi2/n", chi2, z.size, "max |z|", np.abs(z).max())
    return z


def make_chains(oracle, sg, cfg, K):
    """K chains of disorder sample 0 of the workload on each side (same couplings for every 'sample')."""
    L, R, T = cfg.L, cfg.n_replicas, cfg.n_temps
    sim = oracle.OracleSim(L, K, R, T, cfg.betas, cfg.seed)
    gpu = sg.SpinGlass(L, K, R, T, cfg.betas, seed=cfg.seed)
    M = oracle.gen_couplings(L, cfg.seed, 0, oracle.OFFDIAG_SYM, cfg.sigma_D)
    for k in range(K):
        sim.init_sample(k, couplings=M)
        gpu.init_sample(k, couplings=M.astype(np.float32), spins=sim.spins[k].astype(np.float32))
    return sim, gpu


def test_cfg0_thermal_averages_within_errors(sg, oracle):
    """cfg 0 (L=4, 2 replicas x 4 temperatures, 1 HB + 4 OR + PT): 4 chains of 4000 units (BASELINE: one of
    1000; more only sharpens the test), measured after every unit."""
    cfg = W.CONFIGS[0]
    K, n_units = 4, 4000
    sim, gpu = make_chains(oracle, sg, cfg, K)
    ref = run_chain(sim, n_units, cfg.n_or)
    got = run_chain(gpu, n_units, cfg.n_or)
    compare(got, ref, ("e", "q0^2", "|qk|^2"), n_bins=5, family_key="cfg0")
    # PT: the same number of attempts; acceptance rates of the two sides agree
    att_g, acc_g = gpu.pt_stats()
    assert np.array_equal(att_g, sim.attempts)
    rate_g = acc_g.sum(axis=(0, 1)) / att_g.sum(axis=(0, 1))
    rate_o = sim.accepts.sum(axis=(0, 1)) / sim.attempts.sum(axis=(0, 1))
    assert np.abs(rate_g - rate_o).max() < 0.03, (rate_g, rate_o)
    assert gpu.get_counters() == (n_units, n_units)


def test_cfg1_thermal_averages_within_errors(sg, oracle):
    """cfg 1 shape (L=8, 4 replicas x 16 temperatures, beta 0.5..2.0, 1 HB + 8 OR + PT): 4 chains of disorder
    sample 0, 2000 units each, measured every 4th unit; per-temperature <e> and <q0^2>."""
    cfg = W.CONFIGS[1]
    K, n_units = 4, 2000
    sim, gpu = make_chains(oracle, sg, cfg, K)
    ref = run_chain(sim, n_units, cfg.n_or, measure_every=4)
    got = run_chain(gpu, n_units, cfg.n_or, measure_every=4)
    compare(got, ref, ("e", "q0^2", "|qk|^2"), n_bins=5, family_key="cfg1")


def test_family_of_all_comparisons():
    """SURVEY.md section 8(c) as written: `max |z| < 4` is the bar for a family of MORE THAN 50 comparisons (the north star's 3 sigma
    is a per-comparison statement).  The two tests above make 12 + 48 = 60; this one takes the bar over all of them together
    and checks the per-comparison statement in the form it can be checked: no more than 2 of the 60 beyond 3 sigma
    (expected 0.16; P(>= 3) = 6e-4 for a correct code)."""
    if set(FAMILY) != {"cfg0", "cfg1"}:
        pytest.skip("needs both chains of this file (run the whole file)")
    z = np.concatenate([FAMILY["cfg0"], FAMILY["cfg1"]])
    msg = "STATS-MARGIN family: n = %d comparisons, max |z| = %.3f (bar 4), |z| > 3: %d (bar 2), chi^2/n = %.3f" % (
        z.size, np.abs(z).max(), int(np.sum(np.abs(z) > 3)), float((z ** 2).mean()))
    print(msg)
    warnings.warn(msg)
    assert z.size > 50
    assert np.abs(z).max() < 4.0 and np.sum(np.abs(z) > 3) <= 2, msg
