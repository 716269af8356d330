"""Helpers shared by the GPU parity tests (no method arithmetic: masks, construction of the two sides)."""
import numpy as np


def neighbour_dilate(mask, L):
    """mask [..., N] (bool) -> True at every site that has a True nearest neighbour (periodic)."""
    m = mask.reshape(mask.shape[:-1] + (L, L, L))
    out = np.zeros_like(m)
    for ax in (-1, -2, -3):
        out |= np.roll(m, 1, axis=ax) | np.roll(m, -1, axis=ax)
    return out.reshape(mask.shape)


def make_pair(oracle, sgmod, L, S, R, T, betas, seed=1, gen_mode=0, sigma_D=1.0, first_sample=0,
              couplings=None, spins=None, tune=None):
    """Oracle chain and CUDA context with identical inputs.  Inputs flow oracle -> CUDA, never back:
    couplings / spins are drawn by the oracle's generators (or passed in) and copied to the device."""
    sim = oracle.OracleSim(L, S, R, T, betas, seed, store_fp32=True, first_sample=first_sample)
    gpu = sgmod.SpinGlass(L, S, R, T, betas, seed=seed, first_sample=first_sample)
    for knob, value in (tune or ()):           # (sg_tune knob, value) pairs: which sweep kernel serves the calls
        gpu.tune(knob, value)
    for s in range(S):
        sim.init_sample(s, gen_mode, sigma_D,
                        couplings=None if couplings is None else couplings[s],
                        spins=None if spins is None else spins[s])
        gpu.init_sample(s, couplings=sim.M[s].astype(np.float32), spins=sim.spins[s].astype(np.float32))
    return sim, gpu


def gpu_spins(gpu):
    return np.stack([gpu.get_spins(s) for s in range(gpu.S)]).astype(np.float64)


def oracle_spins(sim):
    return np.stack(sim.spins)

