"""The fp32 heat-bath draw of the CUDA path (reading R23) against the fp64 oracle in the TAILS of
the polar uniform, r1 -> 2^-24 and r1 -> 1 - 2^-24, for kappa = beta |h| from 1e-3 to 50 -- where the plain fp32 formula
is ill-conditioned and where the branch-free evaluation has to carry the small one of w = 1 - u, w' = 1 + u to a few ulp.

Set-up: ferromagnetic couplings (M = 1), every spin the same unit vector v, so that every site of the swept colour sees
the field h = 6 v whatever the other sites do (the other colour is frozen: a half-sweep never touches it) and kappa is
6 beta of the copy.  r1 is what Philox draws for (site, copy, HB sweep counter): the oracle's diagnostic hb_uniforms
FINDS sweep counters in which some (site, copy) draws r1 in the last few of its 2^23 values at either end; the
temperature permutation is then rotated so that the copy that holds such a draw visits EVERY kappa of the ladder.
Every site of every copy is compared (1e-5 absolute per component, the north star's bar); the tail draws are reported."""
import numpy as np
import pytest

from tests.util import gpu_spins, make_pair, oracle_spins

pytestmark = pytest.mark.gpu

TAIL = 2.0 ** -20          # a draw counts as "in the tail" when r1 <= TAIL or 1 - r1 <= TAIL


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_1599_b200 import build
    build.build()
    import paper_1309_1599_b200 as mod
    return mod


def test_hb_draw_in_the_tails_of_r1_for_all_kappa(sg, oracle):
    L, R, T, seed = 8, 4, 32, 2024
    N, C = L ** 3, R * T
    betas = np.geomspace(1e-3, 50.0, T) / 6.0                       # kappa = 6 beta: 1e-3 ... 50
    v = np.array([1.0, 2.0, 3.0]) / np.sqrt(14.0)
    spins = np.broadcast_to(v[None, :, None], (C, 3, N)).astype(np.float32).astype(np.float64)
    M = oracle.gen_couplings(L, seed, 0, oracle.FERRO, 0.0)
    idx = np.arange(N)
    colour0 = ((idx % L + (idx // L) % L + idx // (L * L)) % 2) == 0

    # scan HB sweep counters for draws in the extreme tails on colour-0 sites
    hits = []                                                        # (distance from the end, counter, copy, site)
    for k in range(600):
        for c in range(C):
            r1, _ = oracle.hb_uniforms(L, seed, c, k)
            r1 = np.where(colour0, r1, 0.5)
            for i in np.nonzero((r1 <= TAIL) | (1.0 - r1 <= TAIL))[0]:
                hits.append((min(r1[i], 1.0 - r1[i]), k, c, int(i), r1[i] < 0.5))
    lo = sorted(h for h in hits if h[4])[:3]
    hi = sorted(h for h in hits if not h[4])[:3]
    assert len(lo) == 3 and len(hi) == 3, "the scan must find draws in both tails"
    assert lo[0][0] <= 2.0 ** -22 and hi[0][0] <= 2.0 ** -22, (lo[0], hi[0])

    sim, gpu = make_pair(oracle, sg, L, 1, R, T, betas, seed=seed, couplings=[M], spins=[spins], tune=((0, 2),))
    worst_all, worst_tail, n_tail = 0.0, 0.0, 0
    for dist, k, c, i, low in lo + hi:
        r, slot = divmod(c, T)
        for shift in range(T):                                       # copy c visits every temperature of the ladder
            tos = np.tile((np.arange(T) + shift) % T, (R, 1)).astype(np.int32)
            gpu.set_perm(0, tos)
            sim.temp_of_slot[0] = tos
            sim.slot_of_temp[0] = np.argsort(tos, axis=1).astype(np.int32)
            gpu.set_spins(0, spins.astype(np.float32))
            sim.spins[0] = spins.copy()
            gpu.set_counters(k, 0)
            sim.hb_counter = k
            flags = sim.halfsweep(1, 0, want_flags=True)
            gpu.halfsweep(1, 0)
            assert not flags.any()                                   # |h| = 6, n_z = 0.8: nothing is ill-conditioned here
            err = np.abs(gpu_spins(gpu) - oracle_spins(sim)).max(axis=2)[0]      # [C][N]
            worst_all = max(worst_all, err.max())
            worst_tail = max(worst_tail, err[c, i])
            n_tail += 1
            assert err.max() <= 1e-5, (k, c, i, shift, err.max(), np.unravel_index(err.argmax(), err.shape))
            # the tail draw did land next to a pole of h (so the test has the power it claims): |u| -> 1 when kappa is small
            u = float(oracle_spins(sim)[0, c, :, i] @ v)
            kappa = 6.0 * betas[(slot + shift) % T]
            if kappa < 0.1:
                assert (1.0 - abs(u)) < 4.0 * TAIL and (u > 0) == low
    print("HB-TAILS: %d (tail draw, kappa) cases, r1 within %.1e / %.1e of 0 / 1; max error at the tail draws %.2e, over all "
          "draws of those half-sweeps %.2e (bar 1e-5)" % (n_tail, lo[0][0], hi[0][0], worst_tail, worst_all))
