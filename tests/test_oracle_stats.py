"""Pins of the oracle's stochastic parts: the heat-bath law (Eq. (A1)), Schwinger-Dyson (Eq. (A6)),
exact Heisenberg-ring energies for the whole HB+OR+PT chain, overlap statistics, PT acceptance.
CPU only; seeds are fixed, thresholds are 4.5 sigma.  Pin numbers: DESIGN.md section 7."""
import itertools

import numpy as np
import pytest
from scipy import integrate, special, stats

import sg_workloads as W

KAPPAS = [0.1, 0.5, 1.0, 2.0, 5.0, 10.0, 20.0]


def langevin(k):
    return 1.0 / np.tanh(k) - 1.0 / k


# ---------------------------------------------------------------------------------------------
# P8  single spin in a fixed field (north_star check 2)
# ---------------------------------------------------------------------------------------------
def test_hb_update_inverts_the_cdf_of_eq_A1(oracle):
    """u = s.n must satisfy  r1 = int_u^1 e^{kappa u'} du' / int_{-1}^1 e^{kappa u'} du'  (Eq. (A1),
    PAPER.md:325, integrated over the azimuth), the integrals done numerically here."""
    rng = np.random.default_rng(41)
    for kappa in [1e-3, 0.1, 1.0, 3.0, 8.0, 20.0]:
        for _ in range(12):
            h = W.random_unit_vectors(rng, ()) * 2.5
            beta = kappa / 2.5
            r1, r2 = rng.uniform(0.001, 0.999), rng.uniform()
            s = oracle.hb_update(h, beta, r1, r2)
            u = s @ h / 2.5
            assert abs(np.linalg.norm(s) - 1) < 1e-14
            f = lambda x: np.exp(kappa * (x - 1.0))
            num = integrate.quad(f, u, 1.0, epsabs=1e-14, epsrel=1e-13)[0]
            den = integrate.quad(f, -1.0, 1.0, epsabs=1e-14, epsrel=1e-13)[0]
            assert abs(num / den - r1) < 1e-10


def test_hb_update_limits_and_frame(oracle):
    rng = np.random.default_rng(42)
    for _ in range(50):
        n = W.random_unit_vectors(rng, ())
        h = 3.0 * n
        # r1 -> 0: aligned with the field;  r1 -> 1: anti-aligned
        assert np.allclose(oracle.hb_update(h, 1.0, 1e-300, 0.3), n, atol=1e-12)
        assert np.allclose(oracle.hb_update(h, 0.2, 1 - 1e-16, 0.3), -n, atol=1e-6)
        # fixed r1: a circle about n, traversed counter-clockwise (right-handed frame), phi = 2 pi r2
        r1 = rng.uniform(0.1, 0.9)
        a = oracle.hb_update(h, 0.7, r1, 0.0)
        b = oracle.hb_update(h, 0.7, r1, 0.25)
        c = oracle.hb_update(h, 0.7, r1, 0.5)
        u = a @ n
        assert abs(b @ n - u) < 1e-14 and abs(c @ n - u) < 1e-14
        pa, pb, pc = a - u * n, b - u * n, c - u * n
        assert abs(pa @ pb) < 1e-14 and np.allclose(pc, -pa, atol=1e-14)
        assert np.cross(pa, pb) @ n > 0
    # kappa = 0 (beta = 0 or h = 0): uniform law u = 1 - 2 r1; h = 0 is drawn about z^ (reading R8)
    s = oracle.hb_update(np.zeros(3), 1.0, 0.25, 0.0)
    assert np.allclose(s, [np.sqrt(0.75), 0.0, 0.5], atol=1e-15)
    s = oracle.hb_update(np.array([0.0, 2.0, 0.0]), 0.0, 0.25, 0.125)
    assert abs(s[1] - 0.5) < 1e-15 and abs(np.linalg.norm(s) - 1) < 1e-15
    # tiny kappa joins the uniform law continuously
    assert np.allclose(oracle.hb_update(np.array([0, 0, 1e-9]), 1.0, 0.3, 0.6),
                       oracle.hb_update(np.zeros(3), 1.0, 0.3, 0.6), atol=1e-8)


@pytest.mark.parametrize("kappa", KAPPAS)
def test_hb_fixed_field_langevin(oracle, kappa):
    """Colour 1 frozen along d, ferromagnetic couplings: every colour-0 site sees h = 6 d.  Repeated HB
    half-sweeps of colour 0 (Philox stream, lattice path) must give <cos> = coth k - 1/k (north_star 2),
    <cos^2> = 1 - 2 L(k)/k, the full CDF (KS), a uniform azimuth and zero perpendicular mean."""
    L, N = 8, 512
    rng = np.random.default_rng(int(kappa * 1000))
    d = W.random_unit_vectors(rng, ())
    M = oracle.gen_couplings(L, 1, 0, oracle.FERRO, 0.0)
    s = np.ascontiguousarray(np.tile(d[:, None], (1, N)))
    idx = np.arange(N)
    c0 = ((idx % L + (idx // L) % L + idx // (L * L)) % 2) == 0
    beta = kappa / 6.0
    cos, perp = [], []
    for k in range(160):
        oracle.halfsweep(L, M, s, oracle.KIND_HB, 0, beta=beta, seed=77, g=3, hb_counter=k)
        v = s[:, c0]
        cos.append(d @ v)
        perp.append(v - np.outer(d, d @ v))
    assert np.array_equal(s[:, ~c0], np.tile(d[:, None], (1, N // 2)))        # colour 1 untouched
    cos = np.concatenate(cos)
    perp = np.concatenate(perp, axis=1)
    n = cos.size
    Lk = langevin(kappa)
    m2 = 1.0 - 2.0 * Lk / kappa
    assert abs(cos.mean() - Lk) < 4.5 * np.sqrt((m2 - Lk ** 2) / n)
    assert abs((cos ** 2).mean() - m2) < 4.5 * (cos ** 2).std() / np.sqrt(n)
    cdf = lambda u: (np.exp(kappa * (u - 1)) - np.exp(-2 * kappa)) / (1 - np.exp(-2 * kappa))
    assert stats.kstest(cos, cdf).pvalue > 1e-3
    # azimuth in a frame built here from d (any fixed frame will do: uniform is uniform)
    a = np.cross(d, [1.0, 0.0, 0.0]); a /= np.linalg.norm(a)
    b = np.cross(d, a)
    phi = np.arctan2(b @ perp, a @ perp)
    assert stats.kstest(phi, "uniform", args=(-np.pi, 2 * np.pi)).pvalue > 1e-3
    assert np.all(np.abs(perp.mean(axis=1)) < 4.5 * perp.std(axis=1) / np.sqrt(n))
    # polar angle and azimuth independent
    assert abs(np.corrcoef(cos, np.cos(phi))[0, 1]) < 4.5 / np.sqrt(n)


def test_hb_distinct_streams(oracle):
    """site, copy id, sweep counter and seed all enter the counter/key: any change gives new draws."""
    L, N = 4, 64
    M = oracle.gen_couplings(L, 1, 0, oracle.FERRO, 0.0)
    base = dict(beta=0.5, seed=5, g=2, hb_counter=7)
    outs = []
    for delta in [{}, {"seed": 6}, {"g": 3}, {"hb_counter": 8}, {"seed": 5 + (1 << 32)}]:
        s = np.zeros((3, N)); s[2] = 1.0
        oracle.halfsweep(L, M, s, oracle.KIND_HB, 0, **{**base, **delta})
        outs.append(s)
    for a, b in itertools.combinations(outs, 2):
        assert np.abs(a - b).max() > 0.1
    assert len({tuple(np.round(outs[0][:, i], 12)) for i in range(0, N) if outs[0][2, i] != 1.0}) == N // 2


def test_hb_uniforms_are_the_numbers_the_half_sweep_draws(oracle):
    """The test diagnostic hb_uniforms(seed, g, hb_counter) returns, site by site, the (r1, r2) of the lattice heat bath:
    feeding them to the single-spin update with the site's field reproduces the half-sweep, and they are the exactly
    representable 23-bit uniforms of stream 1 (counter (i, g, hb_counter, 1))."""
    L, N = 4, 64
    rng = np.random.default_rng(12)
    M = W.random_couplings(rng, N, "general")
    s0 = W.random_spins(rng, 1, N)[0]
    r1, r2 = oracle.hb_uniforms(L, 5, 2, 7)
    s = s0.copy()
    oracle.halfsweep(L, M, s, oracle.KIND_HB, 1, beta=0.8, seed=5, g=2, hb_counter=7)
    for i in range(N):
        if oracle.lib().sgo_colour(L, i) == 1:
            want = oracle.hb_update(oracle.local_field(L, M, s0, i), 0.8, r1[i], r2[i])
            assert np.array_equal(s[:, i], want)
    for i in (0, 17, 63):
        w = oracle.philox4x32_10((i, 2, 7, 1), (5, 0))
        assert r1[i] == ((w[0] >> 9) + 0.5) / 2 ** 23 and r2[i] == ((w[1] >> 9) + 0.5) / 2 ** 23


# ---------------------------------------------------------------------------------------------
# P9  Schwinger-Dyson (Eq. (A6)), site-averaged, any couplings
# ---------------------------------------------------------------------------------------------
def test_schwinger_dyson_identity(oracle):
    L, N = 4, 64
    rng = np.random.default_rng(51)
    M = W.random_couplings(rng, N, "general")
    for beta in [0.4, 1.0, 2.5]:
        s = W.random_spins(rng, 1, N)[0]
        T = 1.0 / beta
        vals, wrong = [], []
        for k in range(3000):
            for colour in (0, 1):
                _, sd = oracle.halfsweep(L, M, s, oracle.KIND_HB, colour, beta=beta, seed=9, g=1,
                                         hb_counter=k, want_sd=True)
                vals.append(2 * T * sd[0] - (sd[1] - sd[2]))
                wrong.append(2 * 1.1 * T * sd[0] - (sd[1] - sd[2]))
        vals, wrong = np.array(vals[200:]), np.array(wrong[200:])
        err = vals.std() / np.sqrt(vals.size)
        assert abs(vals.mean()) < 4.5 * err
        assert abs(wrong.mean()) > 8 * err            # the test has the power to see a 10 % error in T


# ---------------------------------------------------------------------------------------------
# P10  exact thermal energy of Heisenberg rings (Joyce 1967), whole chain HB + OR + PT
# ---------------------------------------------------------------------------------------------
def ring_energy_per_spin(beta, a):
    """-(1/L) d ln Z / d beta,  Z = sum_l (2l+1) prod_j i_l(beta a_j)  (i_l: modified spherical Bessel)."""
    a = np.asarray(a, dtype=np.float64)
    Z, dZ = 0.0, 0.0
    for l in range(0, 80):
        il = special.spherical_in(l, beta * a)
        dil = special.spherical_in(l, beta * a, derivative=True) * a
        prod = np.prod(il)
        Z += (2 * l + 1) * prod
        dZ += (2 * l + 1) * sum(dil[j] * np.prod(np.delete(il, j)) for j in range(a.size))
    return -dZ / Z / a.size


def test_ring_formula_limits():
    # L -> infinity: e = -(coth b - 1/b); two spins with one bond: Z = sinh(b)/b * 4pi...
    assert abs(ring_energy_per_spin(1.3, np.ones(200)) + langevin(1.3)) < 1e-10
    # L = 2 ring = two spins joined by a double bond 2*beta: e per spin = -L(2 beta)
    assert abs(ring_energy_per_spin(0.7, np.ones(2)) + langevin(1.4)) < 1e-12


def ring_couplings(L, a):
    """M_{x,0} = a_x 1, M_{x,1} = M_{x,2} = 0: L^2 independent periodic rings along x1."""
    N = L ** 3
    M = np.zeros((3, N, 3, 3))
    M[0] = np.asarray(a)[:, None, None] * np.eye(3)
    return M


@pytest.mark.parametrize("L,mode", [(4, "hb_or_pt"), (4, "hb_only"), (2, "hb_or_pt"), (4, "random_bonds")])
def test_heisenberg_rings_exact_energy(oracle, L, mode):
    N = L ** 3
    betas = np.array([0.5, 1.0, 1.6, 2.0])
    rng = np.random.default_rng(61)
    a = np.ones(N) if mode != "random_bonds" else np.round(rng.uniform(0.5, 1.5, N) * rng.choice([-1, 1], N), 3)
    sim = oracle.OracleSim(L, 1, 2, 4, betas, seed=3, store_fp32=False)
    sim.init_sample(0, couplings=ring_couplings(L, a))
    n_units, n_therm = (2500, 250) if L == 4 else (6000, 300)
    e = np.zeros((n_units, 4))
    for k in range(n_units):
        if mode == "hb_only":
            sim.sweep_hb(1)
        else:
            sim.unit(2)
        e[k] = sim.measure()[0][0].mean(axis=0)         # average the two replicas, per temperature
    e = e[n_therm:]
    if mode != "hb_only":
        assert sim.accepts.sum() > 0.05 * sim.attempts.sum()     # PT is really moving copies around
    rings = a.reshape(L, L, L)                          # [x3][x2][x1]: one ring per (x3, x2)
    for t, beta in enumerate(betas):
        exact = np.mean([ring_energy_per_spin(beta, rings[i, j]) for i in range(L) for j in range(L)])
        nb = 25
        bins = e[: (len(e) // nb) * nb, t].reshape(nb, -1).mean(axis=1)
        err = bins.std(ddof=1) / np.sqrt(nb)
        assert err < 0.01
        assert abs(bins.mean() - exact) < 4.5 * err, (L, mode, beta, bins.mean(), exact, err)


# ---------------------------------------------------------------------------------------------
# P12  overlap statistics with zero couplings: <q> = 0, <q^2> = <|q(k)|^2> = 1/(3N)
# ---------------------------------------------------------------------------------------------
def test_overlap_statistics_uncoupled_spins(oracle):
    L, N = 4, 64
    sim = oracle.OracleSim(L, 1, 2, 1, np.array([1.0]), seed=4)
    sim.init_sample(0, couplings=np.zeros((3, N, 3, 3)))
    q0, qk2 = [], []
    for _ in range(4000):
        sim.sweep_hb(1)                                 # h = 0: every sweep is a fresh uniform draw
        _, a, b = sim.measure()
        q0.append(a[0, 0, 0])
        qk2.append((b[0, 0, 0] ** 2).sum(axis=1))
    q0, qk2 = np.array(q0), np.array(qk2)
    n = q0.size
    assert abs(q0.mean()) < 4.5 * q0.std() / np.sqrt(n)
    assert abs((q0 ** 2).mean() - 1 / (3 * N)) < 4.5 * (q0 ** 2).std() / np.sqrt(n)
    for mu in range(3):
        assert abs(qk2[:, mu].mean() - 1 / (3 * N)) < 4.5 * qk2[:, mu].std() / np.sqrt(n)


# ---------------------------------------------------------------------------------------------
# P13  parallel tempering (north_star check 6)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("delta", [-3.0, -1.0, -0.3, -0.05, 0.0, 0.5])
def test_pt_acceptance_probability(oracle, delta):
    """Two temperatures, frozen energies: accept frequency = min(1, exp(dBeta dE))."""
    betas = np.array([0.8, 1.3])
    E = np.array([0.0, -delta / (betas[0] - betas[1])])      # (b0-b1)(E0-E1) = delta
    n, acc = 20000, 0
    for k in range(n):
        sot = np.arange(2, dtype=np.int32); tos = np.arange(2, dtype=np.int32)
        oracle.pt_sweep(betas, E, sot, tos, seed=11, chain=5, pt_counter=k)
        swapped = sot[0] == 1
        assert sorted(sot) == [0, 1] and tos[sot[0]] == 0 and tos[sot[1]] == 1
        acc += swapped
    p = min(1.0, np.exp(delta))
    assert abs(acc / n - p) <= 4.5 * np.sqrt(p * (1 - p) / n) + 1e-12


def test_pt_stationary_distribution_over_permutations(oracle):
    """Frozen energies, PT only: the assignment slot -> temperature must sample
    P(perm) ~ exp(-sum_slot beta_{temp(slot)} E_slot) (Metropolis swaps keep it stationary; pairs are
    visited in order on the updated assignment, reading R11)."""
    betas = np.array([0.5, 0.9, 1.6])
    E = np.array([-1.0, 0.4, 1.3])
    sot = np.arange(3, dtype=np.int32); tos = np.arange(3, dtype=np.int32)
    att = np.zeros(2, dtype=np.uint64); acc = np.zeros(2, dtype=np.uint64)
    counts = {}
    n = 60000
    for k in range(n):
        oracle.pt_sweep(betas, E, sot, tos, seed=12, chain=0, pt_counter=k, attempts=att, accepts=acc)
        assert sorted(sot) == [0, 1, 2] and all(tos[sot[t]] == t for t in range(3))
        if k >= 100:
            counts[tuple(tos)] = counts.get(tuple(tos), 0) + 1
    assert att.tolist() == [n, n] and 0 < acc[0] < n
    perms = list(itertools.permutations(range(3)))
    wts = np.array([np.exp(-sum(betas[p[s]] * E[s] for s in range(3))) for p in perms])
    wts /= wts.sum()
    freq = np.array([counts.get(p, 0) for p in perms]) / (n - 100)
    # successive sweeps are correlated: allow 6 binomial sigma
    assert np.all(np.abs(freq - wts) < 6 * np.sqrt(wts * (1 - wts) / (n - 100)) + 1e-3), (freq, wts)


def test_pt_never_moves_spins_and_counts(oracle):
    L = 4
    betas = np.linspace(0.6, 1.6, 4)
    sim = oracle.OracleSim(L, 2, 2, 4, betas, seed=1)
    for s in range(2):
        sim.init_sample(s)
    before = [x.copy() for x in sim.spins]
    for _ in range(20):
        sim.pt_swap()
    assert all(np.array_equal(a, b) for a, b in zip(before, sim.spins))
    assert sim.pt_counter == 20 and np.all(sim.attempts == 20)
    for s in range(2):
        for r in range(2):
            assert sorted(sim.slot_of_temp[s, r]) == list(range(4))
            assert np.array_equal(sim.temp_of_slot[s, r][sim.slot_of_temp[s, r]], np.arange(4))
    assert sim.accepts.sum() > 0


# ---------------------------------------------------------------------------------------------
# random walk in temperature: pins of oracle.pt_walk_update
# ---------------------------------------------------------------------------------------------
def test_pt_walk_round_trips_by_hand_and_brute_force(oracle):
    """T = 2, every swap accepted: a configuration alternates 0, 1, 0, 1, ...; the one starting at index 1 touches
    index 0 after sweep 1 (label 1), index 1 after sweep 2 (label 2) and completes its first round trip after sweep 3.
    Then: an arbitrary recorded walk against a brute-force count of the pattern 0 ... T-1 ... 0 per configuration."""
    tos = np.array([0, 1], dtype=np.int32); label = np.zeros(2, dtype=np.int32); trips = np.zeros(1, dtype=np.uint64)
    seen = []
    for sweep in range(1, 8):
        tos = tos[::-1].copy()
        oracle.pt_walk_update(tos, label, trips)
        seen.append(int(trips[0]))
    # slot 0: at index 1 after odd sweeps, 0 after even: touches 0 first at sweep 2 -> trips at sweeps 4, 6
    # slot 1: at index 0 after odd sweeps: label 1 at sweep 1 -> trips at sweeps 3, 5, 7
    assert seen == [0, 0, 1, 2, 3, 4, 5]
    rng = np.random.default_rng(2)
    T, n = 5, 4000
    perm = np.arange(T, dtype=np.int32)
    label = np.zeros(T, dtype=np.int32); trips = np.zeros(1, dtype=np.uint64); visits = np.zeros((T, T), dtype=np.uint64)
    hist = []
    for _ in range(n):
        t = rng.integers(0, T - 1)
        if rng.random() < 0.6:
            a, b = np.where(perm == t)[0][0], np.where(perm == t + 1)[0][0]
            perm[a], perm[b] = t + 1, t
        oracle.pt_walk_update(perm, label, trips, visits)
        hist.append(perm.copy())
    hist = np.array(hist)                                         # [n][slot] -> temperature index
    brute = 0
    for slot in range(T):
        ends = [t for t in hist[:, slot] if t in (0, T - 1)]
        state = None
        for t in ends:
            if t == 0:
                if state == "top":
                    brute += 1
                state = "bottom"
            elif state == "bottom":
                state = "top"
    assert int(trips[0]) == brute and brute > 5
    assert np.array_equal(visits, np.array([[np.sum(hist[:, s] == t) for t in range(T)] for s in range(T)], dtype=np.uint64))
    assert visits.sum() == n * T


def test_walk_tau_int_by_hand_and_on_known_processes(oracle):
    """Pins of oracle.walk_tau_int (reading R24).  (a) x = (0, 1, 1, 0) by hand: m = 1/2, C(0) = 1/4,
    C(1) = (-1/4 + 1/4 - 1/4)/3 = -1/12, rho(1) = -1/3, tau(1) = 1/2 - 1/3 = 1/6 and the window closes (1 >= 6/6).
    (b) white noise: tau = 1/2.  (c) AR(1) with coefficient phi: rho(k) = phi^k, tau = 1/2 + phi/(1 - phi).
    (d) a symmetric +-1 walk on the ladder 0..T-1 reflected at the ends (what a chain with acceptance 1 on a flat
    landscape does): rho(k) is the lazy-walk spectrum -- here checked against the exact autocorrelation from the
    transition matrix.  (e) a constant or too short series gives NaN."""
    assert oracle.walk_tau_int([0, 1, 1, 0]) == pytest.approx(1.0 / 6.0, abs=1e-15)
    rng = np.random.default_rng(7)
    n = 400000
    assert oracle.walk_tau_int(rng.integers(0, 8, n)) == pytest.approx(0.5, abs=0.02)
    for phi in (0.5, 0.9):
        x = np.empty(n); x[0] = 0.0
        eps = rng.standard_normal(n)
        for i in range(1, n):
            x[i] = phi * x[i - 1] + eps[i]
        exact = 0.5 + phi / (1.0 - phi)
        assert oracle.walk_tau_int(x) == pytest.approx(exact, rel=0.06)
    # (d) lazy reflecting walk on T sites: P(i -> i+-1) = 1/2, a move off the ladder stays
    T = 6
    P = np.zeros((T, T))
    for i in range(T):
        for j in (i - 1, i + 1):
            P[i, j if 0 <= j < T else i] += 0.5
    pi = np.full(T, 1.0 / T); lab = np.arange(T) - (T - 1) / 2.0
    c0 = float(pi @ lab ** 2)
    rho, v = [], lab.copy()
    for k in range(1, 2000):
        v = P @ v
        rho.append(float(pi @ (lab * v)) / c0)
    exact = 0.5 + sum(rho)                      # rho decays like cos(pi/T)^k: converged long before k = 2000
    steps = rng.integers(0, 2, n) * 2 - 1
    x = np.empty(n, dtype=np.int32); pos = 0
    for i in range(n):
        j = pos + steps[i]
        pos = j if 0 <= j < T else pos
        x[i] = pos
    assert oracle.walk_tau_int(x, window_c=10.0) == pytest.approx(exact, rel=0.08)
    assert np.isnan(oracle.walk_tau_int([3, 3, 3, 3, 3])) and np.isnan(oracle.walk_tau_int([0, 1, 0]))


# ---------------------------------------------------------------------------------------------
# logarithmic data binning (Sect. III): pins of oracle.logbin_index / logbin_observables / accumulate
# ---------------------------------------------------------------------------------------------
def test_logbin_is_the_papers_halving_of_the_time_series(oracle):
    """"i_f contains the last half of the Monte Carlo time series, i_f - 1 the second quarter, i_f - 2 the second octave,
    and so on", each bin "twice the length of the previous": slice a series of 2^k - 1 values by hand."""
    k = 7
    M = 2 ** k - 1
    bins = np.array([oracle.logbin_index(n) for n in range(1, M + 1)])
    assert bins[-1] == k - 1
    assert np.array_equal(np.where(bins == k - 1)[0], np.arange(M - 2 ** (k - 1), M))              # last half
    assert np.array_equal(np.where(bins == k - 2)[0], np.arange(2 ** (k - 2) - 1, 2 ** (k - 1) - 1))  # second quarter
    assert np.array_equal(np.where(bins == k - 3)[0], np.arange(2 ** (k - 3) - 1, 2 ** (k - 2) - 1))  # second octave
    assert [int(np.sum(bins == i)) for i in range(k)] == [2 ** i for i in range(k)]
    assert oracle.logbin_index(1) == 0 and oracle.logbin_index(2 ** 31 - 1) == 30 and oracle.logbin_index(2 ** 31) == 31


def test_logbin_observables_by_hand(oracle):
    """R = 2, T = 1, one pair: e = (1, 3) -> 2; q0 = 1/2 -> q0^2 = 1/4, q0^4 = 1/16; q(k) = (3+4i, 0, 1i) -> (25+0+1)/3.
    R = 3: means over the three pairs.  R = 1: no overlap entries."""
    e = np.array([[[1.0], [3.0]]]); q0 = np.array([[[0.5]]])
    qk = np.zeros((1, 1, 1, 3, 2)); qk[0, 0, 0, 0] = (3.0, 4.0); qk[0, 0, 0, 2] = (0.0, 1.0)
    assert np.allclose(oracle.logbin_observables(e, q0, qk)[0, 0], [2.0, 0.25, 26.0 / 3.0, 0.0625, 0.0, 0.0], rtol=0, atol=1e-15)
    # chiral-glass entries: q_CG^mu(0) = (1, 2, 3) -> (1 + 4 + 9)/3; q_CG^mu(k_nu): two non-zero entries 3+4i (mu=0, nu=1), 2 (mu=2, nu=2)
    # -> (25 + 4)/9
    qc0 = np.array([[[[1.0, 2.0, 3.0]]]]); qck = np.zeros((1, 1, 1, 3, 3, 2)); qck[0, 0, 0, 0, 1] = (3.0, 4.0); qck[0, 0, 0, 2, 2, 0] = 2.0
    assert np.allclose(oracle.logbin_observables(e, q0, qk, qc0, qck)[0, 0, 4:], [14.0 / 3.0, 29.0 / 9.0], rtol=0, atol=1e-15)
    e3 = np.array([[[1.0], [2.0], [6.0]]]); q3 = np.array([[[1.0], [2.0], [3.0]]])
    qk3 = np.zeros((1, 3, 1, 3, 2)); qk3[0, 1, 0, 1, 0] = 3.0
    assert np.allclose(oracle.logbin_observables(e3, q3, qk3)[0, 0, :4], [3.0, 14.0 / 3.0, 1.0, 98.0 / 3.0], rtol=0, atol=1e-14)
    assert np.array_equal(oracle.logbin_observables(np.ones((2, 1, 3)), np.zeros((2, 0, 3)), np.zeros((2, 0, 3, 3, 2)))[..., 1:],
                          np.zeros((2, 3, 5)))


def test_accumulate_bins_a_recorded_series(oracle):
    """OracleSim.accumulate over 15 units of a small chain: bin sums / counts equal the recorded measurements sliced
    as in the paper (bin 3 = last 8, bin 2 = the 4 before, ...)."""
    betas = np.linspace(0.6, 1.6, 4)
    sim = oracle.OracleSim(4, 1, 2, 4, betas, 3)
    sim.init_sample(0)
    rec = []
    for _ in range(15):
        sim.unit(2)
        rec.append(oracle.logbin_observables(*sim.measure(), *sim.measure_chiral()))
        sim.accumulate(with_chirality=True)
    rec = np.array(rec)
    assert sim.n_acc == 15 and list(sim.logbin_counts[:5]) == [1, 2, 4, 8, 0] and np.array_equal(sim.logbin_counts_cg, sim.logbin_counts)
    assert (rec[..., 4] > 0).all() and (rec[..., 5] > 0).all()
    for i, (lo, hi) in enumerate([(0, 1), (1, 3), (3, 7), (7, 15)]):
        assert np.allclose(sim.logbin_sums[i], rec[lo:hi].sum(axis=0), rtol=0, atol=1e-13)
    assert not sim.logbin_sums[4:].any()
