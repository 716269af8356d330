"""Pins of the oracle's deterministic parts: Philox, lattice indexing, local field, energy,
overrelaxation, symmetries, overlap observables.  CPU only.  Pin numbers are DESIGN.md section 7
(SURVEY.md section 8(c)); citations are PAPER.md:<line>."""
import itertools
import os

import numpy as np
import pytest

import sg_workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------------------------------------
# independent numpy construction of the model (shares nothing with oracle/sg_oracle.c)
# ---------------------------------------------------------------------------------------------
def dense_matrix(L, M):
    """A (3N x 3N) with H = -1/2 s^T A s and h = A s, built from the link list (Eq. (1))."""
    N = L ** 3
    A = np.zeros((3 * N, 3 * N))
    for x3, x2, x1 in itertools.product(range(L), repeat=3):
        i = x1 + L * (x2 + L * x3)
        for mu, (d1, d2, d3) in enumerate([(1, 0, 0), (0, 1, 0), (0, 0, 1)]):
            j = (x1 + d1) % L + L * ((x2 + d2) % L + L * ((x3 + d3) % L))
            A[3 * i:3 * i + 3, 3 * j:3 * j + 3] += M[mu, i]
            A[3 * j:3 * j + 3, 3 * i:3 * i + 3] += M[mu, i].T
    return A


def site_major(s):
    """[3][N] -> flat vector (s_0^0, s_0^1, s_0^2, s_1^0, ...)."""
    return np.ascontiguousarray(s.T).reshape(-1)


def colours(L):
    idx = np.arange(L ** 3)
    return (idx % L + (idx // L) % L + idx // (L * L)) % 2


# ---------------------------------------------------------------------------------------------
# P1  Philox4x32-10 known answers; uniforms
# ---------------------------------------------------------------------------------------------
def test_philox_known_answers(oracle):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r if t != "->"]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_uniforms_exact(oracle):
    # r = ((w>>9)+1/2) 2^-23: open interval, symmetric, exactly representable in fp32
    assert oracle.uniform23(0) == 2.0 ** -24
    assert oracle.uniform23(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert oracle.uniform23(0x1FF) == 2.0 ** -24           # low 9 bits are dropped
    for w in [0, 1 << 9, 0x80000000, 0xFFFFFFFF, 0x12345678]:
        r = oracle.uniform23(w)
        assert float(np.float32(r)) == r
    assert oracle.uniform32(0) == 2.0 ** -33
    assert oracle.uniform32(0xFFFFFFFF) == 1.0 - 2.0 ** -33


# ---------------------------------------------------------------------------------------------
# lattice indexing against numpy
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 4, 6])
def test_lattice_indexing(oracle, L):
    lib = oracle.lib()
    col = colours(L)
    for i in range(L ** 3):
        x = (i % L, (i // L) % L, i // (L * L))
        assert lib.sgo_site(L, *x) == i
        assert lib.sgo_colour(L, i) == col[i]
        for mu in range(3):
            for d in (+1, -1):
                y = list(x)
                y[mu] = (y[mu] + d) % L
                j = lib.sgo_neighbour(L, i, mu, d)
                assert j == y[0] + L * (y[1] + L * y[2])
                assert col[j] != col[i]          # every link joins the two colours (even L)


# ---------------------------------------------------------------------------------------------
# P4  field and energy: four routes, dense matrix, exhaustive L=2
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 4])
@pytest.mark.parametrize("kind", ["general", "offdiag_sym"])
def test_energy_routes_and_dense_matrix(oracle, L, kind):
    rng = np.random.default_rng(100 + L)
    N = L ** 3
    M = W.random_couplings(rng, N, kind, fp32=False)
    s = W.random_spins(rng, 1, N, fp32=False)[0]
    A = dense_matrix(L, M)
    v = site_major(s)
    H_dense = -0.5 * v @ A @ v
    H_links = oracle.energy(L, M, s)
    scale = 1e-12 * 3 * N
    assert abs(H_links - H_dense) < scale
    assert abs(oracle.energy_from_fields(L, M, s, -1) - H_dense) < scale
    assert abs(oracle.energy_from_fields(L, M, s, 0) - H_dense) < scale
    assert abs(oracle.energy_from_fields(L, M, s, 1) - H_dense) < scale
    h_dense = (A @ v).reshape(N, 3)
    for i in range(N):
        assert np.allclose(oracle.local_field(L, M, s, i), h_dense[i], rtol=0, atol=1e-12)


def test_exhaustive_L2_axis_configurations(oracle):
    """north_star check (5): all 2^8 configurations s_x = +-z^ on L=2, against a brute-force sum over
    the 24 forward links written out by hand here (double bonds: x+e and x-e coincide, reading R5)."""
    L, N = 2, 8
    rng = np.random.default_rng(7)
    M = W.random_couplings(rng, N, "general", fp32=False)
    coords = [(i % 2, (i // 2) % 2, i // 4) for i in range(N)]
    for bits in range(256):
        sz = np.array([1.0 if (bits >> i) & 1 else -1.0 for i in range(N)])
        s = np.zeros((3, N))
        s[2] = sz
        H = 0.0
        for i, (a, b, c) in enumerate(coords):
            for mu, nb in enumerate([((a + 1) % 2, b, c), (a, (b + 1) % 2, c), (a, b, (c + 1) % 2)]):
                j = nb[0] + 2 * nb[1] + 4 * nb[2]
                H -= sz[i] * M[mu, i, 2, 2] * sz[j]
        assert abs(oracle.energy(L, M, s) - H) < 1e-12


def test_exhaustive_L2_all_axes_sample(oracle):
    """The 6^8 axis configurations are sampled (4096 of them) against the dense matrix."""
    L, N = 2, 8
    rng = np.random.default_rng(8)
    M = W.random_couplings(rng, N, "general", fp32=False)
    A = dense_matrix(L, M)
    axes = np.concatenate([np.eye(3), -np.eye(3)])
    for _ in range(4096):
        s = axes[rng.integers(0, 6, N)].T.copy()
        v = site_major(s)
        assert abs(oracle.energy(L, M, s) + 0.5 * v @ A @ v) < 1e-12


# ---------------------------------------------------------------------------------------------
# P3  ferromagnetic closed forms (the paper's own cross-check idea)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 4, 8])
def test_ferromagnet_closed_forms(oracle, L):
    N = L ** 3
    M = oracle.gen_couplings(L, 1, 0, oracle.FERRO, 0.0)
    assert np.array_equal(M, np.broadcast_to(np.eye(3), (3, N, 3, 3)))
    s = np.zeros((3, N))
    s[1] = 1.0
    assert oracle.energy(L, M, s) / N == -3.0
    s = np.zeros((3, N))
    s[2] = 1.0 - 2.0 * colours(L)
    assert oracle.energy(L, M, s) / N == +3.0
    for i in range(N):                              # field of the aligned state: six neighbours
        s1 = np.zeros((3, N)); s1[0] = 1.0
        assert np.array_equal(oracle.local_field(L, M, s1, i), [6.0, 0.0, 0.0])


# ---------------------------------------------------------------------------------------------
# P2  overrelaxation (Eq. (A2)): energy conserved, |s| = 1, involution
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 4, 6])
def test_or_conserves_energy_and_norm(oracle, L):
    rng = np.random.default_rng(200 + L)
    N = L ** 3
    M = W.random_couplings(rng, N, "general", fp32=False)
    s = W.random_spins(rng, 1, N, fp32=False)[0]
    E0 = oracle.energy(L, M, s)
    for sweep in range(3):
        for colour in (0, 1):
            oracle.halfsweep(L, M, s, oracle.KIND_OR, colour)
            assert abs(oracle.energy(L, M, s) - E0) < 1e-12 * N
    assert np.allclose(np.sum(s * s, axis=0), 1.0, rtol=0, atol=1e-13)


def test_or_single_spin_formula(oracle):
    """Eq. (A2) against numpy: reflection about h; s.h and |s| unchanged; component along h kept."""
    rng = np.random.default_rng(5)
    for _ in range(100):
        h = rng.standard_normal(3) * 3
        s = W.random_unit_vectors(rng, ())
        s2 = oracle.or_update(h, s)
        assert np.allclose(s2, 2 * h * (h @ s) / (h @ h) - s, atol=1e-15)
        assert abs(s2 @ h - s @ h) < 1e-14 * (1 + abs(s @ h))
        assert abs(np.linalg.norm(s2) - 1) < 1e-14
    s = np.array([0.6, 0.0, 0.8])
    assert np.array_equal(oracle.or_update(np.zeros(3), s), s)       # h = 0: unchanged (R8)


def test_or_half_sweep_is_an_involution(oracle):
    L, N = 4, 64
    rng = np.random.default_rng(11)
    M = W.random_couplings(rng, N, "general", fp32=False)
    s0 = W.random_spins(rng, 1, N, fp32=False)[0]
    s = s0.copy()
    oracle.halfsweep(L, M, s, oracle.KIND_OR, 0)
    assert not np.allclose(s, s0)
    assert np.array_equal(s[:, colours(L) == 1], s0[:, colours(L) == 1])   # other colour untouched
    oracle.halfsweep(L, M, s, oracle.KIND_OR, 0)
    assert np.allclose(s, s0, atol=1e-13)


def test_or_sweep_against_numpy_sequential(oracle):
    """A checkerboard half-sweep equals updating the same sites one after another with the dense field
    (same-colour sites do not interact)."""
    L, N = 4, 64
    rng = np.random.default_rng(12)
    M = W.random_couplings(rng, N, "general", fp32=False)
    s = W.random_spins(rng, 1, N, fp32=False)[0]
    A = dense_matrix(L, M)
    ref = s.copy()
    for colour in (0, 1):
        for i in np.nonzero(colours(L) == colour)[0]:
            h = (A @ site_major(ref)).reshape(N, 3)[i]
            ref[:, i] = 2 * h * (h @ ref[:, i]) / (h @ h) - ref[:, i]
    oracle.halfsweep(L, M, s, oracle.KIND_OR, 0)
    oracle.halfsweep(L, M, s, oracle.KIND_OR, 1)
    assert np.allclose(s, ref, atol=1e-12)


# ---------------------------------------------------------------------------------------------
# P5  gauge invariance  s_x -> R_x s_x,  M_{x,mu} -> R_x M_{x,mu} R_{x+mu}^T   (north_star check 3)
# ---------------------------------------------------------------------------------------------
def gauge_transform(L, M, s, Rx):
    N = L ** 3
    idx = np.arange(N)
    x = np.stack([idx % L, (idx // L) % L, idx // (L * L)])
    M2 = np.empty_like(M)
    for mu in range(3):
        y = x.copy()
        y[mu] = (y[mu] + 1) % L
        j = y[0] + L * (y[1] + L * y[2])
        M2[mu] = np.einsum("nab,nbc,ndc->nad", Rx, M[mu], Rx[j])
    s2 = np.einsum("nab,bn->an", Rx, s)
    return np.ascontiguousarray(M2), np.ascontiguousarray(s2)


@pytest.mark.parametrize("L", [2, 4])
def test_gauge_invariance_and_or_covariance(oracle, L):
    rng = np.random.default_rng(300 + L)
    N = L ** 3
    M = W.random_couplings(rng, N, "offdiag_sym", fp32=False)
    s = W.random_spins(rng, 1, N, fp32=False)[0]
    Rx = W.random_rotations(rng, N)
    M2, s2 = gauge_transform(L, M, s, Rx)
    assert abs(oracle.energy(L, M2, s2) - oracle.energy(L, M, s)) < 1e-12 * N
    for i in range(N):                              # h_x -> R_x h_x
        assert np.allclose(oracle.local_field(L, M2, s2, i), Rx[i] @ oracle.local_field(L, M, s, i), atol=1e-12)
    for colour in (0, 1):                           # an OR sweep commutes with the gauge transform
        oracle.halfsweep(L, M, s, oracle.KIND_OR, colour)
        oracle.halfsweep(L, M2, s2, oracle.KIND_OR, colour)
    assert np.allclose(s2, np.einsum("nab,bn->an", Rx, s), atol=1e-12)


# ---------------------------------------------------------------------------------------------
# P6  isotropic limit (north_star check 4), P7 time reversal
# ---------------------------------------------------------------------------------------------
def test_isotropic_global_rotation_invariance(oracle):
    L, N = 4, 64
    rng = np.random.default_rng(21)
    M = W.random_couplings(rng, N, "isotropic", fp32=False)
    s = W.random_spins(rng, 2, N, fp32=False)
    Rg = W.random_rotations(rng, 1, proper=False)[0]
    Rg[:, 0] *= -np.linalg.det(Rg)                  # make it improper: O(3), not only SO(3)
    assert np.isclose(np.linalg.det(Rg), -1.0)
    sr = np.ascontiguousarray(np.einsum("ab,cbn->can", Rg, s))
    assert abs(oracle.energy(L, M, sr[0]) - oracle.energy(L, M, s[0])) < 1e-12 * N
    assert np.allclose(oracle.overlap(L, sr[0], sr[1]), oracle.overlap(L, s[0], s[1]), atol=1e-14)
    a, b = s[0].copy(), sr[0].copy()
    for colour in (0, 1):
        oracle.halfsweep(L, M, a, oracle.KIND_OR, colour)
        oracle.halfsweep(L, M, b, oracle.KIND_OR, colour)
    assert np.allclose(b, Rg @ a, atol=1e-12)
    # with anisotropy the invariance is gone (the test would be vacuous if it held anyway)
    Ma = W.random_couplings(rng, N, "offdiag_sym", fp32=False)
    assert abs(oracle.energy(L, Ma, sr[0]) - oracle.energy(L, Ma, s[0])) > 1e-3


def test_time_reversal(oracle):
    L, N = 4, 64
    rng = np.random.default_rng(22)
    M = W.random_couplings(rng, N, "general", fp32=False)
    s = W.random_spins(rng, 1, N, fp32=False)[0]
    m = np.ascontiguousarray(-s)
    assert abs(oracle.energy(L, M, m) - oracle.energy(L, M, s)) < 1e-12 * N
    oracle.halfsweep(L, M, s, oracle.KIND_OR, 0)
    oracle.halfsweep(L, M, m, oracle.KIND_OR, 0)
    assert np.allclose(m, -s, atol=1e-15)


# ---------------------------------------------------------------------------------------------
# P11  overlap and Fourier modes: closed forms fix normalisation, axis and sign
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [4, 8])
def test_overlap_closed_forms(oracle, L):
    N = L ** 3
    rng = np.random.default_rng(31)
    s = W.random_spins(rng, 1, N, fp32=False)[0]
    o = oracle.overlap(L, s, s)
    assert abs(o[0] - 1.0) < 1e-14 and np.allclose(o[1:], 0.0, atol=1e-14)
    idx = np.arange(N)
    coords = [idx % L, (idx // L) % L, idx // (L * L)]
    sa = np.zeros((3, N)); sa[2] = 1.0
    for mu in range(3):
        th = 2 * np.pi * coords[mu] / L
        sb = np.zeros((3, N)); sb[0] = np.sin(th); sb[2] = np.cos(th)      # q_x = cos(2 pi x_mu / L)
        o = oracle.overlap(L, sa, sb)
        want = np.zeros(7); want[1 + 2 * mu] = 0.5
        assert np.allclose(o, want, atol=1e-14)
        sb = np.zeros((3, N)); sb[0] = np.cos(th); sb[2] = np.sin(th)      # q_x = sin(2 pi x_mu / L)
        o = oracle.overlap(L, sa, sb)
        want = np.zeros(7); want[2 + 2 * mu] = 0.5                          # +i/2: e^{+ik.x} convention
        assert np.allclose(o, want, atol=1e-14)


def test_overlap_against_numpy_fft(oracle):
    L, N = 6, 216
    rng = np.random.default_rng(32)
    s = W.random_spins(rng, 2, N, fp32=False)
    q = np.sum(s[0] * s[1], axis=0).reshape(L, L, L)          # [x3][x2][x1]
    F = np.fft.ifftn(q)                                       # sum q e^{+ik.x}/N
    o = oracle.overlap(L, s[0], s[1])
    assert abs(o[0] - F[0, 0, 0].real) < 1e-14
    for mu, k in enumerate([(0, 0, 1), (0, 1, 0), (1, 0, 0)]):
        assert abs(o[1 + 2 * mu] - F[k].real) < 1e-14 and abs(o[2 + 2 * mu] - F[k].imag) < 1e-14


# ---------------------------------------------------------------------------------------------
# P14  generators
# ---------------------------------------------------------------------------------------------
def test_initial_spins_statistics(oracle):
    L = 16
    s = oracle.gen_spins(L, 1, 5)
    N = L ** 3
    assert np.allclose(np.sum(s * s, axis=0), 1.0, atol=3e-7)          # fp32-rounded unit vectors
    assert np.array_equal(s, s.astype(np.float32).astype(np.float64))
    assert np.all(np.abs(s.mean(axis=1)) < 4.0 / np.sqrt(3 * N))
    cov = s @ s.T / N
    assert np.allclose(cov, np.eye(3) / 3, atol=4.0 / np.sqrt(N))
    from scipy import stats
    assert stats.kstest(s[2], "uniform", args=(-1, 2)).pvalue > 1e-3    # z uniform on [-1,1]
    assert stats.kstest(np.arctan2(s[1], s[0]), "uniform", args=(-np.pi, 2 * np.pi)).pvalue > 1e-3
    assert not np.array_equal(s, oracle.gen_spins(L, 1, 6))            # copy id enters the counter
    assert not np.array_equal(s, oracle.gen_spins(L, 2, 5))            # seed enters the key


@pytest.mark.parametrize("mode,sigma", [(0, 1.0), (0, 2.0 ** 0.5), (1, 0.5), (2, 1.0), (3, 0.5), (0, 0.0)])
def test_coupling_generator_modes(oracle, mode, sigma):
    L = 8
    N = L ** 3
    M = oracle.gen_couplings(L, 1, 3, mode, sigma)
    assert np.array_equal(M, M.astype(np.float32).astype(np.float64))
    n = 3 * N
    tol = 5.0 / np.sqrt(n)
    if mode in (0, 1, 3):
        assert np.array_equal(M, np.swapaxes(M, 2, 3))                # D symmetric
    if mode == 0:
        a = M[..., 0, 0]
        assert np.array_equal(a, M[..., 1, 1]) and np.array_equal(a, M[..., 2, 2])
        assert abs(a.mean()) < tol and abs(a.var() - 1) < 2 * tol
        for p, q in [(0, 1), (0, 2), (1, 2)]:
            d = M[..., p, q]
            assert abs(d.mean()) < tol * max(sigma, 1e-9) + 1e-12 and abs(d.var() - sigma ** 2) < 2 * tol * sigma ** 2 + 1e-12
        if sigma > 0:
            c = np.corrcoef(np.stack([a.ravel(), M[..., 0, 1].ravel(), M[..., 0, 2].ravel(), M[..., 1, 2].ravel()]))
            assert np.all(np.abs(c - np.eye(4)) < tol)
    if mode == 1:
        off = M[..., 0, 1]
        assert abs(off.var() - sigma ** 2) < 2 * tol * sigma ** 2
        assert abs(M[..., 0, 0].var() - (1 + sigma ** 2)) < 3 * tol * (1 + sigma ** 2)
    if mode == 2:
        assert abs(M.mean()) < tol and abs(M.var() - sigma ** 2) < tol
        assert not np.allclose(M, np.swapaxes(M, 2, 3))
    if mode == 3:                                                     # J = +-1, D = +-D
        off = M[..., 0, 1]
        assert set(np.unique(off)) == {-sigma, sigma}
        assert set(np.unique(M[..., 0, 0])) <= {-1 - sigma, -1 + sigma, 1 - sigma, 1 + sigma}
        assert abs(np.mean(off > 0) - 0.5) < tol
    assert not np.array_equal(M, oracle.gen_couplings(L, 1, 4, mode, sigma)) or mode == 4


def test_box_muller_normality(oracle):
    from scipy import stats
    M = oracle.gen_couplings(8, 9, 0, 2, 1.0)          # GENERAL9: nine normals per link
    assert stats.kstest(M.ravel(), "norm").pvalue > 1e-3


# ---------------------------------------------------------------------------------------------
# Schwinger-Dyson terms (Eq. (A6)): pins of oracle.sd_terms
# ---------------------------------------------------------------------------------------------
def test_sd_terms_closed_forms_and_energy_relation(oracle):
    """Ferromagnet, all spins equal: h = 6 s, so <s.h> = 6 and <h^2 - (s.h)^2> = 0; staggered: s.h = -6.
    Any couplings: sum_x s.h = -2 H (each link enters the fields of both its ends).  A spin orthogonal to its
    field contributes h^2 to the second term: checked on the dense numpy route (h = A s)."""
    L = 4
    N = L ** 3
    M = oracle.gen_couplings(L, 1, 0, oracle.FERRO, 0.0)
    s = np.zeros((3, N)); s[2] = 1.0
    assert np.allclose(oracle.sd_terms(L, M, s), [6.0, 0.0], atol=1e-14)
    idx = np.arange(N)
    stag = np.where((idx % L + (idx // L) % L + idx // (L * L)) % 2 == 0, 1.0, -1.0)
    s2 = np.zeros((3, N)); s2[2] = stag
    assert np.allclose(oracle.sd_terms(L, M, s2), [-6.0, 0.0], atol=1e-14)
    rng = np.random.default_rng(12)
    for L in (2, 4):
        N = L ** 3
        M = W.random_couplings(rng, N, "general")
        s = W.random_spins(rng, 1, N, fp32=False)[0]
        a, b = oracle.sd_terms(L, M, s)
        assert abs(a * N + 2.0 * oracle.energy(L, M, s)) < 1e-11 * N
        h = np.stack([oracle.local_field(L, M, s, i) for i in range(N)], axis=1)      # [3][N]
        sh = (s * h).sum(axis=0)
        assert abs(b - ((h * h).sum(axis=0) - sh ** 2).mean()) < 1e-12
        assert b >= 0.0                                                                 # |h|^2 >= (s.h)^2 for unit s


# ---------------------------------------------------------------------------------------------
# packed bimodal couplings: pins of oracle.bimodal_couplings / bimodal_links
# ---------------------------------------------------------------------------------------------
def test_bimodal_byte_decodes_to_the_papers_coupling(oracle):
    """Every one of the 128 bytes: M = J 1 + D with J = +-1 and D symmetric, six independent elements +-D (PAPER.md:65,
    73); the map byte -> matrix is injective (7 bits = 7 signs); two bytes worked by hand; and the decoder reproduces
    the BIMODAL generator from the bytes of its own Philox word."""
    D = 0.5
    links = np.zeros((3, 64), dtype=np.uint8)
    links[0] = np.arange(64); links[1] = np.arange(64, 128); links[2, 0] = 0b1011010
    M = oracle.bimodal_couplings(4, links, D)
    mats = np.concatenate([M[0], M[1]])                     # bytes 0 .. 127
    assert np.array_equal(mats, mats.transpose(0, 2, 1))
    off = mats[:, [0, 0, 1], [1, 2, 2]]
    assert np.array_equal(np.abs(off), np.full((128, 3), D))
    J = np.where(np.arange(128) & 1, 1.0, -1.0)
    dd = mats[:, [0, 1, 2], [0, 1, 2]] - J[:, None]
    assert np.array_equal(np.abs(dd), np.full((128, 3), D))
    assert len({m.tobytes() for m in mats}) == 128
    # byte 0: J = -1, all D elements -D.  byte 0b1011010: J = -1; D00 = +, D11 = -, D22 = +; D01 = +, D02 = -, D12 = +
    assert np.array_equal(mats[0], [[-1.5, -0.5, -0.5], [-0.5, -1.5, -0.5], [-0.5, -0.5, -1.5]])
    assert np.array_equal(M[2, 0], [[-0.5, 0.5, -0.5], [0.5, -1.5, 0.5], [-0.5, 0.5, -0.5]])
    for L, seed, sample, Dg in [(4, 9, 3, 0.5), (2, 1, 0, 1.0), (4, 77, 1, 0.3)]:
        bits = oracle.bimodal_links(L, seed, sample)
        assert np.array_equal(oracle.bimodal_couplings(L, bits, Dg), oracle.gen_couplings(L, seed, sample, oracle.BIMODAL, Dg))
        assert 0.4 < np.unpackbits(bits).mean() * 8 / 7 < 0.6      # the signs are balanced (the top bit is always 0)
