"""Pins of the oracle's chirality observables (Eq. (2)) and of the second-moment correlation
length (Eq. (4)): closed forms, symmetries, and an independent numpy route (np.linalg.det,
np.roll, np.fft) for the indexing.  CPU only."""
import numpy as np
import pytest

import sg_workloads as W


def site_coords(L):
    i = np.arange(L ** 3)
    return i % L, (i // L) % L, i // (L * L)


def numpy_zeta(L, s):
    """zeta[mu][N] by an independent route: determinant of the 3x3 matrix with rows s_{x+mu}, s_x, s_{x-mu}."""
    f = s.reshape(3, L, L, L)                         # [comp][x3][x2][x1]
    out = np.zeros((3, L ** 3))
    for mu in range(3):
        ax = 3 - mu                                   # x1 is the fastest index
        plus, minus = np.roll(f, -1, axis=ax), np.roll(f, 1, axis=ax)
        rows = np.stack([plus, f, minus], axis=0)     # [row][comp][...]
        m = np.moveaxis(rows.reshape(3, 3, -1), -1, 0)
        out[mu] = np.linalg.det(m)
    return out


def test_zeta_of_orthonormal_triads(oracle):
    """s_x = x^, s_{x-mu} = y^, s_{x+mu} = z^: zeta = z^.(x^ x y^) = +1; swapping the two neighbours gives -1;
    coplanar spins give 0 (Eq. (2): an oriented volume)."""
    L = 4
    N = L ** 3
    for mu in range(3):
        i = 21
        ip, im = oracle.lib().sgo_neighbour(L, i, mu, 1), oracle.lib().sgo_neighbour(L, i, mu, -1)
        s = np.zeros((3, N)); s[0, :] = 1.0
        s[:, i] = [1, 0, 0]; s[:, im] = [0, 1, 0]; s[:, ip] = [0, 0, 1]
        assert oracle.chirality(L, s, i, mu) == 1.0
        s[:, im], s[:, ip] = [0, 0, 1], [0, 1, 0]
        assert oracle.chirality(L, s, i, mu) == -1.0
        s[:, ip] = [0.6, 0.8, 0.0]; s[:, im] = [0.0, 1.0, 0.0]
        assert abs(oracle.chirality(L, s, i, mu)) < 1e-16


@pytest.mark.parametrize("L", [2, 4, 6])
def test_zeta_matches_numpy_determinant(oracle, L):
    rng = np.random.default_rng(5 + L)
    s = W.random_spins(rng, 1, L ** 3)[0]
    ref = numpy_zeta(L, s)
    got = np.array([[oracle.chirality(L, s, i, mu) for i in range(L ** 3)] for mu in range(3)])
    assert np.abs(got - ref).max() < 1e-14
    if L == 2:                                        # x+e and x-e coincide: two equal rows
        assert np.abs(got).max() < 1e-15


def test_zeta_symmetries(oracle):
    """Invariant under a global proper rotation, odd under s -> -s and under an improper rotation."""
    L = 4
    rng = np.random.default_rng(8)
    s = W.random_spins(rng, 1, L ** 3, fp32=False)[0]
    Rp = W.random_rotations(rng, 1, proper=True)[0]
    Ri = Rp @ np.diag([1.0, 1.0, -1.0])
    for i, mu in [(0, 0), (13, 1), (63, 2), (37, 0)]:
        z = oracle.chirality(L, s, i, mu)
        assert abs(oracle.chirality(L, Rp @ s, i, mu) - z) < 1e-14
        assert abs(oracle.chirality(L, Ri @ s, i, mu) + z) < 1e-14
        assert abs(oracle.chirality(L, -s, i, mu) + z) < 1e-14


def test_conical_spiral_closed_form(oracle):
    """s_x = (sin a cos(theta x1), sin a sin(theta x1), cos a): zeta_{x,0} = cos a sin^2 a (sin 2 theta - 2 sin theta)
    at every site, zeta_{x,1} = zeta_{x,2} = 0 (spins constant along x2, x3).  Two identical replicas:
    q^_CG^0(0) = zeta^2, every k_min mode vanishes."""
    L, m, a = 8, 1, 0.7
    th = 2 * np.pi * m / L
    x1, _, _ = site_coords(L)
    s = np.stack([np.sin(a) * np.cos(th * x1), np.sin(a) * np.sin(th * x1), np.cos(a) * np.ones(L ** 3)])
    zeta = np.cos(a) * np.sin(a) ** 2 * (np.sin(2 * th) - 2 * np.sin(th))
    for i in (0, 7, 100, 511):
        assert abs(oracle.chirality(L, s, i, 0) - zeta) < 1e-15
        assert abs(oracle.chirality(L, s, i, 1)) < 1e-16 and abs(oracle.chirality(L, s, i, 2)) < 1e-16
    qc0, qck = oracle.chiral_overlap(L, s, s)
    assert np.allclose(qc0, [zeta ** 2, 0, 0], atol=1e-15)
    assert np.abs(qck).max() < 1e-15
    # opposite handedness in replica b (theta -> -theta): kappa = -zeta^2
    sb = s.copy(); sb[1] = -sb[1]
    qc0, _ = oracle.chiral_overlap(L, s, sb)
    assert np.allclose(qc0, [-zeta ** 2, 0, 0], atol=1e-15)


def test_modulated_cone_fixes_fourier_sign_and_axis(oracle):
    """Replica a: uniform conical spiral along x1 (zeta^a_0 = const).  Replica b: the same spiral whose handedness
    is modulated along x2 with period L/2 planes... realised by mirroring s_y on the planes x2 >= L/2; then
    kappa_{x,0} = zeta^2 * sgn(x2) away from nothing else (x2 is not the spiral axis), a square wave along x2 whose
    k_min Fourier coefficient is known in closed form; the axes x1, x3 see nothing."""
    L, a = 8, 0.9
    th = 2 * np.pi / L
    x1, x2, _ = site_coords(L)
    s = np.stack([np.sin(a) * np.cos(th * x1), np.sin(a) * np.sin(th * x1), np.cos(a) * np.ones(L ** 3)])
    sb = s.copy()
    sb[1, x2 >= L // 2] *= -1.0
    zeta2 = (np.cos(a) * np.sin(a) ** 2 * (np.sin(2 * th) - 2 * np.sin(th))) ** 2
    sq = np.where(np.arange(L) >= L // 2, -1.0, 1.0)
    coef = (sq * np.exp(2j * np.pi * np.arange(L) / L)).sum() / L
    qc0, qck = oracle.chiral_overlap(L, s, sb)
    assert abs(qc0[0]) < 1e-15
    assert abs(qck[0, 1, 0] - zeta2 * coef.real) < 1e-15 and abs(qck[0, 1, 1] - zeta2 * coef.imag) < 1e-15
    assert np.abs(qck[0, 0]).max() < 1e-15 and np.abs(qck[0, 2]).max() < 1e-15
    assert np.abs(qck[1:]).max() < 1e-15 and np.abs(qc0[1:]).max() < 1e-15


@pytest.mark.parametrize("L", [4, 6])
def test_chiral_overlap_matches_numpy_fft(oracle, L):
    rng = np.random.default_rng(31 + L)
    sa, sb = W.random_spins(rng, 2, L ** 3)
    kap = numpy_zeta(L, sa) * numpy_zeta(L, sb)                      # [mu][N]
    qc0, qck = oracle.chiral_overlap(L, sa, sb)
    assert np.abs(qc0 - kap.mean(axis=1)).max() < 1e-14
    for mu in range(3):
        F = np.fft.ifftn(kap[mu].reshape(L, L, L))                   # sum kappa e^{+i k.x} / N; axes (x3, x2, x1)
        want = [F[0, 0, 1], F[0, 1, 0], F[1, 0, 0]]
        for nu in range(3):
            assert abs(qck[mu, nu, 0] + 1j * qck[mu, nu, 1] - want[nu]) < 1e-14


def test_chiral_overlap_symmetry_and_statistics(oracle):
    """kappa is symmetric in (a, b); inverting ONE replica flips its sign; for independent uniform spins the mean
    vanishes and <zeta^2> = 2/9 (zeta = det of three independent uniform unit vectors: E[det^2] = 3!/3^3)."""
    L = 6
    rng = np.random.default_rng(77)
    sa, sb = W.random_spins(rng, 2, L ** 3, fp32=False)
    a0, ak = oracle.chiral_overlap(L, sa, sb)
    b0, bk = oracle.chiral_overlap(L, sb, sa)
    assert np.array_equal(a0, b0) and np.array_equal(ak, bk)
    c0, ck = oracle.chiral_overlap(L, -sa, sb)
    assert np.allclose(c0, -a0, atol=1e-16) and np.allclose(ck, -ak, atol=1e-16)
    z2 = []
    for seed in range(40):
        s = W.random_spins(np.random.default_rng(1000 + seed), 1, L ** 3, fp32=False)[0]
        z2.append(oracle.chiral_overlap(L, s, s)[0].mean())          # kappa = zeta^2 for identical replicas
    z2 = np.array(z2)
    assert abs(z2.mean() - 2.0 / 9.0) < 4.5 * z2.std(ddof=1) / np.sqrt(len(z2))


def test_xi_inverts_the_lattice_propagator(oracle):
    """Eq. (4) is built so that a lattice Ornstein-Zernike propagator chi(k) = A / (xi^-2 + 4 sin^2(k/2)) gives
    back xi exactly."""
    for L in (8, 16, 64):
        for xi in (0.3, 1.0, 5.0, 40.0):
            k = 2 * np.pi / L
            chi = lambda kk: 3.7 / (xi ** -2 + 4 * np.sin(kk / 2) ** 2)
            assert abs(oracle.xi(L, chi(0.0), chi(k)) - xi) < 1e-9 * xi
    assert np.isnan(oracle.xi(8, 1.0, 2.0))
