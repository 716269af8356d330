"""Pins of the oracle's gather of a replica pair THROUGH the temperature permutation (OracleSim.measure,
measure_chiral, schwinger_dyson; reading R13: PT moves temperatures, measurement is indexed by temperature,
PAPER.md:338, 79).  The spins are built by hand so that the answer at every temperature is known without
the oracle, and the permutations are NOT involutions (slot_of_temp != temp_of_slot), so that gathering with
the wrong one of the two arrays -- the plausible slip -- gives a different, checkable answer.

    replica 0: temp_of_slot = [1, 2, 0]  =>  slot_of_temp = [2, 0, 1]   (temperature 0 sits in slot 2, ...)
    replica 1: temp_of_slot = [2, 0, 1]  =>  slot_of_temp = [1, 2, 0]
"""
import numpy as np

R, T = 2, 3
TOS = np.array([[1, 2, 0], [2, 0, 1]], dtype=np.int32)
SOT = np.array([[2, 0, 1], [1, 2, 0]], dtype=np.int32)     # written out by hand, checked against TOS below


def _sim(oracle, L, couplings, spins):
    sim = oracle.OracleSim(L, 1, R, T, [0.5, 1.0, 1.5], seed=3)
    sim.init_sample(0, couplings=couplings, spins=spins)
    sim.temp_of_slot[0] = TOS
    sim.slot_of_temp[0] = SOT
    return sim


def test_the_two_hand_written_arrays_are_inverse_and_not_involutions():
    for r in range(R):
        for slot in range(T):
            assert SOT[r, TOS[r, slot]] == slot
        assert not np.array_equal(SOT[r], TOS[r])


def test_overlap_gather_uses_the_slot_that_sits_at_temperature_t(oracle):
    """Copy (r, slot) is the constant field a_slot (replica 0) resp. b_slot (replica 1); all nine a_i.b_k differ.
    q^(0)[t] must be a_{slot_of_temp_0[t]} . b_{slot_of_temp_1[t]}:
        t = 0: a_2.b_1 = 6/sqrt(77);   t = 1: a_0.b_2 = 7/sqrt(213);   t = 2: a_1.b_0 = 2/sqrt(14)
    (gathering with temp_of_slot instead would give a_1.b_2, a_2.b_0, a_0.b_1 = 8/sqrt(213), 3/sqrt(14), 4/sqrt(77))."""
    L = 4
    N = L ** 3
    a = np.eye(3)
    b = np.array([[1, 2, 3], [4, 5, 6], [7, 8, 10]], dtype=np.float64)
    b /= np.linalg.norm(b, axis=1, keepdims=True)
    spins = np.zeros((R * T, 3, N))
    for slot in range(T):
        spins[0 * T + slot] = a[slot][:, None]
        spins[1 * T + slot] = b[slot][:, None]
    sim = _sim(oracle, L, np.zeros((3, N, 3, 3)), spins)
    e, q0, qk = sim.measure()
    want = np.array([6 / np.sqrt(77), 7 / np.sqrt(213), 2 / np.sqrt(14)])
    assert np.abs(q0[0, 0] - want).max() < 1e-15
    assert np.abs(qk).max() < 1e-15                   # constant q_x: every k_min mode vanishes
    wrong = np.array([8 / np.sqrt(213), 3 / np.sqrt(14), 4 / np.sqrt(77)])
    assert np.abs(q0[0, 0] - wrong).min() > 0.05      # the slip is far outside the tolerance


def test_chiral_gather_uses_the_slot_that_sits_at_temperature_t(oracle):
    """Only slot 2 of replica 0 and slot 1 of replica 1 hold the conical spiral (zeta_{x,0} = const, closed form of
    tests/test_oracle_chiral.py); every other copy is uniform (zeta = 0).  Both spirals sit at temperature 0 and nowhere
    else together, so q_CG^0(0)[t] = zeta^2 at t = 0 and 0 at t = 1, 2 (with temp_of_slot as the gather the two spirals
    never meet: all zero)."""
    L, al = 8, 0.7
    N = L ** 3
    th = 2 * np.pi / L
    x1 = np.arange(N) % L
    spiral = np.stack([np.sin(al) * np.cos(th * x1), np.sin(al) * np.sin(th * x1), np.cos(al) * np.ones(N)])
    zeta = np.cos(al) * np.sin(al) ** 2 * (np.sin(2 * th) - 2 * np.sin(th))
    spins = np.zeros((R * T, 3, N))
    spins[:, 2] = 1.0
    spins[0 * T + 2] = spiral
    spins[1 * T + 1] = spiral
    sim = _sim(oracle, L, np.zeros((3, N, 3, 3)), spins)
    qc0, qck = sim.measure_chiral()
    want = np.zeros((T, 3)); want[0, 0] = zeta ** 2
    assert abs(zeta) > 0.1
    assert np.abs(qc0[0, 0] - want).max() < 1e-15 and np.abs(qck).max() < 1e-15


def test_schwinger_dyson_gather_uses_the_slot_that_sits_at_temperature_t(oracle):
    """Ferromagnetic couplings M = 1.  Slot 0 of each replica is aligned (s.h = 6, h.h - (s.h)^2 = 0), the other slots are
    staggered (s.h = -6).  Slot 0 sits at temperature 1 in replica 0 and at temperature 2 in replica 1."""
    L = 4
    N = L ** 3
    idx = np.arange(N)
    stag = 1.0 - 2.0 * ((idx % L + (idx // L) % L + idx // (L * L)) % 2)
    spins = np.zeros((R * T, 3, N))
    spins[:, 2] = stag
    spins[0 * T + 0, 2] = 1.0
    spins[1 * T + 0, 2] = 1.0
    M = oracle.gen_couplings(L, 1, 0, oracle.FERRO, 0.0)
    sim = _sim(oracle, L, M, spins)
    sd = sim.schwinger_dyson()
    want = np.array([[-6.0, 6.0, -6.0], [-6.0, -6.0, 6.0]])
    assert np.array_equal(sd[0, :, :, 0], want)
    assert np.array_equal(sd[0, :, :, 1], np.zeros((R, T)))
    # and the energy gather the same way (e = -s.h / 2): the aligned copy has e = -3 at its temperature
    e, _, _ = sim.measure()
    assert np.array_equal(e[0], -want / 2.0)
