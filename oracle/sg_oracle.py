"""TEST INFRASTRUCTURE: ctypes front end of the fp64 CPU oracle (oracle/sg_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from the CUDA package and the CUDA package imports nothing from here.

`OracleSim` mirrors the call sequence of the C-ABI (include/sg_b200.h) -- init_sample, sweep_or,
sweep_hb, pt_swap, measure -- by driving the per-copy C functions; the book-keeping it adds (which
copy sits at which temperature, the two sweep counters) is DESIGN.md section 2/3 written out.
Citations are PAPER.md:<line>.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sg_oracle.c")
_LIB = os.path.join(_HERE, "libsg_oracle.so")

OFFDIAG_SYM, PAPER_SYM6, GENERAL9, BIMODAL, FERRO = 0, 1, 2, 3, 4
KIND_OR, KIND_HB = 0, 1


def build(force=False):
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP over copies only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        u8p = ctypes.POINTER(ctypes.c_uint8)
        u32p = ctypes.POINTER(ctypes.c_uint32)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        i, u32, u64, d = ctypes.c_int, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_double
        L.sgo_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.sgo_uniform23.argtypes = [u32]; L.sgo_uniform23.restype = d
        L.sgo_uniform32.argtypes = [u32]; L.sgo_uniform32.restype = d
        L.sgo_site.argtypes = [i, i, i, i]; L.sgo_site.restype = i
        L.sgo_colour.argtypes = [i, i]; L.sgo_colour.restype = i
        L.sgo_neighbour.argtypes = [i, i, i, i]; L.sgo_neighbour.restype = i
        L.sgo_gen_couplings.argtypes = [i, u64, u32, i, d, dp]
        L.sgo_gen_spins.argtypes = [i, u64, u32, dp]
        L.sgo_local_field.argtypes = [i, dp, dp, i, dp]
        L.sgo_energy.argtypes = [i, dp, dp]; L.sgo_energy.restype = d
        L.sgo_energy_from_fields.argtypes = [i, dp, dp, i]; L.sgo_energy_from_fields.restype = d
        L.sgo_or_update.argtypes = [dp, dp]
        L.sgo_hb_update.argtypes = [dp, d, d, d, dp]
        L.sgo_halfsweep.argtypes = [i, dp, dp, i, i, d, u64, u32, u32, i, u8p, dp, dp]
        L.sgo_hb_uniforms.argtypes = [i, u64, u32, u32, dp, dp]
        L.sgo_sweep_copies.argtypes = [i, dp, dp, i, i, i, dp, u64, u32, u32, i]
        L.sgo_energy_copies.argtypes = [i, dp, dp, i, dp]
        L.sgo_num_threads.restype = i
        L.sgo_pt_sweep.argtypes = [i, dp, dp, ip, ip, u64, u32, u32, u64p, u64p]
        L.sgo_overlap.argtypes = [i, dp, dp, dp]
        L.sgo_chirality.argtypes = [i, dp, i, i]; L.sgo_chirality.restype = d
        L.sgo_chiral_overlap.argtypes = [i, dp, dp, dp]
        L.sgo_xi.argtypes = [i, d, d]; L.sgo_xi.restype = d
        L.sgo_sd_terms.argtypes = [i, dp, dp, dp]
        L.sgo_pt_walk_update.argtypes = [i, ip, ip, u64p, u64p]
        _lib = L
    return _lib


def _dp(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    assert a.dtype == np.int32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def _u64p(a):
    assert a.dtype == np.uint64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64))


# ---------------------------------------------------------------------------------------------
# thin function-level wrappers (one lattice copy = array [3][N]; couplings = array [3][N][3][3])
# ---------------------------------------------------------------------------------------------
def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*[int(v) for v in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(v) for v in key])
    o = (ctypes.c_uint32 * 4)()
    lib().sgo_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniform23(w):
    return lib().sgo_uniform23(int(w))


def uniform32(w):
    return lib().sgo_uniform32(int(w))


def num_threads():
    return int(lib().sgo_num_threads())


def gen_couplings(L, seed, sample, mode=OFFDIAG_SYM, sigma_D=1.0):
    M = np.zeros((3, L ** 3, 3, 3))
    lib().sgo_gen_couplings(L, int(seed), int(sample), int(mode), float(sigma_D), _dp(M))
    return M


def bimodal_couplings(L, links, D):
    """The paper's own couplings from their packed form (Sect. II.A: J_xy = +-1, D_xy symmetric with
    six independent elements +-D; App. A.3: "a full coupling in a single byte").  links uint8 [3][N]:
    bit 0 of the byte of link (x, mu) is the sign of J (1: +1), bits 1, 2, 3 the signs of D^00, D^11, D^22, bits 4, 5, 6
    those of D^01 = D^10, D^02 = D^20, D^12 = D^21 (1: +D).  Returns M [3][N][3][3] = J 1 + D, every entry rounded to
    fp32 (reading R20) -- the bit assignment is that of gen_couplings(mode=BIMODAL) on the word it draws."""
    links = np.asarray(links, dtype=np.uint8).reshape(3, L ** 3)
    M = np.zeros((3, L ** 3, 3, 3))
    for mu in range(3):
        for i in range(L ** 3):
            b = int(links[mu, i])
            J = 1.0 if (b & 1) else -1.0
            d = [float(D) if ((b >> (k + 1)) & 1) else -float(D) for k in range(6)]
            m = np.array([[J + d[0], d[3], d[4]],
                          [d[3], J + d[1], d[5]],
                          [d[4], d[5], J + d[2]]])
            M[mu, i] = m.astype(np.float32).astype(np.float64)
    return M


def bimodal_links(L, seed, sample):
    """The bytes gen_couplings(mode=BIMODAL) uses: the low 7 bits of word 0 of the coupling stream's first block,
    counter (3 i + mu, sample, 0, 4)."""
    N = L ** 3
    out = np.zeros((3, N), dtype=np.uint8)
    key = (int(seed) & 0xffffffff, int(seed) >> 32)
    for i in range(N):
        for mu in range(3):
            out[mu, i] = philox4x32_10((3 * i + mu, int(sample), 0, 4), key)[0] & 0x7f
    return out


def gen_spins(L, seed, g):
    s = np.zeros((3, L ** 3))
    lib().sgo_gen_spins(L, int(seed), int(g), _dp(s))
    return s


def local_field(L, M, s, i):
    h = np.zeros(3)
    lib().sgo_local_field(L, _dp(M), _dp(s), int(i), _dp(h))
    return h


def energy(L, M, s):
    return float(lib().sgo_energy(L, _dp(M), _dp(s)))


def energy_from_fields(L, M, s, colour=-1):
    return float(lib().sgo_energy_from_fields(L, _dp(M), _dp(s), int(colour)))


def or_update(h, s):
    h = np.ascontiguousarray(h, dtype=np.float64)
    out = np.array(s, dtype=np.float64)
    lib().sgo_or_update(_dp(h), _dp(out))
    return out


def hb_update(h, beta, r1, r2):
    h = np.ascontiguousarray(h, dtype=np.float64)
    out = np.zeros(3)
    lib().sgo_hb_update(_dp(h), float(beta), float(r1), float(r2), _dp(out))
    return out


def halfsweep(L, M, s, kind, colour, beta=0.0, seed=0, g=0, hb_counter=0, store_fp32=False,
              want_flags=False, want_sd=False, hnorm_out=None):
    """In-place half-sweep of one copy `s` ([3][N] float64).  Returns (flags or None, sd or None);
    hnorm_out ([N] float64, optional) receives |h_x| of the updated sites."""
    flags = np.zeros(L ** 3, dtype=np.uint8) if want_flags else None
    sd = np.zeros(3) if want_sd else None
    lib().sgo_halfsweep(L, _dp(M), _dp(s), int(kind), int(colour), float(beta), int(seed), int(g),
                        int(hb_counter), int(bool(store_fp32)),
                        flags.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)) if want_flags else None,
                        _dp(hnorm_out) if hnorm_out is not None else None,
                        _dp(sd) if want_sd else None)
    return flags, sd


def hb_uniforms(L, seed, g, hb_counter):
    """(r1 [N], r2 [N]): the uniforms the heat bath draws at every site of copy g in HB sweep hb_counter (test diagnostic)."""
    r1 = np.zeros(L ** 3); r2 = np.zeros(L ** 3)
    lib().sgo_hb_uniforms(L ** 3, int(seed), int(g), int(hb_counter), _dp(r1), _dp(r2))
    return r1, r2


def sweep_copies(L, M, spins, kind, n_sweeps, beta_of_copy=None, seed=0, g0=0, hb_counter0=0,
                 store_fp32=False):
    """n_sweeps full sweeps of spins[n_copies][3][N] in place (OpenMP over copies)."""
    n = spins.shape[0]
    b = np.ascontiguousarray(beta_of_copy if beta_of_copy is not None else np.zeros(n), dtype=np.float64)
    lib().sgo_sweep_copies(L, _dp(M), _dp(spins), n, int(kind), int(n_sweeps), _dp(b), int(seed),
                           int(g0), int(hb_counter0), int(bool(store_fp32)))


def energy_copies(L, M, spins):
    E = np.zeros(spins.shape[0])
    lib().sgo_energy_copies(L, _dp(M), _dp(spins), spins.shape[0], _dp(E))
    return E


def pt_sweep(betas, E_slot, slot_of_temp, temp_of_slot, seed, chain, pt_counter, attempts=None, accepts=None):
    T = len(betas)
    lib().sgo_pt_sweep(T, _dp(np.ascontiguousarray(betas, dtype=np.float64)),
                       _dp(np.ascontiguousarray(E_slot, dtype=np.float64)), _ip(slot_of_temp), _ip(temp_of_slot),
                       int(seed), int(chain), int(pt_counter),
                       _u64p(attempts) if attempts is not None else None,
                       _u64p(accepts) if accepts is not None else None)


def overlap(L, sa, sb):
    out = np.zeros(7)
    lib().sgo_overlap(L, _dp(sa), _dp(sb), _dp(out))
    return out


def chirality(L, s, i, mu):
    """zeta_{x,mu} of Eq. (2) at site i of one copy s [3][N]."""
    return float(lib().sgo_chirality(L, _dp(s), int(i), int(mu)))


def chiral_overlap(L, sa, sb):
    """(qc0[3], qck[3][3][2]): q^_CG^mu(0) and q^_CG^mu(k_nu) (Re, Im) of two copies."""
    out = np.zeros(21)
    lib().sgo_chiral_overlap(L, _dp(sa), _dp(sb), _dp(out))
    return out[:3].copy(), out[3:].reshape(3, 3, 2).copy()


def xi(L, chi0, chik):
    """Second-moment correlation length, Eq. (4)."""
    return float(lib().sgo_xi(int(L), float(chi0), float(chik)))


def sd_terms(L, M, s):
    """(sum_x s.h / N, sum_x [h.h - (s.h)^2] / N) of one copy: the two site averages of Eq. (A6)."""
    out = np.zeros(2)
    lib().sgo_sd_terms(L, _dp(M), _dp(s), _dp(out))
    return out


def pt_walk_update(temp_of_slot, label, round_trips, visits=None):
    """Round-trip / histogram bookkeeping of one chain after a PT sweep; arrays updated in place:
    temp_of_slot int32 [T], label int32 [T], round_trips uint64 [1], visits uint64 [T][T] or None."""
    T = len(temp_of_slot)
    lib().sgo_pt_walk_update(T, _ip(temp_of_slot), _ip(label), _u64p(round_trips),
                             _u64p(visits) if visits is not None else None)


def logbin_index(n):
    """Bin of the n-th measurement (n = 1, 2, ...) in the logarithmic binning of Sect. III: "each bin
    had twice the length of the previous"; bin i holds the measurements 2^i <= n < 2^(i+1), so that after 2^k - 1
    measurements the last bin k-1 is the last half of the series, bin k-2 the second quarter, and so on."""
    assert n >= 1
    i = 0
    while (n >> (i + 1)) > 0:
        i += 1
    return i


def logbin_observables(e, q0, qk, qc0=None, qck=None):
    """The per (sample, temperature) observables O that are binned, [S][T][6], from one measurement (e [S][R][T],
    q0 [S][P][T], qk [S][P][T][3][2]; optionally the chiral-glass overlaps qc0 [S][P][T][3], qck [S][P][T][3][3][2]):
    O[0] mean over replicas of e; O[1] mean over pairs of q0^2; O[2] mean over pairs and the three k_min directions of
    |q(k_mu)|^2 (the chi(0), chi(k_min) estimators of Eq. (3), up to the factor N); O[3] mean over pairs
    of q0^4; O[4] mean over pairs and the chirality direction mu of q_CG^mu(0)^2; O[5] mean over pairs, mu and the three
    k_min directions nu of |q_CG^mu(k_nu)|^2 ("we averaged over all the values of mu", parallel and orthogonal to k_min,
    PAPER.md:97).  No replica pair (R = 1): the overlap entries are 0.  Without qc0 / qck: O[4] = O[5] = 0."""
    S, R, T = e.shape
    out = np.zeros((S, T, 6))
    out[..., 0] = e.mean(axis=1)
    if q0.shape[1] > 0:
        out[..., 1] = (q0 ** 2).mean(axis=1)
        out[..., 2] = (qk ** 2).sum(axis=-1).mean(axis=-1).mean(axis=1)
        out[..., 3] = (q0 ** 4).mean(axis=1)
        if qc0 is not None:
            out[..., 4] = (qc0 ** 2).mean(axis=-1).mean(axis=1)
            out[..., 5] = (qck ** 2).sum(axis=-1).mean(axis=(-1, -2)).mean(axis=1)
    return out


LOGBINS = 32


def walk_tau_int(series, window_c=6.0):
    """Integrated autocorrelation time of a recorded random walk in temperature (Sect. III: "we measured
    the integrated autocorrelation time (mixing time) of the random walk in temperatures of each sample"; the paper
    gives no formula and cites a textbook, Ref. 31 -- the reading taken, R24, is the standard estimator):
        m = mean(x),  C(0) = sum_i (x_i - m)^2 / n,  C(k) = sum_{i < n-k} (x_i - m)(x_{i+k} - m) / (n - k),
        tau(W) = 1/2 + sum_{k=1}^{W} C(k)/C(0),
    summed up to the first W with W >= window_c * tau(W) (self-consistent window), at most n // 2.  In units of the
    sampling interval of the series (one PT sweep = one MCS).  NaN for n < 4 or a constant series."""
    x = np.asarray(series, dtype=np.float64)
    n = x.size
    if n < 4:
        return float("nan")
    d = x - x.mean()
    c0 = float(np.dot(d, d)) / n
    if not c0 > 0.0:
        return float("nan")
    tau = 0.5
    for k in range(1, n // 2 + 1):
        tau += float(np.dot(d[:n - k], d[k:])) / (n - k) / c0
        if k >= window_c * tau:
            break
    return tau


def replica_pairs(R):
    """Pairs a<b in the order (0,1),(0,2),...,(R-2,R-1) (reading R15)."""
    return [(a, b) for a in range(R) for b in range(a + 1, R)]


# ---------------------------------------------------------------------------------------------
# the chain: S samples x (R replicas x T temperatures) copies, MCS = HB + n_or OR + PT
# (Sect. III; App. A.1)
# ---------------------------------------------------------------------------------------------
class OracleSim:
    """State: couplings M[sample] ([3][N][3][3]), spins[sample] ([C][3][N], copy c = r*T + slot),
    the temperature permutation of every chain (sample, r), the HB and PT sweep counters."""

    def __init__(self, L, n_samples, n_replicas, n_temps, betas, seed, store_fp32=True, first_sample=0):
        assert L >= 2 and L % 2 == 0
        self.L, self.S, self.R, self.T = L, n_samples, n_replicas, n_temps
        self.N, self.C = L ** 3, n_replicas * n_temps
        self.betas = np.ascontiguousarray(betas, dtype=np.float64)
        assert self.betas.shape == (n_temps,)
        self.seed = int(seed)
        self.store_fp32 = store_fp32
        # samples are numbered first_sample .. first_sample+S-1 in every Philox counter, so that a
        # rank holding a shard of the samples draws the same numbers as a single process holding all
        self.first_sample = int(first_sample)
        self.M = [None] * self.S
        self.spins = [None] * self.S
        self.slot_of_temp = np.tile(np.arange(self.T, dtype=np.int32), (self.S, self.R, 1))
        self.temp_of_slot = self.slot_of_temp.copy()
        self.hb_counter = 0
        self.pt_counter = 0
        self.attempts = np.zeros((self.S, self.R, max(self.T - 1, 1)), dtype=np.uint64)
        self.accepts = np.zeros_like(self.attempts)
        self.walk_label = np.zeros((self.S, self.R, self.T), dtype=np.int32)
        self.round_trips = np.zeros((self.S, self.R, 1), dtype=np.uint64)
        self.visits = np.zeros((self.S, self.R, self.T, self.T), dtype=np.uint64)   # [slot][t]
        self.n_acc = 0
        self.logbin_sums = np.zeros((LOGBINS, self.S, self.T, 6))
        self.logbin_counts = np.zeros(LOGBINS, dtype=np.uint64)
        self.logbin_counts_cg = np.zeros(LOGBINS, dtype=np.uint64)

    def g0(self, sample):
        return (self.first_sample + sample) * self.C

    def init_sample(self, sample, gen_mode=OFFDIAG_SYM, sigma_D=1.0, couplings=None, spins=None):
        if couplings is None:
            self.M[sample] = gen_couplings(self.L, self.seed, self.first_sample + sample, gen_mode, sigma_D)
        else:
            self.M[sample] = np.ascontiguousarray(couplings, dtype=np.float64).reshape(3, self.N, 3, 3).copy()
        if spins is None:
            self.spins[sample] = np.stack([gen_spins(self.L, self.seed, self.g0(sample) + c)
                                           for c in range(self.C)])
        else:
            self.spins[sample] = np.ascontiguousarray(spins, dtype=np.float64).reshape(self.C, 3, self.N).copy()
        self.slot_of_temp[sample] = np.arange(self.T, dtype=np.int32)
        self.temp_of_slot[sample] = np.arange(self.T, dtype=np.int32)

    def beta_of_copy(self, sample):
        return self.betas[self.temp_of_slot[sample].reshape(-1)]

    def sweep_or(self, n_sweeps=1):
        for s in range(self.S):
            sweep_copies(self.L, self.M[s], self.spins[s], KIND_OR, n_sweeps, None, self.seed, self.g0(s), 0,
                         self.store_fp32)

    def sweep_hb(self, n_sweeps=1):
        for s in range(self.S):
            sweep_copies(self.L, self.M[s], self.spins[s], KIND_HB, n_sweeps, self.beta_of_copy(s), self.seed,
                         self.g0(s), self.hb_counter, self.store_fp32)
        self.hb_counter += n_sweeps

    def halfsweep(self, kind, colour, want_flags=False, want_hnorm=False):
        """One colour of every copy with the current HB counter (not advanced).  Returns flags [S][C][N]
        (and, with want_hnorm, also |h_x| [S][C][N] of the updated sites, 0 elsewhere)."""
        out = np.zeros((self.S, self.C, self.N), dtype=np.uint8) if want_flags else None
        hn = np.zeros((self.S, self.C, self.N)) if want_hnorm else None
        for s in range(self.S):
            b = self.beta_of_copy(s)
            for c in range(self.C):
                f, _ = halfsweep(self.L, self.M[s], self.spins[s][c], kind, colour, b[c], self.seed,
                                 self.g0(s) + c, self.hb_counter, self.store_fp32, want_flags=want_flags,
                                 hnorm_out=hn[s, c] if want_hnorm else None)
                if want_flags:
                    out[s, c] = f
        return (out, hn) if want_hnorm else out

    def energies(self):
        """Total H of every slot, [S][C]."""
        return np.stack([energy_copies(self.L, self.M[s], self.spins[s]) for s in range(self.S)])

    def pt_swap(self, energies=None):
        E = self.energies() if energies is None else np.asarray(energies, dtype=np.float64)
        for s in range(self.S):
            for r in range(self.R):
                chain = (self.first_sample + s) * self.R + r
                pt_sweep(self.betas, E[s, r * self.T:(r + 1) * self.T], self.slot_of_temp[s, r],
                         self.temp_of_slot[s, r], self.seed, chain, self.pt_counter,
                         self.attempts[s, r], self.accepts[s, r])
                pt_walk_update(self.temp_of_slot[s, r], self.walk_label[s, r], self.round_trips[s, r], self.visits[s, r])
        self.pt_counter += 1

    def measure(self):
        """e[S][R][T] = H/N at temperature t; q0[S][P][T], qk[S][P][T][3][2] for replica pairs a<b with
        both copies at temperature t (readings R15, R16)."""
        E = self.energies()
        pairs = replica_pairs(self.R)
        e = np.zeros((self.S, self.R, self.T))
        q0 = np.zeros((self.S, len(pairs), self.T))
        qk = np.zeros((self.S, len(pairs), self.T, 3, 2))
        for s in range(self.S):
            for r in range(self.R):
                for t in range(self.T):
                    e[s, r, t] = E[s, r * self.T + self.slot_of_temp[s, r, t]] / self.N
            for p, (a, b) in enumerate(pairs):
                for t in range(self.T):
                    sa = self.spins[s][a * self.T + self.slot_of_temp[s, a, t]]
                    sb = self.spins[s][b * self.T + self.slot_of_temp[s, b, t]]
                    o = overlap(self.L, sa, sb)
                    q0[s, p, t] = o[0]
                    qk[s, p, t] = o[1:].reshape(3, 2)
        return e, q0, qk

    def accumulate(self, with_chirality=False):
        """Measure and add into the logarithmic bins: the n-th call goes to bin logbin_index(n); the
        chiral-glass entries O[4], O[5] only with `with_chirality` (their own count per bin)."""
        self.n_acc += 1
        b = logbin_index(self.n_acc)
        cg = self.measure_chiral() if with_chirality else (None, None)
        self.logbin_sums[b] += logbin_observables(*self.measure(), *cg)
        self.logbin_counts[b] += 1
        if with_chirality:
            self.logbin_counts_cg[b] += 1

    def measure_chiral(self):
        """qc0[S][P][T][3], qck[S][P][T][3][3][2]: chiral-glass overlaps of the replica pairs a<b with both
        copies at temperature t (Eq. (2))."""
        pairs = replica_pairs(self.R)
        qc0 = np.zeros((self.S, len(pairs), self.T, 3))
        qck = np.zeros((self.S, len(pairs), self.T, 3, 3, 2))
        for s in range(self.S):
            for p, (a, b) in enumerate(pairs):
                for t in range(self.T):
                    sa = self.spins[s][a * self.T + self.slot_of_temp[s, a, t]]
                    sb = self.spins[s][b * self.T + self.slot_of_temp[s, b, t]]
                    qc0[s, p, t], qck[s, p, t] = chiral_overlap(self.L, sa, sb)
        return qc0, qck

    def schwinger_dyson(self):
        """sd[S][R][T][2]: the two site averages of Eq. (A6) for the copy of replica r at temperature t."""
        out = np.zeros((self.S, self.R, self.T, 2))
        for s in range(self.S):
            for r in range(self.R):
                for t in range(self.T):
                    out[s, r, t] = sd_terms(self.L, self.M[s], self.spins[s][r * self.T + self.slot_of_temp[s, r, t]])
        return out

    def unit(self, n_or):
        """One MCS: 1 HB sweep, n_or OR sweeps, 1 PT sweep."""
        self.sweep_hb(1)
        self.sweep_or(n_or)
        self.pt_swap()
