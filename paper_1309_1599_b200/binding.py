"""ctypes binding of libsg_b200.so: argument marshalling only -- every step of the path runs in the
library's CUDA kernels.  torch is used for device memory (the workspace tensor) and the stream.
Method names follow include/sg_b200.h (sg_init_sample -> init_sample, ...)."""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsg_b200.so")

GEN_OFFDIAG_SYM, GEN_PAPER_SYM6, GEN_GENERAL9, GEN_BIMODAL, GEN_FERRO = 0, 1, 2, 3, 4
KIND_OR, KIND_HB = 0, 1
SHAPE_FUSED_BUFFER = 1
SG_OK, SG_EINVAL, SG_ESTATE, SG_ECUDA, SG_ELIMIT = 0, -1, -2, -3, -4
STATIC_SCRATCH_BYTES, STATIC_MAX_L = 16 << 20, 256
TUNE_SWEEP_IMPL, TUNE_ZCHUNK, TUNE_RES_COPIES, TUNE_PACKED, TUNE_MEASURE_IMPL, TUNE_GRAPH, TUNE_CLUSTER_CTAS = 0, 1, 2, 3, 4, 5, 6
MEASURE_AUTO, MEASURE_STAGED = 0, 1
LOGBINS, LOGBIN_OBS = 32, 6
SWEEP_AUTO, SWEEP_TILED, SWEEP_ZMARCH, SWEEP_RESIDENT, SWEEP_FUSED, SWEEP_CLUSTER = 0, 1, 2, 3, 4, 5

# every symbol include/sg_b200.h declares (checked against the header by tests/test_abi.py)
DECLARED_SYMBOLS = [
    "sg_workspace_bytes", "sg_create", "sg_destroy", "sg_init_sample", "sg_init_sample_bimodal", "sg_sweep_or", "sg_sweep_hb",
    "sg_pt_swap", "sg_pt_publish", "sg_pt_swap_gathered", "sg_energy_by_temp", "sg_run_units", "sg_measure", "sg_accumulate", "sg_get_logbins", "sg_export_replica", "sg_measure_cross", "sg_export_chirality", "sg_chiral_cross", "sg_chiral_cross_static", "sg_measure_chiral", "sg_schwinger_dyson", "sg_correlation_length", "sg_get_spins", "sg_set_spins", "sg_get_couplings", "sg_get_perm",
    "sg_set_perm", "sg_get_energies", "sg_set_energies", "sg_get_counters", "sg_set_counters",
    "sg_halfsweep", "sg_pt_stats", "sg_pt_walk", "sg_pt_visits", "sg_walk_tau_int", "sg_tune", "sg_sweep_impl_used", "sg_sync", "sg_kernel_launches", "sg_graph_replays", "sg_last_cuda_error", "sg_strerror",
    "sg_philox4x32_10",
]


class SgShape(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int32), ("n_samples", ctypes.c_int32), ("n_replicas", ctypes.c_int32),
                ("n_temps", ctypes.c_int32), ("first_sample", ctypes.c_int32), ("first_replica", ctypes.c_int32),
                ("n_replicas_total", ctypes.c_int32), ("flags", ctypes.c_int32),
                ("seed", ctypes.c_uint64), ("first_slot", ctypes.c_int32), ("n_temps_total", ctypes.c_int32)]


class SgError(RuntimeError):
    def __init__(self, code, what, cuda_error=0):
        self.code, self.cuda_error = code, cuda_error
        super().__init__("%s failed: %s (code %d, cudaError %d)" % (what, _strerror(code), code, cuda_error))


_lib = None


def load_library():
    """Loads libsg_b200.so (built by paper_1309_1599_b200/build.py); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = _LIB_PATH
    if not os.path.exists(path):
        raise ImportError("libsg_b200.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(path)
    vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    u64 = ctypes.c_uint64
    shp = ctypes.POINTER(SgShape)
    L.sg_workspace_bytes.argtypes = [shp]; L.sg_workspace_bytes.restype = ctypes.c_size_t
    L.sg_create.argtypes = [ctypes.POINTER(vp), shp, vp, vp, ctypes.c_size_t, vp]; L.sg_create.restype = i
    L.sg_destroy.argtypes = [vp]; L.sg_destroy.restype = i
    L.sg_init_sample.argtypes = [vp, i, i, d, vp, vp]; L.sg_init_sample.restype = i
    L.sg_init_sample_bimodal.argtypes = [vp, i, d, vp, vp]; L.sg_init_sample_bimodal.restype = i
    L.sg_sweep_or.argtypes = [vp, i]; L.sg_sweep_or.restype = i
    L.sg_sweep_hb.argtypes = [vp, i]; L.sg_sweep_hb.restype = i
    L.sg_pt_swap.argtypes = [vp]; L.sg_pt_swap.restype = i
    L.sg_pt_publish.argtypes = [vp, vp]; L.sg_pt_publish.restype = i
    L.sg_pt_swap_gathered.argtypes = [vp, vp]; L.sg_pt_swap_gathered.restype = i
    L.sg_energy_by_temp.argtypes = [vp, vp, vp]; L.sg_energy_by_temp.restype = i
    L.sg_pt_visits.argtypes = [vp, vp]; L.sg_pt_visits.restype = i
    L.sg_walk_tau_int.argtypes = [vp, ctypes.c_int64, d]; L.sg_walk_tau_int.restype = d
    L.sg_measure.argtypes = [vp, vp, vp, vp]; L.sg_measure.restype = i
    L.sg_run_units.argtypes = [vp, i, i]; L.sg_run_units.restype = i
    L.sg_measure_chiral.argtypes = [vp, vp, vp]; L.sg_measure_chiral.restype = i
    L.sg_schwinger_dyson.argtypes = [vp, vp]; L.sg_schwinger_dyson.restype = i
    L.sg_correlation_length.argtypes = [i, ctypes.c_double, ctypes.c_double]; L.sg_correlation_length.restype = ctypes.c_double
    L.sg_get_spins.argtypes = [vp, i, vp]; L.sg_get_spins.restype = i
    L.sg_set_spins.argtypes = [vp, i, vp]; L.sg_set_spins.restype = i
    L.sg_get_couplings.argtypes = [vp, i, vp]; L.sg_get_couplings.restype = i
    L.sg_get_perm.argtypes = [vp, i, vp, vp]; L.sg_get_perm.restype = i
    L.sg_set_perm.argtypes = [vp, i, vp]; L.sg_set_perm.restype = i
    L.sg_get_energies.argtypes = [vp, vp]; L.sg_get_energies.restype = i
    L.sg_set_energies.argtypes = [vp, vp]; L.sg_set_energies.restype = i
    L.sg_get_counters.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64)]; L.sg_get_counters.restype = i
    L.sg_set_counters.argtypes = [vp, u64, u64]; L.sg_set_counters.restype = i
    L.sg_halfsweep.argtypes = [vp, i, i]; L.sg_halfsweep.restype = i
    L.sg_pt_stats.argtypes = [vp, vp, vp]; L.sg_pt_stats.restype = i
    L.sg_accumulate.argtypes = [vp, i]; L.sg_accumulate.restype = i
    L.sg_get_logbins.argtypes = [vp, vp, vp, vp]; L.sg_get_logbins.restype = i
    L.sg_export_replica.argtypes = [vp, i, vp]; L.sg_export_replica.restype = i
    L.sg_measure_cross.argtypes = [vp, i, vp, vp, vp]; L.sg_measure_cross.restype = i
    L.sg_export_chirality.argtypes = [vp, i, vp]; L.sg_export_chirality.restype = i
    L.sg_chiral_cross.argtypes = [vp, vp, vp, vp, vp]; L.sg_chiral_cross.restype = i
    L.sg_chiral_cross_static.argtypes = [i, i, i, vp, vp, vp, vp, ctypes.POINTER(i)]; L.sg_chiral_cross_static.restype = i
    L.sg_pt_walk.argtypes = [vp, vp, vp]; L.sg_pt_walk.restype = i
    L.sg_tune.argtypes = [vp, i, i]; L.sg_tune.restype = i
    L.sg_sweep_impl_used.argtypes = [vp, i, ctypes.POINTER(i)]; L.sg_sweep_impl_used.restype = i
    L.sg_sync.argtypes = [vp]; L.sg_sync.restype = i
    L.sg_kernel_launches.argtypes = [vp]; L.sg_kernel_launches.restype = u64
    L.sg_graph_replays.argtypes = [vp]; L.sg_graph_replays.restype = u64
    L.sg_last_cuda_error.argtypes = [vp]; L.sg_last_cuda_error.restype = i
    L.sg_strerror.argtypes = [i]; L.sg_strerror.restype = ctypes.c_char_p
    L.sg_philox4x32_10.argtypes = [ctypes.POINTER(ctypes.c_uint32)] * 3; L.sg_philox4x32_10.restype = None
    _lib = L
    return L


def _strerror(code):
    return load_library().sg_strerror(int(code)).decode()


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data) if a is not None else None


def workspace_bytes(L, n_samples, n_replicas, n_temps, seed=0, first_sample=0):
    shape = SgShape(L, n_samples, n_replicas, n_temps, first_sample, 0, 0, 0, seed, 0, 0)
    return int(load_library().sg_workspace_bytes(ctypes.byref(shape)))


def walk_tau_int(series, window_c=0.0):
    """integrated autocorrelation time (in PT sweeps) of a recorded walk in temperature (sg_walk_tau_int)."""
    x = np.ascontiguousarray(series, dtype=np.int32)
    return float(load_library().sg_walk_tau_int(_ptr(x), int(x.size), float(window_c)))


def correlation_length(L, chi0, chik):
    """Eq. (4): second-moment correlation length from chi(0), chi(k_min)."""
    return float(load_library().sg_correlation_length(int(L), float(chi0), float(chik)))


def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*[int(v) for v in ctr]); k = (ctypes.c_uint32 * 2)(*[int(v) for v in key])
    o = (ctypes.c_uint32 * 4)()
    load_library().sg_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def chiral_cross_static(L, n_samples, n_temps, za, zb, out=None, stream=None):
    """sg_chiral_cross_static: the chiral-glass overlaps between two export_chirality tensors WITHOUT a context and without
    the library allocating anything -- for callers that hold two zeta buffers on the device but must not (all of HBM is already
    handed out), cannot afford to (cudaMalloc / cudaFree stall every stream of the GPU) or are not allowed to allocate.  The
    partial sums go to a fixed 16 MiB array inside the library (STATIC_SCRATCH_BYTES; every GPU that loads the library holds
    it until the process exits), so n_samples <= 3 per call is always accepted and larger shapes raise SgError(SG_ELIMIT):
    split them by sample.  All calls on a device share that array: order them on one stream, or they race.  The first call on
    a device looks the array's address up; make it during set-up.

    za, zb: float32 device tensors [n_samples][3][L^3][n_temps]; out: float64 device tensor of n_samples * n_temps * 21
    elements (pass one you already own if even torch must not allocate; None = torch.empty).  Asynchronous on `stream` (torch's
    current stream if None).  Returns (qc0 [S][T][3], qck [S][T][3][3][2]) as views of `out`, still on the device."""
    import torch
    S, T, N = int(n_samples), int(n_temps), int(L) ** 3
    for z in (za, zb):
        assert z.is_cuda and z.is_contiguous() and z.dtype == torch.float32 and z.numel() == S * 3 * N * T
    if out is None:
        out = torch.empty(S * T * 21, dtype=torch.float64, device=za.device)
    assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float64 and out.numel() == S * T * 21
    assert out.device == za.device == zb.device == torch.device("cuda", torch.cuda.current_device()), "buffers must be on the current device"
    if stream is None:
        stream = torch.cuda.current_stream(za.device)
    err = ctypes.c_int(0)
    rc = load_library().sg_chiral_cross_static(int(L), S, T, ctypes.c_void_p(za.data_ptr()), ctypes.c_void_p(zb.data_ptr()),
                                               ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(stream.cuda_stream), ctypes.byref(err))
    if rc != SG_OK:
        raise SgError(rc, "sg_chiral_cross_static", int(err.value))
    flat = out.view(-1)
    return flat[:S * T * 3].view(S, T, 3), flat[S * T * 3:].view(S, T, 3, 3, 2)


class SpinGlass:
    """One context of the C-ABI library on the current CUDA device and torch's current stream."""

    def __init__(self, L, n_samples, n_replicas, n_temps, betas, seed=1, first_sample=0, device=None, stream=None,
                 first_replica=0, n_replicas_total=0, first_slot=0, n_temps_total=0, fused_buffer=False):
        import torch
        self._lib = load_library()
        self.L, self.S, self.R, self.T = int(L), int(n_samples), int(n_replicas), int(n_temps)
        self.N, self.C, self.P = self.L ** 3, self.R * self.T, self.R * (self.R - 1) // 2
        self.Tt = int(n_temps_total) if n_temps_total else self.T      # length of the PT chain (> T: temperature-slot sharding)
        self.shape = SgShape(self.L, self.S, self.R, self.T, int(first_sample), int(first_replica), int(n_replicas_total), SHAPE_FUSED_BUFFER if fused_buffer else 0, int(seed),
                             int(first_slot), int(n_temps_total))
        nbytes = int(self._lib.sg_workspace_bytes(ctypes.byref(self.shape)))
        if nbytes == 0:
            raise SgError(SG_EINVAL, "sg_workspace_bytes")
        if not torch.cuda.is_available():
            raise SgError(SG_ECUDA, "sg_create (no CUDA device; there is no CPU fallback)")
        self.device = torch.device(device if device is not None else "cuda:%d" % torch.cuda.current_device())
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) & ~255
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        betas = np.ascontiguousarray(betas, dtype=np.float64)
        if betas.shape != (self.Tt,):
            raise SgError(SG_EINVAL, "sg_create (betas must have n_temps (n_temps_total) entries)")
        self._ctx = ctypes.c_void_p()
        rc = self._lib.sg_create(ctypes.byref(self._ctx), ctypes.byref(self.shape), _ptr(betas), ctypes.c_void_p(aligned),
                                 nbytes, ctypes.c_void_p(self.stream.cuda_stream))
        if rc != SG_OK:
            self._ctx = None
            raise SgError(rc, "sg_create")
        self.workspace_bytes = nbytes

    def _check(self, rc, what):
        if rc != SG_OK:
            raise SgError(rc, what, self._lib.sg_last_cuda_error(self._ctx))

    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.sg_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the five calls of the north star ----
    def init_sample(self, sample, gen_mode=GEN_OFFDIAG_SYM, sigma_D=1.0, couplings=None, spins=None):
        if couplings is not None:
            couplings = np.ascontiguousarray(couplings, dtype=np.float32)
            assert couplings.size == 27 * self.N
        if spins is not None:
            spins = np.ascontiguousarray(spins, dtype=np.float32)
            assert spins.size == 3 * self.N * self.C
        self._check(self._lib.sg_init_sample(self._ctx, int(sample), int(gen_mode), float(sigma_D), _ptr(couplings),
                                             _ptr(spins)), "sg_init_sample")

    def init_sample_bimodal(self, sample, D, links=None, spins=None):
        """The paper's J = +-1, D^ab = +-D couplings from one byte per link (uint8 [3][N]; None: the generator's bytes)."""
        if links is not None:
            links = np.ascontiguousarray(links, dtype=np.uint8)
            assert links.size == 3 * self.N
        if spins is not None:
            spins = np.ascontiguousarray(spins, dtype=np.float32)
            assert spins.size == 3 * self.N * self.C
        self._check(self._lib.sg_init_sample_bimodal(self._ctx, int(sample), float(D), _ptr(links), _ptr(spins)),
                    "sg_init_sample_bimodal")

    def sweep_or(self, n_sweeps=1):
        self._check(self._lib.sg_sweep_or(self._ctx, int(n_sweeps)), "sg_sweep_or")

    def sweep_hb(self, n_sweeps=1):
        self._check(self._lib.sg_sweep_hb(self._ctx, int(n_sweeps)), "sg_sweep_hb")

    def pt_swap(self):
        self._check(self._lib.sg_pt_swap(self._ctx), "sg_pt_swap")

    def pt_publish(self, out=None):
        """Device tensor float64 [S][R][T]: the total energies of this context's slots (the send buffer of the all-gather of a
        slot-sharded chain; asynchronous)."""
        import torch
        if out is None:
            out = torch.empty((self.S, self.R, self.T), dtype=torch.float64, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float64 and out.numel() == self.S * self.C
        self._check(self._lib.sg_pt_publish(self._ctx, ctypes.c_void_p(out.data_ptr())), "sg_pt_publish")
        return out

    def pt_swap_gathered(self, gathered):
        """One PT sweep from the all-gathered energies, device tensor float64 [W][S][R][T], W = n_temps_total / n_temps."""
        assert gathered.is_cuda and gathered.is_contiguous() and gathered.numel() == (self.Tt // self.T) * self.S * self.C
        self._check(self._lib.sg_pt_swap_gathered(self._ctx, ctypes.c_void_p(gathered.data_ptr())), "sg_pt_swap_gathered")

    def energy_by_temp(self, gathered):
        """e [S][R][n_temps_total] = H/N of the copy of replica r at temperature t, from the all-gathered energies."""
        assert gathered.is_cuda and gathered.is_contiguous() and gathered.numel() == (self.Tt // self.T) * self.S * self.C
        e = np.empty((self.S, self.R, self.Tt))
        self._check(self._lib.sg_energy_by_temp(self._ctx, ctypes.c_void_p(gathered.data_ptr()), _ptr(e)), "sg_energy_by_temp")
        return e

    def measure(self):
        e = np.empty((self.S, self.R, self.T)); q0 = np.empty((self.S, self.P, self.T))
        qk = np.empty((self.S, self.P, self.T, 3, 2))
        self._check(self._lib.sg_measure(self._ctx, _ptr(e), _ptr(q0), _ptr(qk)), "sg_measure")
        return e, q0, qk

    def run_units(self, n_units, n_or):
        """n_units MCS (1 HB + n_or OR + PT each) issued from native code."""
        self._check(self._lib.sg_run_units(self._ctx, int(n_units), int(n_or)), "sg_run_units")

    def measure_chiral(self):
        """(qc0 [S][P][T][3], qck [S][P][T][3][3][2]): chiral-glass overlaps, Eq. (2) PAPER.md:81-85."""
        qc0 = np.empty((self.S, self.P, self.T, 3)); qck = np.empty((self.S, self.P, self.T, 3, 3, 2))
        self._check(self._lib.sg_measure_chiral(self._ctx, _ptr(qc0), _ptr(qck)), "sg_measure_chiral")
        return qc0, qck

    def schwinger_dyson(self):
        """sd [S][R][T][2]: site averages of s.h and of h.h - (s.h)^2 per (replica, temperature), Eq. (A6)."""
        sd = np.empty((self.S, self.R, self.Tt, 2))      # by the chain's temperatures; zeros for those another slot shard holds
        self._check(self._lib.sg_schwinger_dyson(self._ctx, _ptr(sd)), "sg_schwinger_dyson")
        return sd

    def unit(self, n_or):
        """One MCS: 1 HB sweep, n_or OR sweeps, 1 PT sweep."""
        self.sweep_hb(1)
        self.sweep_or(n_or)
        self.pt_swap()

    # ---- state access ----
    def get_spins(self, sample):
        out = np.empty((self.C, 3, self.N), dtype=np.float32)
        self._check(self._lib.sg_get_spins(self._ctx, int(sample), _ptr(out)), "sg_get_spins")
        return out

    def set_spins(self, sample, spins):
        spins = np.ascontiguousarray(spins, dtype=np.float32)
        assert spins.size == 3 * self.N * self.C
        self._check(self._lib.sg_set_spins(self._ctx, int(sample), _ptr(spins)), "sg_set_spins")

    def get_couplings(self, sample):
        out = np.empty((3, self.N, 3, 3), dtype=np.float32)
        self._check(self._lib.sg_get_couplings(self._ctx, int(sample), _ptr(out)), "sg_get_couplings")
        return out

    def get_perm(self, sample):
        tos = np.empty((self.R, self.Tt), dtype=np.int32); sot = np.empty((self.R, self.Tt), dtype=np.int32)
        self._check(self._lib.sg_get_perm(self._ctx, int(sample), _ptr(tos), _ptr(sot)), "sg_get_perm")
        return tos, sot

    def set_perm(self, sample, temp_of_slot):
        tos = np.ascontiguousarray(temp_of_slot, dtype=np.int32)
        assert tos.shape == (self.R, self.Tt)
        self._check(self._lib.sg_set_perm(self._ctx, int(sample), _ptr(tos)), "sg_set_perm")

    def get_energies(self):
        E = np.empty((self.S, self.C))
        self._check(self._lib.sg_get_energies(self._ctx, _ptr(E)), "sg_get_energies")
        return E

    def set_energies(self, E):
        E = np.ascontiguousarray(E, dtype=np.float64)
        assert E.shape == (self.S, self.C)
        self._check(self._lib.sg_set_energies(self._ctx, _ptr(E)), "sg_set_energies")

    def get_counters(self):
        hb, pt = ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self._lib.sg_get_counters(self._ctx, ctypes.byref(hb), ctypes.byref(pt)), "sg_get_counters")
        return int(hb.value), int(pt.value)

    def set_counters(self, hb, pt):
        self._check(self._lib.sg_set_counters(self._ctx, int(hb), int(pt)), "sg_set_counters")

    def halfsweep(self, kind, colour):
        self._check(self._lib.sg_halfsweep(self._ctx, int(kind), int(colour)), "sg_halfsweep")

    def pt_stats(self):
        n = max(self.Tt - 1, 1)
        att = np.zeros((self.S, self.R, n), dtype=np.uint64); acc = np.zeros((self.S, self.R, n), dtype=np.uint64)
        self._check(self._lib.sg_pt_stats(self._ctx, _ptr(att), _ptr(acc)), "sg_pt_stats")
        return att, acc

    def accumulate(self, with_chirality=False):
        """Measure and add into the device-side logarithmic bins; asynchronous."""
        self._check(self._lib.sg_accumulate(self._ctx, int(bool(with_chirality))), "sg_accumulate")

    def get_logbins(self):
        """(sums float64 [LOGBINS][S][T][LOGBIN_OBS], counts uint64 [LOGBINS], counts_cg uint64 [LOGBINS])."""
        sums = np.zeros((LOGBINS, self.S, self.T, LOGBIN_OBS)); counts = np.zeros(LOGBINS, dtype=np.uint64)
        counts_cg = np.zeros(LOGBINS, dtype=np.uint64)
        self._check(self._lib.sg_get_logbins(self._ctx, _ptr(sums), _ptr(counts), _ptr(counts_cg)), "sg_get_logbins")
        return sums, counts, counts_cg

    def export_buffer(self):
        """Uninitialised device tensor of the shape export_replica / export_chirality fill (a receive buffer)."""
        import torch
        return torch.empty((self.S, 3, self.N, self.Tt), dtype=torch.float32, device=self.device)

    def export_replica(self, r, out=None):
        """Device tensor float32 [S][3][N][T]: the configurations of local replica r ordered by temperature (asynchronous)."""
        import torch
        if out is None:
            out = torch.empty((self.S, 3, self.N, self.Tt), dtype=torch.float32, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float32 and out.numel() == self.S * 3 * self.N * self.Tt
        self._check(self._lib.sg_export_replica(self._ctx, int(r), ctypes.c_void_p(out.data_ptr())), "sg_export_replica")
        return out

    def measure_cross(self, r, remote):
        """(q0 [S][T], qk [S][T][3][2]) between local replica r and a partner's export_replica tensor (on this device)."""
        assert remote.is_cuda and remote.is_contiguous() and remote.numel() == self.S * 3 * self.N * self.Tt
        q0 = np.empty((self.S, self.Tt)); qk = np.empty((self.S, self.Tt, 3, 2))
        self._check(self._lib.sg_measure_cross(self._ctx, int(r), ctypes.c_void_p(remote.data_ptr()), _ptr(q0), _ptr(qk)),
                    "sg_measure_cross")
        return q0, qk

    def export_chirality(self, r, out=None):
        """Device tensor float32 [S][3][N][T]: zeta_{x,mu} of local replica r ordered by temperature (asynchronous)."""
        import torch
        if out is None:
            out = torch.empty((self.S, 3, self.N, self.Tt), dtype=torch.float32, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float32 and out.numel() == self.S * 3 * self.N * self.Tt
        self._check(self._lib.sg_export_chirality(self._ctx, int(r), ctypes.c_void_p(out.data_ptr())), "sg_export_chirality")
        return out

    def chiral_cross(self, za, zb):
        """(qc0 [S][T][3], qck [S][T][3][3][2]) between two export_chirality tensors (both on this device); T = the temperatures of
        the whole chain (n_temps_total in a slot-sharded context)."""
        for z in (za, zb):
            assert z.is_cuda and z.is_contiguous() and z.numel() == self.S * 3 * self.N * self.Tt
        qc0 = np.empty((self.S, self.Tt, 3)); qck = np.empty((self.S, self.Tt, 3, 3, 2))
        self._check(self._lib.sg_chiral_cross(self._ctx, ctypes.c_void_p(za.data_ptr()), ctypes.c_void_p(zb.data_ptr()), _ptr(qc0), _ptr(qck)),
                    "sg_chiral_cross")
        return qc0, qck

    def pt_walk(self):
        """(round_trips uint64 [S][R], label int32 [S][R][T]) of the random walk in temperature."""
        trips = np.zeros((self.S, self.R), dtype=np.uint64); lab = np.zeros((self.S, self.R, self.Tt), dtype=np.int32)
        self._check(self._lib.sg_pt_walk(self._ctx, _ptr(trips), _ptr(lab)), "sg_pt_walk")
        return trips, lab

    def pt_visits(self):
        """visits uint64 [S][R][T][T]: PT sweeps configuration `slot` has spent at temperature index t."""
        v = np.zeros((self.S, self.R, self.Tt, self.Tt), dtype=np.uint64)
        self._check(self._lib.sg_pt_visits(self._ctx, _ptr(v)), "sg_pt_visits")
        return v

    def tune(self, knob, value):
        self._check(self._lib.sg_tune(self._ctx, int(knob), int(value)), "sg_tune")

    def sweep_impl_used(self, kind=KIND_OR):
        """(SWEEP_* constant of the kernel that served the last sweep_or / sweep_hb call, cudaError of the cluster launch that
        made the automatic choice fall back, 0 if none)."""
        err = ctypes.c_int(0)
        rc = self._lib.sg_sweep_impl_used(self._ctx, int(kind), ctypes.byref(err))
        if rc < 0:
            raise SgError(rc, "sg_sweep_impl_used")
        return int(rc), int(err.value)

    def sync(self):
        self._check(self._lib.sg_sync(self._ctx), "sg_sync")

    def kernel_launches(self):
        return int(self._lib.sg_kernel_launches(self._ctx))

    def graph_replays(self):
        """Units run_units has issued as CUDA-graph replays so far."""
        return int(self._lib.sg_graph_replays(self._ctx))
