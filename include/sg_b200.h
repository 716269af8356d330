/*
 * sg_b200.h -- C ABI of the B200-native spin-glass sweep library (libsg_b200.so).
 *
 * The library performs the Monte Carlo hot path of arXiv:1309.1599 (citations: PAPER.md:<line>):
 * checkerboard heat-bath (Eq. (A1)) and overrelaxation (Eq. (A2))
 * sweeps of unit 3-vector spins on an L^3 periodic lattice with one 3x3 coupling matrix per link
 * (Eq. (1); local field: footnote 64), parallel-tempering swaps
 * and the energy / overlap / k_min Fourier-mode reductions.  Every step runs in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback: without a CUDA device every compute
 * call returns SG_ECUDA.
 *
 * Conventions (DESIGN.md sections 2-3).
 *   N = L^3, L even >= 2.  Site index i = x1 + L*(x2 + L*x3), colour (x1+x2+x3)&1.  S samples,
 *   R replicas, T temperatures, C = R*T copies per sample, copy c = r*T + slot, P = R(R-1)/2 replica
 *   pairs (a<b) in the order (0,1),(0,2),...,(R-2,R-1).  A PT sweep exchanges the *temperatures* of two
 *   slots; spins never move.  temp_of_slot / slot_of_temp are the per-chain permutation and its inverse.
 *
 * Host-visible layouts are logical and fixed here; the device layout is private to the library.
 *   couplings  float [3][N][3][3]   M[mu][i][a][b]: link (i, mu) joins i and i+e_mu, a acts on s_i
 *   spins      float [C][3][N]      by slot
 *
 * Ownership.  The caller owns all device memory (one workspace of sg_workspace_bytes() bytes, 256-byte
 * aligned, e.g. a torch tensor's data_ptr()) and the CUDA stream; the library never calls cudaMalloc for
 * state and never frees caller memory.  Host input arrays are consumed before the call returns; host
 * output arrays are caller-allocated.  Sweeps and PT are asynchronous on the stream; calls that return
 * data to the host synchronise the stream.
 *
 * Errors.  Every call returns SG_OK (0) or a negative code; nothing is printed, nothing throws.
 */
#ifndef SG_B200_H
#define SG_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sg_ctx sg_ctx; /* opaque; owns only small host book-keeping */

typedef struct {
    int32_t L;            /* lattice size, even, >= 2 */
    int32_t n_samples;    /* S: disorder samples held by this context */
    int32_t n_replicas;   /* R >= 1 */
    int32_t n_temps;      /* T >= 1 */
    int32_t first_sample; /* global number of local sample 0 (enters every Philox counter; lets ranks
                             shard the samples and still draw the single-process numbers) */
    int32_t first_replica;     /* global number of local replica 0 (replica sharding of one sample, see n_replicas_total) */
    int32_t n_replicas_total;  /* replicas of the whole job; 0 = n_replicas (no replica sharding).  A context that holds the
                                  replicas [first_replica, first_replica + n_replicas) of every sample draws exactly the numbers
                                  (initial spins, heat bath, PT) a single context holding all n_replicas_total would: the PT chains
                                  of a sample are per replica, so its replicas can live on different GPUs with no
                                  exchange inside the Monte Carlo; overlaps are measured between the replicas a context holds */
    int32_t flags;             /* 0, or SG_SHAPE_FUSED_BUFFER: the workspace also holds the second state buffer and the ring
                                  couplings of the colour-fused sweep (SG_SWEEP_FUSED; L a multiple of 8, else SG_EINVAL):
                                  sg_workspace_bytes grows by the size of the spins plus N/4 * 224 bytes per sample */
    uint64_t seed;             /* Philox key */
    int32_t first_slot;        /* temperature-slot sharding of one chain (App. A.3: "each GPU updates only 2
                                  lattices ... N_GPU = N_T"): the context holds the configurations (slots) [first_slot, first_slot +
                                  n_temps) of every replica; the chain itself has n_temps_total temperatures */
    int32_t n_temps_total;     /* length of the chain; 0 = n_temps (no slot sharding).  Else a multiple of n_temps, first_slot a
                                  multiple of n_temps, betas passed to sg_create has n_temps_total entries.  Such a context draws
                                  the numbers a single context holding the whole chain would (heat bath and initial spins are
                                  keyed by the global copy id); it keeps the WHOLE temperature assignment of its chains, and
                                  the PT step is sg_pt_publish -> all-gather of the energies -> sg_pt_swap_gathered, the same
                                  decisions on every shard (identical Philox counters).  sg_pt_swap, sg_run_units, sg_measure,
                                  sg_accumulate, sg_measure_chiral return SG_EINVAL in such a context; sg_schwinger_dyson reports the held slots;
                                  overlaps go through sg_export_replica / sg_measure_cross, chiral-glass overlaps through
                                  sg_export_chirality / sg_chiral_cross */
} sg_shape;

enum {
    SG_OK = 0,
    SG_EINVAL = -1, /* bad argument: odd or too small L, counts <= 0, non-finite or non-monotone betas,
                       NULL where not allowed, sample out of range, workspace too small or misaligned */
    SG_ESTATE = -2, /* a sample was used before sg_init_sample */
    SG_ECUDA = -3,  /* a CUDA call failed (no device, launch failure, ...); see sg_last_cuda_error */
    SG_ELIMIT = -4  /* sg_chiral_cross_static only: the shape needs more than the fixed SG_STATIC_SCRATCH_BYTES */
};

/* coupling generator modes of sg_init_sample */
enum {
    SG_GEN_OFFDIAG_SYM = 0, /* M = a*1 + sigma_D * symmetric off-diagonal D, Gaussian (BASELINE configs) */
    SG_GEN_PAPER_SYM6 = 1,  /* M = a*1 + sigma_D * symmetric D with six independent Gaussian elements    */
    SG_GEN_GENERAL9 = 2,    /* nine independent Gaussian entries (non-symmetric)                         */
    SG_GEN_BIMODAL = 3,     /* the paper's J = +-1, D^{ab} = +-sigma_D                                    */
    SG_GEN_FERRO = 4        /* M = 1                                                                      */
};

enum { SG_KIND_OR = 0, SG_KIND_HB = 1 };
enum { SG_SHAPE_FUSED_BUFFER = 1 };   /* sg_shape.flags */

/* Device bytes the caller must provide for `shape`; 0 if the shape is invalid. */
size_t sg_workspace_bytes(const sg_shape* shape);

/* Create a context.  betas: host double[T], finite, strictly monotone (neighbouring
 * temperatures are adjacent entries).  dev_workspace: device pointer, 256-byte aligned, `bytes` >=
 * sg_workspace_bytes(shape); its contents are overwritten.  cuda_stream: a cudaStream_t (may be NULL =
 * the legacy default stream).  On success *out is the new context. */
int sg_create(sg_ctx** out, const sg_shape* shape, const double* betas, void* dev_workspace, size_t bytes,
              void* cuda_stream);
int sg_destroy(sg_ctx* ctx);

/* S0.  Sets the quenched couplings and the initial spins of local sample `sample` and
 * resets its temperature assignment to the identity.
 *   couplings == NULL: generated from (seed, first_sample+sample) with gen_mode / sigma_D;
 *                else: host float [3][N][3][3], copied (gen_mode, sigma_D ignored).
 *   spins     == NULL: uniform on S^2 from Philox stream 3; else host float [C][3][N], copied. */
int sg_init_sample(sg_ctx* ctx, int sample, int gen_mode, double sigma_D, const float* couplings,
                   const float* spins);

/* The paper's own couplings in their packed form (Sect. II.A: J_xy = +-1 and a
 * symmetric D_xy with six independent elements +-D; App. A.3: "a full coupling in a single byte").
 *   links: host uint8 [3][N], one byte per forward link (x, mu); bit 0 = sign of J (1: +1), bits 1, 2, 3 = signs of
 *          D^00, D^11, D^22, bits 4, 5, 6 = signs of D^01 = D^10, D^02 = D^20, D^12 = D^21 (1: +D); bit 7 must be 0 (else
 *          SG_EINVAL).  NULL: the bytes generator mode SG_GEN_BIMODAL draws for (seed, first_sample + sample).  Copied.
 *   D >= 0, finite.  spins as in sg_init_sample.
 * The sample behaves exactly as after sg_init_sample with the fp32 matrices M = fl32(J 1 + D) (which are stored too and
 * serve sg_get_couplings and every kernel but the one below).  When EVERY sample of the context has been initialised
 * this way with the same D, L is a multiple of 8 and sg_tune(SG_TUNE_PACKED, 1) was called, the z-marching sweep reads
 * 8 bytes per site (6 link bytes + pad) instead of 224 and its producer warp decodes them into the shared-memory blocks
 * the updating warps read: the same fp32 operands, hence the same spins bit for bit. */
int sg_init_sample_bimodal(sg_ctx* ctx, int sample, double D, const uint8_t* links, const float* spins);

/* S1 (Eq. (A2)).  n_sweeps full overrelaxation sweeps of every copy of every sample:
 * colour 0 half-sweep then colour 1.  The last half-sweep also reduces the total energy of every copy. */
int sg_sweep_or(sg_ctx* ctx, int n_sweeps);

/* S2 (Eq. (A1)).  n_sweeps full heat-bath sweeps at each copy's current temperature;
 * the HB counter advances by one per sweep.  Energies are reduced as in sg_sweep_or. */
int sg_sweep_hb(sg_ctx* ctx, int n_sweeps);

/* S4.  One parallel-tempering sweep of every chain (sample, replica): pairs t = 0..T-2 in
 * order, Metropolis acceptance min(1, exp((beta_t - beta_{t+1})(E_i - E_j))) on the total energies, which
 * are recomputed first if stale.  The PT counter advances by one. */
int sg_pt_swap(sg_ctx* ctx);

/* S4 when the slots of a chain are sharded over contexts (sg_shape.first_slot / n_temps_total; "the
 * exchange with the master of a double precision number" per lattice and MCS, here an all-gather).
 * sg_pt_publish: the total energies of this context's slots, double [S][R][n_temps] (recomputed first if stale), written
 *   to the DEVICE buffer dev_out (caller-owned; the send buffer of the all-gather).  Asynchronous on the stream.
 * sg_pt_swap_gathered: one PT sweep of every chain from the all-gathered energies, DEVICE buffer double [W][S][R][n_temps],
 *   W = n_temps_total / n_temps, block w written by the context with first_slot = w * n_temps.  Every shard must call it
 *   with the same buffer contents: all take the same decisions (PT stream keyed by chain, pair and PT counter), each keeps
 *   the whole assignment and the statistics, and updates the betas of its own slots.  The PT counter advances by one.
 *   Also valid without slot sharding (W = 1).  Asynchronous.
 * sg_energy_by_temp: e = H/N of the copy of replica r at temperature t from such a gathered buffer through the current
 *   assignment, host double [S][R][n_temps_total]; synchronises.
 * Errors: SG_EINVAL (NULL), SG_ESTATE, SG_ECUDA. */
int sg_pt_publish(sg_ctx* ctx, void* dev_out);
int sg_pt_swap_gathered(sg_ctx* ctx, const void* dev_all);
int sg_energy_by_temp(sg_ctx* ctx, const void* dev_all, double* e);

/* n_units Monte Carlo steps (MCS, Sect. III, App. A.1): each is sg_sweep_hb(ctx, 1);
 * sg_sweep_or(ctx, n_or); sg_pt_swap(ctx), issued from native code so that small lattices are not bound by the
 * caller's per-call overhead; for small lattices (resident kernel) and n_units >= 8 one unit is captured in a CUDA graph and
 * replayed (SG_TUNE_GRAPH).  Asynchronous on the stream; identical results to the three calls made
 * one by one. */
int sg_run_units(sg_ctx* ctx, int n_units, int n_or);

/* S3 + S5.  Host outputs (any may be NULL):
 *   e  double [S][R][T]        H/N of the copy of replica r at temperature t
 *   q0 double [S][P][T]        q^(0)   = sum_x s^a_x.s^b_x / N, both copies at temperature t
 *   qk double [S][P][T][3][2]  q^(k_mu) = sum_x q_x exp(+i 2 pi x_mu / L) / N, (Re, Im), mu = 0,1,2
 * Synchronises the stream. */
int sg_measure(sg_ctx* ctx, double* e, double* q0, double* qk);

/* Logarithmic data binning on the device (Sect. III: "Each bin had twice the
 * length of the previous ... i_f contains the last half of the Monte Carlo time series, i_f - 1 the second quarter").
 * sg_accumulate measures as sg_measure does (energies recomputed if stale, overlaps of all replica pairs) and adds, per
 * (sample, temperature), the observables below into bin floor(log2 n) of the n-th call since creation (n = 1, 2, ...):
 *   O[0] = mean over replicas of e,  O[1] = mean over pairs of q^(0)^2,  O[2] = mean over pairs and the three k_min
 *   directions of |q^(k_mu)|^2 (Eq. (3) up to the factor N),  O[3] = mean over pairs of q^(0)^4   (0 when R = 1);
 *   with_chirality != 0 also (as sg_measure_chiral measures them; "we averaged over all the values of mu")
 *   O[4] = mean over pairs and mu of q^_CG^mu(0)^2,  O[5] = mean over pairs, mu and the three k_min directions nu of
 *   |q^_CG^mu(k_nu)|^2.   chi = N <O>, xi by sg_correlation_length(L, <O[1]>, <O[2]>) resp. (L, <O[4]>, <O[5]>).
 * ASYNCHRONOUS on the stream: nothing crosses to the host.  fp64 sums in call order.  Errors: SG_EINVAL, SG_ESTATE.
 * sg_get_logbins: sums double [SG_LOGBINS][S][T][SG_LOGBIN_OBS]; counts uint64 [SG_LOGBINS] = calls that fell into each
 * bin, counts_cg = those of them made with chirality (the divisor of O[4], O[5]); host outputs, any may be NULL;
 * synchronises. */
#define SG_LOGBINS 32
#define SG_LOGBIN_OBS 6
int sg_accumulate(sg_ctx* ctx, int with_chirality);
int sg_get_logbins(sg_ctx* ctx, double* sums, uint64_t* counts, uint64_t* counts_cg);

/* Chiral-glass overlaps (Sect. II.B, Eq. (2)):
 *   zeta_{x,mu}  = s_{x+e_mu} . (s_x x s_{x-e_mu}),  kappa_{x,mu} = zeta^a_{x,mu} zeta^b_{x,mu}
 *   qc0 double [S][P][T][3]        q^_CG^mu(0)    = sum_x kappa_{x,mu} / N
 *   qck double [S][P][T][3][3][2]  q^_CG^mu(k_nu) = sum_x kappa_{x,mu} exp(+i 2 pi x_nu / L) / N, (Re, Im)
 * for the replica pairs a < b in the order of sg_measure, both copies at temperature t (found through the
 * temperature permutation), mu = chirality direction, nu = direction of k_min.  Host outputs, either may
 * be NULL.  fp32 triple products, fp64 sums in a fixed order.  For L = 2 every zeta vanishes up to rounding (x+e = x-e).
 * Synchronises the stream.  Errors: SG_EINVAL (ctx NULL), SG_ESTATE (a sample not initialised), SG_ECUDA. */
int sg_measure_chiral(sg_ctx* ctx, double* qc0, double* qck);

/* Overlaps between replicas held by different contexts (replica sharding: sg_shape.first_replica; q_x = s^a_x . s^b_x,
 * q^(k) as in sg_measure).
 * sg_export_replica: the configurations of local replica r ordered by TEMPERATURE, float [S][3][N][T] (temperature index
 *   fastest, site index i lexicographic), written to the DEVICE buffer dev_out (caller-owned, S*3*N*T floats; e.g. the
 *   send buffer of an all-gather over NVLink).  Asynchronous on the stream.
 * sg_measure_cross: between local replica r (through its own temperature permutation) and such a device buffer of a
 *   partner replica (same sample numbers, same temperatures): q0 double [S][T], qk double [S][T][3][2] (Re, Im), host
 *   outputs, either may be NULL.  fp32 products, fp64 sums in a fixed order.  Synchronises.
 * Errors: SG_EINVAL (NULL, r out of range, T > 256 for sg_measure_cross), SG_ESTATE, SG_ECUDA. */
int sg_export_replica(sg_ctx* ctx, int r, void* dev_out);
int sg_measure_cross(sg_ctx* ctx, int r, const void* dev_remote, double* q0, double* qk);
/* The same for the chiral-glass overlaps (Eq. (2)): sg_export_chirality writes zeta_{x,mu} of local replica r
 * ordered by temperature, float [S][3][N][T] (mu, site, temperature; temperature fastest) to the device buffer dev_out
 * (asynchronous); sg_chiral_cross forms kappa = zeta^a zeta^b between two such device buffers (one local, one the partner's):
 * qc0 double [S][T][3], qck double [S][T][3][3][2] as in sg_measure_chiral, host outputs, either may be NULL; synchronises.
 * In a context sharded by temperature slot T is n_temps_total throughout: sg_export_chirality writes zeta for the temperatures
 * whose configuration the shard holds and ZEROS for the others, so the element-wise sum of the shards' buffers (an all-reduce)
 * is the replica ordered by temperature; sg_chiral_cross of a shard's own (zero-padded) export of replica a with the summed
 * buffer of replica b gives the overlaps at the shard's temperatures and exact zeros elsewhere, and the sum of these over
 * the shards completes every temperature (multi.overlaps_sharded(chirality=True); Eq. (2) was measured on exactly the runs the
 * paper sharded this way).
 * Errors: SG_EINVAL (NULL, r out of range, T > 256), SG_ESTATE, SG_ECUDA. */
int sg_export_chirality(sg_ctx* ctx, int r, void* dev_out);
int sg_chiral_cross(sg_ctx* ctx, const void* dev_a, const void* dev_b, double* qc0, double* qck);

/* sg_chiral_cross without a context and without any allocation (the arithmetic of sg_chiral_cross, Eq. (2)).
 *
 * Who this is for.  Everything above needs an sg_ctx on top of a caller-allocated workspace, and a context itself pins host
 * memory when it is created (cudaHostAlloc) and creates streams and events the first time some calls are used.  Some callers
 * of this library cannot make allocating calls, or cannot afford them, at the point where they want the chiral-glass overlaps
 * of two zeta buffers they already hold on the device (their own sg_export_chirality output, or a partner rank's that
 * arrived through an all-gather or a peer copy):
 *   - a measurement process that runs next to the Monte Carlo ranks on a GPU whose HBM has been handed out in full (the sweep
 *     workspaces sized to the 180 GB, or a framework's memory pool that owns all of it): a cudaMalloc there fails, or succeeds
 *     only by making the pool give memory back;
 *   - a caller in the middle of a run for whom cudaMalloc / cudaFree are too expensive: both synchronise the whole device, so
 *     every sweep in flight on every other stream of the GPU waits for them;
 *   - code that is not allowed to touch the allocator at all (a callback, a plug-in of a host application that manages device
 *     memory itself and audits its use).
 * For them the partial sums that sg_chiral_cross keeps in the context's workspace live in a fixed array that is part of the
 * library image: SG_STATIC_SCRATCH_BYTES (16 MiB) of device memory, held by every GPU on which the library is loaded from the
 * moment its CUDA module loads until the process exits, whether or not this call is ever made.
 *
 *   L, n_samples (S), n_temps (T)   shape of the two buffers: L even, 2 <= L <= SG_STATIC_MAX_L, S >= 1, 1 <= T <= 256
 *   dev_a, dev_b   DEVICE, float [S][3][N][T] as sg_export_chirality writes them (mu, site, temperature; temperature fastest);
 *                  read only; they may be the same buffer
 *   dev_out        DEVICE, double [S*T*21], caller-owned, 8-byte aligned: qc0 [S][T][3] followed by qck [S][T][3][3][2] with the
 *                  meaning and normalisation of sg_chiral_cross.  Written asynchronously on the stream; NOT copied to the host
 *                  (the caller reads it in stream order).  Must not overlap the inputs.
 *   cuda_stream    a cudaStream_t (NULL = the legacy default stream); the buffers must belong to the CURRENT device
 *   cuda_error     may be NULL; on SG_ECUDA receives the cudaError_t (there is no context to keep it)
 *
 * Capacity.  4096 + S * 128 * ((256/T)*T) * 21 * 8 bytes (256/T an integer division) must not exceed
 * SG_STATIC_SCRATCH_BYTES: S <= 3 samples per call is accepted for every T, more only where (256/T)*T is small.  A larger job
 * is split by sample by the caller (one call per group of samples, ordered on one stream): the slice [s][3][N][T] of each input
 * is contiguous, and each call writes a complete [qc0 | qck] block for its own samples.  Beyond the capacity the call returns
 * SG_ELIMIT and does nothing; it never falls back to allocating.
 *
 * First call on a device.  The device address of the array is looked up once per device (cudaGetSymbolAddress, with that
 * device current) by the first call made on it; that look-up loads the library's CUDA module if nothing has yet.  Make this
 * first call during set-up, before any stream capture is begun.  Later calls only launch kernels (three per call) and call
 * no cudaMalloc, cudaFree, cudaHostAlloc, stream or event creation, nor any library routine that allocates.
 *
 * Sharing.  There is ONE array per device and every call on that device uses it, from any thread and any stream.  Calls
 * that can overlap on the GPU (different streams without an ordering between them, or different host threads) race on it and
 * return garbage: order them on one stream or with events.  The array keeps whatever the last call left in it; nothing in it
 * has to start at zero, because every element a call reads has been written by the same call first (the Fourier phase table
 * and all partial sums of the shape at hand), so leftovers of a call with another shape are harmless.
 * Results equal sg_chiral_cross to rounding (same products and summation order; the phase table is computed on the device,
 * within an ulp of the host's).  Errors: SG_EINVAL (NULL, odd or out-of-range L, S < 1, T outside 1..256, misaligned output),
 * SG_ELIMIT, SG_ECUDA. */
#define SG_STATIC_SCRATCH_BYTES (16u << 20)
#define SG_STATIC_MAX_L 256
int sg_chiral_cross_static(int L, int n_samples, int n_temps, const void* dev_a, const void* dev_b, void* dev_out,
                           void* cuda_stream, int* cuda_error);

/* Schwinger-Dyson monitor (App. A.4, Eq. (A6)):
 *   2 T <s_x.h_x> - <(h_x)^2 - (s_x.h_x)^2> = 0 in equilibrium, "averaged over all the sites in the lattice".
 *   sd double [S][R][T][2]   sd[..][0] = sum_x s_x.h_x / N,  sd[..][1] = sum_x [h_x.h_x - (s_x.h_x)^2] / N
 * of the copy of replica r at temperature t (current configuration; the caller averages over time and forms
 * 2 sd[0]/beta_t - sd[1]).  Host output, required.  fp32 fields, fp64 sums in a fixed order.  Synchronises.
 * In a context sharded by temperature slot T is n_temps_total and the entries of the temperatures whose configuration another
 * shard holds are exact zeros: the sum over the shards (an all-reduce of S*R*T*2 doubles, multi.schwinger_dyson_sharded) is the
 * whole chain's monitor -- the paper's check ran on its temperature-sharded L = 64 runs. */
int sg_schwinger_dyson(sg_ctx* ctx, double* sd);

/* Second-moment correlation length, Eq. (4) PAPER.md:93-97 (host arithmetic, no device work):
 *   xi = sqrt(chi(0)/chi(k_min) - 1) / (2 sin(pi/L)),   chi(k) = N <|q^(k)|^2>  (Eq. (3))
 * for either overlap field.  NaN when chi0 < chik. */
double sg_correlation_length(int L, double chi0, double chik);

/* ---- state access: tests, checkpoint / resume (all synchronise) ---- */
int sg_get_spins(sg_ctx* ctx, int sample, float* out /* [C][3][N] */);
int sg_set_spins(sg_ctx* ctx, int sample, const float* in /* [C][3][N] */);
int sg_get_couplings(sg_ctx* ctx, int sample, float* out /* [3][N][3][3] */);
int sg_get_perm(sg_ctx* ctx, int sample, int32_t* temp_of_slot /* [R][T] */, int32_t* slot_of_temp /* [R][T] */);
int sg_set_perm(sg_ctx* ctx, int sample, const int32_t* temp_of_slot /* [R][T], a permutation per chain */);
/* Total H of every slot, double [S][C]; recomputed if stale. */
int sg_get_energies(sg_ctx* ctx, double* E);
/* Test hook: overwrite the cached energies (marks them fresh), so that sg_pt_swap can be fed given values. */
int sg_set_energies(sg_ctx* ctx, const double* E /* [S][C] */);
int sg_get_counters(sg_ctx* ctx, uint64_t* hb_counter, uint64_t* pt_counter);
int sg_set_counters(sg_ctx* ctx, uint64_t hb_counter, uint64_t pt_counter);
/* One half-sweep of one colour (kind SG_KIND_OR / SG_KIND_HB) of every copy with the current HB counter,
 * which is not advanced: repeated HB calls on one colour are draws in a fixed field. */
int sg_halfsweep(sg_ctx* ctx, int kind, int colour);
/* PT statistics since creation, uint64 [S][R][T-1] each (either may be NULL). */
int sg_pt_stats(sg_ctx* ctx, uint64_t* attempts, uint64_t* accepts);
/* Random walk in temperature (Sect. III: "the random walk in temperatures
 * of each sample"), kept by every sg_pt_swap since creation.  Each configuration (slot) of a chain (sample, replica)
 * carries a label: 0 = has not touched an end of the ladder yet, 1 = last touched temperature index 0, 2 = last touched
 * index T-1.  A round trip is index 0 -> index T-1 -> index 0.
 *   round_trips uint64 [S][R]     completed round trips, summed over the chain's T configurations
 *   label       int32  [S][R][T]  current label of every slot
 * Host outputs, either may be NULL.  Integer work: bit-exact against the oracle.  Synchronises. */
int sg_pt_walk(sg_ctx* ctx, uint64_t* round_trips, int32_t* label);
/* Histogram of that walk ("In a thermalized sample, all the replicas stay a significant amount of time at each
 * temperature"): visits uint64 [S][R][T][T], visits[..][slot][t] = PT sweeps since creation after which the
 * configuration in `slot` sat at temperature index t.  Kept on the device by every PT sweep when S*R*T*T*8 bytes <= 64 MiB
 * (else SG_EINVAL).  Host output, required.  Integer work: bit-exact against the oracle.  Synchronises. */
int sg_pt_visits(sg_ctx* ctx, uint64_t* visits);
/* Integrated autocorrelation time of a recorded random walk in temperature ("the integrated autocorrelation
 * time (mixing time) of the random walk in temperatures of each sample"; host arithmetic, no device work).
 *   series: host int32 [n], the temperature index of one configuration after each PT sweep (e.g. temp_of_slot over time)
 *   tau = 1/2 + sum_{k=1}^{W} rho(k),  rho(k) = C(k)/C(0),  C(k) = sum_{i<n-k} (x_i - m)(x_{i+k} - m) / (n - k),
 *   m the mean of the series, summed up to the first W with W >= window_c * tau(W) (self-consistent window; window_c <= 0
 *   means 6) or W = n/2.  Returns tau in PT sweeps; NaN when n < 4 or the series is constant. */
double sg_walk_tau_int(const int32_t* series, int64_t n, double window_c);

/* ---- tuning (results do not depend on it beyond floating-point summation order) ----
 * SG_TUNE_SWEEP_IMPL: which half-sweep kernel serves sg_sweep_or / sg_sweep_hb / the energy pass.
 *   SG_SWEEP_AUTO     the resident kernel when the lattice of 8 copies fits in shared memory (N * 96 B <= 200 KB: L <= 12), else the
 *                     z-marching kernel when L is a multiple of 8, else the tiled kernel (default); at L = 16 with at least 15
 *                     (sample, copy group) pairs the overrelaxation sweeps go to the cluster-resident kernel (SG_SWEEP_CLUSTER)
 *   SG_SWEEP_TILED    the tiled kernel (any even L)
 *   SG_SWEEP_ZMARCH   the z-marching kernel; SG_EINVAL unless L is a multiple of 8
 *   SG_SWEEP_RESIDENT all n sweeps of an sg_sweep_or / sg_sweep_hb call in ONE launch, the lattice of a (sample, group of
 *                     32 copies) held in shared memory; SG_EINVAL unless the lattice of 4 copies fits (N * 48 B <= 200 KB).
 *                     sg_halfsweep and the stand-alone energy pass keep using the z-marching / tiled kernel.
 *   SG_SWEEP_FUSED    sg_sweep_or only: both colours of a sweep in ONE pass of the colour-fused z-marching kernel (SURVEY.md
 *                     section 8(f1): every spin read once and written once per sweep; the new colour-0 values of the one-site
 *                     ring around a CTA's column are recomputed, the sweep runs out of place between two state buffers);
 *                     heat bath, sg_halfsweep and the energy pass as SG_SWEEP_ZMARCH.  SG_EINVAL unless the context was created
 *                     with sg_shape.flags = SG_SHAPE_FUSED_BUFFER.  Measured SLOWER than SG_SWEEP_ZMARCH (DESIGN.md section 10:
 *                     28.7 instead of 38.5 bytes per update from HBM, but 4.9 instead of 3.1 instructions): opt-in.
 *   SG_SWEEP_CLUSTER  L = 16 only (else SG_EINVAL): all n sweeps of an sg_sweep_or / sg_sweep_hb call in ONE launch, the lattice of a
 *                     (sample, group of 32 copies) held in the shared memory of thread-block clusters (SG_TUNE_CLUSTER_CTAS: 4 CTAs
 *                     holding 4 planes of 16 copies each, or 8 CTAs holding 2 planes of 32 copies); the x3 neighbours across a
 *                     cut are read from the neighbouring CTA's shared memory.
 * All kernels perform the same arithmetic in the same order: the spins do not depend on the choice.  The ENERGIES do, in the
 * last bits: each kernel sums its per-CTA partials of E in its own fixed order (they agree to ~1e-7 * N relative to |E|), and E
 * feeds the PT acceptance.  SG_SWEEP_AUTO looks at the LOCAL shape (the cluster kernel needs n_samples * copy groups >= 15 in this
 * context; SG_TUNE_ZCHUNK = 0 picks the chunk from the local grid), so the same job split over ranks by sample, replica or slot
 * may run another kernel per shard than the single context would, and a PT decision whose random number falls within that
 * rounding of the threshold can then differ.  A shard reproduces the single-context chain BIT FOR BIT only when both pin
 * SG_TUNE_SWEEP_IMPL (SG_SWEEP_ZMARCH or SG_SWEEP_TILED) and SG_TUNE_ZCHUNK to the same explicit values; left on AUTO the two
 * chains are equally valid samples of the same Markov chain but not guaranteed identical.
 * sg_sweep_impl_used reports which kernel served the last sg_sweep_or / sg_sweep_hb call (below).
 * SG_TUNE_ZCHUNK: planes per CTA of the z-marching kernel; 0 = automatic, else even, >= 4 and a divisor of L.
 * SG_TUNE_RES_COPIES: copies per CTA of the resident kernel: 0 = automatic, else 4, 8, 16 or 32 (SG_EINVAL if the lattice
 *   of that many copies does not fit in shared memory).
 * SG_TUNE_PACKED: 1 = the z-marching sweep reads the packed bytes when every sample was initialised by
 *   sg_init_sample_bimodal with one and the same D; 0 (default) = always the fp32 matrices, which measured 3-7 % faster
 *   at 32 and more copies per sample.  Same spins bit for bit.
 * SG_TUNE_MEASURE_IMPL: which kernel forms the overlaps of sg_measure / sg_accumulate.
 *   SG_MEASURE_AUTO    the streaming row kernel (thread = (lattice row, temperature), every replica's spin loaded once for
 *                      all pairs) when 2 <= R <= 4, else the staged kernel (default)
 *   SG_MEASURE_STAGED  the staged kernel (sites of all copies through shared memory; any R)
 *   Same fp32 products.  The staged kernel adds them in fp64 from the single site on; the streaming kernel adds the L sites of a
 *   lattice row (and their x1 phases, rounded to fp32) in fp32 and goes on in fp64.  |difference of any q^| <= L * 2^-24 in the worst
 *   case (every rounding of every row in the same direction: 3.8e-6 at L = 64), ~1e-8 in practice (roundings of different rows are
 *   independent); the tests hold it to 2e-7 absolute at cfg 4's full size, for random copies and for identical copies (q^(0) = 1, the
 *   coherent worst case), and both kernels to 1e-6 against the oracle.
 * SG_TUNE_CLUSTER_CTAS: shape of the cluster-resident kernel (L = 16): 4 (default) = clusters of 4 CTAs, each holding 4 planes of
 *   16 copies (two clusters per copy group); 8 = clusters of 8 CTAs, each holding 2 planes of all 32 copies.  Same spins.
 * SG_TUNE_GRAPH: 1 (default) = sg_run_units captures one unit in a CUDA graph and replays it (the sweep counters patched in
 *   the captured parameter blocks) when the resident kernel serves the sweeps and n_units >= 8; 0 = always issue the launches
 *   one by one.  Same launches, same results. */
enum { SG_TUNE_SWEEP_IMPL = 0, SG_TUNE_ZCHUNK = 1, SG_TUNE_RES_COPIES = 2, SG_TUNE_PACKED = 3, SG_TUNE_MEASURE_IMPL = 4, SG_TUNE_GRAPH = 5, SG_TUNE_CLUSTER_CTAS = 6 };
enum { SG_MEASURE_AUTO = 0, SG_MEASURE_STAGED = 1 };
enum { SG_SWEEP_AUTO = 0, SG_SWEEP_TILED = 1, SG_SWEEP_ZMARCH = 2, SG_SWEEP_RESIDENT = 3, SG_SWEEP_FUSED = 4, SG_SWEEP_CLUSTER = 5 };
int sg_tune(sg_ctx* ctx, int knob, int value);

/* ---- utilities ---- */
/* Which kernel served the last sg_sweep_or (kind = SG_KIND_OR) or sg_sweep_hb (SG_KIND_HB) call, sg_run_units included: one of
 * SG_SWEEP_TILED / ZMARCH / RESIDENT / FUSED / CLUSTER; 0 (SG_SWEEP_AUTO) before the first such call; SG_EINVAL for a NULL context
 * or another kind.  cluster_fallback_cuda (may be NULL) receives the cudaError_t of the cluster launch that made the automatic
 * choice give up k_sweep_cres in this context (that sweep call itself went on with the z-marching kernel and returned SG_OK;
 * sg_last_cuda_error is not set by it), 0 if that never happened.  The automatic choice tries the cluster kernel again after
 * the next sg_tune(SG_TUNE_SWEEP_IMPL / SG_TUNE_CLUSTER_CTAS, ...).  Host book-keeping only: no device work. */
int sg_sweep_impl_used(const sg_ctx* ctx, int kind, int* cluster_fallback_cuda);
int sg_sync(sg_ctx* ctx);                       /* cudaStreamSynchronize on the context's stream        */
uint64_t sg_kernel_launches(const sg_ctx* ctx); /* kernels launched by this context so far              */
uint64_t sg_graph_replays(const sg_ctx* ctx);   /* units sg_run_units issued as replays of a captured CUDA graph so far (0 when
                                                   every unit was issued launch by launch: SG_TUNE_GRAPH off, fewer than 8 units,
                                                   a lattice the resident kernel does not serve, or a capture that failed)   */
int sg_last_cuda_error(const sg_ctx* ctx);      /* cudaError_t of the last failed CUDA call, 0 if none  */
const char* sg_strerror(int code);              /* static string for an SG_* code                       */
/* Philox4x32-10 block on the host (the library's own implementation; known-answer tests). */
void sg_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

#ifdef __cplusplus
}
#endif
#endif /* SG_B200_H */
