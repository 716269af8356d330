// sg_api.cu -- host side of libsg_b200: the C ABI of include/sg_b200.h.
// Context book-keeping, workspace carving, the coupling generator (host fp64 Philox + Box-Muller,
// DESIGN.md section 3.2) and the kernel launches.  No CPU implementation of any sweep exists here:
// without a device every compute call fails with SG_ECUDA.
#include "../../include/sg_b200.h"

#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "sg_kernels.cuh"
#include "sg_measure.cuh"
#include "sg_sweep_res.cuh"
#include "sg_sweep_fz.cuh"
#include "sg_sweep_cres.cuh"

using namespace sg;

struct sg_ctx {
    sg_shape shape;
    int L, N, Nh, S, R, T, C, NG, Cp, P;
    int Rt, Cg;           // replicas / copies per sample of the whole job (replica sharding; = R, C otherwise)
    int Tt, slot0;        // length of the PT chain and first slot held (temperature-slot sharding; = T, 0 otherwise); T = slots held
    unsigned long long* visits;   // [S][R][Tt][Tt] histogram of the walk in temperature, nullptr when too large
    uint32_t g_first;     // global copy id of (local sample 0, local copy 0)
    cudaStream_t stream;
    // device arrays (carved from the caller's workspace)
    float* spins; float* spins2; float* Jr; float* Jg; float* Jt; unsigned char* Jp; float* Mraw; float* staging; float* beta_slot;
    double* betas; double* E; double* Epart; double* SDpart; double* phase; double* Mpart; double* result;
    double* h_result = nullptr;   // pinned host mirror of `result`: one device-to-host copy per measurement call
    size_t result_doubles = 0;
    int* slot_of_temp; int* temp_of_slot;
    unsigned long long* attempts; unsigned long long* accepts;
    int* walk_label; unsigned long long* round_trips;
    double* logbin; uint64_t n_acc;
    double* Xpart;
    uint64_t n_acc_cg[SG_LOGBINS];   // calls with chirality per bin
    // sweep geometry
    int tile_sites, ntiles, log2L;
    // z-marching sweep (L a multiple of 8): tuning knobs and the derived chunking
    int sweep_impl;   // SG_SWEEP_AUTO / SG_SWEEP_TILED / SG_SWEEP_ZMARCH / SG_SWEEP_RESIDENT
    int res_ok, res_auto;   // the lattice of 4 (explicit request) / 8 (automatic choice) copies fits in shared memory
    int res_cpc, res_cpc_req;   // copies per CTA of the resident kernel (4, 8, 16, 32); requested, 0 = automatic
    int zm_zc_req;    // requested planes per chunk, 0 = automatic
    int zm_ok, zm_ZC, zm_nzc;
    uint32_t zm_attr_set = 0;
    uint32_t fz_attr_set = 0;   // the same for k_sweep_fz
    uint32_t cres_attr_set = 0; // and for k_sweep_cres
    int cres_cs = 4;                 // SG_TUNE_CLUSTER_CTAS: CTAs per cluster of k_sweep_cres (4: half groups, 4 planes each; 8: whole groups, 2 planes)
    bool cres_unavailable = false;   // a cluster launch failed on this device: the automatic choice stops using it (until the next sg_tune of the sweep kernel)
    int cres_fail_cuda = 0;          // the cudaError_t of that launch (sg_sweep_impl_used reports it; last_cuda is cleared: the call succeeded)
    uint64_t graph_replays = 0;      // units issued by sg_run_units as replays of a captured CUDA graph (sg_graph_replays)
    int served_impl[2] = { 0, 0 };   // SG_SWEEP_* of the kernel that served the last sg_sweep_or [0] / sg_sweep_hb [1] (0: none yet)
    int fz_ZC, fz_nzc;          // chunking of the colour-fused sweep   // template instances of k_sweep_zm whose shared-memory attribute this context has set on its device
    // measure geometry
    int nchunk, chunk_sites, MS;
    int mq_nchunk, mq_rows_per_cta, mq_Tw, mq_rows_t;   // k_measure_rows: row chunks per sample, rows per CTA, temperatures and rows per CTA pass
    uint32_t mq_attr_set = 0;
    // host state
    std::vector<double> h_betas;
    std::vector<char> inited;
    std::vector<double> bimodal_D;   // per sample: D of its packed bimodal couplings (sg_init_sample_bimodal), NaN if not packed
    int measure_impl = 0;            // SG_TUNE_MEASURE_IMPL
    int packed_on;                   // SG_TUNE_PACKED: 1 = the z-marching sweep reads the packed bytes when every sample is packed
    uint64_t hb_counter, pt_counter, launches;
    bool energies_fresh;
    int last_cuda;
    // CUDA-graph replay of a unit (sg_run_units): while `capturing`, every launch whose parameter block carries the HB or
    // PT counter notes its graph node, so that the counter can be patched before each replay
    struct CounterNode { cudaGraphNode_t node; int which; size_t offset, size; };
    bool capturing = false;
    std::vector<CounterNode> counter_nodes;
    // sg_set_spins: a group is uploaded in UP_CHUNKS site chunks on a copy stream of the library's own, each transposed on the
    // context's stream as soon as it has landed (events), so the PCIe link does not wait for the transposition kernels
    static constexpr int UP_CHUNKS = 4;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_copied[UP_CHUNKS] = {}, ev_done[UP_CHUNKS] = {}, ev_start = nullptr;
    int upload_state = 0;                // 0 = not tried, 1 = pipelined upload available, -1 = not available (plain path)
    cudaStream_t gstream = nullptr;      // capture / replay stream when the context's own stream is the legacy default stream
    cudaEvent_t gevent = nullptr;
    int graph_mode = 1;                  // SG_TUNE_GRAPH: 1 = sg_run_units replays a captured unit when it pays
};

namespace {

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

bool shape_ok(const sg_shape* s)
{
    if (!s) return false;
    if (s->L < 2 || (s->L & 1) || s->L > 1024) return false;
    if (s->n_samples <= 0 || s->n_replicas <= 0 || s->n_temps <= 0 || s->first_sample < 0) return false;
    if ((s->flags & ~SG_SHAPE_FUSED_BUFFER) != 0 || s->first_replica < 0) return false;
    if ((s->flags & SG_SHAPE_FUSED_BUFFER) && s->L % 8 != 0) return false;
    if (s->n_replicas_total != 0 && s->first_replica + s->n_replicas > s->n_replicas_total) return false;
    if (s->n_replicas_total == 0 && s->first_replica != 0) return false;
    if (s->first_slot < 0 || s->n_temps_total < 0) return false;
    if (s->n_temps_total == 0 && s->first_slot != 0) return false;
    if (s->n_temps_total != 0 && (s->n_temps_total % s->n_temps != 0 || s->first_slot % s->n_temps != 0 ||
                                  s->first_slot + s->n_temps > s->n_temps_total)) return false;
    const double N = (double)s->L * s->L * s->L;
    const double C = (double)s->n_replicas * s->n_temps;
    const double Cjob = (double)(s->n_replicas_total ? s->n_replicas_total : s->n_replicas) * (s->n_temps_total ? s->n_temps_total : s->n_temps);
    if (N > 2.0e9 || Cjob > 1.0e6) return false;
    if (((double)s->first_sample + s->n_samples) * Cjob > 4.0e9) return false;   // copy ids are 32-bit counters
    if ((double)s->n_samples * std::ceil(C / 32.0) * N * 96.0 > 4.0e11) return false;
    return true;
}

struct Geometry {
    int L, N, Nh, S, R, T, Tt, C, NG, Cp, P, tile_sites, ntiles, nchunk, chunk_sites, MS;
    int mq_nchunk, mq_rows_per_cta, mq_Tw, mq_rows_t;
    bool fused;     // SG_SHAPE_FUSED_BUFFER
};

Geometry geometry(const sg_shape* s)
{
    Geometry g;
    g.L = s->L; g.N = s->L * s->L * s->L; g.Nh = g.N / 2;
    g.S = s->n_samples; g.R = s->n_replicas; g.T = s->n_temps; g.C = g.R * g.T;
    g.Tt = s->n_temps_total ? s->n_temps_total : s->n_temps;
    g.fused = (s->flags & SG_SHAPE_FUSED_BUFFER) != 0;
    g.NG = (g.C + G - 1) / G; g.Cp = g.NG * G; g.P = g.R * (g.R - 1) / 2;
    // sweep tiles: 128 consecutive same-colour sites per CTA (4 passes of 32 site slots)
    g.tile_sites = 128;
    g.ntiles = (g.Nh + g.tile_sites - 1) / g.tile_sites;
    // measure chunks
    g.nchunk = g.N / 32; if (g.nchunk < 1) g.nchunk = 1; if (g.nchunk > 256) g.nchunk = 256;   // >= 2 batches of sites per CTA, enough CTAs for small lattices
    g.chunk_sites = (g.N + g.nchunk - 1) / g.nchunk;
    g.MS = 11500 / (3 * g.Cp); if (g.MS < 1) g.MS = 1; if (g.MS > 16) g.MS = 16;
    // k_measure_rows: a CTA pass = rows_t lattice rows x Tw temperatures; a CTA takes `rounds` passes of consecutive rows.
    // At most 256 chunks per sample (the partials array), at least ~4 CTAs per SM over the job when the lattice allows,
    // and a few passes per CTA to amortise its final reduction.
    g.mq_Tw = g.T < MROWS_THREADS ? g.T : MROWS_THREADS;
    g.mq_rows_t = MROWS_THREADS / g.mq_Tw;
    {
        const int rows = g.L * g.L;
        int rounds = (rows + 256 * g.mq_rows_t - 1) / (256 * g.mq_rows_t);
        while (rounds < 4 && (long)g.S * (rows / (g.mq_rows_t * (rounds + 1))) >= 592) ++rounds;
        g.mq_rows_per_cta = g.mq_rows_t * rounds;
        g.mq_nchunk = (rows + g.mq_rows_per_cta - 1) / g.mq_rows_per_cta;
    }
    return g;
}

// histogram of the walk in temperature, [S][R][Tt][Tt] uint64: kept when it is at most 64 MiB
size_t visits_bytes(const Geometry& g)
{
    const double b = (double)g.S * g.R * (double)g.Tt * g.Tt * sizeof(unsigned long long);
    return (b <= 64.0 * 1024 * 1024) ? (size_t)b : 0;
}

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) { size_t o = off; off += align256(bytes); return o; }
};

struct Offsets {
    size_t spins, spins2, Jr, Jg, Jt, Jp, Mraw, staging, beta_slot, betas, E, Epart, SDpart, phase, Mpart, result, sot, tos, att, acc, wlab, trips, visits, logbin, xpart, total;
};

Offsets offsets(const Geometry& g)
{
    Carve c; Offsets o;
    o.spins = c.take((size_t)g.S * g.NG * g.N * SITE_FLOATS * sizeof(float));
    // the colour-fused sweep (L a multiple of 8) is out of place: a second state buffer, and the couplings of the ring sites
    o.spins2 = c.take(g.fused ? (size_t)g.S * g.NG * g.N * SITE_FLOATS * sizeof(float) : 0);
    o.Jr = c.take(g.fused ? (size_t)g.S * (g.N / 4) * JG * sizeof(float) : 0);
    o.Jg = c.take((size_t)g.S * 2 * g.Nh * JG * sizeof(float));
    o.Jt = c.take((g.L % 8 == 0) ? (size_t)g.S * 2 * g.Nh * JG * sizeof(float) : 0);
    o.Jp = c.take((g.L % 8 == 0) ? (size_t)g.S * g.N * 8 : 0);
    o.Mraw = c.take((size_t)g.S * 3 * g.N * 9 * sizeof(float));
    size_t stg = (size_t)G * 3 * g.N * sizeof(float);
    o.staging = c.take(stg);
    o.beta_slot = c.take((size_t)g.S * g.Cp * sizeof(float));
    o.betas = c.take((size_t)g.Tt * sizeof(double));
    o.E = c.take((size_t)g.S * g.Cp * sizeof(double));
    o.Epart = c.take((size_t)g.S * g.NG * g.ntiles * G * sizeof(double));
    o.SDpart = c.take((size_t)g.S * g.NG * 2 * g.ntiles * G * 2 * sizeof(double));
    o.phase = c.take((size_t)g.L * 2 * sizeof(double));
    {   // 21 per item and chunk (chirality), 7 per item and row chunk (overlap)
        const size_t items = (g.P * g.T > 0 ? (size_t)g.P * g.T : 1);
        const size_t a = (size_t)g.nchunk * 21, b = (size_t)g.mq_nchunk * 7;
        o.Mpart = c.take((size_t)g.S * items * (a > b ? a : b) * sizeof(double));
    }
    o.result = c.take(((size_t)g.S * g.R * g.Tt + (size_t)g.S * g.P * g.Tt * 21 + (size_t)g.S * g.Tt * 21 + 1) * sizeof(double));
    o.sot = c.take((size_t)g.S * g.R * g.Tt * sizeof(int));
    o.tos = c.take((size_t)g.S * g.R * g.Tt * sizeof(int));
    size_t st = (size_t)g.S * g.R * (g.Tt > 1 ? g.Tt - 1 : 1) * sizeof(unsigned long long);
    o.att = c.take(st);
    o.acc = c.take(st);
    o.wlab = c.take((size_t)g.S * g.R * g.Tt * sizeof(int));
    o.trips = c.take((size_t)g.S * g.R * sizeof(unsigned long long));
    o.visits = c.take(visits_bytes(g));
    o.logbin = c.take((size_t)SG_LOGBINS * g.S * g.T * SG_LOGBIN_OBS * sizeof(double));
    o.xpart = c.take((size_t)g.S * XCHUNKS * XTHREADS * 21 * sizeof(double));   // rows * T <= XTHREADS when T <= XTHREADS
    o.total = c.off;
    return o;
}

int cuda_fail(sg_ctx* ctx, cudaError_t e)
{
    if (ctx) ctx->last_cuda = (int)e;
    return SG_ECUDA;
}

#define SG_CUDA(ctx, call)                                    \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail((ctx), e__); \
    } while (0)

#define SG_LAUNCHED(ctx)                                      \
    do {                                                      \
        (ctx)->launches += 1;                                 \
        cudaError_t e__ = cudaGetLastError();                 \
        if (e__ != cudaSuccess) return cuda_fail((ctx), e__); \
    } while (0)

// during the capture of a unit: remember the node of the launch just made if its parameter block holds a sweep counter
// (which: 0 = HB counter, 1 = PT counter; offset / size: of the counter inside / of the parameter block)
void note_counter_node(sg_ctx* ctx, cudaStream_t stream, int which, size_t offset, size_t size)
{
    if (!ctx->capturing) return;
#if CUDART_VERSION >= 13000
    // CUDA 13 changes the signature of cudaStreamGetCaptureInfo (an edge-data argument).  Until this call is ported and tested
    // there, the capture is marked unusable and sg_run_units issues its units launch by launch: slower for small lattices, same results.
    (void)stream; (void)which; (void)offset; (void)size;
    ctx->counter_nodes.push_back({ nullptr, -1, 0, 0 });
#else
    cudaStreamCaptureStatus st;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    if (cudaStreamGetCaptureInfo(stream, &st, nullptr, nullptr, &deps, &ndeps) != cudaSuccess || st != cudaStreamCaptureStatusActive || ndeps != 1) {
        ctx->counter_nodes.push_back({ nullptr, -1, 0, 0 });     // marks the capture as unusable
        return;
    }
    ctx->counter_nodes.push_back({ deps[0], which, offset, size });
#endif
}

int ilog2_exact(int L)
{
    int l = 0;
    while ((1 << l) < L) ++l;
    return ((1 << l) == L) ? l : 0;
}

// ---- coupling generator (host, fp64) ----
const double kPi = 3.14159265358979323846;

void link_normals(uint64_t seed, uint32_t link, uint32_t sample, double n[12], uint32_t w0[4])
{
    const uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);
    for (uint32_t j = 0; j < 3; ++j) {
        uint32_t w[4];
        philox4x32_10(link, sample, j, STREAM_COUPLINGS, k0, k1, w);
        if (j == 0) std::memcpy(w0, w, sizeof(w));
        for (int pair = 0; pair < 2; ++pair) {
            const double u0 = ((double)w[2 * pair] + 0.5) / 4294967296.0;
            const double u1 = ((double)w[2 * pair + 1] + 0.5) / 4294967296.0;
            const double rad = std::sqrt(-2.0 * std::log(u0));
            n[4 * j + 2 * pair] = rad * std::cos(2.0 * kPi * u1);
            n[4 * j + 2 * pair + 1] = rad * std::sin(2.0 * kPi * u1);
        }
    }
}

// the paper's coupling of one link from its byte (layout in include/sg_b200.h)
void bimodal_matrix(uint32_t b, double D, double m[9])
{
    const double J = (b & 1u) ? 1.0 : -1.0;
    double d[6];
    for (int k = 0; k < 6; ++k) d[k] = ((b >> (k + 1)) & 1u) ? D : -D;
    m[0] = J + d[0]; m[4] = J + d[1]; m[8] = J + d[2];
    m[1] = m[3] = d[3]; m[2] = m[6] = d[4]; m[5] = m[7] = d[5];
}

void generate_couplings(int L, uint64_t seed, uint32_t sample, int mode, double sd, float* M)
{
    const int N = L * L * L;
    for (int i = 0; i < N; ++i)
        for (int mu = 0; mu < 3; ++mu) {
            double n[12], m[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
            uint32_t w0[4];
            link_normals(seed, (uint32_t)(3 * i + mu), sample, n, w0);
            switch (mode) {
            case SG_GEN_OFFDIAG_SYM:
                m[0] = m[4] = m[8] = n[0];
                m[1] = m[3] = sd * n[1]; m[2] = m[6] = sd * n[2]; m[5] = m[7] = sd * n[3];
                break;
            case SG_GEN_PAPER_SYM6:
                m[0] = n[0] + sd * n[1]; m[4] = n[0] + sd * n[2]; m[8] = n[0] + sd * n[3];
                m[1] = m[3] = sd * n[4]; m[2] = m[6] = sd * n[5]; m[5] = m[7] = sd * n[6];
                break;
            case SG_GEN_GENERAL9:
                for (int e = 0; e < 9; ++e) m[e] = sd * n[e];
                break;
            case SG_GEN_BIMODAL:
                bimodal_matrix(w0[0] & 0x7fu, sd, m);
                break;
            default:
                m[0] = m[4] = m[8] = 1.0;
            }
            float* dst = M + ((size_t)mu * N + i) * 9;
            for (int e = 0; e < 9; ++e) dst[e] = (float)m[e];
        }
}

template <int KIND, bool WITH_E>
void launch_sweep_l(sg_ctx* ctx, const SweepParams& p, dim3 grid)
{
    switch (ctx->log2L) {
    case 1: k_sweep<KIND, WITH_E, 1><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    case 2: k_sweep<KIND, WITH_E, 2><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    case 3: k_sweep<KIND, WITH_E, 3><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    case 4: k_sweep<KIND, WITH_E, 4><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    case 5: k_sweep<KIND, WITH_E, 5><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    case 6: k_sweep<KIND, WITH_E, 6><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    case 7: k_sweep<KIND, WITH_E, 7><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    default: k_sweep<KIND, WITH_E, 0><<<grid, SWEEP_THREADS, 0, ctx->stream>>>(p); break;
    }
}

// ---- z-marching sweep: 8 x 8 columns, ring of NST other-colour planes and NJ coupling stages ----
constexpr int ZM_TX = 8, ZM_TY = 8, ZM_NST = 5, ZM_NJ = 3;

void zm_plan(sg_ctx* ctx)
{
    const int L = ctx->L;
    ctx->zm_ok = (L % 8 == 0) ? 1 : 0;
    ctx->zm_ZC = 0; ctx->zm_nzc = 0;
    if (!ctx->zm_ok) return;
    int ZC = 0;
    if (ctx->zm_zc_req > 0) {
        ZC = ctx->zm_zc_req;
    } else {
        // the longest chunk that still gives every SM several CTAs' worth of work in turn (2 CTAs per SM x 148 SMs
        // per wave); a chunk re-reads 2 planes of other-colour sites per ZC planes
        // Candidates are the even divisors of L that are >= 4 (the kernel steps through a chunk in pairs of planes
        // from an even z0): the longest one that reaches the CTA count, else the shortest candidate.
        const long per_plane_col = (long)ctx->S * ctx->NG * (L / ZM_TX) * (L / ZM_TY);
        int shortest = L;
        for (int cand = L; cand >= 4; --cand) {
            if ((cand & 1) || L % cand != 0) continue;
            shortest = cand;
            if (cand <= 8 || per_plane_col * (L / cand) >= 6 * 296) { ZC = cand; break; }
        }
        if (ZC == 0) ZC = shortest;
    }
    if (ZC < 2 || (ZC & 1) || L % ZC != 0) { ctx->zm_ok = 0; return; }     // never launch a chunking the kernel cannot step through
    ctx->zm_ZC = ZC; ctx->zm_nzc = L / ZC;
}

template <int KIND, bool WITH_E, bool PACKED>
int launch_zm_p(sg_ctx* ctx, const ZmParams& p, dim3 grid)
{
    auto kern = k_sweep_zm<KIND, WITH_E, ZM_TX, ZM_TY, ZM_NST, ZM_NJ, PACKED>;
    constexpr size_t smem = zm_smem_bytes<ZM_TX, ZM_TY, ZM_NST, ZM_NJ>();
    // the attribute is per (function, device): remembered per context (a context lives on one device, is driven by one
    // host thread at a time) and per template instance
    constexpr uint32_t bit = 1u << ((KIND * 2 + (WITH_E ? 1 : 0)) * 2 + (PACKED ? 1 : 0));
    if (!(ctx->zm_attr_set & bit)) {
        SG_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->zm_attr_set |= bit;
    }
    kern<<<grid, ZmGeom<ZM_TX, ZM_TY>::THREADS, smem, ctx->stream>>>(p);
    return SG_OK;
}

// the caller asked for the packed path and every sample holds packed bimodal couplings of one and the same D
bool use_packed(const sg_ctx* ctx)
{
    if (!ctx->packed_on || !ctx->Jp) return false;
    for (double d : ctx->bimodal_D)
        if (!(d == ctx->bimodal_D[0])) return false;     // NaN (not packed) fails too
    return true;
}

template <int KIND, bool WITH_E>
int launch_zm(sg_ctx* ctx, const ZmParams& p, dim3 grid)
{
    return use_packed(ctx) ? launch_zm_p<KIND, WITH_E, true>(ctx, p, grid) : launch_zm_p<KIND, WITH_E, false>(ctx, p, grid);
}

int half_sweep_zm(sg_ctx* ctx, int kind, int colour, bool with_energy)
{
    ZmParams p;
    p.spins = ctx->spins; p.Jt = ctx->Jt; p.beta_slot = ctx->beta_slot; p.Epart = ctx->Epart;
    p.Jp = ctx->Jp; p.bimA = p.bimB = p.bimD = 0.f;
    if (use_packed(ctx)) { const double D = ctx->bimodal_D[0]; p.bimA = (float)(1.0 + D); p.bimB = (float)(1.0 - D); p.bimD = (float)D; }
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.C = ctx->C;
    p.ntx = ctx->L / ZM_TX; p.nty = ctx->L / ZM_TY; p.nzc = ctx->zm_nzc; p.ZC = ctx->zm_ZC;
    p.colour = colour;
    p.key0 = (uint32_t)(ctx->shape.seed & 0xffffffffu); p.key1 = (uint32_t)(ctx->shape.seed >> 32);
    p.hb_counter = (uint32_t)ctx->hb_counter;
    p.g_first = ctx->g_first; p.Cg = ctx->Cg; p.Tl = ctx->T; p.Tpad = ctx->Tt - ctx->T;
    const int nblk = p.ntx * p.nty * p.nzc;
    const dim3 grid(nblk * ctx->NG, ctx->S);
    int rc;
    if (kind == KIND_OR) rc = with_energy ? launch_zm<KIND_OR, true>(ctx, p, grid) : launch_zm<KIND_OR, false>(ctx, p, grid);
    else if (kind == KIND_HB) rc = with_energy ? launch_zm<KIND_HB, true>(ctx, p, grid) : launch_zm<KIND_HB, false>(ctx, p, grid);
    else rc = launch_zm<KIND_ENERGY, true>(ctx, p, grid);
    if (rc != SG_OK) return rc;
    SG_LAUNCHED(ctx);
    if (kind == KIND_HB) note_counter_node(ctx, ctx->stream, 0, offsetof(ZmParams, hb_counter), sizeof(ZmParams));
    if (with_energy || kind == KIND_ENERGY) {
        k_reduce_energy<<<ctx->S * ctx->NG, 256, 0, ctx->stream>>>(ctx->Epart, ctx->E, nblk);
        SG_LAUNCHED(ctx);
        ctx->energies_fresh = true;
    } else {
        ctx->energies_fresh = false;
    }
    return SG_OK;
}

// ---- colour-fused overrelaxation sweep (sg_sweep_fz.cuh): one pass per sweep, out of place ----
constexpr int FZ_NSO = 4, FZ_NSN = 3, FZ_NJ = 3;

void fz_plan(sg_ctx* ctx)
{
    const int L = ctx->L;
    ctx->fz_ZC = 0; ctx->fz_nzc = 0;
    if (L % 8 != 0 || !ctx->spins2) return;
    int ZC = 0;
    if (ctx->zm_zc_req > 0) {
        ZC = ctx->zm_zc_req;
    } else {
        // the longest chunk (a chunk recomputes 2 colour-0 planes per ZC) that still gives every SM a few CTAs in turn (1 per SM resident)
        const long per_chunk = (long)ctx->S * ctx->NG * (L / 8) * (L / 8);
        for (int cand = L; cand >= 4; --cand) {
            if ((cand & 1) || L % cand != 0) continue;
            ZC = cand;
            if (per_chunk * (L / cand) >= 4 * 148) break;
        }
    }
    if (ZC < 2 || (ZC & 1) || L % ZC != 0) return;
    ctx->fz_ZC = ZC; ctx->fz_nzc = L / ZC;
}

int sweep_fused(sg_ctx* ctx, bool with_energy)
{
    FzParams p;
    p.src = ctx->spins; p.dst = ctx->spins2; p.Jt = ctx->Jt; p.Jr = ctx->Jr; p.Epart = ctx->Epart;
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG;
    p.ntx = ctx->L / 8; p.nty = ctx->L / 8; p.nzc = ctx->fz_nzc; p.ZC = ctx->fz_ZC;
    const int nblk = p.ntx * p.nty * p.nzc;
    const dim3 grid(nblk * ctx->NG, ctx->S);
    constexpr size_t smem = fz_smem_bytes<FZ_NSO, FZ_NSN, FZ_NJ>();
    auto k0 = k_sweep_fz<false, FZ_NSO, FZ_NSN, FZ_NJ>;
    auto k1 = k_sweep_fz<true, FZ_NSO, FZ_NSN, FZ_NJ>;
    const uint32_t bit = with_energy ? 2u : 1u;
    if (!(ctx->fz_attr_set & bit)) {
        SG_CUDA(ctx, cudaFuncSetAttribute(with_energy ? k1 : k0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->fz_attr_set |= bit;
    }
    if (with_energy) k1<<<grid, FzGeom::THREADS, smem, ctx->stream>>>(p);
    else k0<<<grid, FzGeom::THREADS, smem, ctx->stream>>>(p);
    SG_LAUNCHED(ctx);
    float* t = ctx->spins; ctx->spins = ctx->spins2; ctx->spins2 = t;      // the new state
    if (with_energy) {
        k_reduce_energy<<<ctx->S * ctx->NG, 256, 0, ctx->stream>>>(ctx->Epart, ctx->E, nblk);
        SG_LAUNCHED(ctx);
        ctx->energies_fresh = true;
    } else {
        ctx->energies_fresh = false;
    }
    return SG_OK;
}

// one half-sweep of every copy; with_energy also reduces E (valid because a whole colour is swept)
int half_sweep(sg_ctx* ctx, int kind, int colour, bool with_energy)
{
    if (ctx->zm_ok && ctx->sweep_impl != SG_SWEEP_TILED) return half_sweep_zm(ctx, kind, colour, with_energy);
    SweepParams p;
    p.spins = ctx->spins; p.Jg = ctx->Jg; p.beta_slot = ctx->beta_slot; p.Epart = ctx->Epart;
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.ntiles = ctx->ntiles;
    p.tile_sites = ctx->tile_sites; p.colour = colour; p.C = ctx->C;
    p.key0 = (uint32_t)(ctx->shape.seed & 0xffffffffu); p.key1 = (uint32_t)(ctx->shape.seed >> 32);
    p.hb_counter = (uint32_t)ctx->hb_counter;
    p.g_first = ctx->g_first; p.Cg = ctx->Cg; p.Tl = ctx->T; p.Tpad = ctx->Tt - ctx->T;
    const dim3 grid(ctx->ntiles * ctx->NG, ctx->S);
    if (kind == KIND_OR) {
        if (with_energy) launch_sweep_l<KIND_OR, true>(ctx, p, grid);
        else launch_sweep_l<KIND_OR, false>(ctx, p, grid);
    } else if (kind == KIND_HB) {
        if (with_energy) launch_sweep_l<KIND_HB, true>(ctx, p, grid);
        else launch_sweep_l<KIND_HB, false>(ctx, p, grid);
    } else {
        launch_sweep_l<KIND_ENERGY, true>(ctx, p, grid);
    }
    SG_LAUNCHED(ctx);
    if (kind == KIND_HB) note_counter_node(ctx, ctx->stream, 0, offsetof(SweepParams, hb_counter), sizeof(SweepParams));
    if (with_energy || kind == KIND_ENERGY) {
        k_reduce_energy<<<ctx->S * ctx->NG, 256, 0, ctx->stream>>>(ctx->Epart, ctx->E, ctx->ntiles);
        SG_LAUNCHED(ctx);
        ctx->energies_fresh = true;
    } else {
        ctx->energies_fresh = false;
    }
    return SG_OK;
}

// n doubles of ctx->result to the host and a stream synchronisation; returns where they are (pinned mirror), or
// nullptr with *rc set on failure / when no mirror exists (the caller then copies piecewise)
const double* fetch_result(sg_ctx* ctx, size_t n, int* rc)
{
    *rc = SG_OK;
    if (!ctx->h_result || n > ctx->result_doubles) return nullptr;
    cudaError_t e = cudaMemcpyAsync(ctx->h_result, ctx->result, n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { *rc = cuda_fail(ctx, e); return nullptr; }
    return ctx->h_result;
}

int all_inited(const sg_ctx* ctx)
{
    for (char c : ctx->inited)
        if (!c) return SG_ESTATE;
    return SG_OK;
}

int ensure_energies(sg_ctx* ctx)
{
    if (ctx->energies_fresh) return SG_OK;
    return half_sweep(ctx, KIND_ENERGY, 0, true);
}

int fill_beta_slot(sg_ctx* ctx)
{
    const int n = ctx->S * ctx->Cp;
    k_fill_beta_slot<<<(n + 255) / 256, 256, 0, ctx->stream>>>(ctx->betas, ctx->temp_of_slot, ctx->beta_slot, ctx->S,
                                                              ctx->R, ctx->Tt, ctx->T, ctx->slot0, ctx->Cp);
    SG_LAUNCHED(ctx);
    return SG_OK;
}

// ---- shared-memory-resident multi-sweep kernel (sg_sweep_res.cuh): n sweeps of one kind in ONE launch ----
constexpr size_t RES_SMEM_MAX = 200 * 1024;   // + 8.4 KB static reduction scratch <= 227 KB per CTA

template <int KIND, int CPC>
int launch_res_c(sg_ctx* ctx, const ResParams& p)
{
    // the couplings ride along in shared memory when they fit beside the lattice (L <= 8: no global load left in the sweep loop)
    const bool jsmem = res_smem_bytes(ctx->N, CPC) + res_jsmem_bytes(ctx->N) <= RES_SMEM_MAX;
    const size_t smem = res_smem_bytes(ctx->N, CPC) + (jsmem ? res_jsmem_bytes(ctx->N) : 0);
    const dim3 grid(ctx->NG * (G / CPC), ctx->S);
#define SG_RES_CASE(LG)                                                                                              \
    if (jsmem) {                                                                                                     \
        auto kern = k_sweep_res<KIND, LG, CPC, true>;                                                                \
        SG_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES_SMEM_MAX));    \
        kern<<<grid, RES_THREADS, smem, ctx->stream>>>(p);                                                           \
    } else {                                                                                                         \
        auto kern = k_sweep_res<KIND, LG, CPC>;                                                                      \
        SG_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES_SMEM_MAX));    \
        kern<<<grid, RES_THREADS, smem, ctx->stream>>>(p);                                                           \
    }
    switch (ctx->log2L) {
    case 1: SG_RES_CASE(1) break;
    case 2: SG_RES_CASE(2) break;
    case 3: SG_RES_CASE(3) break;
    default: SG_RES_CASE(0) break;
    }
#undef SG_RES_CASE
    return SG_OK;
}

template <int KIND>
int launch_res(sg_ctx* ctx, const ResParams& p)
{
    switch (ctx->res_cpc) {
    case 4: return launch_res_c<KIND, 4>(ctx, p);
    case 8: return launch_res_c<KIND, 8>(ctx, p);
    case 16: return launch_res_c<KIND, 16>(ctx, p);
    default: return launch_res_c<KIND, 32>(ctx, p);
    }
}

// copies per CTA of the resident kernel: 8 (full 32-byte sectors, several CTAs per SM), 4 when even that leaves most
// SMs idle; a request through sg_tune(SG_TUNE_RES_COPIES) wins if its lattice fits
void res_plan(sg_ctx* ctx)
{
    ctx->res_ok = (res_smem_bytes(ctx->N, 4) <= RES_SMEM_MAX) ? 1 : 0;     // an explicit request is honoured down to 4 copies
    ctx->res_auto = (res_smem_bytes(ctx->N, 8) <= RES_SMEM_MAX) ? 1 : 0;   // automatic choice: full 32-byte sectors only
    int cpc = ctx->res_cpc_req;
    if (cpc == 0) cpc = ((long)ctx->S * ctx->NG * (G / 8) < 148) ? 4 : 8;
    while (cpc > 4 && res_smem_bytes(ctx->N, cpc) > RES_SMEM_MAX) cpc /= 2;
    ctx->res_cpc = cpc;
}

bool use_resident(const sg_ctx* ctx)
{
    return (ctx->res_auto && ctx->sweep_impl == SG_SWEEP_AUTO) || (ctx->res_ok && ctx->sweep_impl == SG_SWEEP_RESIDENT);
}

int sweeps_resident(sg_ctx* ctx, int kind, int n_sweeps)
{
    ResParams p;
    p.spins = ctx->spins; p.Jg = ctx->Jg; p.beta_slot = ctx->beta_slot; p.E = ctx->E;
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.C = ctx->C; p.Cp = ctx->Cp;
    p.n_sweeps = n_sweeps; p.n_hb = 0;
    p.key0 = (uint32_t)(ctx->shape.seed & 0xffffffffu); p.key1 = (uint32_t)(ctx->shape.seed >> 32);
    p.hb_counter = (uint32_t)ctx->hb_counter;
    p.g_first = ctx->g_first; p.Cg = ctx->Cg; p.Tl = ctx->T; p.Tpad = ctx->Tt - ctx->T;
    if (int rc = (kind == KIND_HB) ? launch_res<1>(ctx, p) : launch_res<0>(ctx, p)) return rc;
    SG_LAUNCHED(ctx);
    if (kind == KIND_HB) note_counter_node(ctx, ctx->stream, 0, offsetof(ResParams, hb_counter), sizeof(ResParams));
    if (kind == KIND_HB) ctx->hb_counter += (uint64_t)n_sweeps;
    ctx->energies_fresh = true;
    return SG_OK;
}

// the sweeps of a whole unit -- n_hb heat-bath sweeps, then n_or overrelaxation sweeps -- in ONE launch of the resident kernel
int sweeps_resident_unit(sg_ctx* ctx, int n_hb, int n_or)
{
    ResParams p;
    p.spins = ctx->spins; p.Jg = ctx->Jg; p.beta_slot = ctx->beta_slot; p.E = ctx->E;
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.C = ctx->C; p.Cp = ctx->Cp;
    p.n_sweeps = n_or; p.n_hb = n_hb;
    p.key0 = (uint32_t)(ctx->shape.seed & 0xffffffffu); p.key1 = (uint32_t)(ctx->shape.seed >> 32);
    p.hb_counter = (uint32_t)ctx->hb_counter;
    p.g_first = ctx->g_first; p.Cg = ctx->Cg; p.Tl = ctx->T; p.Tpad = ctx->Tt - ctx->T;
    if (int rc = launch_res<2>(ctx, p)) return rc;
    SG_LAUNCHED(ctx);
    note_counter_node(ctx, ctx->stream, 0, offsetof(ResParams, hb_counter), sizeof(ResParams));
    ctx->hb_counter += (uint64_t)n_hb;
    ctx->energies_fresh = true;
    return SG_OK;
}

// ---- cluster-resident multi-sweep kernel (sg_sweep_cres.cuh): L = 16, the lattice of a copy group in the shared memory of 8 CTAs ----
// explicit request: both sweep kinds; automatic choice: overrelaxation only (measured at cfg 2: 96 against 101 us per OR sweep,
// 241 against 164 us per heat-bath sweep -- 15 clusters = 120 of the 148 SMs run at once), and only when the clusters fill the GPU
bool use_cluster(const sg_ctx* ctx, int kind)
{
    if (ctx->L != CresGeom::L) return false;
    if (ctx->sweep_impl == SG_SWEEP_CLUSTER) return true;
    return ctx->sweep_impl == SG_SWEEP_AUTO && !ctx->cres_unavailable && kind == KIND_OR && (long)ctx->S * ctx->NG >= 15;
}

template <int KIND, int CS>
int launch_cres(sg_ctx* ctx, const CresParams& p)
{
    using Gm = CresGeomT<CS>;
    auto kern = k_sweep_cres<KIND, CS>;
    const uint32_t bit = 1u << (KIND * 2 + (CS == 8 ? 1 : 0));
    if (!(ctx->cres_attr_set & bit)) {
        SG_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Gm::SMEM));
        ctx->cres_attr_set |= bit;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(CS * (G / Gm::NC) * ctx->NG, ctx->S);
    cfg.blockDim = dim3(Gm::THREADS);
    cfg.dynamicSmemBytes = Gm::SMEM;
    cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    SG_CUDA(ctx, cudaLaunchKernelEx(&cfg, kern, p));
    return SG_OK;
}

int sweeps_cluster(sg_ctx* ctx, int kind, int n_sweeps)
{
    CresParams p;
    p.spins = ctx->spins; p.Jg = ctx->Jg; p.beta_slot = ctx->beta_slot; p.Epart = ctx->Epart;
    p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.Cp = ctx->Cp; p.Cg = ctx->Cg; p.Tl = ctx->T; p.Tpad = ctx->Tt - ctx->T;
    p.n_sweeps = n_sweeps;
    p.key0 = (uint32_t)(ctx->shape.seed & 0xffffffffu); p.key1 = (uint32_t)(ctx->shape.seed >> 32);
    p.hb_counter = (uint32_t)ctx->hb_counter; p.g_first = ctx->g_first;
    int rc;
    if (ctx->cres_cs == 8) rc = (kind == KIND_HB) ? launch_cres<KIND_HB, 8>(ctx, p) : launch_cres<KIND_OR, 8>(ctx, p);
    else rc = (kind == KIND_HB) ? launch_cres<KIND_HB, 4>(ctx, p) : launch_cres<KIND_OR, 4>(ctx, p);
    if (rc != SG_OK) return rc;
    SG_LAUNCHED(ctx);
    if (kind == KIND_HB) note_counter_node(ctx, ctx->stream, 0, offsetof(CresParams, hb_counter), sizeof(CresParams));
    k_reduce_energy<<<ctx->S * ctx->NG, 256, 0, ctx->stream>>>(ctx->Epart, ctx->E, ctx->cres_cs);
    SG_LAUNCHED(ctx);
    if (kind == KIND_HB) ctx->hb_counter += (uint64_t)n_sweeps;
    ctx->energies_fresh = true;
    return SG_OK;
}

int sweeps(sg_ctx* ctx, int kind, int n_sweeps)
{
    if (!ctx || n_sweeps < 0) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    if (n_sweeps == 0) return SG_OK;
    int& served = ctx->served_impl[kind == KIND_HB ? 1 : 0];
    if (use_resident(ctx)) { served = SG_SWEEP_RESIDENT; return sweeps_resident(ctx, kind, n_sweeps); }
    if (use_cluster(ctx, kind)) {
        const int rc = sweeps_cluster(ctx, kind, n_sweeps);
        // the automatic choice falls back to the z-marching kernel where 8-CTA clusters of 192 KB cannot be launched
        // (the launch call itself fails: nothing ran); an explicit request reports the error
        if (rc == SG_OK) served = SG_SWEEP_CLUSTER;
        if (rc == SG_OK || ctx->sweep_impl == SG_SWEEP_CLUSTER || ctx->capturing) return rc;
        cudaGetLastError();
        ctx->cres_unavailable = true;
        ctx->cres_fail_cuda = ctx->last_cuda;     // kept for sg_sweep_impl_used; this call goes on and succeeds,
        ctx->last_cuda = 0;                       // so sg_last_cuda_error must not report a failure for it
    }
    if (kind == KIND_OR && ctx->sweep_impl == SG_SWEEP_FUSED && ctx->fz_ZC > 0 && !use_packed(ctx)) {
        served = SG_SWEEP_FUSED;
        for (int k = 0; k < n_sweeps; ++k)
            if (int rc = sweep_fused(ctx, k == n_sweeps - 1)) return rc;
        return SG_OK;
    }
    served = (ctx->zm_ok && ctx->sweep_impl != SG_SWEEP_TILED) ? SG_SWEEP_ZMARCH : SG_SWEEP_TILED;
    for (int k = 0; k < n_sweeps; ++k) {
        if (int rc = half_sweep(ctx, kind, 0, false)) return rc;
        if (int rc = half_sweep(ctx, kind, 1, k == n_sweeps - 1)) return rc;
        if (kind == KIND_HB) ctx->hb_counter += 1;
    }
    return SG_OK;
}

// the streaming overlap pass (sg_measure.cuh) for R = 2, 3, 4 replicas
template <int R_>
int launch_measure_rows(sg_ctx* ctx)
{
    MeasureRowsParams p;
    p.spins = ctx->spins; p.slot_of_temp = ctx->slot_of_temp; p.phase = ctx->phase; p.Mpart = ctx->Mpart;
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.R = ctx->R; p.T = ctx->T; p.P = ctx->P;
    p.nchunk = ctx->mq_nchunk; p.rows_per_cta = ctx->mq_rows_per_cta; p.Tw = ctx->mq_Tw; p.rows_t = ctx->mq_rows_t;
    const size_t smem = mrows_smem_bytes(ctx->L, R_);
    auto kern = k_measure_rows<R_>;
    if (!(ctx->mq_attr_set & (1u << R_))) {
        SG_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->mq_attr_set |= 1u << R_;
    }
    const int tz = (ctx->T + ctx->mq_Tw - 1) / ctx->mq_Tw;
    kern<<<dim3(ctx->mq_nchunk, ctx->S, tz), MROWS_THREADS, smem, ctx->stream>>>(p);
    SG_LAUNCHED(ctx);
    return SG_OK;
}

}  // namespace

extern "C" {

size_t sg_workspace_bytes(const sg_shape* shape)
{
    if (!shape_ok(shape)) return 0;
    return offsets(geometry(shape)).total;
}

int sg_create(sg_ctx** out, const sg_shape* shape, const double* betas, void* dev_workspace, size_t bytes,
              void* cuda_stream)
{
    if (!out) return SG_EINVAL;
    *out = nullptr;
    if (!shape_ok(shape) || !betas || !dev_workspace) return SG_EINVAL;
    if (((uintptr_t)dev_workspace & 255) != 0) return SG_EINVAL;
    const int n_betas = shape->n_temps_total ? shape->n_temps_total : shape->n_temps;   // the whole chain
    for (int t = 0; t < n_betas; ++t)
        if (!std::isfinite(betas[t])) return SG_EINVAL;
    if (n_betas > 1) {
        const bool up = betas[1] > betas[0];
        for (int t = 1; t < n_betas; ++t)
            if (up ? !(betas[t] > betas[t - 1]) : !(betas[t] < betas[t - 1])) return SG_EINVAL;
    }
    const Geometry g = geometry(shape);
    const Offsets o = offsets(g);
    if (bytes < o.total) return SG_EINVAL;

    sg_ctx* ctx = new (std::nothrow) sg_ctx();
    if (!ctx) return SG_EINVAL;
    ctx->shape = *shape;
    ctx->L = g.L; ctx->N = g.N; ctx->Nh = g.Nh; ctx->S = g.S; ctx->R = g.R; ctx->T = g.T; ctx->C = g.C;
    ctx->NG = g.NG; ctx->Cp = g.Cp; ctx->P = g.P;
    ctx->Tt = g.Tt; ctx->slot0 = shape->first_slot;
    ctx->Rt = shape->n_replicas_total ? shape->n_replicas_total : g.R; ctx->Cg = ctx->Rt * g.Tt;
    ctx->g_first = (uint32_t)shape->first_sample * (uint32_t)ctx->Cg + (uint32_t)shape->first_replica * (uint32_t)g.Tt + (uint32_t)shape->first_slot;
    ctx->tile_sites = g.tile_sites; ctx->ntiles = g.ntiles; ctx->log2L = ilog2_exact(g.L);
    ctx->nchunk = g.nchunk; ctx->chunk_sites = g.chunk_sites; ctx->MS = g.MS;
    ctx->mq_nchunk = g.mq_nchunk; ctx->mq_rows_per_cta = g.mq_rows_per_cta; ctx->mq_Tw = g.mq_Tw; ctx->mq_rows_t = g.mq_rows_t;
    ctx->stream = (cudaStream_t)cuda_stream;
    char* base = (char*)dev_workspace;
    ctx->spins2 = g.fused ? (float*)(base + o.spins2) : nullptr; ctx->Jr = g.fused ? (float*)(base + o.Jr) : nullptr;
    ctx->spins = (float*)(base + o.spins); ctx->Jg = (float*)(base + o.Jg); ctx->Jt = (g.L % 8 == 0) ? (float*)(base + o.Jt) : nullptr; ctx->Jp = (g.L % 8 == 0) ? (unsigned char*)(base + o.Jp) : nullptr; ctx->Mraw = (float*)(base + o.Mraw);
    ctx->staging = (float*)(base + o.staging); ctx->beta_slot = (float*)(base + o.beta_slot);
    ctx->betas = (double*)(base + o.betas); ctx->E = (double*)(base + o.E); ctx->Epart = (double*)(base + o.Epart);
    ctx->SDpart = (double*)(base + o.SDpart);
    ctx->phase = (double*)(base + o.phase); ctx->Mpart = (double*)(base + o.Mpart);
    ctx->result = (double*)(base + o.result);
    ctx->result_doubles = (size_t)g.S * g.R * g.Tt + (size_t)g.S * g.P * g.Tt * 21 + (size_t)g.S * g.Tt * 21 + 1;
    if (cudaHostAlloc((void**)&ctx->h_result, ctx->result_doubles * sizeof(double), cudaHostAllocDefault) != cudaSuccess) {
        ctx->h_result = nullptr;   // fall back to direct copies into the caller's arrays
        cudaGetLastError();
    }
    ctx->slot_of_temp = (int*)(base + o.sot); ctx->temp_of_slot = (int*)(base + o.tos);
    ctx->attempts = (unsigned long long*)(base + o.att); ctx->accepts = (unsigned long long*)(base + o.acc);
    ctx->walk_label = (int*)(base + o.wlab); ctx->round_trips = (unsigned long long*)(base + o.trips);
    ctx->visits = visits_bytes(g) ? (unsigned long long*)(base + o.visits) : nullptr;
    ctx->logbin = (double*)(base + o.logbin); ctx->n_acc = 0;
    ctx->Xpart = (double*)(base + o.xpart);
    for (int b = 0; b < SG_LOGBINS; ++b) ctx->n_acc_cg[b] = 0;
    ctx->h_betas.assign(betas, betas + g.Tt);
    ctx->inited.assign(g.S, 0);
    ctx->bimodal_D.assign(g.S, std::nan("")); ctx->packed_on = 0;
    ctx->hb_counter = ctx->pt_counter = ctx->launches = 0;
    ctx->sweep_impl = SG_SWEEP_AUTO; ctx->zm_zc_req = 0;
    ctx->res_cpc_req = 0;
    res_plan(ctx);
    zm_plan(ctx);
    fz_plan(ctx);
    ctx->energies_fresh = false;
    ctx->last_cuda = 0;

    // small tables: betas, Fourier phases, identity permutations, zeroed statistics
    std::vector<double> phase(2 * (size_t)g.L);
    for (int x = 0; x < g.L; ++x) {
        phase[2 * x] = std::cos(2.0 * kPi * (double)x / (double)g.L);
        phase[2 * x + 1] = std::sin(2.0 * kPi * (double)x / (double)g.L);
    }
    std::vector<int> ident((size_t)g.S * g.R * g.Tt);
    for (size_t k = 0; k < ident.size(); ++k) ident[k] = (int)(k % g.Tt);
    cudaError_t e = cudaMemcpyAsync(ctx->betas, betas, g.Tt * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->phase, phase.data(), phase.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->slot_of_temp, ident.data(), ident.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->temp_of_slot, ident.data(), ident.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream);
    const size_t st = (size_t)g.S * g.R * (g.Tt > 1 ? g.Tt - 1 : 1) * sizeof(unsigned long long);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->attempts, 0, st, ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->accepts, 0, st, ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->walk_label, 0, (size_t)g.S * g.R * g.Tt * sizeof(int), ctx->stream);
    if (e == cudaSuccess && ctx->visits) e = cudaMemsetAsync(ctx->visits, 0, visits_bytes(g), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->round_trips, 0, (size_t)g.S * g.R * sizeof(unsigned long long), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->logbin, 0, (size_t)SG_LOGBINS * g.S * g.T * SG_LOGBIN_OBS * sizeof(double), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->E, 0, (size_t)g.S * g.Cp * sizeof(double), ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);   // the host vectors above go out of scope
    if (e != cudaSuccess) { delete ctx; return SG_ECUDA; }
    int rc = fill_beta_slot(ctx);
    if (rc != SG_OK) { delete ctx; return rc; }
    *out = ctx;
    return SG_OK;
}

int sg_destroy(sg_ctx* ctx)
{
    if (!ctx) return SG_EINVAL;
    cudaStreamSynchronize(ctx->stream);
    if (ctx->gstream) { cudaStreamSynchronize(ctx->gstream); cudaStreamDestroy(ctx->gstream); }
    if (ctx->gevent) cudaEventDestroy(ctx->gevent);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    for (int k = 0; k < sg_ctx::UP_CHUNKS; ++k) {
        if (ctx->ev_copied[k]) cudaEventDestroy(ctx->ev_copied[k]);
        if (ctx->ev_done[k]) cudaEventDestroy(ctx->ev_done[k]);
    }
    if (ctx->h_result) cudaFreeHost(ctx->h_result);
    delete ctx;
    return SG_OK;
}

// the streams and events of the pipelined upload, created on first use
static bool upload_ready(sg_ctx* ctx)
{
    if (ctx->upload_state != 0) return ctx->upload_state > 0;
    ctx->upload_state = -1;
    if (cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); ctx->copy_stream = nullptr; return false; }
    bool ok = cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming) == cudaSuccess;
    for (int k = 0; ok && k < sg_ctx::UP_CHUNKS; ++k)
        ok = cudaEventCreateWithFlags(&ctx->ev_copied[k], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&ctx->ev_done[k], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { cudaGetLastError(); return false; }
    ctx->upload_state = 1;
    return true;
}

// large lattices: chunks of sites, copy of chunk k+1 (copy stream) under the transposition of chunk k (context's stream)
static int set_spins_pipelined(sg_ctx* ctx, int sample, const float* in)
{
    constexpr int K = sg_ctx::UP_CHUNKS;
    const int N = ctx->N, nchunk_sites = (N + K - 1) / K;
    const size_t copy_floats = (size_t)3 * N;
    SG_CUDA(ctx, cudaEventRecord(ctx->ev_start, ctx->stream));             // the staging buffer may still be in use by earlier work
    SG_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_start, 0));
    bool used[K] = {};
    for (int grp = 0; grp < ctx->NG; ++grp) {
        const int c0 = grp * G, nc = (ctx->C - c0 < G) ? ctx->C - c0 : G;
        float* dev = ctx->spins + ((size_t)(sample * ctx->NG + grp) * N) * SITE_FLOATS;
        for (int k = 0; k < K; ++k) {
            const int i_first = k * nchunk_sites, n = (N - i_first < nchunk_sites) ? N - i_first : nchunk_sites;
            if (n <= 0) break;
            float* stg = ctx->staging + (size_t)G * 3 * i_first;           // region of chunk k: [c][3][n]
            if (used[k]) SG_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_done[k], 0));
            if (nc < G) SG_CUDA(ctx, cudaMemsetAsync(stg, 0, (size_t)G * 3 * n * sizeof(float), ctx->copy_stream));
            SG_CUDA(ctx, cudaMemcpy2DAsync(stg, (size_t)n * sizeof(float), in + (size_t)c0 * copy_floats + i_first, (size_t)N * sizeof(float),
                                           (size_t)n * sizeof(float), (size_t)nc * 3, cudaMemcpyHostToDevice, ctx->copy_stream));
            SG_CUDA(ctx, cudaEventRecord(ctx->ev_copied[k], ctx->copy_stream));
            SG_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_copied[k], 0));
            k_spins_from_staging_chunk<<<dim3((n + 31) / 32, 3), dim3(32, 8), 0, ctx->stream>>>(stg, dev, N, ctx->L, i_first, n);
            SG_LAUNCHED(ctx);
            SG_CUDA(ctx, cudaEventRecord(ctx->ev_done[k], ctx->stream));
            used[k] = true;
        }
    }
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->energies_fresh = false;
    return SG_OK;
}

int sg_set_spins(sg_ctx* ctx, int sample, const float* in)
{
    if (!ctx || !in || sample < 0 || sample >= ctx->S) return SG_EINVAL;
    if (ctx->N >= 32768 && upload_ready(ctx)) return set_spins_pipelined(ctx, sample, in);
    const size_t copy_floats = (size_t)3 * ctx->N;
    for (int grp = 0; grp < ctx->NG; ++grp) {
        const int c0 = grp * G, nc = (ctx->C - c0 < G) ? ctx->C - c0 : G;
        if (nc < G) SG_CUDA(ctx, cudaMemsetAsync(ctx->staging, 0, (size_t)G * copy_floats * sizeof(float), ctx->stream));
        SG_CUDA(ctx, cudaMemcpyAsync(ctx->staging, in + (size_t)c0 * copy_floats, (size_t)nc * copy_floats * sizeof(float),
                                     cudaMemcpyHostToDevice, ctx->stream));
        float* dev = ctx->spins + ((size_t)(sample * ctx->NG + grp) * ctx->N) * SITE_FLOATS;
        k_spins_from_staging<<<dim3((ctx->N + 31) / 32, 3), dim3(32, 8), 0, ctx->stream>>>(ctx->staging, dev, ctx->N, ctx->L);
        SG_LAUNCHED(ctx);
    }
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->energies_fresh = false;
    return SG_OK;
}

int sg_get_spins(sg_ctx* ctx, int sample, float* out)
{
    if (!ctx || !out || sample < 0 || sample >= ctx->S) return SG_EINVAL;
    if (!ctx->inited[sample]) return SG_ESTATE;
    const size_t copy_floats = (size_t)3 * ctx->N;
    for (int grp = 0; grp < ctx->NG; ++grp) {
        const int c0 = grp * G, nc = (ctx->C - c0 < G) ? ctx->C - c0 : G;
        const float* dev = ctx->spins + ((size_t)(sample * ctx->NG + grp) * ctx->N) * SITE_FLOATS;
        k_spins_to_staging<<<dim3((ctx->N + 31) / 32, 3), dim3(32, 8), 0, ctx->stream>>>(dev, ctx->staging, ctx->N, ctx->L);
        SG_LAUNCHED(ctx);
        SG_CUDA(ctx, cudaMemcpyAsync(out + (size_t)c0 * copy_floats, ctx->staging, (size_t)nc * copy_floats * sizeof(float),
                                     cudaMemcpyDeviceToHost, ctx->stream));
        SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return SG_OK;
}

int sg_init_sample(sg_ctx* ctx, int sample, int gen_mode, double sigma_D, const float* couplings, const float* spins)
{
    if (!ctx || sample < 0 || sample >= ctx->S) return SG_EINVAL;
    if (!couplings && (gen_mode < SG_GEN_OFFDIAG_SYM || gen_mode > SG_GEN_FERRO || !std::isfinite(sigma_D))) return SG_EINVAL;
    const size_t mfloats = (size_t)3 * ctx->N * 9;
    float* Mdev = ctx->Mraw + (size_t)sample * mfloats;
    std::vector<float> gen;
    const float* src = couplings;
    if (!src) {
        gen.resize(mfloats);
        generate_couplings(ctx->L, ctx->shape.seed, (uint32_t)(ctx->shape.first_sample + sample), gen_mode, sigma_D, gen.data());
        src = gen.data();
    }
    ctx->bimodal_D[sample] = std::nan("");
    SG_CUDA(ctx, cudaMemcpyAsync(Mdev, src, mfloats * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    k_gather_couplings<<<(ctx->N + 127) / 128, 128, 0, ctx->stream>>>(Mdev, ctx->Jg + (size_t)sample * 2 * ctx->Nh * JG,
                                                                           ctx->Jt ? ctx->Jt + (size_t)sample * 2 * ctx->Nh * JG : nullptr, ctx->L);
    SG_LAUNCHED(ctx);
    if (ctx->Jr) {
        const size_t n = (size_t)(ctx->N / 4);
        k_gather_ring_couplings<<<(unsigned)((n + 127) / 128), 128, 0, ctx->stream>>>(ctx->Jg + (size_t)sample * 2 * ctx->Nh * JG,
                                                                                   ctx->Jr + (size_t)sample * n * JG, ctx->L);
        SG_LAUNCHED(ctx);
    }

    if (spins) {
        if (int rc = sg_set_spins(ctx, sample, spins)) return rc;
    } else {
        const size_t nthr = (size_t)ctx->NG * ctx->N * 8;
        const uint32_t g_sample = ctx->g_first + (uint32_t)sample * (uint32_t)ctx->Cg;
        k_init_spins<<<(unsigned)((nthr + 255) / 256), 256, 0, ctx->stream>>>(
            ctx->spins + (size_t)sample * ctx->NG * ctx->N * SITE_FLOATS, ctx->L, ctx->N, ctx->NG, ctx->C, g_sample, ctx->T, ctx->Tt - ctx->T,
            (uint32_t)(ctx->shape.seed & 0xffffffffu), (uint32_t)(ctx->shape.seed >> 32));
        SG_LAUNCHED(ctx);
    }
    // identity temperature assignment for this sample
    std::vector<int> ident((size_t)ctx->R * ctx->Tt);
    for (size_t k = 0; k < ident.size(); ++k) ident[k] = (int)(k % ctx->Tt);
    const size_t off = (size_t)sample * ctx->R * ctx->Tt;
    SG_CUDA(ctx, cudaMemcpyAsync(ctx->slot_of_temp + off, ident.data(), ident.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    SG_CUDA(ctx, cudaMemcpyAsync(ctx->temp_of_slot + off, ident.data(), ident.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (int rc = fill_beta_slot(ctx)) return rc;
    ctx->inited[sample] = 1;
    ctx->energies_fresh = false;
    return SG_OK;
}

int sg_init_sample_bimodal(sg_ctx* ctx, int sample, double D, const uint8_t* links, const float* spins)
{
    if (!ctx || sample < 0 || sample >= ctx->S || !std::isfinite(D) || D < 0.0) return SG_EINVAL;
    const int L = ctx->L, N = ctx->N;
    std::vector<uint8_t> bits((size_t)3 * N);
    if (links) {
        for (size_t k = 0; k < bits.size(); ++k) {
            if (links[k] & 0x80u) return SG_EINVAL;
            bits[k] = links[k];
        }
    } else {   // the bytes of generator mode SG_GEN_BIMODAL: low 7 bits of word 0 of the link's first Philox block
        const uint32_t k0 = (uint32_t)(ctx->shape.seed & 0xffffffffu), k1 = (uint32_t)(ctx->shape.seed >> 32);
        for (int i = 0; i < N; ++i)
            for (int mu = 0; mu < 3; ++mu) {
                uint32_t w[4];
                philox4x32_10((uint32_t)(3 * i + mu), (uint32_t)(ctx->shape.first_sample + sample), 0u, STREAM_COUPLINGS, k0, k1, w);
                bits[(size_t)mu * N + i] = (uint8_t)(w[0] & 0x7fu);
            }
    }
    // the fp32 matrices serve every kernel but the packed z-marching sweep (and sg_get_couplings)
    std::vector<float> M((size_t)3 * N * 9);
    for (size_t k = 0; k < bits.size(); ++k) {
        double m[9];
        bimodal_matrix(bits[k], D, m);
        for (int e = 0; e < 9; ++e) M[k * 9 + e] = (float)m[e];
    }
    if (int rc = sg_init_sample(ctx, sample, SG_GEN_FERRO, 0.0, M.data(), spins)) return rc;
    if (ctx->Jp) {
        // per-site gathered bytes in the tile-major order of Jt: (+x1, -x1, +x2, -x2, +x3, -x3, 0, 0); D is symmetric,
        // so the backward link's byte serves as it is
        std::vector<uint8_t> pk((size_t)N * 8, 0);
        const int nt = L >> 3;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    const int i = x + L * (y + L * z), colour = (x + y + z) & 1;
                    const int bw[3] = { ((x == 0) ? L - 1 : x - 1) + L * (y + L * z), x + L * (((y == 0) ? L - 1 : y - 1) + L * z),
                                        x + L * (y + L * ((z == 0) ? L - 1 : z - 1)) };
                    const size_t t = ((((size_t)colour * nt + (y >> 3)) * nt + (x >> 3)) * L + z) * 32 + (y & 7) * 4 + ((x & 7) >> 1);
                    for (int mu = 0; mu < 3; ++mu) {
                        pk[t * 8 + 2 * mu] = bits[(size_t)mu * N + i];
                        pk[t * 8 + 2 * mu + 1] = bits[(size_t)mu * N + bw[mu]];
                    }
                }
        SG_CUDA(ctx, cudaMemcpyAsync(ctx->Jp + (size_t)sample * N * 8, pk.data(), pk.size(), cudaMemcpyHostToDevice, ctx->stream));
        SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    ctx->bimodal_D[sample] = D;
    return SG_OK;
}

int sg_sweep_or(sg_ctx* ctx, int n_sweeps) { return sweeps(ctx, KIND_OR, n_sweeps); }
int sg_sweep_hb(sg_ctx* ctx, int n_sweeps) { return sweeps(ctx, KIND_HB, n_sweeps); }

int sg_halfsweep(sg_ctx* ctx, int kind, int colour)
{
    if (!ctx || (kind != SG_KIND_OR && kind != SG_KIND_HB) || (colour != 0 && colour != 1)) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    return half_sweep(ctx, kind, colour, false);
}

// one PT sweep of every chain from the energies E: local (E_wstride unused) or all-gathered [W][S][R][T] (slot sharding)
static int pt_launch(sg_ctx* ctx, const double* E, long long E_sstride, long long E_wstride)
{
    PtParams p;
    p.betas = ctx->betas; p.E = E; p.slot_of_temp = ctx->slot_of_temp; p.temp_of_slot = ctx->temp_of_slot;
    p.beta_slot = ctx->beta_slot; p.attempts = ctx->attempts; p.accepts = ctx->accepts;
    p.walk_label = ctx->walk_label; p.round_trips = ctx->round_trips; p.visits = ctx->visits;
    p.S = ctx->S; p.R = ctx->R; p.T = ctx->Tt; p.Cp = ctx->Cp;
    p.Tl = ctx->T; p.slot0 = ctx->slot0; p.E_sstride = E_sstride; p.E_wstride = E_wstride;
    p.key0 = (uint32_t)(ctx->shape.seed & 0xffffffffu); p.key1 = (uint32_t)(ctx->shape.seed >> 32);
    p.pt_counter = (uint32_t)ctx->pt_counter;
    p.chain_first = (uint32_t)ctx->shape.first_sample * (uint32_t)ctx->Rt + (uint32_t)ctx->shape.first_replica; p.Rt = ctx->Rt;
    const int chains = ctx->S * ctx->R;
    const size_t smem = (size_t)ctx->Tt * PT_SMEM_PER_TEMP;
    if (smem <= 40 * 1024) k_pt_swap<<<chains, 32, smem, ctx->stream>>>(p);             // a warp per chain, the chain in shared memory
    else k_pt_swap_serial<<<(chains + 63) / 64, 64, 0, ctx->stream>>>(p);
    SG_LAUNCHED(ctx);
    note_counter_node(ctx, ctx->stream, 1, offsetof(PtParams, pt_counter), sizeof(PtParams));
    ctx->pt_counter += 1;
    return SG_OK;
}

int sg_pt_swap(sg_ctx* ctx)
{
    if (!ctx || ctx->Tt != ctx->T) return SG_EINVAL;     // a slot-sharded chain needs the other shards' energies: sg_pt_swap_gathered
    if (int rc = all_inited(ctx)) return rc;
    if (int rc = ensure_energies(ctx)) return rc;
    return pt_launch(ctx, ctx->E, ctx->Cp, 0);
}

int sg_pt_publish(sg_ctx* ctx, void* dev_out)
{
    if (!ctx || !dev_out) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    if (int rc = ensure_energies(ctx)) return rc;
    SG_CUDA(ctx, cudaMemcpy2DAsync(dev_out, (size_t)ctx->C * sizeof(double), ctx->E, (size_t)ctx->Cp * sizeof(double),
                                   (size_t)ctx->C * sizeof(double), ctx->S, cudaMemcpyDeviceToDevice, ctx->stream));
    return SG_OK;
}

int sg_pt_swap_gathered(sg_ctx* ctx, const void* dev_all)
{
    if (!ctx || !dev_all) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    return pt_launch(ctx, (const double*)dev_all, (long long)ctx->R * ctx->T, (long long)ctx->S * ctx->R * ctx->T);
}

int sg_energy_by_temp(sg_ctx* ctx, const void* dev_all, double* e)
{
    if (!ctx || !dev_all || !e) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    const int n = ctx->S * ctx->R * ctx->Tt;
    k_energy_by_temp<<<(n + 127) / 128, 128, 0, ctx->stream>>>((const double*)dev_all, ctx->slot_of_temp, ctx->result, ctx->S, ctx->R, ctx->Tt,
                                                            ctx->T, ctx->N);
    SG_LAUNCHED(ctx);
    SG_CUDA(ctx, cudaMemcpyAsync(e, ctx->result, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

static int one_unit(sg_ctx* ctx, int n_or)
{
    if (n_or > 0 && use_resident(ctx)) {              // small lattices: the unit's sweeps in one launch
        if (int rc = all_inited(ctx)) return rc;
        ctx->served_impl[0] = ctx->served_impl[1] = SG_SWEEP_RESIDENT;
        if (int rc = sweeps_resident_unit(ctx, 1, n_or)) return rc;
        return sg_pt_swap(ctx);
    }
    if (int rc = sg_sweep_hb(ctx, 1)) return rc;
    if (int rc = sg_sweep_or(ctx, n_or)) return rc;
    return sg_pt_swap(ctx);
}

// Units u0 .. n_units-1 as replays of ONE captured unit ("CUDA-graph capture of a unit").  The launches
// of a unit are the same from unit to unit except for the HB and PT sweep counters inside two or three parameter blocks; those
// nodes are noted during the capture (note_counter_node) and patched before every replay.  Returns SG_OK with *done = false
// when the capture is not possible (the caller then issues the units one by one).
static int replay_units(sg_ctx* ctx, int n_units, int n_or, bool* done)
{
    *done = false;
    cudaStream_t user = ctx->stream, cap = ctx->stream;
    if (user == nullptr || user == cudaStreamLegacy || user == cudaStreamPerThread) {
        // the legacy default stream cannot be captured: replay on a stream of our own, ordered after / before the caller's by events
        if (!ctx->gstream) {
            if (cudaStreamCreateWithFlags(&ctx->gstream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); ctx->gstream = nullptr; return SG_OK; }
            if (cudaEventCreateWithFlags(&ctx->gevent, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); cudaStreamDestroy(ctx->gstream); ctx->gstream = nullptr; return SG_OK; }
        }
        cap = ctx->gstream;
        SG_CUDA(ctx, cudaEventRecord(ctx->gevent, user));
        SG_CUDA(ctx, cudaStreamWaitEvent(cap, ctx->gevent, 0));
    }
    const uint64_t hb0 = ctx->hb_counter, pt0 = ctx->pt_counter, launches0 = ctx->launches;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    ctx->counter_nodes.clear();
    if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return SG_OK; }
    ctx->stream = cap; ctx->capturing = true;
    const int rc_cap = one_unit(ctx, n_or);
    ctx->capturing = false; ctx->stream = user;
    const cudaError_t e_end = cudaStreamEndCapture(cap, &graph);
    const uint64_t per_unit = ctx->launches - launches0;
    ctx->hb_counter = hb0; ctx->pt_counter = pt0; ctx->launches = launches0;      // nothing ran
    bool ok = rc_cap == SG_OK && e_end == cudaSuccess && graph != nullptr;
    for (const auto& cn : ctx->counter_nodes) ok = ok && cn.node != nullptr;
    if (ok && cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) ok = false;
    struct Patch { cudaKernelNodeParams np; std::vector<unsigned char> block; void* args[1]; int which; size_t offset; uint32_t base; };
    std::vector<Patch> patches(ok ? ctx->counter_nodes.size() : 0);
    for (size_t k = 0; ok && k < patches.size(); ++k) {
        const auto& cn = ctx->counter_nodes[k];
        Patch& pa = patches[k];
        if (cudaGraphKernelNodeGetParams(cn.node, &pa.np) != cudaSuccess || !pa.np.kernelParams) { ok = false; break; }
        pa.block.assign((const unsigned char*)pa.np.kernelParams[0], (const unsigned char*)pa.np.kernelParams[0] + cn.size);
        pa.which = cn.which; pa.offset = cn.offset;
        std::memcpy(&pa.base, pa.block.data() + cn.offset, sizeof(uint32_t));     // the counter the capture saw
    }
    int rc = SG_OK;
    if (ok) {
        for (int u = 0; u < n_units && rc == SG_OK; ++u) {
            for (Patch& pa : patches) {
                const uint32_t v = pa.base + (uint32_t)u;     // both counters advance by one per unit
                std::memcpy(pa.block.data() + pa.offset, &v, sizeof(uint32_t));
                pa.args[0] = pa.block.data();
                pa.np.kernelParams = pa.args; pa.np.extra = nullptr;
                cudaGraphNode_t node = ctx->counter_nodes[&pa - patches.data()].node;
                if (cudaGraphExecKernelNodeSetParams(exec, node, &pa.np) != cudaSuccess) { rc = cuda_fail(ctx, cudaGetLastError()); break; }
            }
            if (rc != SG_OK) break;
            const cudaError_t e = cudaGraphLaunch(exec, cap);
            if (e != cudaSuccess) { rc = cuda_fail(ctx, e); break; }
            ctx->hb_counter += 1; ctx->pt_counter += 1; ctx->launches += per_unit; ctx->graph_replays += 1;
        }
        ctx->energies_fresh = true;
        *done = (rc == SG_OK);
    } else {
        cudaGetLastError();
    }
    if (exec) cudaGraphExecDestroy(exec);
    if (graph) cudaGraphDestroy(graph);
    ctx->counter_nodes.clear();
    if (cap != user) {
        cudaEventRecord(ctx->gevent, cap);
        cudaStreamWaitEvent(user, ctx->gevent, 0);
    }
    return rc;
}

int sg_run_units(sg_ctx* ctx, int n_units, int n_or)
{
    if (!ctx || n_units < 0 || n_or < 0 || ctx->Tt != ctx->T) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    int u = 0;
    // Replaying a captured unit pays when a unit is a handful of short launches (the resident kernel: L <= 12) and there are
    // enough units to amortise the capture; the first unit always runs directly (it sets the kernels' attributes).
    if (ctx->graph_mode && n_units >= 8 && use_resident(ctx)) {
        if (int rc = one_unit(ctx, n_or)) return rc;
        u = 1;
        bool done = false;
        if (int rc = replay_units(ctx, n_units - 1, n_or, &done)) return rc;
        if (done) return SG_OK;
    }
    for (; u < n_units; ++u)
        if (int rc = one_unit(ctx, n_or)) return rc;
    return SG_OK;
}

// S3 + S5 into ctx->result = [ e | q0 | qk ] (asynchronous); with_q = false skips the overlap pass
static int launch_measure(sg_ctx* ctx, bool with_q)
{
    if (ctx->Tt != ctx->T) return SG_EINVAL;      // slot-sharded: sg_energy_by_temp, sg_export_replica / sg_measure_cross
    if (int rc = all_inited(ctx)) return rc;
    if (int rc = ensure_energies(ctx)) return rc;
    const int PT = ctx->P * ctx->T;
    int nchunk = ctx->nchunk;
    if (PT > 0 && with_q) {
        const bool rows = ctx->measure_impl != SG_MEASURE_STAGED && ctx->R >= 2 && ctx->R <= 4 && mrows_smem_bytes(ctx->L, ctx->R) <= 200 * 1024;
        if (rows) {
            int rc = (ctx->R == 2) ? launch_measure_rows<2>(ctx) : (ctx->R == 3) ? launch_measure_rows<3>(ctx) : launch_measure_rows<4>(ctx);
            if (rc != SG_OK) return rc;
            nchunk = ctx->mq_nchunk;
        } else {
            MeasureParams p;
            p.spins = ctx->spins; p.slot_of_temp = ctx->slot_of_temp; p.phase = ctx->phase; p.Mpart = ctx->Mpart;
            p.L = ctx->L; p.N = ctx->N; p.NG = ctx->NG; p.Cp = ctx->Cp; p.R = ctx->R; p.T = ctx->T; p.P = ctx->P;
            p.nchunk = ctx->nchunk; p.chunk_sites = ctx->chunk_sites; p.MS = ctx->MS;
            int threads = ((PT + 31) / 32) * 32;
            if (threads > 512) threads = 512;
            const int nbatch = (PT + threads - 1) / threads;
            const size_t smem = (size_t)ctx->MS * 3 * ctx->Cp * sizeof(float) + (size_t)ctx->MS * 6 * sizeof(double);
            if (smem > 48 * 1024) return SG_EINVAL;
            k_measure<<<dim3(ctx->nchunk, ctx->S, nbatch), threads, smem, ctx->stream>>>(p);
            SG_LAUNCHED(ctx);
        }
    }
    const int nE = ctx->S * ctx->R * ctx->T, nQ = ctx->S * PT;
    const int total = nE + nQ * 7;
    k_reduce_measure<<<(total + 127) / 128, 128, 0, ctx->stream>>>(ctx->Mpart, ctx->E, ctx->slot_of_temp, ctx->result, ctx->S,
                                                                 ctx->R, ctx->T, ctx->P, ctx->Cp, nchunk, ctx->N);
    SG_LAUNCHED(ctx);
    return SG_OK;
}

int sg_measure(sg_ctx* ctx, double* e, double* q0, double* qk)
{
    if (!ctx) return SG_EINVAL;
    if (int rc = launch_measure(ctx, q0 || qk)) return rc;
    const int PT = ctx->P * ctx->T;
    const int nE = ctx->S * ctx->R * ctx->T, nQ = ctx->S * PT;
    {
        int rc;
        if (const double* h = fetch_result(ctx, (size_t)nE + (size_t)nQ * 7, &rc)) {
            if (e) std::memcpy(e, h, (size_t)nE * sizeof(double));
            if (q0 && nQ) std::memcpy(q0, h + nE, (size_t)nQ * sizeof(double));
            if (qk && nQ) std::memcpy(qk, h + nE + nQ, (size_t)nQ * 6 * sizeof(double));
            return SG_OK;
        }
        if (rc != SG_OK) return rc;
    }
    if (e) SG_CUDA(ctx, cudaMemcpyAsync(e, ctx->result, (size_t)nE * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (q0 && nQ) SG_CUDA(ctx, cudaMemcpyAsync(q0, ctx->result + nE, (size_t)nQ * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (qk && nQ) SG_CUDA(ctx, cudaMemcpyAsync(qk, ctx->result + nE + nQ, (size_t)nQ * 6 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

static int launch_measure_chiral(sg_ctx* ctx);

int sg_accumulate(sg_ctx* ctx, int with_chirality)
{
    if (!ctx) return SG_EINVAL;
    if (int rc = launch_measure(ctx, true)) return rc;
    const uint64_t n = ctx->n_acc + 1;
    int b = 0;
    while (b + 1 < SG_LOGBINS && (n >> (b + 1)) != 0) ++b;
    const int items = ctx->S * ctx->T;
    double* bin = ctx->logbin + (size_t)b * items * SG_LOGBIN_OBS;
    k_logbin_add<<<(items + 127) / 128, 128, 0, ctx->stream>>>(ctx->result, bin, ctx->S, ctx->R, ctx->T, ctx->P);
    SG_LAUNCHED(ctx);
    if (with_chirality) {
        if (ctx->P > 0) {     // the result buffer is reused: stream order keeps the two passes apart
            if (int rc = launch_measure_chiral(ctx)) return rc;
            k_logbin_add_chiral<<<(items + 127) / 128, 128, 0, ctx->stream>>>(ctx->result, bin, ctx->S, ctx->T, ctx->P);
            SG_LAUNCHED(ctx);
        }
        ctx->n_acc_cg[b] += 1;
    }
    ctx->n_acc = n;
    return SG_OK;
}

int sg_get_logbins(sg_ctx* ctx, double* sums, uint64_t* counts, uint64_t* counts_cg)
{
    if (!ctx) return SG_EINVAL;
    if (counts) {
        for (int b = 0; b < SG_LOGBINS; ++b) {
            const uint64_t lo = 1ull << b, hi = (b + 1 < SG_LOGBINS) ? (1ull << (b + 1)) : ~0ull;   // measurements lo <= n < hi
            counts[b] = (ctx->n_acc < lo) ? 0 : ((ctx->n_acc < hi ? ctx->n_acc + 1 : hi) - lo);
        }
    }
    if (counts_cg)
        for (int b = 0; b < SG_LOGBINS; ++b) counts_cg[b] = ctx->n_acc_cg[b];
    if (sums) SG_CUDA(ctx, cudaMemcpyAsync(sums, ctx->logbin, (size_t)SG_LOGBINS * ctx->S * ctx->T * SG_LOGBIN_OBS * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

// chiral-glass overlaps into ctx->result = [ qc0 | qck ] (asynchronous); requires P*T > 0
static int launch_measure_chiral(sg_ctx* ctx)
{
    const int PT = ctx->P * ctx->T;
    const int nQ = ctx->S * PT;
    ChiralParams p;
    p.spins = ctx->spins; p.slot_of_temp = ctx->slot_of_temp; p.phase = ctx->phase; p.Mpart = ctx->Mpart;
    p.L = ctx->L; p.N = ctx->N; p.NG = ctx->NG; p.Cp = ctx->Cp; p.R = ctx->R; p.T = ctx->T; p.P = ctx->P;
    p.nchunk = ctx->nchunk; p.chunk_sites = ctx->chunk_sites; p.MS = ctx->MS;
    int threads = ((PT + 31) / 32) * 32;
    if (threads > 512) threads = 512;
    if (threads < 128) threads = 128;        // the zeta stage wants a few warps even when there are few items
    const int nbatch = (PT + threads - 1) / threads;
    const size_t smem = (size_t)ctx->MS * 3 * ctx->Cp * sizeof(float) + (size_t)ctx->MS * 6 * sizeof(double) + (size_t)ctx->MS * 8 * sizeof(int);
    if (smem > 48 * 1024) return SG_EINVAL;
    k_measure_chiral<<<dim3(ctx->nchunk, ctx->S, nbatch), threads, smem, ctx->stream>>>(p);
    SG_LAUNCHED(ctx);
    k_reduce_chiral<<<(nQ * 21 + 127) / 128, 128, 0, ctx->stream>>>(ctx->Mpart, ctx->result, ctx->S, PT, ctx->nchunk, ctx->N);
    SG_LAUNCHED(ctx);
    return SG_OK;
}

int sg_measure_chiral(sg_ctx* ctx, double* qc0, double* qck)
{
    if (!ctx || ctx->Tt != ctx->T) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    const int PT = ctx->P * ctx->T;
    const int nQ = ctx->S * PT;
    if (PT == 0) return SG_OK;
    if (int rc = launch_measure_chiral(ctx)) return rc;
    {
        int rc;
        if (const double* h = fetch_result(ctx, (size_t)nQ * 21, &rc)) {
            if (qc0) std::memcpy(qc0, h, (size_t)nQ * 3 * sizeof(double));
            if (qck) std::memcpy(qck, h + (size_t)nQ * 3, (size_t)nQ * 18 * sizeof(double));
            return SG_OK;
        }
        if (rc != SG_OK) return rc;
    }
    if (qc0) SG_CUDA(ctx, cudaMemcpyAsync(qc0, ctx->result, (size_t)nQ * 3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (qck) SG_CUDA(ctx, cudaMemcpyAsync(qck, ctx->result + (size_t)nQ * 3, (size_t)nQ * 18 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_export_replica(sg_ctx* ctx, int r, void* dev_out)
{
    if (!ctx || !dev_out || r < 0 || r >= ctx->R) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    const size_t n = (size_t)ctx->N * ctx->Tt;
    k_export_by_temp<<<dim3((unsigned)((n + 255) / 256), ctx->S), 256, 0, ctx->stream>>>(ctx->spins, ctx->slot_of_temp, (float*)dev_out, ctx->L,
                                                                                      ctx->N, ctx->NG, ctx->R, ctx->Tt, ctx->T, ctx->slot0, r);
    SG_LAUNCHED(ctx);
    return SG_OK;
}

int sg_measure_cross(sg_ctx* ctx, int r, const void* dev_remote, double* q0, double* qk)
{
    if (!ctx || !dev_remote || r < 0 || r >= ctx->R || ctx->Tt > XTHREADS) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    CrossParams p;
    p.spins = ctx->spins; p.slot_of_temp = ctx->slot_of_temp; p.remote = (const float*)dev_remote; p.phase = ctx->phase; p.Xpart = ctx->Xpart;
    p.L = ctx->L; p.N = ctx->N; p.NG = ctx->NG; p.R = ctx->R; p.T = ctx->Tt; p.r = r; p.Tl = ctx->T; p.slot0 = ctx->slot0;
    const int rows = XTHREADS / ctx->Tt;
    k_overlap_cross<<<dim3(XCHUNKS, ctx->S), XTHREADS, 0, ctx->stream>>>(p);
    SG_LAUNCHED(ctx);
    const int total = ctx->S * ctx->Tt * 7;
    k_reduce_cross<<<(total + 127) / 128, 128, 0, ctx->stream>>>(ctx->Xpart, ctx->result, ctx->S, ctx->Tt, XCHUNKS * rows, ctx->N);
    SG_LAUNCHED(ctx);
    const size_t nQ = (size_t)ctx->S * ctx->Tt;
    if (q0) SG_CUDA(ctx, cudaMemcpyAsync(q0, ctx->result, nQ * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (qk) SG_CUDA(ctx, cudaMemcpyAsync(qk, ctx->result + nQ, nQ * 6 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_export_chirality(sg_ctx* ctx, int r, void* dev_out)
{
    if (!ctx || !dev_out || r < 0 || r >= ctx->R) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    const size_t n = (size_t)ctx->N * ctx->Tt;
    k_export_zeta_by_temp<<<dim3((unsigned)((n + 255) / 256), ctx->S), 256, 0, ctx->stream>>>(ctx->spins, ctx->slot_of_temp, (float*)dev_out,
                                                                                           ctx->L, ctx->N, ctx->NG, ctx->R, ctx->Tt, ctx->T, ctx->slot0, r);
    SG_LAUNCHED(ctx);
    return SG_OK;
}

int sg_chiral_cross(sg_ctx* ctx, const void* dev_a, const void* dev_b, double* qc0, double* qck)
{
    if (!ctx || !dev_a || !dev_b || ctx->Tt > XTHREADS) return SG_EINVAL;
    const int Tt = ctx->Tt;                  // the buffers are ordered by the temperatures of the whole chain (= T unless sharded by slot)
    const int rows = XTHREADS / Tt;
    k_chiral_cross<<<dim3(XCHUNKS, ctx->S), XTHREADS, 0, ctx->stream>>>((const float*)dev_a, (const float*)dev_b, ctx->phase, ctx->Xpart, ctx->L,
                                                                       ctx->N, Tt);
    SG_LAUNCHED(ctx);
    const int total = ctx->S * Tt * 21;
    k_reduce_chiral_cross<<<(total + 127) / 128, 128, 0, ctx->stream>>>(ctx->Xpart, ctx->result, ctx->S, Tt, XCHUNKS * rows, ctx->N);
    SG_LAUNCHED(ctx);
    const size_t nQ = (size_t)ctx->S * Tt;
    if (qc0) SG_CUDA(ctx, cudaMemcpyAsync(qc0, ctx->result, nQ * 3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (qck) SG_CUDA(ctx, cudaMemcpyAsync(qck, ctx->result + nQ * 3, nQ * 18 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_schwinger_dyson(sg_ctx* ctx, double* sd)
{
    if (!ctx || !sd) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    SdParams p;
    p.spins = ctx->spins; p.Jg = ctx->Jg; p.SDpart = ctx->SDpart;
    p.L = ctx->L; p.N = ctx->N; p.Nh = ctx->Nh; p.NG = ctx->NG; p.ntiles = ctx->ntiles; p.tile_sites = ctx->tile_sites;
    k_sd<<<dim3(ctx->NG * ctx->ntiles, ctx->S, 2), SWEEP_THREADS, 0, ctx->stream>>>(p);
    SG_LAUNCHED(ctx);
    const int total = ctx->S * ctx->R * ctx->Tt * 2;      // by the temperatures of the whole chain (zeros for those held by other shards)
    k_reduce_sd<<<(total + 127) / 128, 128, 0, ctx->stream>>>(ctx->SDpart, ctx->slot_of_temp, ctx->result, ctx->S, ctx->R, ctx->Tt, ctx->T,
                                                              ctx->slot0, ctx->NG, ctx->ntiles, ctx->N);
    SG_LAUNCHED(ctx);
    {
        int rc;
        if (const double* h = fetch_result(ctx, (size_t)total, &rc)) { std::memcpy(sd, h, (size_t)total * sizeof(double)); return SG_OK; }
        if (rc != SG_OK) return rc;
    }
    SG_CUDA(ctx, cudaMemcpyAsync(sd, ctx->result, (size_t)total * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

double sg_correlation_length(int L, double chi0, double chik)
{
    return std::sqrt(chi0 / chik - 1.0) / (2.0 * std::sin(3.14159265358979323846 / (double)L));
}

int sg_get_couplings(sg_ctx* ctx, int sample, float* out)
{
    if (!ctx || !out || sample < 0 || sample >= ctx->S) return SG_EINVAL;
    if (!ctx->inited[sample]) return SG_ESTATE;
    const size_t mfloats = (size_t)3 * ctx->N * 9;
    SG_CUDA(ctx, cudaMemcpyAsync(out, ctx->Mraw + (size_t)sample * mfloats, mfloats * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_get_perm(sg_ctx* ctx, int sample, int32_t* temp_of_slot, int32_t* slot_of_temp)
{
    if (!ctx || sample < 0 || sample >= ctx->S) return SG_EINVAL;
    const size_t n = (size_t)ctx->R * ctx->Tt, off = (size_t)sample * n;
    if (temp_of_slot) SG_CUDA(ctx, cudaMemcpyAsync(temp_of_slot, ctx->temp_of_slot + off, n * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    if (slot_of_temp) SG_CUDA(ctx, cudaMemcpyAsync(slot_of_temp, ctx->slot_of_temp + off, n * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_set_perm(sg_ctx* ctx, int sample, const int32_t* temp_of_slot)
{
    if (!ctx || !temp_of_slot || sample < 0 || sample >= ctx->S) return SG_EINVAL;
    const int R = ctx->R, T = ctx->Tt;
    std::vector<int> tos(temp_of_slot, temp_of_slot + (size_t)R * T), sot((size_t)R * T, -1);
    for (int r = 0; r < R; ++r)
        for (int s = 0; s < T; ++s) {
            const int t = tos[(size_t)r * T + s];
            if (t < 0 || t >= T || sot[(size_t)r * T + t] != -1) return SG_EINVAL;
            sot[(size_t)r * T + t] = s;
        }
    const size_t off = (size_t)sample * R * T;
    SG_CUDA(ctx, cudaMemcpyAsync(ctx->temp_of_slot + off, tos.data(), tos.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    SG_CUDA(ctx, cudaMemcpyAsync(ctx->slot_of_temp + off, sot.data(), sot.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return fill_beta_slot(ctx);
}

int sg_get_energies(sg_ctx* ctx, double* E)
{
    if (!ctx || !E) return SG_EINVAL;
    if (int rc = all_inited(ctx)) return rc;
    if (int rc = ensure_energies(ctx)) return rc;
    SG_CUDA(ctx, cudaMemcpy2DAsync(E, (size_t)ctx->C * sizeof(double), ctx->E, (size_t)ctx->Cp * sizeof(double),
                                   (size_t)ctx->C * sizeof(double), ctx->S, cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_set_energies(sg_ctx* ctx, const double* E)
{
    if (!ctx || !E) return SG_EINVAL;
    SG_CUDA(ctx, cudaMemcpy2DAsync(ctx->E, (size_t)ctx->Cp * sizeof(double), E, (size_t)ctx->C * sizeof(double),
                                   (size_t)ctx->C * sizeof(double), ctx->S, cudaMemcpyHostToDevice, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->energies_fresh = true;
    return SG_OK;
}

int sg_get_counters(sg_ctx* ctx, uint64_t* hb_counter, uint64_t* pt_counter)
{
    if (!ctx) return SG_EINVAL;
    if (hb_counter) *hb_counter = ctx->hb_counter;
    if (pt_counter) *pt_counter = ctx->pt_counter;
    return SG_OK;
}

int sg_set_counters(sg_ctx* ctx, uint64_t hb_counter, uint64_t pt_counter)
{
    if (!ctx) return SG_EINVAL;
    ctx->hb_counter = hb_counter;
    ctx->pt_counter = pt_counter;
    return SG_OK;
}

int sg_pt_stats(sg_ctx* ctx, uint64_t* attempts, uint64_t* accepts)
{
    if (!ctx) return SG_EINVAL;
    if (ctx->Tt < 2) return SG_OK;
    const size_t n = (size_t)ctx->S * ctx->R * (ctx->Tt - 1) * sizeof(unsigned long long);
    if (attempts) SG_CUDA(ctx, cudaMemcpyAsync(attempts, ctx->attempts, n, cudaMemcpyDeviceToHost, ctx->stream));
    if (accepts) SG_CUDA(ctx, cudaMemcpyAsync(accepts, ctx->accepts, n, cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_pt_walk(sg_ctx* ctx, uint64_t* round_trips, int32_t* label)
{
    if (!ctx) return SG_EINVAL;
    if (round_trips) SG_CUDA(ctx, cudaMemcpyAsync(round_trips, ctx->round_trips, (size_t)ctx->S * ctx->R * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
    if (label) SG_CUDA(ctx, cudaMemcpyAsync(label, ctx->walk_label, (size_t)ctx->S * ctx->R * ctx->Tt * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_pt_visits(sg_ctx* ctx, uint64_t* visits)
{
    if (!ctx || !visits || !ctx->visits) return SG_EINVAL;
    SG_CUDA(ctx, cudaMemcpyAsync(visits, ctx->visits, (size_t)ctx->S * ctx->R * ctx->Tt * ctx->Tt * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

// Integrated autocorrelation time of a recorded walk in temperature: tau = 1/2 + sum_{k=1..W} rho(k), with the
// self-consistent window W >= c tau(W) (Madras-Sokal; Ref. 31 of the paper is a textbook treatment of the same estimator)
double sg_walk_tau_int(const int32_t* series, int64_t n, double window_c)
{
    if (!series || n < 4) return std::nan("");
    const double c = window_c > 0.0 ? window_c : 6.0;
    double m = 0.0;
    for (int64_t i = 0; i < n; ++i) m += (double)series[i];
    m /= (double)n;
    double c0 = 0.0;
    for (int64_t i = 0; i < n; ++i) { const double d = (double)series[i] - m; c0 += d * d; }
    c0 /= (double)n;
    if (!(c0 > 0.0)) return std::nan("");
    double tau = 0.5;
    for (int64_t k = 1; k <= n / 2; ++k) {
        double ck = 0.0;
        for (int64_t i = 0; i + k < n; ++i) ck += ((double)series[i] - m) * ((double)series[i + k] - m);
        ck /= (double)(n - k);
        tau += ck / c0;
        if ((double)k >= c * tau) break;
    }
    return tau;
}

int sg_tune(sg_ctx* ctx, int knob, int value)
{
    if (!ctx) return SG_EINVAL;
    switch (knob) {
    case SG_TUNE_SWEEP_IMPL:
        if (value != SG_SWEEP_AUTO && value != SG_SWEEP_TILED && value != SG_SWEEP_ZMARCH && value != SG_SWEEP_RESIDENT && value != SG_SWEEP_FUSED && value != SG_SWEEP_CLUSTER) return SG_EINVAL;
        if ((value == SG_SWEEP_ZMARCH || value == SG_SWEEP_FUSED) && ctx->L % 8 != 0) return SG_EINVAL;
        if (value == SG_SWEEP_FUSED && !ctx->spins2) return SG_EINVAL;
        if (value == SG_SWEEP_CLUSTER && ctx->L != CresGeom::L) return SG_EINVAL;
        if (value == SG_SWEEP_RESIDENT && !ctx->res_ok) return SG_EINVAL;
        ctx->sweep_impl = value;
        ctx->cres_unavailable = false;      // a fresh choice re-arms the automatic use of the cluster kernel
        return SG_OK;
    case SG_TUNE_RES_COPIES:
        if (value != 0 && value != 4 && value != 8 && value != 16 && value != 32) return SG_EINVAL;
        if (value > 0 && res_smem_bytes(ctx->N, value) > RES_SMEM_MAX) return SG_EINVAL;
        ctx->res_cpc_req = value;
        res_plan(ctx);
        return SG_OK;
    case SG_TUNE_PACKED:
        if (value != 0 && value != 1) return SG_EINVAL;
        ctx->packed_on = value;
        return SG_OK;
    case SG_TUNE_MEASURE_IMPL:
        if (value != SG_MEASURE_AUTO && value != SG_MEASURE_STAGED) return SG_EINVAL;
        ctx->measure_impl = value;
        return SG_OK;
    case SG_TUNE_CLUSTER_CTAS:
        if (value != 4 && value != 8) return SG_EINVAL;
        ctx->cres_cs = value;
        ctx->cres_unavailable = false;      // the other cluster shape may launch where this one did not
        return SG_OK;
    case SG_TUNE_GRAPH:
        if (value != 0 && value != 1) return SG_EINVAL;
        ctx->graph_mode = value;
        return SG_OK;
    case SG_TUNE_ZCHUNK:
        if (value < 0) return SG_EINVAL;
        if (value > 0 && (ctx->L % 8 != 0 || value < 4 || (value & 1) || ctx->L % value != 0)) return SG_EINVAL;
        ctx->zm_zc_req = value;
        zm_plan(ctx);
        fz_plan(ctx);
        return SG_OK;
    default:
        return SG_EINVAL;
    }
}

int sg_sync(sg_ctx* ctx)
{
    if (!ctx) return SG_EINVAL;
    SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SG_OK;
}

int sg_sweep_impl_used(const sg_ctx* ctx, int kind, int* cluster_fallback_cuda)
{
    if (!ctx || (kind != SG_KIND_OR && kind != SG_KIND_HB)) return SG_EINVAL;
    if (cluster_fallback_cuda) *cluster_fallback_cuda = ctx->cres_unavailable ? ctx->cres_fail_cuda : 0;
    return ctx->served_impl[kind == SG_KIND_HB ? 1 : 0];
}

uint64_t sg_kernel_launches(const sg_ctx* ctx) { return ctx ? ctx->launches : 0; }
uint64_t sg_graph_replays(const sg_ctx* ctx) { return ctx ? ctx->graph_replays : 0; }
int sg_last_cuda_error(const sg_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }

}  // extern "C"

// ---- sg_chiral_cross_static: the allocation-free variant of sg_chiral_cross (include/sg_b200.h) ----
// The partial sums of k_chiral_cross and the Fourier phase table, which a context keeps in the caller's workspace, live here in
// an array that is part of the library image.  In HOST code the name g_static_scratch is only a handle for the runtime, not a
// device address (a kernel handed `g_static_scratch` from the host would fault, or scribble over host memory where the GPU can
// reach it): the device address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[SG_STATIC_SCRATCH_BYTES];

namespace {
constexpr size_t STATIC_PHASE_BYTES = 4096;      // double [SG_STATIC_MAX_L][2] at the head of the array, partial sums behind it
static_assert((size_t)SG_STATIC_MAX_L * 2 * sizeof(double) <= STATIC_PHASE_BYTES, "phase table");
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;                                   // guards the table below (set-up only; the calls do not hold it)
unsigned char* g_static_addr[STATIC_MAX_DEVICES] = {};       // device address of g_static_scratch on device d; nullptr = not set up

// Set-up of the current device on the first call made on it.  No allocation: the array already exists on every device that
// has the module loaded; cudaGetSymbolAddress only reports where (and loads the module if this is the library's first CUDA call).
int static_scratch_of_current_device(unsigned char** out, cudaError_t* err)
{
    int dev = -1;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return SG_ECUDA;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) { *err = cudaErrorInvalidDevice; return SG_ECUDA; }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_static_scratch);
        if (*err != cudaSuccess || !p) { if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol; return SG_ECUDA; }
        g_static_addr[dev] = (unsigned char*)p;
    }
    *out = g_static_addr[dev];
    return SG_OK;
}
}  // namespace

// phase[x] = (cos, sin)(2 pi x / L), the table sg_create uploads for a context, here written by the device for itself
__global__ void k_static_phase(double* __restrict__ phase, int L)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= L) return;
    double sn, cs;
    sincospi(2.0 * (double)x / (double)L, &sn, &cs);
    phase[2 * x] = cs;
    phase[2 * x + 1] = sn;
}

extern "C" {

int sg_chiral_cross_static(int L, int n_samples, int n_temps, const void* dev_a, const void* dev_b, void* dev_out,
                           void* cuda_stream, int* cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    if (!dev_a || !dev_b || !dev_out || ((uintptr_t)dev_out & 7)) return SG_EINVAL;
    if (L < 2 || (L & 1) || L > SG_STATIC_MAX_L || n_samples < 1 || n_temps < 1 || n_temps > XTHREADS) return SG_EINVAL;
    const int S = n_samples, T = n_temps, N = L * L * L;
    const int rows = XTHREADS / T;
    // the partial sums k_chiral_cross writes and k_reduce_chiral_cross reads: [S][XCHUNKS * rows][T][21] doubles
    const unsigned long long need = (unsigned long long)S * XCHUNKS * rows * T * 21ull * sizeof(double);
    if (need > (unsigned long long)SG_STATIC_SCRATCH_BYTES - STATIC_PHASE_BYTES) return SG_ELIMIT;
    if ((long long)S * T * 21 > 0x7fffffffLL) return SG_ELIMIT;     // unreachable under the byte limit; keeps the int arithmetic below honest
    unsigned char* base = nullptr;
    cudaError_t e = cudaSuccess;
    if (int rc = static_scratch_of_current_device(&base, &e)) { if (cuda_error) *cuda_error = (int)e; return rc; }
    double* phase = (double*)base;
    double* xpart = (double*)(base + STATIC_PHASE_BYTES);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // Every element read below is written first by this call: the phase table for this L, then all S * XCHUNKS * rows * T * 21
    // partial sums (chunks past the end of the lattice store zeros), so the leftovers of earlier calls never matter.
    k_static_phase<<<(L + 127) / 128, 128, 0, stream>>>(phase, L);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        k_chiral_cross<<<dim3(XCHUNKS, S), XTHREADS, 0, stream>>>((const float*)dev_a, (const float*)dev_b, phase, xpart, L, N, T);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        const int total = S * T * 21;
        k_reduce_chiral_cross<<<(total + 127) / 128, 128, 0, stream>>>(xpart, (double*)dev_out, S, T, XCHUNKS * rows, N);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { if (cuda_error) *cuda_error = (int)e; return SG_ECUDA; }
    return SG_OK;
}

const char* sg_strerror(int code)
{
    switch (code) {
    case SG_OK: return "ok";
    case SG_EINVAL: return "invalid argument";
    case SG_ESTATE: return "sample not initialised";
    case SG_ECUDA: return "CUDA call failed (see sg_last_cuda_error)";
    case SG_ELIMIT: return "shape exceeds the fixed scratch array of the allocation-free entry point (SG_STATIC_SCRATCH_BYTES): split the call by sample";
    default: return "unknown error";
    }
}

void sg_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1], out);
}

}  // extern "C"
