// sg_kernels.cuh -- the CUDA kernels of libsg_b200 (sm_100a).  DESIGN.md section 10 states, for each
// kernel, the roofline that bounds it and its algorithmic bytes per spin update.
#pragma once
#include "sg_device.cuh"
#include "sg_sweep_zm.cuh"

namespace sg {

// ------------------------------------------------------------------------------------------------
// Sweep kernel (S1, S2, S3): one checkerboard half-sweep of every copy of every sample.
//
// Work decomposition.  A CTA owns TILE consecutive same-colour sites (h-order: along x1, then x2, x3)
// of ONE (sample, copy group); its 256 threads are 32 site slots x 8 lanes, a lane holding the float4 of
// 4 consecutive copies.  Every spin access of a warp instruction is four full, aligned 128-byte lines
// (one per site), for every L, with no colour-split arrays; stores are full lines.  The six matrices
// of a site are shared by the 8 lanes (one broadcast LDG.128 per 4 floats) and used for 4 copies each.
// ------------------------------------------------------------------------------------------------
constexpr int SWEEP_THREADS = 256;
constexpr int SLOTS = SWEEP_THREADS / 8;   // site slots per pass

struct SweepParams {
    float* spins;            // [S][NG][2][Nh][3][G]
    const float* Jg;         // [S][2][Nh][JG]
    const float* beta_slot;  // [S][Cp]
    double* Epart;           // [S][NG][ntiles][G]
    int L, N, Nh, NG, ntiles, tile_sites;
    int colour;
    int C;                   // copies per sample (R*T); Cp = NG*G
    int Cg;                  // copies per sample of the whole job (all replicas, sg_shape.n_replicas_total): stride of the global copy id
    int Tl, Tpad;            // slots per replica held here, n_temps_total - Tl (copy_gid)
    uint32_t key0, key1, hb_counter;
    uint32_t g_first;        // global copy id of (local sample 0, copy 0) = first_sample*C
};

template <int KIND, bool WITH_E, int LOG2L>
__global__ void __launch_bounds__(SWEEP_THREADS) k_sweep(const SweepParams p)
{
    const int tid = threadIdx.x;
    const int q = tid & 7;        // copy quad: copies 4q..4q+3 of the group
    const int slot = tid >> 3;    // site slot
    // the copy group is the fastest block index: the CTAs that share a tile's couplings run together
    const int grp = blockIdx.x % p.NG, tile = blockIdx.x / p.NG, sample = blockIdx.y;
    const int L = p.L;

    float* const sp = p.spins + ((size_t)(sample * p.NG + grp) * p.N) * SITE_FLOATS + q * 4;
    const float* const Jc = p.Jg + ((size_t)(sample * 2 + p.colour) * p.Nh) * JG;

    float4 beta4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (KIND == KIND_HB) beta4 = ldg4(p.beta_slot + (size_t)sample * p.NG * G + grp * G + q * 4);

    float eacc[4] = { 0.f, 0.f, 0.f, 0.f };

    const int h_end = min(p.Nh, (tile + 1) * p.tile_sites);
    for (int h = tile * p.tile_sites + slot; h < h_end; h += SLOTS) {
        int x, y, z;
        site_of<LOG2L>(h, p.colour, L, x, y, z);
        const int xp = (x + 1 == L) ? 0 : x + 1, xm = (x == 0) ? L - 1 : x - 1;
        const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
        const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
        const int row = L * (y + L * z);
        const int i = x + row;
        int nb[6];
        nb[0] = xp + row;            nb[1] = xm + row;
        nb[2] = x + L * (yp + L * z); nb[3] = x + L * (ym + L * z);
        nb[4] = x + L * (y + L * zp); nb[5] = x + L * (y + L * zm);

        // couplings of this site: 14 broadcast 16-byte loads (54 floats + 2 pad)
        float J[JG];
        {
            const float* jp = Jc + (size_t)h * JG;
#pragma unroll
            for (int v = 0; v < JG / 4; ++v) {
                const float4 t4 = ldg4(jp + 4 * v);
                J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
            }
        }
        float* const own = sp + ((size_t)p.colour * p.Nh + h) * SITE_FLOATS;
        float s[3][4];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float4 t4 = ld4(own + a * G);
            s[a][0] = t4.x; s[a][1] = t4.y; s[a][2] = t4.z; s[a][3] = t4.w;
        }
        float hf[3][4];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int j = 0; j < 4; ++j) hf[a][j] = 0.f;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float* np_ = sp + ((size_t)(1 - p.colour) * p.Nh + (nb[k] >> 1)) * SITE_FLOATS;
            float n[3][4];
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const float4 t4 = ld4(np_ + b * G);
                n[b][0] = t4.x; n[b][1] = t4.y; n[b][2] = t4.z; n[b][3] = t4.w;
            }
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    fma4(J[9 * k + 3 * a + b], n[b], hf[a]);
        }

        if (KIND == KIND_OR) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                or_update(hf[0][j], hf[1][j], hf[2][j], s[0][j], s[1][j], s[2][j]);
                if (WITH_E) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));   // of the stored spin
            }
        } else if (KIND == KIND_HB) {
            const float bt[4] = { beta4.x, beta4.y, beta4.z, beta4.w };
            const uint32_t gbase = p.g_first + (uint32_t)sample * (uint32_t)p.Cg;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                uint32_t w[4];
                philox4x32_10((uint32_t)i, copy_gid(gbase, grp * G + q * 4 + j, p.Tl, p.Tpad), p.hb_counter, STREAM_HB, p.key0, p.key1, w);
                hb_update(hf[0][j], hf[1][j], hf[2][j], bt[j], uniform23(w[0]), uniform23(w[1]),
                          s[0][j], s[1][j], s[2][j]);
                if (WITH_E) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
            }
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
        }
        if (KIND != KIND_ENERGY) {
#pragma unroll
            for (int a = 0; a < 3; ++a) st4(own + a * G, make_float4(s[a][0], s[a][1], s[a][2], s[a][3]));
        }
    }

    if (WITH_E || KIND == KIND_ENERGY) {
        // per-copy sum over the CTA's sites: fixed order, fp64 across threads (no float atomics)
        __shared__ double red[SLOTS][G + 1];
#pragma unroll
        for (int j = 0; j < 4; ++j) red[slot][q * 4 + j] = (double)eacc[j];
        __syncthreads();
        if (tid < G) {
            double acc = 0.0;
            for (int r = 0; r < SLOTS; ++r) acc += red[r][tid];
            p.Epart[((size_t)(sample * p.NG + grp) * p.ntiles + tile) * G + tid] = acc;
        }
    }
}

// E[sample][copy] = - sum over tiles of the per-CTA partial sums of s.h over ONE colour
// (every link joins the two colours, so one colour's sum of s_x.h_x counts each link once).
__global__ void k_reduce_energy(const double* __restrict__ Epart, double* __restrict__ E, int ntiles)
{
    // grid = S*NG blocks of 256 threads = 8 tile ranges x 32 copies
    __shared__ double part[8][G];
    const int col = threadIdx.x & 31, rng = threadIdx.x >> 5;
    const double* src = Epart + (size_t)blockIdx.x * ntiles * G;
    const int per = (ntiles + 7) / 8;
    double acc = 0.0;
    for (int t = rng * per; t < min(ntiles, (rng + 1) * per); ++t) acc += src[(size_t)t * G + col];
    part[rng][col] = acc;
    __syncthreads();
    if (rng == 0) {
        double tot = 0.0;
        for (int r = 0; r < 8; ++r) tot += part[r][col];
        E[(size_t)blockIdx.x * G + col] = -tot;
    }
}

// ------------------------------------------------------------------------------------------------
// S0: initial spins uniform on S^2, Philox stream 3, counter (i, g, 0, 3)
// ------------------------------------------------------------------------------------------------
__global__ void k_init_spins(float* __restrict__ spins_sample /* [NG][2][Nh][3][G] of one sample */, int L, int N, int NG,
                             int C, uint32_t g_sample, int Tl, int Tpad, uint32_t key0, uint32_t key1)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;   // over NG*N*8 (site, quad)
    if (t >= (size_t)NG * N * 8) return;
    const int q = (int)(t & 7);
    const size_t si = t >> 3;
    const int i = (int)(si % N), grp = (int)(si / N);
    float out[3][4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = grp * G + q * 4 + j;
        uint32_t w[4];
        philox4x32_10((uint32_t)i, copy_gid(g_sample, c, Tl, Tpad), 0u, STREAM_SPINS, key0, key1, w);
        const float zc = 1.0f - 2.0f * uniform23(w[0]);
        const float rho = sqrtf(fmaxf(1.0f - zc * zc, 0.0f));
        float sn, cs;
        sincospif(2.0f * uniform23(w[1]), &sn, &cs);
        const bool live = c < C;     // padding copies of the last group stay zero
        out[0][j] = live ? rho * cs : 0.f;
        out[1][j] = live ? rho * sn : 0.f;
        out[2][j] = live ? zc : 0.f;
    }
    float* dst = spins_sample + ((size_t)grp * N + site_slot(i, L, N >> 1)) * SITE_FLOATS + q * 4;
#pragma unroll
    for (int a = 0; a < 3; ++a) st4(dst + a * G, make_float4(out[a][0], out[a][1], out[a][2], out[a][3]));
}

// host layout [c][3][N] (32 copies of one group, staged on the device) <-> device layout [2][Nh][3][G]
// block (32, 8); tile = 32 sites x 32 copies per component
__global__ void k_spins_from_staging(const float* __restrict__ stg, float* __restrict__ dev, int N, int L)
{
    __shared__ float tile[32][33];
    const int comp = blockIdx.y;
    const int i0 = blockIdx.x * 32;
    for (int c = threadIdx.y; c < 32; c += 8) {
        const int i = i0 + threadIdx.x;
        tile[c][threadIdx.x] = (i < N) ? stg[((size_t)c * 3 + comp) * N + i] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int i = i0 + r;
        if (i < N) dev[site_slot(i, L, N >> 1) * SITE_FLOATS + comp * G + threadIdx.x] = tile[threadIdx.x][r];
    }
}

// the same for the sites [i_first, i_first + n) only, staged as [c][3][n] (sg_set_spins uploads a group in site chunks so that
// the host-to-device copy of one chunk overlaps the transposition of the previous one)
__global__ void k_spins_from_staging_chunk(const float* __restrict__ stg, float* __restrict__ dev, int N, int L, int i_first, int n)
{
    __shared__ float tile[32][33];
    const int comp = blockIdx.y;
    const int j0 = blockIdx.x * 32;
    for (int c = threadIdx.y; c < 32; c += 8) {
        const int j = j0 + threadIdx.x;
        tile[c][threadIdx.x] = (j < n) ? stg[((size_t)c * 3 + comp) * n + j] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int j = j0 + r;
        if (j < n) dev[site_slot(i_first + j, L, N >> 1) * SITE_FLOATS + comp * G + threadIdx.x] = tile[threadIdx.x][r];
    }
}

__global__ void k_spins_to_staging(const float* __restrict__ dev, float* __restrict__ stg, int N, int L)
{
    __shared__ float tile[32][33];
    const int comp = blockIdx.y;
    const int i0 = blockIdx.x * 32;
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int i = i0 + r;
        tile[r][threadIdx.x] = (i < N) ? dev[site_slot(i, L, N >> 1) * SITE_FLOATS + comp * G + threadIdx.x] : 0.f;
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += 8) {
        const int i = i0 + threadIdx.x;
        if (i < N) stg[((size_t)c * 3 + comp) * N + i] = tile[threadIdx.x][c];
    }
}

// raw couplings M[3][N][9] of one sample -> gathered per-site blocks Jg[2][Nh][JG]
// (and, when Jt_sample != nullptr, the tile-major copy Jt[2][L/8][L/8][L][8][4][JG] of the z-marching sweep)
__global__ void k_gather_couplings(const float* __restrict__ M, float* __restrict__ Jg_sample, float* __restrict__ Jt_sample, int L)
{
    const int N = L * L * L, Nh = N >> 1;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int x = i % L, y = (i / L) % L, z = i / (L * L);
    const int colour = (x + y + z) & 1;
    float* dst = Jg_sample + ((size_t)colour * Nh + (i >> 1)) * JG;
    const int bw[3] = { ((x == 0) ? L - 1 : x - 1) + L * (y + L * z), x + L * (((y == 0) ? L - 1 : y - 1) + L * z),
                        x + L * (y + L * ((z == 0) ? L - 1 : z - 1)) };
    for (int mu = 0; mu < 3; ++mu) {
        const float* mf = M + ((size_t)mu * N + i) * 9;        // link (x, mu): acts as M
        const float* mb = M + ((size_t)mu * N + bw[mu]) * 9;   // link (x-e_mu, mu): acts as M^T
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                dst[(2 * mu) * 9 + 3 * a + b] = mf[3 * a + b];
                dst[(2 * mu + 1) * 9 + 3 * a + b] = mb[3 * b + a];
            }
    }
    dst[54] = 0.f; dst[55] = 0.f;
    if (Jt_sample) {
        const int nt = L >> 3;
        const size_t t = ((((size_t)colour * nt + (y >> 3)) * nt + (x >> 3)) * L + z) * 32 + (y & 7) * 4 + ((x & 7) >> 1);
        float* d2 = Jt_sample + t * JG;
        for (int e = 0; e < JG; ++e) d2[e] = dst[e];
    }
}

// ------------------------------------------------------------------------------------------------
// S4: parallel tempering.  The pairs of a chain (sample, replica) are taken in order on the updated
// assignment, so a chain is sequential; everything around that dependence is not.  k_pt_swap gives a warp to a chain:
// the lanes stage the chain's assignment, energies, beta differences and uniforms (one Philox block per pair) in shared
// memory, lane 0 walks the T-1 pairs there (fp64 exp, no global round trips), the lanes write the new assignment, the
// betas of the slots, the statistics and the random-walk labels back.  k_pt_swap_serial (one thread per chain, straight
// from global memory) is the same arithmetic for chains too long for shared memory.
// Temperature-slot sharding (sg_shape.first_slot / n_temps_total): every context of the chain runs the
// SAME kernel on the all-gathered energies (E + w*E_wstride: the block of the context with slot window w) and keeps the
// whole assignment; only beta_slot is restricted to the slots [slot0, slot0 + Tl) it holds.
// ------------------------------------------------------------------------------------------------
struct PtParams {
    const double* betas;   // [T]
    const double* E;       // local: [S][Cp], copy r*T + slot; gathered: [W][S][R][Tl]
    int* slot_of_temp;     // [S][R][T]
    int* temp_of_slot;     // [S][R][T]
    float* beta_slot;      // [S][Cp], local copy r*Tl + (slot - slot0)
    unsigned long long* attempts;  // [S][R][T-1]
    unsigned long long* accepts;
    int* walk_label;                 // [S][R][T]: 0 = no end touched yet, 1 = last touched index 0, 2 = last touched index T-1
    unsigned long long* round_trips; // [S][R]: completed walks 0 -> T-1 -> 0, summed over the chain's configurations
    unsigned long long* visits;      // [S][R][T][T]: PT sweeps configuration `slot` has spent at temperature index t (after the sweep)
    int S, R, T, Cp, Rt;   // T: length of the chain (n_temps_total); Rt: replicas of the whole job (sg_shape.n_replicas_total)
    int Tl, slot0;         // slots per replica held by this context and the first of them (Tl = T, slot0 = 0 unless slot-sharded)
    long long E_sstride, E_wstride;   // E of (sample, r, slot) = E[(slot / Tl) * E_wstride + sample * E_sstride + r * Tl + slot % Tl]
    uint32_t key0, key1, pt_counter, chain_first;   // chain id of (local sample 0, r = 0) = first_sample*Rt + first_replica
};

__device__ __forceinline__ double pt_energy(const PtParams& p, int sample, int r, int slot)
{
    return p.E[(long long)(slot / p.Tl) * p.E_wstride + (long long)sample * p.E_sstride + r * p.Tl + slot % p.Tl];
}

__device__ __forceinline__ double pt_uniform(const PtParams& p, int sample, int r, int t)
{
    uint32_t w[4];
    philox4x32_10((uint32_t)t, p.chain_first + (uint32_t)(sample * p.Rt + r), p.pt_counter, STREAM_PT, p.key0, p.key1, w);
    return ((double)(w[0] >> 9) + 0.5) * (1.0 / 8388608.0);
}

constexpr int PT_SMEM_PER_TEMP = 4 * sizeof(double) + 2 * sizeof(int) + sizeof(double);   // E, rr, dbeta, ln rr, sot, flags (+ slack)

__global__ void __launch_bounds__(32) k_pt_swap(const PtParams p)
{
    extern __shared__ __align__(16) unsigned char pt_sm[];
    const int chain = blockIdx.x, lane = threadIdx.x, T = p.T;
    const int sample = chain / p.R, r = chain % p.R;
    double* const Es = reinterpret_cast<double*>(pt_sm);          // [T] energy of configuration `slot`
    double* const rr = Es + T;                                    // [T] uniform of pair t
    double* const db = rr + T;                                    // [T] beta_t - beta_{t+1}
    double* const lr = db + T;                                    // [T] ln of the uniform of pair t
    int* const sot = reinterpret_cast<int*>(lr + T);              // [T]
    unsigned char* const acc = reinterpret_cast<unsigned char*>(sot + T);   // [T] pair t accepted
    int* const sot_g = p.slot_of_temp + (size_t)chain * T;
    int* const tos_g = p.temp_of_slot + (size_t)chain * T;
    for (int t = lane; t < T; t += 32) {
        Es[t] = pt_energy(p, sample, r, t);
        sot[t] = sot_g[t];
        if (t + 1 < T) { rr[t] = pt_uniform(p, sample, r, t); lr[t] = log(rr[t]); db[t] = p.betas[t] - p.betas[t + 1]; }
    }
    __syncwarp();
    if (lane == 0) {
        int i = sot[0];                    // the configuration now at temperature index t
        double Ei = Es[i];
        for (int t = 0; t + 1 < T; ++t) {
            const int j = sot[t + 1];
            const double Ej = Es[j];
            const double delta = db[t] * (Ei - Ej);
            // r < exp(delta) <=> ln r < delta.  The logarithms were taken by the lanes in parallel; the sequential walk only compares.
            // Both sides carry ~1e-16 of rounding, so outside a band of 1e-12 the comparison of the logarithms IS the decision of
            // the rule as specified (r < exp(delta) in fp64); inside it (one decision in ~1e12) the rule itself is evaluated.
            const double gap = lr[t] - delta;
            const bool accept = (delta >= 0.0) || ((fabs(gap) > 1e-12) ? (gap < 0.0) : (rr[t] < exp(delta)));
            acc[t] = accept ? 1 : 0;
            if (accept) { sot[t] = j; sot[t + 1] = i; }     // i moves on to index t + 1
            else { i = j; Ei = Ej; }
        }
    }
    __syncwarp();
    float* const bs = p.beta_slot + (size_t)sample * p.Cp + r * p.Tl;
    int* const lab = p.walk_label + (size_t)chain * T;
    unsigned long long trips = 0ull;
    for (int t = lane; t < T; t += 32) {
        const int slot = sot[t];
        sot_g[t] = slot;
        tos_g[slot] = t;
        if (slot >= p.slot0 && slot < p.slot0 + p.Tl) bs[slot - p.slot0] = (float)p.betas[t];
        if (t + 1 < T) {
            p.attempts[(size_t)chain * (T - 1) + t] += 1ull;
            if (acc[t]) p.accepts[(size_t)chain * (T - 1) + t] += 1ull;
        }
        // random walk in temperature of every configuration of the chain
        if (t == 0) {
            if (lab[slot] == 2) trips += 1ull;
            lab[slot] = 1;
        } else if (t == T - 1 && lab[slot] == 1) {
            lab[slot] = 2;
        }
        if (p.visits) p.visits[((size_t)chain * T + slot) * T + t] += 1ull;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) trips += __shfl_xor_sync(0xffffffffu, trips, o);
    if (lane == 0) p.round_trips[chain] += trips;
}

__global__ void k_pt_swap_serial(const PtParams p)
{
    const int chain = blockIdx.x * blockDim.x + threadIdx.x;
    if (chain >= p.S * p.R) return;
    const int sample = chain / p.R, r = chain % p.R;
    int* sot = p.slot_of_temp + (size_t)chain * p.T;
    int* tos = p.temp_of_slot + (size_t)chain * p.T;
    float* bs = p.beta_slot + (size_t)sample * p.Cp + r * p.Tl;
    for (int t = 0; t + 1 < p.T; ++t) {
        const int i = sot[t], j = sot[t + 1];
        const double delta = (p.betas[t] - p.betas[t + 1]) * (pt_energy(p, sample, r, i) - pt_energy(p, sample, r, j));
        const double rr = pt_uniform(p, sample, r, t);
        const bool accept = (delta >= 0.0) || (rr < exp(delta));
        p.attempts[(size_t)chain * (p.T - 1) + t] += 1ull;
        if (accept) {
            sot[t] = j; sot[t + 1] = i;
            tos[j] = t; tos[i] = t + 1;
            if (j >= p.slot0 && j < p.slot0 + p.Tl) bs[j - p.slot0] = (float)p.betas[t];
            if (i >= p.slot0 && i < p.slot0 + p.Tl) bs[i - p.slot0] = (float)p.betas[t + 1];
            p.accepts[(size_t)chain * (p.T - 1) + t] += 1ull;
        }
    }
    int* lab = p.walk_label + (size_t)chain * p.T;
    unsigned long long trips = 0ull;
    for (int slot = 0; slot < p.T; ++slot) {
        const int t = tos[slot];
        if (t == 0) {
            if (lab[slot] == 2) trips += 1ull;
            lab[slot] = 1;
        } else if (t == p.T - 1 && lab[slot] == 1) {
            lab[slot] = 2;
        }
        if (p.visits) p.visits[((size_t)chain * p.T + slot) * p.T + t] += 1ull;
    }
    p.round_trips[chain] += trips;
}

// e[sample][r][t] = E(configuration of replica r at temperature index t) / N from the all-gathered energies [W][S][R][Tl]
__global__ void k_energy_by_temp(const double* __restrict__ Eall, const int* __restrict__ slot_of_temp, double* __restrict__ out,
                                 int S, int R, int T, int Tl, int N)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= S * R * T) return;
    const int sample = u / (R * T), r = (u / T) % R;
    const int slot = slot_of_temp[u];
    out[u] = Eall[(size_t)(slot / Tl) * S * R * Tl + ((size_t)sample * R + r) * Tl + slot % Tl] * (1.0 / (double)N);   // as k_reduce_measure
}

// beta_slot[sample][r*Tl + s] = beta[temp_of_slot[sample][r][slot0 + s]], for all chains (after init / set_perm);
// T = length of the chain, Tl = slots per replica held by this context
__global__ void k_fill_beta_slot(const double* __restrict__ betas, const int* __restrict__ temp_of_slot,
                                 float* __restrict__ beta_slot, int S, int R, int T, int Tl, int slot0, int Cp)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= S * Cp) return;
    const int sample = t / Cp, c = t % Cp;
    float b = 0.f;
    if (c < R * Tl) b = (float)betas[temp_of_slot[((size_t)sample * R + c / Tl) * T + slot0 + c % Tl]];
    beta_slot[t] = b;
}

// ------------------------------------------------------------------------------------------------
// S5: overlap and k_min Fourier modes.  One work item = (replica pair, temperature);
// a CTA stages MS sites of all Cp copies in shared memory, every thread looks its two copies up
// through the temperature permutation.  Partial sums per site chunk, reduced in fixed order.
// ------------------------------------------------------------------------------------------------
struct MeasureParams {
    const float* spins;        // [S][NG][2][Nh][3][G]
    const int* slot_of_temp;   // [S][R][T]
    const double* phase;       // [L][2] cos, sin of 2 pi x / L
    double* Mpart;             // [S][nchunk][PT][7]
    int L, N, NG, Cp, R, T, P, nchunk, chunk_sites, MS;
};

__global__ void k_measure(const MeasureParams p)
{
    extern __shared__ float sm[];   // [MS][3][Cp] spins, then [MS][3][2] doubles: phases of the batch's sites
    double* const ph = reinterpret_cast<double*>(sm + (size_t)p.MS * 3 * p.Cp);
    const int chunk = blockIdx.x, sample = blockIdx.y;
    const int PT = p.P * p.T;
    const int item = blockIdx.z * blockDim.x + threadIdx.x;
    int ca = 0, cb = 0;
    const bool live = item < PT;
    if (live) {
        const int pr = item / p.T, t = item % p.T;
        int a = 0, rem = pr;                       // pair index -> (a, b), a < b, lexicographic
        while (rem >= p.R - 1 - a) { rem -= p.R - 1 - a; ++a; }
        const int b = a + 1 + rem;
        ca = a * p.T + p.slot_of_temp[((size_t)sample * p.R + a) * p.T + t];
        cb = b * p.T + p.slot_of_temp[((size_t)sample * p.R + b) * p.T + t];
    }
    double acc[7] = { 0, 0, 0, 0, 0, 0, 0 };
    const int i_begin = chunk * p.chunk_sites, i_end = min(p.N, i_begin + p.chunk_sites);
    const float* base = p.spins + (size_t)sample * p.NG * p.N * SITE_FLOATS;
    const int row = 3 * p.Cp;
    for (int i0 = i_begin; i0 < i_end; i0 += p.MS) {
        const int ms = min(p.MS, i_end - i0);
        __syncthreads();
        // a warp copies the three 128-byte lines of one (site, copy group) per pass
        for (int r = threadIdx.x >> 5; r < ms * p.NG; r += blockDim.x >> 5) {
            const int m = r / p.NG, grp = r - m * p.NG, lane = threadIdx.x & 31;
            const float* src = base + ((size_t)grp * p.N + site_slot(i0 + m, p.L, p.N >> 1)) * SITE_FLOATS + lane;
            float* dst = sm + m * row + grp * G + lane;
            dst[0] = src[0]; dst[p.Cp] = src[G]; dst[2 * p.Cp] = src[2 * G];
        }
        for (int u = threadIdx.x; u < ms * 3; u += blockDim.x) {   // e^{i 2 pi x_mu / L} of the batch's sites, once per batch
            const int m = u / 3, mu = u % 3, i = i0 + m;
            const int xm = (mu == 0) ? i % p.L : ((mu == 1) ? (i / p.L) % p.L : i / (p.L * p.L));
            ph[m * 6 + 2 * mu] = p.phase[2 * xm];
            ph[m * 6 + 2 * mu + 1] = p.phase[2 * xm + 1];
        }
        __syncthreads();
        if (live) {
            for (int m = 0; m < ms; ++m) {
                const float* s = sm + m * row;
                const float qf = fmaf(s[ca], s[cb], fmaf(s[p.Cp + ca], s[p.Cp + cb], s[2 * p.Cp + ca] * s[2 * p.Cp + cb]));
                const double qx = (double)qf;
                acc[0] += qx;
#pragma unroll
                for (int k = 0; k < 6; ++k) acc[1 + k] = fma(qx, ph[m * 6 + k], acc[1 + k]);
            }
        }
    }
    if (live) {
        double* dst = p.Mpart + (((size_t)sample * p.nchunk + chunk) * PT + item) * 7;
#pragma unroll
        for (int k = 0; k < 7; ++k) dst[k] = acc[k];
    }
}

// result = [ e[S][R][T] | q0[S][P][T] | qk[S][P][T][3][2] ]
__global__ void k_reduce_measure(const double* __restrict__ Mpart, const double* __restrict__ E,
                                 const int* __restrict__ slot_of_temp, double* __restrict__ result,
                                 int S, int R, int T, int P, int Cp, int nchunk, int N)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int nE = S * R * T, PT = P * T, nQ = S * PT;
    const double invN = 1.0 / (double)N;
    if (t < nE) {
        const int sample = t / (R * T), r = (t / T) % R;
        result[t] = E[(size_t)sample * Cp + r * T + slot_of_temp[t]] * invN;
    } else if (t < nE + nQ * 7) {
        const int u = t - nE;
        const int k = u % 7, item = (u / 7) % PT, sample = u / (7 * PT);
        double acc = 0.0;
        for (int c = 0; c < nchunk; ++c) acc += Mpart[(((size_t)sample * nchunk + c) * PT + item) * 7 + k];
        acc *= invN;
        if (k == 0) result[nE + (size_t)sample * PT + item] = acc;
        else result[nE + nQ + ((size_t)sample * PT + item) * 6 + (k - 1)] = acc;
    }
}

// ------------------------------------------------------------------------------------------------
// Overlaps between replicas held by DIFFERENT contexts (replica sharding; q_x = s^a_x . s^b_x,
// PAPER.md:79).  k_export_by_temp writes the configurations of local replica r ordered by temperature,
// out[sample][a][i][t] (t fastest), so that the partner needs no permutation; k_overlap_cross forms, per temperature,
// the sums of q_x and q_x e^{i 2 pi x_mu / L} between local replica r (through its own permutation) and such a
// buffer.  Thread = (site row, temperature): private fp64 sums, partials reduced in a fixed order by k_reduce_cross.
// ------------------------------------------------------------------------------------------------
__global__ void k_export_by_temp(const float* __restrict__ spins, const int* __restrict__ slot_of_temp, float* __restrict__ out,
                                 int L, int N, int NG, int R, int T, int Tl, int slot0, int r)
{
    // T: length of the chain; the context holds the slots [slot0, slot0 + Tl) (all of them unless slot-sharded).
    // A temperature whose configuration lives elsewhere is written as zeros, so that the sum of the shards' buffers
    // is the whole replica.
    const int sample = blockIdx.y;
    const size_t f = (size_t)blockIdx.x * blockDim.x + threadIdx.x;      // (site, temperature), temperature fastest
    if (f >= (size_t)N * T) return;
    const int i = (int)(f / T), t = (int)(f - (size_t)i * T);
    const int slot = slot_of_temp[((size_t)sample * R + r) * T + t] - slot0;
    const bool here = slot >= 0 && slot < Tl;
    const int c = r * Tl + (here ? slot : 0);
    const float* src = spins + (((size_t)sample * NG + c / G) * N + site_slot(i, L, N >> 1)) * SITE_FLOATS + (c % G);
    float* dst = out + (size_t)sample * 3 * N * T + f;
#pragma unroll
    for (int a = 0; a < 3; ++a) dst[(size_t)a * N * T] = here ? src[a * G] : 0.f;
}

constexpr int XCHUNKS = 128, XTHREADS = 256;     // k_overlap_cross: site chunks per sample, threads per CTA

struct CrossParams {
    const float* spins;        // [S][NG][2][Nh][3][G]
    const int* slot_of_temp;   // [S][R][T]
    const float* remote;       // [S][3][N][T] by temperature (k_export_by_temp of the partner)
    const double* phase;       // [L][2]
    double* Xpart;             // [S][XCHUNKS * rows][T][7]
    int L, N, NG, R, T, r;
    int Tl, slot0;             // slots per replica held here and the first of them (T, 0 unless slot-sharded)
};

__global__ void __launch_bounds__(XTHREADS) k_overlap_cross(const CrossParams p)
{
    const int chunk = blockIdx.x, sample = blockIdx.y;
    const int Tw = min(p.T, XTHREADS), rows = XTHREADS / Tw;
    const int tx = threadIdx.x % Tw, row = threadIdx.x / Tw;
    if (row >= rows) return;
    const int per = (p.N + XCHUNKS - 1) / XCHUNKS;
    const int i_begin = chunk * per, i_end = min(p.N, i_begin + per);
    const float* base = p.spins + (size_t)sample * p.NG * p.N * SITE_FLOATS;
    const float* rem = p.remote + (size_t)sample * 3 * p.N * p.T;
    const size_t plane = (size_t)p.N * p.T;
    for (int t = tx; t < p.T; t += Tw) {
        const int slot = p.slot_of_temp[((size_t)sample * p.R + p.r) * p.T + t] - p.slot0;
        const bool here = slot >= 0 && slot < p.Tl;      // else the configuration at t lives in another shard: sums stay 0
        const int c = p.r * p.Tl + (here ? slot : 0);
        const float* loc = base + (size_t)(c / G) * p.N * SITE_FLOATS + (c % G);
        double acc[7] = { 0, 0, 0, 0, 0, 0, 0 };
        for (int i = i_begin + row; here && i < i_end; i += rows) {
            const float* s = loc + site_slot(i, p.L, p.N >> 1) * SITE_FLOATS;
            const size_t f = (size_t)i * p.T + t;
            const float qf = fmaf(s[0], rem[f], fmaf(s[G], rem[plane + f], s[2 * G] * rem[2 * plane + f]));
            const double qx = (double)qf;
            const int x = i % p.L, y = (i / p.L) % p.L, z = i / (p.L * p.L);
            acc[0] += qx;
            acc[1] = fma(qx, p.phase[2 * x], acc[1]); acc[2] = fma(qx, p.phase[2 * x + 1], acc[2]);
            acc[3] = fma(qx, p.phase[2 * y], acc[3]); acc[4] = fma(qx, p.phase[2 * y + 1], acc[4]);
            acc[5] = fma(qx, p.phase[2 * z], acc[5]); acc[6] = fma(qx, p.phase[2 * z + 1], acc[6]);
        }
        double* dst = p.Xpart + ((((size_t)sample * XCHUNKS + chunk) * rows + row) * p.T + t) * 7;
#pragma unroll
        for (int k = 0; k < 7; ++k) dst[k] = acc[k];
    }
}

// result = [ q0[S][T] | qk[S][T][3][2] ]
__global__ void k_reduce_cross(const double* __restrict__ Xpart, double* __restrict__ result, int S, int T, int nparts, int N)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= S * T * 7) return;
    const int k = u % 7, t = (u / 7) % T, sample = u / (7 * T);
    double acc = 0.0;
    for (int c = 0; c < nparts; ++c) acc += Xpart[(((size_t)sample * nparts + c) * T + t) * 7 + k];
    acc /= (double)N;
    if (k == 0) result[(size_t)sample * T + t] = acc;
    else result[(size_t)S * T + ((size_t)sample * T + t) * 6 + (k - 1)] = acc;
}

// The chiral-glass counterpart (Eq. (2)): k_export_zeta_by_temp writes zeta_{x,mu} of local replica r ordered by
// temperature, out[sample][mu][i][t]; k_chiral_cross forms, per temperature, the 21 sums of kappa_{x,mu} = zeta^a zeta^b and
// kappa e^{i 2 pi x_nu / L} between two such buffers (either may be the partner's).  Same thread mapping as k_overlap_cross.
// T: temperatures of the chain; Tl, slot0: slots per replica held by this context and the first of them (T, 0 unless the chain is
// sharded by slot): a temperature whose configuration lives in another shard gets zeros, as in k_export_by_temp, so that the sum
// of the shards' exports is the replica ordered by temperature.
__global__ void k_export_zeta_by_temp(const float* __restrict__ spins, const int* __restrict__ slot_of_temp, float* __restrict__ out,
                                      int L, int N, int NG, int R, int T, int Tl, int slot0, int r)
{
    const int sample = blockIdx.y;
    const size_t f = (size_t)blockIdx.x * blockDim.x + threadIdx.x;      // (site, temperature), temperature fastest
    if (f >= (size_t)N * T) return;
    const int i = (int)(f / T), t = (int)(f - (size_t)i * T);
    const int slot = slot_of_temp[((size_t)sample * R + r) * T + t] - slot0;
    if (slot < 0 || slot >= Tl) {
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) out[(size_t)sample * 3 * N * T + (size_t)mu * N * T + f] = 0.f;
        return;
    }
    const int c = r * Tl + slot;
    const float* gb = spins + ((size_t)sample * NG + c / G) * N * SITE_FLOATS + (c % G);
    const int Nh = N >> 1;
    const float* c0 = gb + site_slot(i, L, Nh) * SITE_FLOATS;
    const float bx = c0[0], by = c0[G], bz = c0[2 * G];
    float* dst = out + (size_t)sample * 3 * N * T + f;
#pragma unroll
    for (int mu = 0; mu < 3; ++mu) {
        const int st = (mu == 0) ? 1 : ((mu == 1) ? L : L * L);
        const int xm = (mu == 0) ? i % L : ((mu == 1) ? (i / L) % L : i / (L * L));
        const int ip = (xm + 1 == L) ? i - (L - 1) * st : i + st, im = (xm == 0) ? i + (L - 1) * st : i - st;
        const float* pa = gb + site_slot(ip, L, Nh) * SITE_FLOATS;   // s_{x+e_mu}
        const float* pc = gb + site_slot(im, L, Nh) * SITE_FLOATS;   // s_{x-e_mu}
        const float ax = pa[0], ay = pa[G], az = pa[2 * G];
        const float cx = pc[0], cy = pc[G], cz = pc[2 * G];
        dst[(size_t)mu * N * T] = fmaf(ax, fmaf(by, cz, -bz * cy), fmaf(ay, fmaf(bz, cx, -bx * cz), az * fmaf(bx, cy, -by * cx)));
    }
}

__global__ void __launch_bounds__(XTHREADS) k_chiral_cross(const float* __restrict__ za, const float* __restrict__ zb, const double* __restrict__ phase,
                                                           double* __restrict__ Xpart /* [S][XCHUNKS * rows][T][21] */, int L, int N, int T)
{
    const int chunk = blockIdx.x, sample = blockIdx.y;
    const int Tw = min(T, XTHREADS), rows = XTHREADS / Tw;
    const int tx = threadIdx.x % Tw, row = threadIdx.x / Tw;
    if (row >= rows) return;
    const int per = (N + XCHUNKS - 1) / XCHUNKS;
    const int i_begin = chunk * per, i_end = min(N, i_begin + per);
    const size_t plane = (size_t)N * T;
    const float* a = za + (size_t)sample * 3 * plane;
    const float* b = zb + (size_t)sample * 3 * plane;
    for (int t = tx; t < T; t += Tw) {
        double acc[21];
#pragma unroll
        for (int k = 0; k < 21; ++k) acc[k] = 0.0;
        for (int i = i_begin + row; i < i_end; i += rows) {
            const size_t f = (size_t)i * T + t;
            const int xs[3] = { i % L, (i / L) % L, i / (L * L) };
#pragma unroll
            for (int mu = 0; mu < 3; ++mu) {
                const double kap = (double)(a[mu * plane + f] * b[mu * plane + f]);
                acc[mu] += kap;
#pragma unroll
                for (int nu = 0; nu < 3; ++nu) {
                    acc[3 + (mu * 3 + nu) * 2] = fma(kap, phase[2 * xs[nu]], acc[3 + (mu * 3 + nu) * 2]);
                    acc[4 + (mu * 3 + nu) * 2] = fma(kap, phase[2 * xs[nu] + 1], acc[4 + (mu * 3 + nu) * 2]);
                }
            }
        }
        double* dst = Xpart + ((((size_t)sample * XCHUNKS + chunk) * rows + row) * T + t) * 21;
#pragma unroll
        for (int k = 0; k < 21; ++k) dst[k] = acc[k];
    }
}

// result = [ qc0[S][T][3] | qck[S][T][3][3][2] ]
__global__ void k_reduce_chiral_cross(const double* __restrict__ Xpart, double* __restrict__ result, int S, int T, int nparts, int N)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= S * T * 21) return;
    const int k = u % 21, t = (u / 21) % T, sample = u / (21 * T);
    double acc = 0.0;
    for (int c = 0; c < nparts; ++c) acc += Xpart[(((size_t)sample * nparts + c) * T + t) * 21 + k];
    acc /= (double)N;
    if (k < 3) result[((size_t)sample * T + t) * 3 + k] = acc;
    else result[(size_t)S * T * 3 + ((size_t)sample * T + t) * 18 + (k - 3)] = acc;
}

// Logarithmic data binning (Sect. III): adds the observables of one measurement (the `result` of
// k_reduce_measure) into bin[S][T][6] (entries 0-3): mean over replicas of e, mean over pairs of q0^2, mean over pairs and the
// three k_min directions of |q(k_mu)|^2, mean over pairs of q0^4.  Thread = (sample, temperature); fp64, fixed order.
__global__ void k_logbin_add(const double* __restrict__ result, double* __restrict__ bin, int S, int R, int T, int P)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= S * T) return;
    const int sample = u / T, t = u % T;
    const int nE = S * R * T, PT = P * T, nQ = S * PT;
    double e = 0.0, q2 = 0.0, qk2 = 0.0, q4 = 0.0;
    for (int r = 0; r < R; ++r) e += result[((size_t)sample * R + r) * T + t];
    e /= (double)R;
    for (int pr = 0; pr < P; ++pr) {
        const size_t item = (size_t)sample * PT + (size_t)pr * T + t;
        const double q = result[nE + item];
        q2 += q * q;
        q4 += (q * q) * (q * q);
        const double* k = result + nE + nQ + item * 6;
        double m = 0.0;
        for (int mu = 0; mu < 3; ++mu) m += k[2 * mu] * k[2 * mu] + k[2 * mu + 1] * k[2 * mu + 1];
        qk2 += m / 3.0;
    }
    if (P > 0) { q2 /= (double)P; qk2 /= (double)P; q4 /= (double)P; }
    double* o = bin + (size_t)u * 6;
    o[0] += e; o[1] += q2; o[2] += qk2; o[3] += q4;
}

// The chiral-glass entries 4, 5 of the same bins from the `result` of k_reduce_chiral ([ qc0[S][P][T][3] | qck[S][P][T][3][3][2] ]):
// mean over pairs and mu of q_CG^mu(0)^2; mean over pairs, mu and the three k_min directions of |q_CG^mu(k_nu)|^2.
__global__ void k_logbin_add_chiral(const double* __restrict__ result, double* __restrict__ bin, int S, int T, int P)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= S * T || P == 0) return;
    const int sample = u / T, t = u % T;
    const int PT = P * T;
    const size_t nQ = (size_t)S * PT;
    double c0 = 0.0, ck = 0.0;
    for (int pr = 0; pr < P; ++pr) {
        const size_t item = (size_t)sample * PT + (size_t)pr * T + t;
        const double* a = result + item * 3;
        c0 += (a[0] * a[0] + a[1] * a[1] + a[2] * a[2]) / 3.0;
        const double* k = result + nQ * 3 + item * 18;
        double m = 0.0;
        for (int j = 0; j < 18; ++j) m += k[j] * k[j];
        ck += m / 9.0;
    }
    double* o = bin + (size_t)u * 6;
    o[4] += c0 / (double)P; o[5] += ck / (double)P;
}

// ------------------------------------------------------------------------------------------------
// Chirality observables (Eq. (2)): zeta_{x,mu} = s_{x+e_mu} . (s_x x s_{x-e_mu}),
// kappa_{x,mu} = zeta^a zeta^b, q^_CG^mu(k) = sum_x kappa_{x,mu} e^{ik.x}/N at k = 0 and k_nu = 2 pi e_nu/L.
// Same structure as k_measure: a CTA owns a chunk of sites; per batch of MS sites the threads first
// compute zeta_{x,mu} of EVERY copy (thread = copy lane: coalesced 128-byte lines, the stencil's re-reads
// hit L1/L2) into shared memory, then thread = (replica pair, temperature) looks its two copies up
// through the temperature permutation and accumulates the 21 sums in fp64.
// ------------------------------------------------------------------------------------------------
struct ChiralParams {
    const float* spins;        // [S][NG][2][Nh][3][G]
    const int* slot_of_temp;   // [S][R][T]
    const double* phase;       // [L][2]
    double* Mpart;             // [S][nchunk][PT][21]
    int L, N, NG, Cp, R, T, P, nchunk, chunk_sites, MS;
};

__global__ void k_measure_chiral(const ChiralParams p)
{
    extern __shared__ float sm[];   // [MS][3][Cp]: zeta_{x,mu} of every copy; then [MS][3][2] doubles: phases
    double* const phs = reinterpret_cast<double*>(sm + (size_t)p.MS * 3 * p.Cp);
    int* const nbs = reinterpret_cast<int*>(phs + (size_t)p.MS * 6);   // [MS][8]: site positions of the stencil
    const int chunk = blockIdx.x, sample = blockIdx.y;
    const int PT = p.P * p.T;
    const int item = blockIdx.z * blockDim.x + threadIdx.x;
    int ca = 0, cb = 0;
    const bool live = item < PT;
    if (live) {
        const int pr = item / p.T, t = item % p.T;
        int a = 0, rem = pr;
        while (rem >= p.R - 1 - a) { rem -= p.R - 1 - a; ++a; }
        const int b = a + 1 + rem;
        ca = a * p.T + p.slot_of_temp[((size_t)sample * p.R + a) * p.T + t];
        cb = b * p.T + p.slot_of_temp[((size_t)sample * p.R + b) * p.T + t];
    }
    double acc[21];
#pragma unroll
    for (int k = 0; k < 21; ++k) acc[k] = 0.0;
    const int i_begin = chunk * p.chunk_sites, i_end = min(p.N, i_begin + p.chunk_sites);
    const float* base = p.spins + (size_t)sample * p.NG * p.N * SITE_FLOATS;
    const int row = 3 * p.Cp, L = p.L, Nh = p.N >> 1;
    for (int i0 = i_begin; i0 < i_end; i0 += p.MS) {
        const int ms = min(p.MS, i_end - i0);
        __syncthreads();
        // positions (own, x1+-1, x2+-1, x3+-1) of the batch's sites in the colour-split order, once per batch
        for (int u = threadIdx.x; u < ms * 7; u += blockDim.x) {
            const int m = u / 7, k = u % 7, i = i0 + m;
            int j = i;
            if (k > 0) {
                const int mu = (k - 1) >> 1, up = (k - 1) & 1 ? 0 : 1;
                const int st = (mu == 0) ? 1 : ((mu == 1) ? L : L * L);
                const int xm = (mu == 0) ? i % L : ((mu == 1) ? (i / L) % L : i / (L * L));
                j = up ? ((xm + 1 == L) ? i - (L - 1) * st : i + st) : ((xm == 0) ? i + (L - 1) * st : i - st);
            }
            nbs[m * 8 + k] = (int)site_slot(j, L, Nh);
        }
        __syncthreads();
        // a warp computes zeta_{x,mu} of the 32 copies of one (site, copy group) per pass
        for (int r = threadIdx.x >> 5; r < ms * p.NG; r += blockDim.x >> 5) {
            const int m = r / p.NG, grp = r - m * p.NG, lane = threadIdx.x & 31;
            const float* gb = base + (size_t)grp * p.N * SITE_FLOATS + lane;
            const int* nb = nbs + m * 8;
            const float* c0 = gb + (size_t)nb[0] * SITE_FLOATS;
            const float bx = c0[0], by = c0[G], bz = c0[2 * G];
#pragma unroll
            for (int mu = 0; mu < 3; ++mu) {
                const float* pa = gb + (size_t)nb[1 + 2 * mu] * SITE_FLOATS;   // s_{x+e_mu}
                const float* pc = gb + (size_t)nb[2 + 2 * mu] * SITE_FLOATS;   // s_{x-e_mu}
                const float ax = pa[0], ay = pa[G], az = pa[2 * G];
                const float cx = pc[0], cy = pc[G], cz = pc[2 * G];
                // a . (b x c)
                const float z = fmaf(ax, fmaf(by, cz, -bz * cy), fmaf(ay, fmaf(bz, cx, -bx * cz), az * fmaf(bx, cy, -by * cx)));
                sm[m * row + mu * p.Cp + grp * G + lane] = z;
            }
        }
        for (int u = threadIdx.x; u < ms * 3; u += blockDim.x) {
            const int m = u / 3, nu = u % 3, i = i0 + m;
            const int xn = (nu == 0) ? i % L : ((nu == 1) ? (i / L) % L : i / (L * L));
            phs[m * 6 + 2 * nu] = p.phase[2 * xn];
            phs[m * 6 + 2 * nu + 1] = p.phase[2 * xn + 1];
        }
        __syncthreads();
        if (live) {
            for (int m = 0; m < ms; ++m) {
                const float* z = sm + m * row;
                double ph[3][2];
#pragma unroll
                for (int nu = 0; nu < 3; ++nu) { ph[nu][0] = phs[m * 6 + 2 * nu]; ph[nu][1] = phs[m * 6 + 2 * nu + 1]; }
#pragma unroll
                for (int mu = 0; mu < 3; ++mu) {
                    const double kap = (double)(z[mu * p.Cp + ca] * z[mu * p.Cp + cb]);
                    acc[mu] += kap;
#pragma unroll
                    for (int nu = 0; nu < 3; ++nu) {
                        acc[3 + 2 * (3 * mu + nu)] = fma(kap, ph[nu][0], acc[3 + 2 * (3 * mu + nu)]);
                        acc[4 + 2 * (3 * mu + nu)] = fma(kap, ph[nu][1], acc[4 + 2 * (3 * mu + nu)]);
                    }
                }
            }
        }
    }
    if (live) {
        double* dst = p.Mpart + (((size_t)sample * p.nchunk + chunk) * PT + item) * 21;
#pragma unroll
        for (int k = 0; k < 21; ++k) dst[k] = acc[k];
    }
}

// result = [ qc0[S][P][T][3] | qck[S][P][T][3][3][2] ]: fixed-order sum over the chunks, times 1/N
__global__ void k_reduce_chiral(const double* __restrict__ Mpart, double* __restrict__ result, int S, int PT, int nchunk, int N)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int nQ = S * PT;
    if (t >= nQ * 21) return;
    const int k = t % 21, item = (t / 21) % PT, sample = t / (21 * PT);
    double acc = 0.0;
    for (int c = 0; c < nchunk; ++c) acc += Mpart[(((size_t)sample * nchunk + c) * PT + item) * 21 + k];
    acc /= (double)N;
    if (k < 3) result[((size_t)sample * PT + item) * 3 + k] = acc;
    else result[(size_t)nQ * 3 + ((size_t)sample * PT + item) * 18 + (k - 3)] = acc;
}

// ------------------------------------------------------------------------------------------------
// Schwinger-Dyson monitor (Eq. (A6)): per copy, the site sums of s.h and of
// h.h - (s.h)^2 over BOTH colours (blockIdx.z = colour).  Same decomposition as k_sweep (a CTA = a tile of
// same-colour sites of one copy group; neighbours through L1/L2); a read-only pass, off the timed path.
// ------------------------------------------------------------------------------------------------
struct SdParams {
    const float* spins;      // [S][NG][2][Nh][3][G]
    const float* Jg;         // [S][2][Nh][JG]
    double* SDpart;          // [S][NG][2*ntiles][G][2]
    int L, N, Nh, NG, ntiles, tile_sites;
};

__global__ void __launch_bounds__(SWEEP_THREADS) k_sd(const SdParams p)
{
    const int tid = threadIdx.x, q = tid & 7, slot = tid >> 3;
    const int grp = blockIdx.x % p.NG, tile = blockIdx.x / p.NG, sample = blockIdx.y, colour = blockIdx.z;
    const int L = p.L;
    const float* const sp = p.spins + ((size_t)(sample * p.NG + grp) * p.N) * SITE_FLOATS + q * 4;
    const float* const Jc = p.Jg + ((size_t)(sample * 2 + colour) * p.Nh) * JG;
    float acc_a[4] = { 0.f, 0.f, 0.f, 0.f }, acc_b[4] = { 0.f, 0.f, 0.f, 0.f };
    const int h_end = min(p.Nh, (tile + 1) * p.tile_sites);
    for (int h = tile * p.tile_sites + slot; h < h_end; h += SLOTS) {
        int x, y, z;
        site_of<0>(h, colour, L, x, y, z);
        const int xp = (x + 1 == L) ? 0 : x + 1, xm = (x == 0) ? L - 1 : x - 1;
        const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
        const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
        const int row = L * (y + L * z);
        const int nb[6] = { xp + row, xm + row, x + L * (yp + L * z), x + L * (ym + L * z), x + L * (y + L * zp), x + L * (y + L * zm) };
        float J[JG];
        const float* jp = Jc + (size_t)h * JG;
#pragma unroll
        for (int v = 0; v < JG / 4; ++v) {
            const float4 t4 = ldg4(jp + 4 * v);
            J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
        }
        const float* const own = sp + ((size_t)colour * p.Nh + h) * SITE_FLOATS;
        float s[3][4], hf[3][4];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float4 t4 = ld4(own + a * G);
            s[a][0] = t4.x; s[a][1] = t4.y; s[a][2] = t4.z; s[a][3] = t4.w;
#pragma unroll
            for (int j = 0; j < 4; ++j) hf[a][j] = 0.f;
        }
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float* np_ = sp + ((size_t)(1 - colour) * p.Nh + (nb[k] >> 1)) * SITE_FLOATS;
            float n[3][4];
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const float4 t4 = ld4(np_ + b * G);
                n[b][0] = t4.x; n[b][1] = t4.y; n[b][2] = t4.z; n[b][3] = t4.w;
            }
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    fma4(J[9 * k + 3 * a + b], n[b], hf[a]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float sh = fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
            const float hh = fmaf(hf[0][j], hf[0][j], fmaf(hf[1][j], hf[1][j], hf[2][j] * hf[2][j]));
            acc_a[j] += sh;
            acc_b[j] += fmaf(-sh, sh, hh);
        }
    }
    __shared__ double red[SLOTS][G + 1];
    for (int k = 0; k < 2; ++k) {
        __syncthreads();
#pragma unroll
        for (int j = 0; j < 4; ++j) red[slot][q * 4 + j] = (double)(k ? acc_b[j] : acc_a[j]);
        __syncthreads();
        if (tid < G) {
            double acc = 0.0;
            for (int r = 0; r < SLOTS; ++r) acc += red[r][tid];
            p.SDpart[((((size_t)(sample * p.NG + grp) * 2 + colour) * p.ntiles + tile) * G + tid) * 2 + k] = acc;
        }
    }
}

// sd[S][R][T][2] = (sum_x s.h / N, sum_x [h.h - (s.h)^2] / N) of the copy of replica r at temperature t
// T: temperatures of the chain; Tl, slot0: slots per replica held here and the first of them (T, 0 unless sharded by slot): exact zeros
// for the temperatures whose configuration lives in another shard, so that the sum over the shards completes every temperature
__global__ void k_reduce_sd(const double* __restrict__ SDpart, const int* __restrict__ slot_of_temp, double* __restrict__ result,
                            int S, int R, int T, int Tl, int slot0, int NG, int ntiles, int N)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= S * R * T * 2) return;
    const int k = u & 1, t = (u >> 1) % T, r = (u / (2 * T)) % R, sample = u / (2 * T * R);
    const int slot = slot_of_temp[((size_t)sample * R + r) * T + t] - slot0;
    if (slot < 0 || slot >= Tl) { result[u] = 0.0; return; }
    const int c = r * Tl + slot;
    const int grp = c / G, lane = c % G;
    double acc = 0.0;
    for (int b = 0; b < 2 * ntiles; ++b) acc += SDpart[((((size_t)(sample * NG + grp)) * 2 * ntiles + b) * G + lane) * 2 + k];
    result[u] = acc / (double)N;
}

}  // namespace sg
