// sg_sweep_res.cuh -- the shared-memory-resident multi-sweep kernel of libsg_b200 for small lattices
// (multi-sweep fusion where the state fits on chip).
//
// Why.  For L <= 8 a half-sweep is a few thousand site updates per copy group: one launch per half-sweep is
// pure launch and pipeline latency (cfg 1: 16 CTAs per launch, 15 us each, 0.05 of the HBM roofline).  Copies
// are independent between parallel-tempering swaps, so a CTA can keep the WHOLE lattice of one
// (sample, group of 32 copies) in shared memory -- N sites x 384 bytes: 24 KB at L = 4, 192 KB at L = 8 -- and
// run all n sweeps of an sg_sweep_or / sg_sweep_hb call in one launch: spins cross HBM once per call instead of
// once per half-sweep, and the per-copy energies come out of the last half-sweep with no second kernel.
// The couplings (224 bytes per site, shared by the 32 copies) are read through L1/L2 every half-sweep.
//
// Same arithmetic, in the same order, as k_sweep / k_sweep_zm (field: neighbours +x1,-x1,+x2,-x2,+x3,-x3, rows,
// columns), so the spins after a call are bit-identical to the other two kernels'; only the energy summation
// order differs.  Thread = (site slot, quad of copies).  A CTA takes CPC = 32, 16, 8 or 4 consecutive copies of a
// group (CPC/4 quads x 1024/CPC site slots): small problems are spread over more SMs by giving each CTA fewer
// copies (cfg 1 has only 16 (sample, group) pairs for 148 SMs); CPC >= 8 keeps every global access a full 32-byte sector.
#pragma once
#include "sg_device.cuh"

namespace sg {

struct ResParams {
    float* spins;            // [S][NG][2][Nh][3][G]
    const float* Jg;         // [S][2][Nh][JG]
    const float* beta_slot;  // [S][Cp]
    double* E;               // [S][Cp]: total H of every slot, written by the last half-sweep
    int L, N, Nh, NG, C, Cp, Cg;   // Cg: copies per sample of the whole job (stride of the global copy id)
    int Tl, Tpad;                  // slots per replica held here, n_temps_total - Tl (copy_gid)
    int n_sweeps;                  // sweeps of the kernel's kind; KIND_ = 2 (a whole unit): overrelaxation sweeps ...
    int n_hb;                      // ... after n_hb heat-bath sweeps, all in one launch
    uint32_t key0, key1, hb_counter, g_first;
};

constexpr int RES_THREADS = 256;

inline size_t res_smem_bytes(int N, int cpc) { return (size_t)N * 3 * cpc * sizeof(float); }
// JSMEM: the couplings of the sample (both colours) resident in shared memory too, one block per site padded from 56 to
// RES_JPAD floats (60 words: the blocks of 8 consecutive sites start in 8 different bank groups)
constexpr int RES_JPAD = 60;
inline size_t res_jsmem_bytes(int N) { return (size_t)N * RES_JPAD * sizeof(float); }

template <int KIND_, int LOG2L, int CPC, bool JSMEM = false>
__global__ void __launch_bounds__(RES_THREADS) k_sweep_res(const ResParams p)
{
    constexpr int QUADS = CPC / 4, RES_SLOTS = RES_THREADS / QUADS, SUBS = G / CPC, SITE = 3 * CPC;
    extern __shared__ __align__(16) float lat[];      // [2][Nh][3][CPC]: the lattice of this CTA's copies; JSMEM: then [2][Nh][RES_JPAD] couplings
    __shared__ double red[RES_SLOTS * (CPC + 1)];
    const int tid = threadIdx.x, q = tid % QUADS, slot = tid / QUADS;
    const int grp = blockIdx.x / SUBS, sub = blockIdx.x % SUBS, sample = blockIdx.y;
    const int c_first = grp * G + sub * CPC;          // first copy of this CTA inside the sample
    if (c_first >= p.C) return;                       // padding copies only
    const int L = p.L;
    float* const gl = p.spins + ((size_t)(sample * p.NG + grp) * p.N) * SITE_FLOATS + sub * CPC;
    for (int e = tid; e < p.N * 3 * QUADS; e += RES_THREADS) {
        const int qq = e % QUADS, line = e / QUADS;   // line = site * 3 + component
        st4(lat + line * CPC + qq * 4, ld4(gl + (size_t)line * G + qq * 4));
    }
    float* const Js = lat + (size_t)p.N * SITE;       // JSMEM: the sample's coupling blocks, by colour then h
    if (JSMEM) {
        const float* const Jsrc = p.Jg + (size_t)sample * 2 * p.Nh * JG;
        for (int e = tid; e < p.N * (JG / 4); e += RES_THREADS) {
            const int v = e % (JG / 4), site = e / (JG / 4);
            st4(Js + (size_t)site * RES_JPAD + 4 * v, ldg4(Jsrc + (size_t)site * JG + 4 * v));
        }
    }
    __syncthreads();

    float* const sp = lat + q * 4;
    float4 beta4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (KIND_ != 0) beta4 = ldg4(p.beta_slot + (size_t)sample * p.Cp + c_first + q * 4);
    uint32_t gid[4];                                  // global ids of this thread's four copies
#pragma unroll
    for (int j = 0; j < 4; ++j) gid[j] = copy_gid(p.g_first + (uint32_t)sample * (uint32_t)p.Cg, c_first + q * 4 + j, p.Tl, p.Tpad);
    float eacc[4] = { 0.f, 0.f, 0.f, 0.f };

    const int n_total = (KIND_ == 2) ? p.n_hb + p.n_sweeps : p.n_sweeps;
    for (int sw = 0; sw < n_total; ++sw) {
        const bool heat_bath = (KIND_ == 1) || (KIND_ == 2 && sw < p.n_hb);
        for (int colour = 0; colour < 2; ++colour) {
            const bool last = (sw == n_total - 1) && (colour == 1);
            const float* const Jc = p.Jg + ((size_t)(sample * 2 + colour) * p.Nh) * JG;
            for (int h = slot; h < p.Nh; h += RES_SLOTS) {
                int x, y, z;
                site_of<LOG2L>(h, colour, L, x, y, z);
                const int xp = (x + 1 == L) ? 0 : x + 1, xm = (x == 0) ? L - 1 : x - 1;
                const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
                const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
                const int row = L * (y + L * z);
                const int i = x + row;
                const int nb[6] = { xp + row, xm + row, x + L * (yp + L * z), x + L * (ym + L * z),
                                    x + L * (y + L * zp), x + L * (y + L * zm) };
                float J[JG];
                if (JSMEM) {
                    const float* jp = Js + (size_t)(colour * p.Nh + h) * RES_JPAD;
#pragma unroll
                    for (int v = 0; v < JG / 4; ++v) {
                        const float4 t4 = ld4(jp + 4 * v);
                        J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
                    }
                } else {
                    const float* jp = Jc + (size_t)h * JG;
#pragma unroll
                    for (int v = 0; v < JG / 4; ++v) {
                        const float4 t4 = ldg4(jp + 4 * v);
                        J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
                    }
                }
                float* const own = sp + (colour * p.Nh + h) * SITE;
                float s[3][4], hf[3][4];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float4 t4 = ld4(own + a * CPC);
                    s[a][0] = t4.x; s[a][1] = t4.y; s[a][2] = t4.z; s[a][3] = t4.w;
#pragma unroll
                    for (int j = 0; j < 4; ++j) hf[a][j] = 0.f;
                }
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    const float* np_ = sp + ((1 - colour) * p.Nh + (nb[k] >> 1)) * SITE;
                    float n[3][4];
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        const float4 t4 = ld4(np_ + b * CPC);
                        n[b][0] = t4.x; n[b][1] = t4.y; n[b][2] = t4.z; n[b][3] = t4.w;
                    }
#pragma unroll
                    for (int a = 0; a < 3; ++a)
#pragma unroll
                        for (int b = 0; b < 3; ++b)
                    fma4(J[9 * k + 3 * a + b], n[b], hf[a]);
                }
                if (!heat_bath) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        or_update(hf[0][j], hf[1][j], hf[2][j], s[0][j], s[1][j], s[2][j]);
                        if (last) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));   // of the stored spin
                    }
                } else {
                    const float bt[4] = { beta4.x, beta4.y, beta4.z, beta4.w };
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        uint32_t w[4];
                        philox4x32_10((uint32_t)i, gid[j], p.hb_counter + (uint32_t)sw, STREAM_HB, p.key0, p.key1, w);
                        hb_update(hf[0][j], hf[1][j], hf[2][j], bt[j], uniform23(w[0]), uniform23(w[1]), s[0][j], s[1][j], s[2][j]);
                        if (last) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
                    }
                }
#pragma unroll
                for (int a = 0; a < 3; ++a) st4(own + a * CPC, make_float4(s[a][0], s[a][1], s[a][2], s[a][3]));
            }
            __syncthreads();      // the other colour reads what this colour wrote
        }
    }

    for (int e = tid; e < p.N * 3 * QUADS; e += RES_THREADS) {
        const int qq = e % QUADS, line = e / QUADS;
        st4(gl + (size_t)line * G + qq * 4, ld4(lat + line * CPC + qq * 4));
    }
    // E = - sum over the colour-1 sites of s.h (every link joins the two colours): fixed order, fp64 across threads
#pragma unroll
    for (int j = 0; j < 4; ++j) red[slot * (CPC + 1) + q * 4 + j] = (double)eacc[j];
    __syncthreads();
    if (tid < CPC) {
        double acc = 0.0;
        for (int r = 0; r < RES_SLOTS; ++r) acc += red[r * (CPC + 1) + tid];
        p.E[(size_t)sample * p.Cp + c_first + tid] = -acc;
    }
}

}  // namespace sg
