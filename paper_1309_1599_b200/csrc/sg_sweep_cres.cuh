// sg_sweep_cres.cuh -- the CLUSTER-resident multi-sweep kernel of libsg_b200 for L = 16.
//
// Why.  A group of 32 copies of an L = 16 lattice is 4096 sites x 384 bytes = 1.5 MB: too large for one CTA's shared
// memory (k_sweep_res stops at L = 12), exactly the shared memory of 8 SMs.  The z-marching kernel streams it from
// HBM / L2 twice per sweep and, at 16 planes, spends a quarter of its time filling and draining its pipeline (cfg 2:
// 0.71 of the streaming roofline).  Copies are independent between parallel-tempering swaps, so here
// thread-block clusters keep the lattice on chip for ALL n sweeps of an sg_sweep_or / sg_sweep_hb call: every CTA of a
// cluster holds a slab of consecutive planes (both colours, 192 KB), the x3 neighbours that lie across a cut are read from
// the neighbouring CTA's shared memory (mapa + ld.shared::cluster), a cluster barrier separates the two colours, and the
// couplings (shared by the copies of a site) are streamed 64 sites at a time through a two-stage ring of bulk copies.
// Spins cross HBM once per call; per update the SM reads 7-14 bytes of couplings from L2 and nothing else.
//
// Same arithmetic, in the same order, as k_sweep / k_sweep_zm / k_sweep_res (field: neighbours +x1,-x1,+x2,-x2,+x3,-x3),
// so the spins after a call are bit-identical to the other kernels'.  Thread = (site of the pass, quad of copies).
#pragma once
#include "sg_sweep_zm.cuh"

namespace sg {

// Two shapes of the same kernel (CS = CTAs per cluster):
//   CS = 8: a CTA holds 2 planes of all 32 copies of the group; every plane borders a cut (one neighbour in six is remote); an
//           8-CTA cluster must sit inside one GPC: 15 clusters = 120 of the 148 SMs run at once
//   CS = 4: a CTA holds 4 planes of 16 copies (half a group: two clusters per group); only the outer two planes border a cut
//           (one neighbour in twelve is remote); 4-CTA clusters pack 132-148 SMs.  Its 64-byte half lines cannot be bulk-copied:
//           the slab is loaded and stored with 16-byte accesses, once per call.
template <int CS_>
struct CresGeomT {
    static constexpr int L = 16, CS = CS_, PZ = L / CS;             // cluster size, planes per CTA
    static constexpr int NC = (CS == 8) ? 32 : 16;                  // copies per CTA
    static constexpr int QUADS = NC / 4;
    static constexpr int PLANE_C = L * L / 2;                       // 128 sites of one colour per plane
    static constexpr int SITES_C = PZ * PLANE_C;                    // sites of one colour per CTA: 256 / 512
    static constexpr int SITE_BYTES = 3 * NC * 4;                   // 384 / 192
    static constexpr int COMP_BYTES = NC * 4;                       // one component of a site
    static constexpr int COLOUR_BYTES = SITES_C * SITE_BYTES;       // 98304
    static constexpr int SLAB_BYTES = 2 * COLOUR_BYTES;             // 196608
    static constexpr int THREADS = 512;
    static constexpr int WARPS = THREADS / 32;
    static constexpr int PASS_SITES = THREADS / QUADS;              // 64 / 128 sites per pass
    static constexpr int PASSES = SITES_C / PASS_SITES;             // 4 passes per half-sweep
    static constexpr int PIECE_SITES = 64;                          // couplings are staged 64 sites at a time
    static constexpr int PP = PASS_SITES / PIECE_SITES;             // pieces per pass: 1 / 2
    static constexpr int JPIECE = PIECE_SITES * JG * 4;             // 14336
    static constexpr int NJ = 2;
    static constexpr int WARPS_PER_PIECE = WARPS / PP;
    static constexpr size_t SMEM = (size_t)SLAB_BYTES + NJ * JPIECE + 8 * (2 * NJ + 1) + 64;
};
using CresGeom = CresGeomT<8>;

struct CresParams {
    float* spins;            // [S][NG][2][Nh][3][G]
    const float* Jg;         // [S][2][Nh][JG]
    const float* beta_slot;  // [S][Cp]
    double* Epart;           // [S][NG][CS][G]: per-CTA partial sums of s.h over the colour-1 sites (CS = 4: the two half groups fill G)
    int N, Nh, NG, Cp, Cg, Tl, Tpad;
    int n_sweeps;
    uint32_t key0, key1, hb_counter, g_first;
};

__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
__device__ __forceinline__ float4 ld_dsmem4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

template <int KIND_, int CS_>
__global__ void __launch_bounds__(CresGeomT<CS_>::THREADS, 1) k_sweep_cres(const CresParams p)
{
    using Gm = CresGeomT<CS_>;
    constexpr int L = Gm::L;
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* const slab = smem;                                // [2 colours][SITES_C sites][3][NC] floats
    unsigned char* const jring = smem + Gm::SLAB_BYTES;              // NJ pieces of couplings
    const uint32_t bars = smem_u32(jring + Gm::NJ * Gm::JPIECE);     // full_j[NJ] empty_j[NJ] slab
    auto full_j = [&](int s) { return bars + 8u * s; };
    auto empty_j = [&](int s) { return bars + 8u * (Gm::NJ + s); };
    const uint32_t bar_slab = bars + 8u * (2 * Gm::NJ);

    const int tid = threadIdx.x, q = tid % Gm::QUADS, slot = tid / Gm::QUADS;
    const uint32_t rank = cluster_rank();
    constexpr int HALVES = G / Gm::NC;                               // clusters per copy group: 1 / 2
    const int grp = blockIdx.x / (Gm::CS * HALVES), half = (blockIdx.x / Gm::CS) % HALVES, sample = blockIdx.y;
    const int c_first = grp * G + half * Gm::NC;                     // first copy of this CTA inside the sample
    float* const gl = p.spins + ((size_t)(sample * p.NG + grp) * p.N) * SITE_FLOATS;     // the group's lattice in HBM

    if (tid == 0) {
        for (int s = 0; s < Gm::NJ; ++s) { mbar_init(full_j(s), 1); mbar_init(empty_j(s), Gm::WARPS_PER_PIECE); }
        mbar_init(bar_slab, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // couplings: piece g = (half-sweep * PASSES + pass) * PP + part covers 64 colour sites h = SITES_C rank + 64 (pass PP + part) ...;
    // it lives in stage g % NJ and is read by the WARPS / PP warps that update those sites
    const int n_pieces = p.n_sweeps * 2 * Gm::PASSES * Gm::PP;
    auto issue_j = [&](int g) {
        const int colour = (g / (Gm::PASSES * Gm::PP)) & 1, piece = g % (Gm::PASSES * Gm::PP);
        const float* src = p.Jg + ((size_t)(sample * 2 + colour) * p.Nh + (size_t)rank * Gm::SITES_C + (size_t)piece * Gm::PIECE_SITES) * JG;
        mbar_expect_tx(full_j(g % Gm::NJ), Gm::JPIECE);
        bulk_g2s(smem_u32(jring + (size_t)(g % Gm::NJ) * Gm::JPIECE), src, Gm::JPIECE, full_j(g % Gm::NJ));
    };
    if (tid == 0) {
        if (Gm::NC == G) {
            // the slab: the CTA's sites of each colour are contiguous in the colour-split site order
            mbar_expect_tx(bar_slab, Gm::SLAB_BYTES);
            for (int c = 0; c < 2; ++c)
                bulk_g2s(smem_u32(slab + (size_t)c * Gm::COLOUR_BYTES), gl + ((size_t)c * p.Nh + (size_t)rank * Gm::SITES_C) * SITE_FLOATS,
                         Gm::COLOUR_BYTES, bar_slab);
        }
        for (int g = 0; g < Gm::NJ && g < n_pieces; ++g) issue_j(g);
    }
    if (Gm::NC != G) {
        // half lines (64 of every 128 bytes): 16-byte loads, once per call
        for (int c = 0; c < 2; ++c) {
            const float* const src = gl + ((size_t)c * p.Nh + (size_t)rank * Gm::SITES_C) * SITE_FLOATS + half * Gm::NC;
            float* const dstc = reinterpret_cast<float*>(slab + (size_t)c * Gm::COLOUR_BYTES);
            for (int e = tid; e < Gm::SITES_C * 3 * Gm::QUADS; e += Gm::THREADS) {
                const int qq = e % Gm::QUADS, line = e / Gm::QUADS;                 // line = site * 3 + component
                st4(dstc + (size_t)line * Gm::NC + qq * 4, ld4(src + (size_t)line * G + qq * 4));
            }
        }
        __syncthreads();
    }

    float4 beta4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (KIND_ == KIND_HB) beta4 = ldg4(p.beta_slot + (size_t)sample * p.Cp + c_first + q * 4);
    uint32_t gid[4] = { 0u, 0u, 0u, 0u };
    if (KIND_ == KIND_HB) {
#pragma unroll
        for (int j = 0; j < 4; ++j) gid[j] = copy_gid(p.g_first + (uint32_t)sample * (uint32_t)p.Cg, c_first + q * 4 + j, p.Tl, p.Tpad);
    }
    float eacc[4] = { 0.f, 0.f, 0.f, 0.f };

    if (Gm::NC == G) mbar_wait(bar_slab, 0);
    cluster_sync_all();          // every CTA of the cluster holds its planes before anyone reads across the cut

    const uint32_t slab_u32 = smem_u32(slab);
    int t = 0;
    for (int sw = 0; sw < p.n_sweeps; ++sw) {
        for (int colour = 0; colour < 2; ++colour) {
            const bool last = (sw == p.n_sweeps - 1) && (colour == 1);
            unsigned char* const mine = slab + (size_t)colour * Gm::COLOUR_BYTES + q * 16;
            const uint32_t other = (uint32_t)((1 - colour) * Gm::COLOUR_BYTES + q * 16);      // byte offset of the other colour (this quad)
#pragma unroll 1
            for (int pass = 0; pass < Gm::PASSES; ++pass, ++t) {
                const int hl = pass * Gm::PASS_SITES + slot;               // site of this thread among the CTA's SITES_C of the colour
                const int zl = hl >> 7, m = hl & 127, y = m >> 3, xh = m & 7;
                const int z = (int)rank * Gm::PZ + zl;
                const int x = 2 * xh + ((y + z + colour) & 1);
                const int i = x + L * (y + L * z);
                const int rowo = zl * Gm::PLANE_C + y * 8;
                const uint32_t o_xp = other + (uint32_t)(rowo + (((x + 1) & 15) >> 1)) * Gm::SITE_BYTES;
                const uint32_t o_xm = other + (uint32_t)(rowo + (((x + 15) & 15) >> 1)) * Gm::SITE_BYTES;
                const uint32_t o_yp = other + (uint32_t)(zl * Gm::PLANE_C + ((y + 1) & 15) * 8 + xh) * Gm::SITE_BYTES;
                const uint32_t o_ym = other + (uint32_t)(zl * Gm::PLANE_C + ((y + 15) & 15) * 8 + xh) * Gm::SITE_BYTES;
                // x3 neighbours: inside the CTA, except below its first plane and above its last one -- there it is the last / first
                // plane of CTA rank -+ 1 (same offset in that CTA's shared memory window)
                const bool up_remote = (zl == Gm::PZ - 1), dn_remote = (zl == 0);
                const uint32_t o_zp = other + (uint32_t)((up_remote ? 0 : zl + 1) * Gm::PLANE_C + y * 8 + xh) * Gm::SITE_BYTES;
                const uint32_t o_zm = other + (uint32_t)((dn_remote ? Gm::PZ - 1 : zl - 1) * Gm::PLANE_C + y * 8 + xh) * Gm::SITE_BYTES;
                float nbz[3][4];                                           // the remote spin first: it has the longest way
                if (up_remote || dn_remote) {                              // uniform over the pass (a pass is one plane or half of one)
                    const uint32_t rz = up_remote ? dsmem_addr(slab_u32 + o_zp, (rank + 1) & (Gm::CS - 1))
                                                  : dsmem_addr(slab_u32 + o_zm, (rank + Gm::CS - 1) & (Gm::CS - 1));
#pragma unroll
                    for (int bb = 0; bb < 3; ++bb) {
                        const float4 t4 = ld_dsmem4(rz + bb * Gm::COMP_BYTES);
                        nbz[bb][0] = t4.x; nbz[bb][1] = t4.y; nbz[bb][2] = t4.z; nbz[bb][3] = t4.w;
                    }
                }
                const int part = slot / Gm::PIECE_SITES;                   // which 64-site piece of the pass this thread's site is in
                const int g = t * Gm::PP + part;
                const int sj = g % Gm::NJ;
                mbar_wait(full_j(sj), (g / Gm::NJ) & 1);
                float J[JG];
                {
                    const unsigned char* Jp = jring + (size_t)sj * Gm::JPIECE + (slot % Gm::PIECE_SITES) * (JG * 4);
#pragma unroll
                    for (int v = 0; v < JG / 4; ++v) {
                        const float4 t4 = lds4(Jp + 16 * v);
                        J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
                    }
                }
                __syncwarp();
                if ((tid & 31) == 0) mbar_arrive(empty_j(sj));
                if (tid == part * (Gm::THREADS / Gm::PP) && g + Gm::NJ < n_pieces) {   // refill the stage once every warp that reads it holds its couplings
                    mbar_wait(empty_j(sj), (g / Gm::NJ) & 1);
                    issue_j(g + Gm::NJ);
                }

                float hf[3][4], s[3][4];
                unsigned char* const own = mine + (size_t)hl * Gm::SITE_BYTES;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float4 t4 = lds4(own + a * Gm::COMP_BYTES);
                    s[a][0] = t4.x; s[a][1] = t4.y; s[a][2] = t4.z; s[a][3] = t4.w;
#pragma unroll
                    for (int j = 0; j < 4; ++j) hf[a][j] = 0.f;
                }
                const uint32_t offs[4] = { o_xp, o_xm, o_yp, o_ym };
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    float n[3][4];
                    if (k < 4 || (k == 4 && !up_remote) || (k == 5 && !dn_remote)) {
                        const unsigned char* np_ = slab + (k < 4 ? offs[k] : (k == 4 ? o_zp : o_zm));
#pragma unroll
                        for (int bb = 0; bb < 3; ++bb) {
                            const float4 t4 = lds4(np_ + bb * Gm::COMP_BYTES);
                            n[bb][0] = t4.x; n[bb][1] = t4.y; n[bb][2] = t4.z; n[bb][3] = t4.w;
                        }
                    } else {
#pragma unroll
                        for (int bb = 0; bb < 3; ++bb)
#pragma unroll
                            for (int j = 0; j < 4; ++j) n[bb][j] = nbz[bb][j];
                    }
#pragma unroll
                    for (int a = 0; a < 3; ++a)
#pragma unroll
                        for (int bb = 0; bb < 3; ++bb)
                            fma4(J[9 * k + 3 * a + bb], n[bb], hf[a]);
                }
                if (KIND_ == KIND_OR) {
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
                for (int a = 0; a < 3; ++a) *reinterpret_cast<float4*>(own + a * Gm::COMP_BYTES) = make_float4(s[a][0], s[a][1], s[a][2], s[a][3]);
            }
            cluster_sync_all();      // the other colour -- here and across the cut -- reads what this colour wrote
        }
    }

    // the slab back to HBM (coalesced 16-byte stores; the two colours are contiguous there as they are here)
    for (int c = 0; c < 2; ++c) {
        float* const dst = gl + ((size_t)c * p.Nh + (size_t)rank * Gm::SITES_C) * SITE_FLOATS + half * Gm::NC;
        const float* const src = reinterpret_cast<const float*>(slab + (size_t)c * Gm::COLOUR_BYTES);
        for (int e = tid; e < Gm::SITES_C * 3 * Gm::QUADS; e += Gm::THREADS) {
            const int qq = e % Gm::QUADS, line = e / Gm::QUADS;
            st4(dst + (size_t)line * G + qq * 4, *reinterpret_cast<const float4*>(src + (size_t)line * Gm::NC + qq * 4));
        }
    }
    // per-copy sums of s.h over this CTA's colour-1 sites: fixed order, fp64 across threads; k_reduce_energy adds the 8 CTAs
    __syncthreads();
    double* red = reinterpret_cast<double*>(jring);         // [PASS_SITES][NC + 1]: the coupling ring is dead
#pragma unroll
    for (int j = 0; j < 4; ++j) red[slot * (Gm::NC + 1) + q * 4 + j] = (double)eacc[j];
    __syncthreads();
    if (tid < Gm::NC) {
        double acc = 0.0;
        for (int r = 0; r < Gm::PASS_SITES; ++r) acc += red[r * (Gm::NC + 1) + tid];
        p.Epart[((size_t)(sample * p.NG + grp) * Gm::CS + rank) * G + half * Gm::NC + tid] = acc;
    }
}

}  // namespace sg
