// sg_sweep_fz.cuh -- the colour-fused z-marching overrelaxation sweep (L a multiple of 8).
//
// Why.  Two half-sweeps stream every spin of a sample through the SMs twice: 36 + 216/C bytes per update.  A sweep that
// updates colour 0 of plane k and then colour 1 of plane k-1 in ONE pass reads every spin once and writes it once:
// 24 + 216/C bytes per update, the only way past the streaming roofline of the half-sweep kernel (sg_sweep_zm.cuh).
// A colour-1 site needs the NEW colour-0 values of its six neighbours.  A CTA owns an 8 x 8 column and marches along x3;
// the new colour-0 values just outside the column belong to the neighbouring CTAs, which run unsynchronised.  They are
// recomputed here: per plane the CTA updates the 32 colour-0 sites of its tile AND the 16 colour-0 sites of the one-site
// ring around it (the same inputs and the same instruction sequence as the owner: bit-identical values), keeps them in
// shared memory only, and updates its 32 colour-1 sites of the plane below from them: 80 site updates for 64 stored ones.
// Since a CTA reads old values of sites other CTAs overwrite, the sweep is OUT OF PLACE: it reads `src`, writes `dst`,
// and the library swaps the two buffers afterwards.
//
// Step n = 0 .. ZC+1 of a chunk of ZC planes starting at z0 (pz = z0 - 1 + n, all x3 periodic):
//   A(n)  colour 0 of plane pz over the tile and its ring, from the OLD colour-1 sites of planes pz-1, pz, pz+1
//   B(n)  colour 1 of plane pz-1 over the tile (n >= 2), from the NEW colour-0 sites of planes pz-2, pz-1, pz
// so the colour-0 planes z0-1 and z0+ZC are computed twice (by this chunk and by its x3 neighbours): (ZC+2)/ZC work.
// A thread (site, copy quad) handles the colour-0 site (x1, x2, pz) and the colour-1 site right below it, so the x3
// neighbours of both updates and the own spin of the second are values the thread already holds in registers:
//   U  = old colour 1 at (x1, x2, pz+1)   read from shared memory for A(n); it is M of step n+2
//   M  = old colour 1 at (x1, x2, pz-1)   x3-1 neighbour of A(n) and own spin of B(n)
//   N0 = new colour 0 at (x1, x2, pz)     result of A(n), x3+1 neighbour of B(n); it is P0 of step n+2
//   P0 = new colour 0 at (x1, x2, pz-2)   x3-1 neighbour of B(n)
// Shared memory per CTA: a ring of NSO stages of OLD colour-1 planes (tile + two-site diamond halo, 12 rows x 6 slots),
// a ring of NSN stages of NEW colour-0 planes (tile + ring, 10 rows x 5 slots), NJ stages of couplings (32 + 16 + 32
// site blocks); one producer warp feeds the first and the last with bulk copies completing on mbarriers.
#pragma once
#include "sg_sweep_zm.cuh"

namespace sg {

struct FzGeom {
    static constexpr int TX = 8, TY = 8;
    static constexpr int SITE_BYTES = SITE_FLOATS * 4;             // 384
    static constexpr int OROW = 6, OROWS = 12;                     // old colour 1: xx in [-2, 9] -> slot (xx+2)>>1, yy in [-2, 9]
    static constexpr int OSTAGE = OROW * OROWS * SITE_BYTES;       // 27648
    static constexpr int OLOADED = (8 * 6 + 2 * 5 + 2 * 4) * SITE_BYTES;   // 66 sites really loaded per plane
    static constexpr int NROW = 5, NROWS = 10;                     // new colour 0: xx in [-1, 8] -> slot (xx+1)>>1, yy in [-1, 8]
    static constexpr int NSTAGE = NROW * NROWS * SITE_BYTES;       // 19200
    static constexpr int JSITE = JG * 4;                           // 224
    static constexpr int JA = 32 * JSITE, JR = 16 * JSITE, JB = 32 * JSITE;
    static constexpr int JSTAGE = JA + JR + JB;                    // 17920: A interior | A ring | B
    static constexpr int WARPS_I = 8, WARPS_R = 4;                 // interior (A + B) and ring (A only) consumer warps
    static constexpr int CONSUMERS = (WARPS_I + WARPS_R) * 32;     // 384
    static constexpr int THREADS = CONSUMERS;                      // no producer warp: the first ring warp issues the bulk copies
                                                                   // (384 threads leave 168 registers per thread; 416 would cap them at 128)
};

template <int NSO, int NSN, int NJ>
constexpr size_t fz_smem_bytes()
{
    return (size_t)NSO * FzGeom::OSTAGE + (size_t)NSN * FzGeom::NSTAGE + (size_t)NJ * FzGeom::JSTAGE + 8 * (2 * NSO + 2 * NJ) + 128;
}

struct FzParams {
    const float* src;        // [S][NG][2][Nh][3][G]: the state before the sweep
    float* dst;              // same layout: the state after it
    const float* Jt;         // [S][2][L/8][L/8][L][8][4][JG]
    const float* Jr;         // [S][L/8][L/8][L][16][JG]: colour-0 ring sites of every (tile, plane): rows x2 = -1, 8, columns x1 = -1, 8
    double* Epart;           // [S][NG][nblk][G]
    int L, N, Nh, NG;
    int ntx, nty, nzc, ZC;
};

// local coordinates (xx, yy) of ring site rs = 0..15 of a plane whose colour-0 sites have (xx + yy + par) even
// (par = parity of the plane): rows x2 = -1 and 8 (4 sites each, x1 ascending), columns x1 = -1 and 8 (x2 ascending)
__host__ __device__ inline void fz_ring_site(int rs, int par, int& xx, int& yy)
{
    const int side = rs >> 2, j = rs & 3;
    if (side == 0) { yy = -1; xx = 2 * j + ((par + 1) & 1); }
    else if (side == 1) { yy = 8; xx = 2 * j + (par & 1); }
    else if (side == 2) { xx = -1; yy = 2 * j + ((par + 1) & 1); }
    else { xx = 8; yy = 2 * j + (par & 1); }
}

// gathered couplings Jg[2][Nh][JG] of one sample -> Jr[L/8][L/8][L][16][JG] (the blocks of the colour-0 ring sites)
__global__ void k_gather_ring_couplings(const float* __restrict__ Jg_sample, float* __restrict__ Jr_sample, int L)
{
    const int nt = L >> 3;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;     // (tile y, tile x, plane, ring site)
    if (t >= (size_t)nt * nt * L * 16) return;
    const int rs = (int)(t & 15);
    const int z = (int)((t >> 4) % L);
    const int tile = (int)((t >> 4) / L), tx = tile % nt, ty = tile / nt;
    int xx, yy;
    fz_ring_site(rs, z & 1, xx, yy);
    const int x = (tx * 8 + xx + L) % L, y = (ty * 8 + yy + L) % L;
    const int i = x + L * (y + L * z);                                  // a colour-0 site by construction
    const float* src = Jg_sample + (size_t)(i >> 1) * JG;
    float* dst = Jr_sample + t * JG;
    for (int e = 0; e < JG; ++e) dst[e] = src[e];
}

// field of 4 copies: hf[a][j] += sum_b J[9 nbk + 3 a + b] n[b][j], in the order of the half-sweep kernels
__device__ __forceinline__ void fz_acc(const float (&J)[JG], int nbk, const float (&n)[3][4], float (&hf)[3][4])
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int bb = 0; bb < 3; ++bb)
            fma4(J[9 * nbk + 3 * a + bb], n[bb], hf[a]);
}
__device__ __forceinline__ void fz_lds_spin(const unsigned char* p, float (&n)[3][4])
{
#pragma unroll
    for (int bb = 0; bb < 3; ++bb) {
        const float4 t4 = lds4(p + bb * (G * 4));
        n[bb][0] = t4.x; n[bb][1] = t4.y; n[bb][2] = t4.z; n[bb][3] = t4.w;
    }
}
__device__ __forceinline__ void fz_sts_spin(unsigned char* p, const float (&s)[3][4])
{
#pragma unroll
    for (int a = 0; a < 3; ++a) *reinterpret_cast<float4*>(p + a * (G * 4)) = make_float4(s[a][0], s[a][1], s[a][2], s[a][3]);
}
__device__ __forceinline__ void fz_lds_J(const unsigned char* p, float (&J)[JG])
{
#pragma unroll
    for (int v = 0; v < JG / 4; ++v) {
        const float4 t4 = lds4(p + 16 * v);
        J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
    }
}
__device__ __forceinline__ void fz_ldg_spin(const float* p, float (&s)[3][4])
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float4 t4 = ld4(p + a * G);
        s[a][0] = t4.x; s[a][1] = t4.y; s[a][2] = t4.z; s[a][3] = t4.w;
    }
}
__device__ __forceinline__ void fz_stg_spin(float* p, const float (&s)[3][4])
{
#pragma unroll
    for (int a = 0; a < 3; ++a) st4(p + a * G, make_float4(s[a][0], s[a][1], s[a][2], s[a][3]));
}
__device__ __forceinline__ void fz_or4(const float (&hf)[3][4], float (&s)[3][4])
{
#pragma unroll
    for (int j = 0; j < 4; ++j) or_update(hf[0][j], hf[1][j], hf[2][j], s[0][j], s[1][j], s[2][j]);
}

template <bool WITH_E, int NSO, int NSN, int NJ>
__global__ void __launch_bounds__(FzGeom::THREADS, 1) k_sweep_fz(const FzParams p)
{
    using Gm = FzGeom;
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* const oring = smem;                                            // NSO stages: old colour-1 planes
    unsigned char* const nring = oring + (size_t)NSO * Gm::OSTAGE;                // NSN stages: new colour-0 planes
    unsigned char* const jring = nring + (size_t)NSN * Gm::NSTAGE;                // NJ stages: couplings
    const uint32_t bars = smem_u32(jring + (size_t)NJ * Gm::JSTAGE);              // full_o[NSO] empty_o[NSO] full_j[NJ] empty_j[NJ]
    auto full_o = [&](int s) { return bars + 8u * s; };
    auto empty_o = [&](int s) { return bars + 8u * (NSO + s); };
    auto full_j = [&](int s) { return bars + 8u * (2 * NSO + s); };
    auto empty_j = [&](int s) { return bars + 8u * (2 * NSO + NJ + s); };

    const int tid = threadIdx.x;
    int b = blockIdx.x;                               // block -> (chunk, tile, group), group fastest (as k_sweep_zm)
    const int ntile = p.ntx * p.nty;
    const int grp = b % p.NG; b /= p.NG;
    const int zc = b / ntile; b -= zc * ntile;
    const int blk = zc * ntile + b;
    const int TXI = b % p.ntx, TYI = b / p.ntx;
    const int X0 = TXI * 8, Y0 = TYI * 8;
    const int sample = blockIdx.y;
    const int L = p.L, Lh = L >> 1, ZC = p.ZC, z0 = zc * ZC;
    constexpr int NW = Gm::WARPS_I + Gm::WARPS_R;

    if (tid == 0) {
        for (int s = 0; s < NSO; ++s) { mbar_init(full_o(s), 1); mbar_init(empty_o(s), NW); }
        for (int s = 0; s < NJ; ++s) { mbar_init(full_j(s), 1); mbar_init(empty_j(s), NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const size_t grp_off = ((size_t)(sample * p.NG + grp) * p.N) * SITE_FLOATS;
    const float* const src_grp = p.src + grp_off;
    float* const dst_grp = p.dst + grp_off;
    auto wrapz = [&](int z) { return (z < 0) ? z + L : ((z >= L) ? z - L : z); };

    // ---------------- producer duty (first ring warp, at the start of every step) ----------------
    const int lane = tid & 31;
    const uint64_t pol_last = policy_evict_last();
    const float* const c1 = src_grp + (size_t)p.Nh * SITE_FLOATS;          // old colour-1 sites
    const size_t tile_lin = (size_t)TYI * p.ntx + TXI;
    const unsigned char* const Jt0 = reinterpret_cast<const unsigned char*>(p.Jt) + (((size_t)(sample * 2 + 0) * ntile + tile_lin) * L) * Gm::JA;
    const unsigned char* const Jt1 = reinterpret_cast<const unsigned char*>(p.Jt) + (((size_t)(sample * 2 + 1) * ntile + tile_lin) * L) * Gm::JB;
    const unsigned char* const Jr0 = reinterpret_cast<const unsigned char*>(p.Jr) + (((size_t)sample * ntile + tile_lin) * L) * Gm::JR;
    // old colour-1 plane m of the chunk (x3 = z0 - 2 + m) into stage m % NSO: one row of the diamond per lane
    auto load_o = [&](int m) {
        const int st = m % NSO;
        if (m >= NSO) mbar_wait(empty_o(st), ((m / NSO) - 1) & 1);
        if (lane == 0) mbar_expect_tx(full_o(st), Gm::OLOADED);
        __syncwarp();
        const int z = wrapz(z0 - 2 + m);
        if (lane < Gm::OROWS) {
            const int yy = lane - 2;
            int y = Y0 + yy; y = (y < 0) ? y + L : ((y >= L) ? y - L : y);
            // slots [sa, sb] of the row hold colour-1 sites: h = X0/2 - 1 + slot (periodic)
            int sa, sb;
            if (yy >= 0 && yy < 8) { sa = 0; sb = 5; }
            else if (yy == -1 || yy == 8) { sa = ((yy + z) & 1) ? 1 : 0; sb = sa + 4; }
            else { sa = 1; sb = 4; }
            const size_t rowh = (size_t)Lh * (y + (size_t)L * z);
            const uint32_t dst = smem_u32(oring + (size_t)st * Gm::OSTAGE) + lane * Gm::OROW * Gm::SITE_BYTES;
            const int hb = (X0 >> 1) - 1;
            if (sa == 0 && X0 == 0) {                                       // the first site wraps
                bulk_g2s_hint(dst, c1 + (rowh + (Lh - 1)) * SITE_FLOATS, Gm::SITE_BYTES, full_o(st), pol_last);
                sa = 1;
            }
            if (sb == 5 && X0 + 8 == L) {                                   // the last site wraps
                bulk_g2s_hint(dst + 5 * Gm::SITE_BYTES, c1 + rowh * SITE_FLOATS, Gm::SITE_BYTES, full_o(st), pol_last);
                sb = 4;
            }
            bulk_g2s_hint(dst + sa * Gm::SITE_BYTES, c1 + (rowh + (hb + sa)) * SITE_FLOATS, (sb - sa + 1) * Gm::SITE_BYTES, full_o(st), pol_last);
        }
    };
    // couplings of step n: colour 0 of plane pz (tile, ring), colour 1 of plane pz - 1
    auto load_j = [&](int n) {
        const int st = n % NJ;
        if (n >= NJ) mbar_wait(empty_j(st), ((n / NJ) - 1) & 1);
        if (lane == 0) {
            const int pz = wrapz(z0 - 1 + n), pzm = wrapz(z0 - 2 + n);
            const uint32_t dst = smem_u32(jring + (size_t)st * Gm::JSTAGE);
            mbar_expect_tx(full_j(st), Gm::JSTAGE);
            bulk_g2s_hint(dst, Jt0 + (size_t)pz * Gm::JA, Gm::JA, full_j(st), pol_last);
            bulk_g2s_hint(dst + Gm::JA, Jr0 + (size_t)pz * Gm::JR, Gm::JR, full_j(st), pol_last);
            bulk_g2s_hint(dst + Gm::JA + Gm::JR, Jt1 + (size_t)pzm * Gm::JB, Gm::JB, full_j(st), pol_last);
        }
        __syncwarp();
    };
    const bool duty = (tid >> 5) == Gm::WARPS_I;
    if (duty) {
        for (int m = 0; m < NSO; ++m) load_o(m);
        for (int n = 0; n < NJ - 1; ++n) load_j(n);
    }

    const int q = tid & 7;
    const int warp = tid >> 5;
    const bool interior = warp < Gm::WARPS_I;
    auto Ooff = [&](int xx, int yy) { return (uint32_t)(((yy + 2) * Gm::OROW + ((xx + 2) >> 1)) * Gm::SITE_BYTES + q * 16); };
    auto Noff = [&](int xx, int yy) { return (uint32_t)(((yy + 1) * Gm::NROW + ((xx + 1) >> 1)) * Gm::SITE_BYTES + q * 16); };
    // position of the colour-c site (x, y, z) in a group's array, in floats
    auto gpos = [&](int c, int x, int y, int z) { return ((size_t)c * p.Nh + (size_t)(x >> 1) + (size_t)Lh * (y + (size_t)L * z)) * SITE_FLOATS + q * 4; };

    // per parity d = n & 1 of the step: local coordinates of this thread's column and the offsets derived from them
    int cxx[2], cyy[2], gx[2], gy[2];
    uint32_t oA[2][5];          // old colour 1 in the stage of plane pz: +x1, -x1, +x2, -x2; [4]: the column itself (planes pz +- 1)
    uint32_t nW[2];             // new colour 0 of the column in the stage of plane pz
    uint32_t nB[2][4];          // interior: new colour 0 around the column in the stage of plane pz - 1: +x1, -x1, +x2, -x2
    uint32_t jA, jB = 0;        // coupling blocks inside a coupling stage
    if (interior) {
        const int ks = tid >> 3, ky = ks >> 2, kx = ks & 3;
        jA = ks * Gm::JSITE; jB = Gm::JA + Gm::JR + ks * Gm::JSITE;
#pragma unroll
        for (int d = 0; d < 2; ++d) { cxx[d] = 2 * kx + ((ky + d + 1) & 1); cyy[d] = ky; }
    } else {
        const int rs = (tid - Gm::WARPS_I * 32) >> 3;
        jA = Gm::JA + rs * Gm::JSITE;
#pragma unroll
        for (int d = 0; d < 2; ++d) fz_ring_site(rs, (d + 1) & 1, cxx[d], cyy[d]);      // parity of pz = z0 - 1 + n is that of n + 1
    }
#pragma unroll
    for (int d = 0; d < 2; ++d) {
        const int xx = cxx[d], yy = cyy[d];
        oA[d][0] = Ooff(xx + 1, yy); oA[d][1] = Ooff(xx - 1, yy); oA[d][2] = Ooff(xx, yy + 1); oA[d][3] = Ooff(xx, yy - 1);
        oA[d][4] = Ooff(xx, yy);
        nW[d] = Noff(xx, yy);
        nB[d][0] = Noff(xx + 1, yy); nB[d][1] = Noff(xx - 1, yy); nB[d][2] = Noff(xx, yy + 1); nB[d][3] = Noff(xx, yy - 1);
        int x = X0 + xx, y = Y0 + yy;
        gx[d] = (x < 0) ? x + L : ((x >= L) ? x - L : x);
        gy[d] = (y < 0) ? y + L : ((y >= L) ? y - L : y);
    }

    float M[2][3][4], P0[2][3][4];
    float eacc[4] = { 0.f, 0.f, 0.f, 0.f };
    // prologue: M of steps 0 and 1 = old colour 1 of the column in planes z0 - 2 and z0 - 1 (stages 0 and 1)
    mbar_wait(full_o(0), 0);
    mbar_wait(full_o(1 % NSO), 0);
    fz_lds_spin(oring + 0 * Gm::OSTAGE + oA[0][4], M[0]);
    fz_lds_spin(oring + (size_t)(1 % NSO) * Gm::OSTAGE + oA[1][4], M[1]);
#pragma unroll
    for (int d = 0; d < 2; ++d)
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int j = 0; j < 4; ++j) P0[d][a][j] = 0.f;
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(empty_o(0));          // plane z0 - 2 serves nothing else

    float own[2][3][4];         // old colour 0 of the column in plane pz, fetched two steps ahead
    fz_ldg_spin(src_grp + gpos(0, gx[0], gy[0], wrapz(z0 - 1)), own[0]);
    fz_ldg_spin(src_grp + gpos(0, gx[1], gy[1], wrapz(z0)), own[1]);

    for (int n2 = 0; n2 < ZC + 2; n2 += 2) {
#pragma unroll
        for (int d = 0; d < 2; ++d) {
            const int n = n2 + d;
            const int pz = wrapz(z0 - 1 + n);
            const int so_cur = (n + 1) % NSO, so_up = (n + 2) % NSO, sj = n % NJ, sn = n % NSN;
            if (duty) {                   // the planes and couplings of the steps to come, into the stages the last steps freed
                if (n + NSO < ZC + 4) load_o(n + NSO);
                if (n + NJ - 1 < ZC + 2) load_j(n + NJ - 1);
            }
            mbar_wait(full_o(so_up), ((n + 2) / NSO) & 1);
            mbar_wait(full_j(sj), (n / NJ) & 1);
            const unsigned char* const Oc = oring + (size_t)so_cur * Gm::OSTAGE;
            const unsigned char* const Ou = oring + (size_t)so_up * Gm::OSTAGE;
            const unsigned char* const Jst = jring + (size_t)sj * Gm::JSTAGE;

            // ---- A(n): colour 0 of plane pz ----
            float J[JG], hf[3][4], nb[3][4], U[3][4], s0[3][4];
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 4; ++j) { hf[a][j] = 0.f; s0[a][j] = own[d][a][j]; }
            // the own spin of step n + 2 (same column): two steps ahead of its use
            fz_ldg_spin(src_grp + gpos(0, gx[d], gy[d], wrapz(wrapz(z0 + 1 + n))), own[d]);
            fz_lds_J(Jst + jA, J);
#pragma unroll
            for (int k = 0; k < 4; ++k) { fz_lds_spin(Oc + oA[d][k], nb); fz_acc(J, k, nb, hf); }
            fz_lds_spin(Ou + oA[d][4], U);
            fz_acc(J, 4, U, hf);
            fz_acc(J, 5, M[d], hf);
            fz_or4(hf, s0);
            fz_sts_spin(nring + (size_t)sn * Gm::NSTAGE + nW[d], s0);
            if (interior && n >= 1 && n <= ZC) fz_stg_spin(dst_grp + gpos(0, gx[d], gy[d], pz), s0);
            __syncwarp();
            if ((tid & 31) == 0) {
                mbar_arrive(empty_o(so_cur));                         // plane pz: its in-plane use was the last one
                if (!interior) mbar_arrive(empty_j(sj));
            }
            asm volatile("bar.sync 1, %0;" ::"r"(Gm::CONSUMERS) : "memory");    // every new colour-0 value of plane pz is in place

            // ---- B(n): colour 1 of plane pz - 1 (interior warps) ----
            if (interior) {
                if (n >= 2) {
                    const unsigned char* const Nm = nring + (size_t)((n - 1) % NSN) * Gm::NSTAGE;
                    float s1[3][4];
#pragma unroll
                    for (int a = 0; a < 3; ++a)
#pragma unroll
                        for (int j = 0; j < 4; ++j) { hf[a][j] = 0.f; s1[a][j] = M[d][a][j]; }
                    fz_lds_J(Jst + jB, J);
#pragma unroll
                    for (int k = 0; k < 4; ++k) { fz_lds_spin(Nm + nB[d][k], nb); fz_acc(J, k, nb, hf); }
                    fz_acc(J, 4, s0, hf);
                    fz_acc(J, 5, P0[d], hf);
                    fz_or4(hf, s1);
                    if (WITH_E) {
#pragma unroll
                        for (int j = 0; j < 4; ++j) eacc[j] += fmaf(hf[0][j], s1[0][j], fmaf(hf[1][j], s1[1][j], hf[2][j] * s1[2][j]));
                    }
                    fz_stg_spin(dst_grp + gpos(1, gx[d], gy[d], wrapz(z0 - 2 + n)), s1);
                }
                __syncwarp();
                if ((tid & 31) == 0) mbar_arrive(empty_j(sj));
            }
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 4; ++j) { M[d][a][j] = U[a][j]; P0[d][a][j] = s0[a][j]; }
        }
    }

    if (WITH_E) {
        // per-copy sum over the CTA's colour-1 sites (E = -sum over one colour of s.h): fixed order, fp64 across threads
        asm volatile("bar.sync 1, %0;" ::"r"(Gm::CONSUMERS) : "memory");
        double* red = reinterpret_cast<double*>(oring);        // [32][G+1]; the rings are dead
        if (interior) {
            const int ks = tid >> 3;
#pragma unroll
            for (int j = 0; j < 4; ++j) red[ks * (G + 1) + q * 4 + j] = (double)eacc[j];
        }
        asm volatile("bar.sync 1, %0;" ::"r"(Gm::CONSUMERS) : "memory");
        if (tid < G) {
            double acc = 0.0;
            for (int r = 0; r < 32; ++r) acc += red[r * (G + 1) + tid];
            const int nblk = ntile * p.nzc;
            p.Epart[((size_t)(sample * p.NG + grp) * nblk + blk) * G + tid] = acc;
        }
    }
}

}  // namespace sg
