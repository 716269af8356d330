// sg_sweep_zm.cuh -- the z-marching half-sweep kernel (S1, S2, S3) of libsg_b200 for L a multiple of 8.
//
// Why.  A half-sweep is HBM-bound at 36 + 216/C bytes per update, but only if every
// spin is fetched from L2 about once: the first kernel (k_sweep, sg_kernels.cuh) pulled 78 B per update
// through the L2 -> SM crossbar, which saturates near 6300 B/clk on this chip, before HBM does.  Here a CTA
// owns a TX x TY column of one copy group and marches along x3.  Per plane it needs the 32-copy lines of
//   * the TX*TY/2 sites it updates (read once, by the updating thread, prefetched into registers), and
//   * the other-colour sites of that plane, tile plus a one-site halo (TX*TY/2 + TX + TY lines),
// and every other-colour plane serves three consecutive steps (as the x3+1 neighbours, the in-plane
// neighbours, the x3-1 neighbours).  A producer warp streams those planes, and the per-site coupling
// blocks, into a shared-memory ring with bulk asynchronous copies (cp.async.bulk -> UBLKCP) that complete
// on mbarriers; the consumer warps read neighbours and couplings from shared memory only.
// L2 -> SM traffic: 12 (own) + 12 (TX*TY/2+TX+TY)/(TX*TY/2) (other) + 7 (couplings) + 12 (write) = 49 B
// per update for 8 x 8 columns.
#pragma once
#include "sg_device.cuh"

namespace sg {

enum : int { KIND_OR = 0, KIND_HB = 1, KIND_ENERGY = 2 };

// ---- mbarrier / bulk-copy primitives (PTX; sm_90+) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ float4 lds4(const unsigned char* p) { return *reinterpret_cast<const float4*>(p); }

// L2 eviction policy for the bulk copies: other-colour planes and coupling blocks are re-read within microseconds (by the
// neighbour tiles' halos, by the other copy groups of the tile), the own-colour stream is not: evict_last on the former
// measured -0.9 % on the OR half-sweep at cfg 4 (616.2 -> 610.8 us); evict_first on the own loads / stores changed nothing.
__device__ __forceinline__ uint64_t policy_evict_last()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// global -> shared bulk copy of `bytes` (multiple of 16, 16-byte aligned both sides) with an L2 policy, completing on `bar`
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol)
                 : "memory");
}

// Geometry of one ring stage: the other-colour sites of a plane, tile + halo.
//   interior row yy (0..TY-1): ROW = TX/2+1 slots, slot = yy*ROW + ((xx+1)>>1), xx in [-1, TX]
//   halo rows yy = -1, TY     : TX/2 slots each, slot = TY*ROW + (yy<0 ? 0 : TX/2) + (xx>>1)
template <int TX, int TY>
struct ZmGeom {
    static constexpr int ROW = TX / 2 + 1;
    static constexpr int SLOTS = TY * ROW + TX;
    static constexpr int OWN = TX * TY / 2;
    static constexpr int SITE_BYTES = SITE_FLOATS * 4;            // 384
    static constexpr int STAGE_BYTES = SLOTS * SITE_BYTES;        // 18432 for 8 x 8
    static constexpr int JSITE_BYTES = JG * 4;                    // 224
    static constexpr int JSTAGE_BYTES = OWN * JSITE_BYTES;        // 7168 for 8 x 8
    static constexpr int PJSITE_BYTES = 8;                        // packed bimodal couplings: 6 link bytes + 2 pad
    static constexpr int PJSTAGE_BYTES = OWN * PJSITE_BYTES;      // 256 for 8 x 8
    static constexpr int CONSUMERS = OWN * 8;                     // threads: (site, copy quad)
    static constexpr int THREADS = CONSUMERS + 32;                // + one producer warp
    static constexpr int NWARPS_C = CONSUMERS / 32;
};

template <int TX, int TY, int NST, int NJ>
constexpr size_t zm_smem_bytes()
{
    return (size_t)NST * ZmGeom<TX, TY>::STAGE_BYTES + (size_t)NJ * ZmGeom<TX, TY>::JSTAGE_BYTES + 8 * (2 * NST + 2 * NJ) + 128;
}

struct ZmParams {
    float* spins;            // [S][NG][2][Nh][3][G]
    const float* Jt;         // [S][2][L/TY][L/TX][L][TY][TX/2][JG]
    const unsigned char* Jp; // [S][2][L/TY][L/TX][L][TY][TX/2][8]: packed bimodal couplings (PACKED kernels only)
    float bimA, bimB, bimD;  // fl32(1 + D), fl32(1 - D), fl32(D) of the packed couplings
    const float* beta_slot;  // [S][Cp]
    double* Epart;           // [S][NG][nblk][G]
    int L, N, Nh, NG, C, Cg; // Cg: copies per sample of the whole job (stride of the global copy id)
    int Tl, Tpad;            // slots per replica held here, n_temps_total - Tl (copy_gid)
    int ntx, nty, nzc, ZC;   // tiles along x1, x2; chunks along x3 of ZC planes each
    int colour;
    uint32_t key0, key1, hb_counter, g_first;
};

// the single-site update of 4 copies held by one thread (shared by the update kinds)
template <int KIND, bool WITH_E>
__device__ __forceinline__ void zm_update(const float (&hf)[3][4], float (&s)[3][4], float (&eacc)[4], const float4& beta4,
                                          uint32_t i, const uint32_t (&gid)[4], const ZmParams& p)
{
    if (KIND == KIND_OR) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            or_update(hf[0][j], hf[1][j], hf[2][j], s[0][j], s[1][j], s[2][j]);
            // s.h of the STORED spin (equal to the old s.h only in exact arithmetic), so that E is the energy of the stored state
            if (WITH_E) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
        }
    } else if (KIND == KIND_HB) {
        const float bt[4] = { beta4.x, beta4.y, beta4.z, beta4.w };
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t w[4];
            philox4x32_10(i, gid[j], p.hb_counter, STREAM_HB, p.key0, p.key1, w);
            hb_update(hf[0][j], hf[1][j], hf[2][j], bt[j], uniform23(w[0]), uniform23(w[1]), s[0][j], s[1][j], s[2][j]);
            if (WITH_E) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
        }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) eacc[j] += fmaf(hf[0][j], s[0][j], fmaf(hf[1][j], s[1][j], hf[2][j] * s[2][j]));
    }
}

// The paper's bimodal coupling from its byte: bit 0 the sign of J = +-1 (1: +), bits 1-3 the
// signs of D^00, D^11, D^22, bits 4-6 those of D^01, D^02, D^12 (1: +D); M = J 1 + D, D symmetric.  The nine fp32
// values are those of the unpacked array (fl32(J + d) = +-A or +-B), so the field FMAs see identical operands.
__device__ __forceinline__ void bimodal_decode(uint32_t b, float A, float B, float D, float* __restrict__ m)
{
    const uint32_t jb = b & 1u;
    const uint32_t sj = (jb ^ 1u) << 31;
    float dg[3], of[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const uint32_t db = (b >> (1 + a)) & 1u;
        dg[a] = __uint_as_float(__float_as_uint(db == jb ? A : B) ^ sj);      // J + d = J (1 + d/J)
        of[a] = __uint_as_float(__float_as_uint(D) ^ ((((b >> (4 + a)) & 1u) ^ 1u) << 31));
    }
    m[0] = dg[0]; m[1] = of[0]; m[2] = of[1];
    m[3] = of[0]; m[4] = dg[1]; m[5] = of[2];
    m[6] = of[1]; m[7] = of[2]; m[8] = dg[2];
}

template <int KIND, bool WITH_E, int TX, int TY, int NST, int NJ, bool PACKED = false>
__global__ void __launch_bounds__(ZmGeom<TX, TY>::THREADS, 2) k_sweep_zm(const ZmParams p)
{
    using Gm = ZmGeom<TX, TY>;
    constexpr int JST = Gm::JSTAGE_BYTES;                                  // bytes of one coupling stage in shared memory
    static_assert(!PACKED || Gm::OWN == 32, "the packed path decodes one site per producer lane");
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* const ring = smem;                                       // NST stages of other-colour planes
    unsigned char* const jring = smem + (size_t)NST * Gm::STAGE_BYTES;      // NJ stages of coupling blocks
    const uint32_t bars = smem_u32(jring + (size_t)NJ * JST);  // full_o[NST] empty_o[NST] full_j[NJ] empty_j[NJ]
    auto full_o = [&](int s) { return bars + 8u * s; };
    auto empty_o = [&](int s) { return bars + 8u * (NST + s); };
    auto full_j = [&](int s) { return bars + 8u * (2 * NST + s); };
    auto empty_j = [&](int s) { return bars + 8u * (2 * NST + NJ + s); };

    const int tid = threadIdx.x;
    // block -> (chunk, tile, group).  The group is fastest so that the CTAs that share a tile's couplings run next to each
    // other in time (one DRAM read of the couplings per tile, not per group); the chunk is slowest, so that the ~296 CTAs
    // in flight cover ~6 whole rows of neighbouring tiles in the SAME range of planes and find each other's x1 / x2 halo
    // lines in L2 (tile-outer, chunk-inner order: 3 rows of tiles per range; measured 610 -> 593 us at cfg 4).
    int b = blockIdx.x;
    const int ntile_ = p.ntx * p.nty;
    const int grp = b % p.NG; b /= p.NG;
    const int zc = b / ntile_; b -= zc * ntile_;
    const int blk_ = zc * ntile_ + b;
    const int X0 = (b % p.ntx) * TX, Y0 = (b / p.ntx) * TY;
    const int sample = blockIdx.y;
    const int L = p.L, z0 = zc * p.ZC, ZC = p.ZC;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(full_o(s), 1); mbar_init(empty_o(s), Gm::NWARPS_C); }
        for (int s = 0; s < NJ; ++s) { mbar_init(full_j(s), 1); mbar_init(empty_j(s), Gm::NWARPS_C); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const float* const spins_grp = p.spins + ((size_t)(sample * p.NG + grp) * p.N) * SITE_FLOATS;
    const int Lh = L >> 1;

    if (tid >= Gm::CONSUMERS) {
        // ---------------- producer warp ----------------
        // Other-colour sites of a lattice row are contiguous in HBM (colour-split site order), so a plane is
        // TY row segments of ROW sites (split in two where the x1 halo wraps), two halo rows of TX/2 sites,
        // and the couplings of a plane are one block of the tile-major array: 11 to 19 bulk copies per step.
        const int lane = tid - Gm::CONSUMERS;
        const uint64_t pol_last = policy_evict_last();
        const float* const other = spins_grp + (size_t)(1 - p.colour) * p.Nh * SITE_FLOATS;
        const size_t tile_first = (((size_t)(sample * 2 + p.colour) * p.nty + Y0 / TY) * p.ntx + X0 / TX) * L;   // in plane blocks
        const unsigned char* const Jtile = reinterpret_cast<const unsigned char*>(p.Jt) + tile_first * JST;
        // packed bimodal couplings: lane = site of the plane, 8 bytes per site read straight from global memory one step
        // ahead and decoded by this (otherwise idle) warp into the fp32 blocks the consumers read
        const uint2* const Ptile = reinterpret_cast<const uint2*>(p.Jp + tile_first * Gm::PJSTAGE_BYTES) + lane;
        uint2 pk_next = make_uint2(0u, 0u);
        if constexpr (PACKED) pk_next = __ldg(Ptile + (size_t)z0 * Gm::OWN);
        for (int n = 0; n < ZC + 2; ++n) {
            // other-colour plane n of the chunk: x3 = z0 - 1 + n (periodic)
            {
                const int st = n % NST;
                if (n >= NST) mbar_wait(empty_o(st), ((n / NST) - 1) & 1);
                if (lane == 0) mbar_expect_tx(full_o(st), Gm::STAGE_BYTES);
                __syncwarp();
                int z = z0 - 1 + n;
                z = (z < 0) ? z + L : ((z >= L) ? z - L : z);
                const uint32_t dst0 = smem_u32(ring + (size_t)st * Gm::STAGE_BYTES);
                if (lane < TY) {
                    const int yy = lane;
                    const int e = (yy + z + p.colour) & 1;          // first other-colour x1 of the row: X0 - 1 + e
                    const size_t rowh = (size_t)Lh * (Y0 + yy + (size_t)L * z);
                    const uint32_t dst = dst0 + yy * Gm::ROW * Gm::SITE_BYTES;
                    if (e == 0) {
                        // sites X0-1, X0+1, .., X0+TX-1: the first one wraps for the leftmost tile
                        if (X0 == 0) {
                            bulk_g2s_hint(dst, other + (rowh + (Lh - 1)) * SITE_FLOATS, Gm::SITE_BYTES, full_o(st), pol_last);
                            bulk_g2s_hint(dst + Gm::SITE_BYTES, other + (rowh + 0) * SITE_FLOATS, (Gm::ROW - 1) * Gm::SITE_BYTES, full_o(st), pol_last);
                        } else {
                            bulk_g2s_hint(dst, other + (rowh + ((X0 - 1) >> 1)) * SITE_FLOATS, Gm::ROW * Gm::SITE_BYTES, full_o(st), pol_last);
                        }
                    } else {
                        // sites X0, X0+2, .., X0+TX: the last one wraps for the rightmost tile
                        if (X0 + TX == L) {
                            bulk_g2s_hint(dst, other + (rowh + (X0 >> 1)) * SITE_FLOATS, (Gm::ROW - 1) * Gm::SITE_BYTES, full_o(st), pol_last);
                            bulk_g2s_hint(dst + (Gm::ROW - 1) * Gm::SITE_BYTES, other + rowh * SITE_FLOATS, Gm::SITE_BYTES, full_o(st), pol_last);
                        } else {
                            bulk_g2s_hint(dst, other + (rowh + (X0 >> 1)) * SITE_FLOATS, Gm::ROW * Gm::SITE_BYTES, full_o(st), pol_last);
                        }
                    }
                } else if (lane < TY + 2) {
                    // halo rows x2 = Y0-1 and Y0+TY (periodic): TX/2 sites X0 + e, X0 + e + 2, ..
                    const int up = lane - TY;
                    int y = up ? Y0 + TY : Y0 - 1;
                    y = (y < 0) ? y + L : ((y >= L) ? y - L : y);
                    const size_t rowh = (size_t)Lh * (y + (size_t)L * z);
                    bulk_g2s_hint(dst0 + (TY * Gm::ROW + up * (TX / 2)) * Gm::SITE_BYTES, other + (rowh + (X0 >> 1)) * SITE_FLOATS,
                             (TX / 2) * Gm::SITE_BYTES, full_o(st), pol_last);
                }
            }
            // coupling blocks of step k = n - 2: one contiguous block of the tile-major array
            const int k = n - 2;
            if (k >= 0) {
                const int st = k % NJ;
                if constexpr (PACKED) {
                    const uint2 pk = pk_next;
                    if (k + 1 < ZC) pk_next = __ldg(Ptile + (size_t)(z0 + k + 1) * Gm::OWN);
                    float J[JG];
#pragma unroll
                    for (int nbk = 0; nbk < 6; ++nbk)     // bytes 0-3: +x1, -x1, +x2, -x2; 4-5: +x3, -x3
                        bimodal_decode(((nbk < 4) ? (pk.x >> (8 * nbk)) : (pk.y >> (8 * (nbk - 4)))) & 0x7fu, p.bimA, p.bimB, p.bimD, &J[9 * nbk]);
                    J[54] = 0.f; J[55] = 0.f;
                    if (k >= NJ) mbar_wait(empty_j(st), ((k / NJ) - 1) & 1);
                    float* const dstJ = reinterpret_cast<float*>(jring + (size_t)st * JST) + lane * JG;
#pragma unroll
                    for (int v = 0; v < JG / 4; ++v) st4(dstJ + 4 * v, make_float4(J[4 * v], J[4 * v + 1], J[4 * v + 2], J[4 * v + 3]));
                    __syncwarp();
                    if (lane == 0) mbar_arrive(full_j(st));
                } else {
                    if (k >= NJ) mbar_wait(empty_j(st), ((k / NJ) - 1) & 1);
                    if (lane == 0) {
                        mbar_expect_tx(full_j(st), JST);
                        bulk_g2s_hint(smem_u32(jring + (size_t)st * JST), Jtile + (size_t)(z0 + k) * JST, JST, full_j(st), pol_last);
                    }
                    __syncwarp();
                }
            }
        }
        return;
    }

    // ---------------- consumer warps: thread = (own-colour site of the plane, copy quad) ----------------
    const int q = tid & 7, ks = tid >> 3;
    const int ky = ks / (TX / 2), kx = ks - ky * (TX / 2);
    const int Y = Y0 + ky;
    float4 beta4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (KIND == KIND_HB) beta4 = ldg4(p.beta_slot + (size_t)sample * p.NG * G + grp * G + q * 4);
    uint32_t gid[4] = { 0u, 0u, 0u, 0u };             // global ids of this thread's four copies (heat bath only)
    if (KIND == KIND_HB) {
#pragma unroll
        for (int j = 0; j < 4; ++j) gid[j] = copy_gid(p.g_first + (uint32_t)sample * (uint32_t)p.Cg, grp * G + q * 4 + j, p.Tl, p.Tpad);
    }
    float eacc[4] = { 0.f, 0.f, 0.f, 0.f };

    // Own spin of step k: site (X0 + 2 kx + off, Y, z0 + k), off = (ky + z + colour) & 1.  In the colour-split
    // order its position is (X0/2 + kx) + (L/2)(Y + L z) whatever off is: a constant stride per plane.
    const size_t plane = (size_t)Lh * L * SITE_FLOATS;
    float* own = const_cast<float*>(spins_grp) +
                 ((size_t)p.colour * p.Nh + (size_t)(X0 >> 1) + kx + (size_t)Lh * (Y + (size_t)L * z0)) * SITE_FLOATS + q * 4;
    float4 pre[2][3];   // register prefetch of the own spins, two steps deep
#pragma unroll
    for (int d = 0; d < 2; ++d)
#pragma unroll
        for (int a = 0; a < 3; ++a) pre[d][a] = (d < ZC) ? ld4(own + d * plane + a * G) : make_float4(0.f, 0.f, 0.f, 0.f);

    // Byte offsets of the six neighbours inside a stage, for even and odd steps (z0 and ZC are even, so the
    // parity of the step is the parity of x3 - z0): +x1, -x1, +x2, -x2 in the plane's own stage, x3 +- 1 in
    // the next / previous stage at the slot of (x1, x2).
    uint32_t o_xm[2], o_yp[2], o_ym[2], o_z[2];
#pragma unroll
    for (int d = 0; d < 2; ++d) {
        const int off = (ky + z0 + d + p.colour) & 1;
        o_xm[d] = (uint32_t)((ky * Gm::ROW + kx) * Gm::SITE_BYTES + q * 16);
        o_z[d] = (uint32_t)((ky * Gm::ROW + kx + off) * Gm::SITE_BYTES + q * 16);
        o_ym[d] = (uint32_t)(((ky > 0) ? (ky - 1) * Gm::ROW + kx + off : TY * Gm::ROW + kx) * Gm::SITE_BYTES + q * 16);
        o_yp[d] = (uint32_t)(((ky < TY - 1) ? (ky + 1) * Gm::ROW + kx + off : TY * Gm::ROW + TX / 2 + kx) * Gm::SITE_BYTES + q * 16);
    }
    const uint32_t i0 = (uint32_t)(X0 + 2 * kx + L * (Y + L * z0));   // site index of step k: i0 + off + L^2 k (heat bath only)

    mbar_wait(full_o(0 % NST), 0);
    mbar_wait(full_o(1 % NST), 0);
    // rotating stage indices and phase parities: planes k (x3-1), k+1 (in-plane), k+2 (x3+1); coupling stage of step k
    int sm_ = 0, s0_ = 1 % NST, sp_ = 2 % NST, sj_ = 0;
    uint32_t par_p = (2 / NST) & 1, par_j = 0;

    for (int k2 = 0; k2 < ZC; k2 += 2) {
#pragma unroll
        for (int d = 0; d < 2; ++d) {
            const int k = k2 + d;      // ZC is even (sg_tune / zm_plan), so k < ZC for both steps of the pair
            float s[3][4];
            mbar_wait(full_o(sp_), par_p);
            mbar_wait(full_j(sj_), par_j);
            const unsigned char* const Pm = ring + sm_ * Gm::STAGE_BYTES;
            const unsigned char* const P0 = ring + s0_ * Gm::STAGE_BYTES;
            const unsigned char* const Pp = ring + sp_ * Gm::STAGE_BYTES;
            const unsigned char* nbp[6] = { P0 + o_xm[d] + Gm::SITE_BYTES, P0 + o_xm[d], P0 + o_yp[d], P0 + o_ym[d],
                                            Pp + o_z[d], Pm + o_z[d] };
            const unsigned char* const Jp = jring + sj_ * JST + ks * Gm::JSITE_BYTES;

            float hf[3][4];
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 4; ++j) hf[a][j] = 0.f;
            float J[JG];
#pragma unroll
            for (int v = 0; v < JG / 4; ++v) {
                const float4 t4 = lds4(Jp + 16 * v);
                J[4 * v] = t4.x; J[4 * v + 1] = t4.y; J[4 * v + 2] = t4.z; J[4 * v + 3] = t4.w;
            }
#pragma unroll
            for (int nbk = 0; nbk < 6; ++nbk) {
                float n[3][4];
#pragma unroll
                for (int bb = 0; bb < 3; ++bb) {
                    const float4 t4 = lds4(nbp[nbk] + bb * (G * 4));
                    n[bb][0] = t4.x; n[bb][1] = t4.y; n[bb][2] = t4.z; n[bb][3] = t4.w;
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int bb = 0; bb < 3; ++bb) fma4(J[9 * nbk + 3 * a + bb], n[bb], hf[a]);
            }
            // the stage of plane k and the coupling stage are dead for this warp once the loads above retire
            __syncwarp();
            if ((tid & 31) == 0) { mbar_arrive(empty_o(sm_)); mbar_arrive(empty_j(sj_)); }
            sm_ = s0_; s0_ = sp_;
            sp_ = (sp_ + 1 == NST) ? 0 : sp_ + 1; par_p ^= (sp_ == 0) ? 1u : 0u;
            sj_ = (sj_ + 1 == NJ) ? 0 : sj_ + 1; par_j ^= (sj_ == 0) ? 1u : 0u;

            const uint32_t i = i0 + (uint32_t)((ky + z0 + d + p.colour) & 1) + (uint32_t)(L * L) * (uint32_t)k;
            // the own spin is needed only now (s.h and the reflection): take it from the prefetch registers ...
#pragma unroll
            for (int a = 0; a < 3; ++a) { s[a][0] = pre[d][a].x; s[a][1] = pre[d][a].y; s[a][2] = pre[d][a].z; s[a][3] = pre[d][a].w; }
            zm_update<KIND, WITH_E>(hf, s, eacc, beta4, i, gid, p);
            if (KIND != KIND_ENERGY) {
#pragma unroll
                for (int a = 0; a < 3; ++a) st4(own + a * G, make_float4(s[a][0], s[a][1], s[a][2], s[a][3]));
            }
            // ... and refill them for step k + 2 once they are dead: still two field computations ahead of the next use.
            // Unconditional (a predicated load would force copies of the old values): past the end of the chunk it re-reads
            // the plane just written, an L2 hit whose value is never used.
            {
                const float* const nxt = own + ((k + 2 < ZC) ? 2 * plane : 0);
#pragma unroll
                for (int a = 0; a < 3; ++a) pre[d][a] = ld4(nxt + a * G);
            }
            own += plane;
        }
    }

    if (WITH_E || KIND == KIND_ENERGY) {
        // per-copy sum over the CTA's sites: fixed order, fp64 across threads (no float atomics).
        // The ring is dead by now for every consumer warp (all full barriers were waited, all reads retired
        // before the named barrier below), so its first bytes serve as the reduction scratch.
        asm volatile("bar.sync 1, %0;" ::"r"(Gm::CONSUMERS) : "memory");
        double* red = reinterpret_cast<double*>(ring);   // [OWN][G+1]
#pragma unroll
        for (int j = 0; j < 4; ++j) red[ks * (G + 1) + q * 4 + j] = (double)eacc[j];
        asm volatile("bar.sync 1, %0;" ::"r"(Gm::CONSUMERS) : "memory");
        if (tid < G) {
            double acc = 0.0;
            for (int r = 0; r < Gm::OWN; ++r) acc += red[r * (G + 1) + tid];
            const int nblk = p.ntx * p.nty * p.nzc;
            const int blk = blk_;
            p.Epart[((size_t)(sample * p.NG + grp) * nblk + blk) * G + tid] = acc;
        }
    }
}

}  // namespace sg
