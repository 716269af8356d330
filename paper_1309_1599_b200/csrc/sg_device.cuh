// sg_device.cuh -- device-side building blocks of libsg_b200: Philox4x32-10, the single-spin updates
// (Eq. (A1), (A2) of arXiv:1309.1599) and the private HBM layout.
// Shares no code with oracle/ (the fp64 CPU oracle); see DESIGN.md sections 3, 9, 10.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sg {

// ------------------------------------------------------------------------------------------------
// HBM layout (private)
//   spins  float [S][NG][2][N/2][3][G]  G = 32 consecutive copy ids: one aligned 128-byte line per
//                                   (site, component, group); a site of a group is 384 contiguous bytes.
//                                   Sites are split by colour, then ordered by h = i>>1, so that the
//                                   same-colour sites of a lattice row (x2, x3) are L/2 contiguous
//                                   384-byte blocks: one bulk copy fetches a whole row segment.
//   Jg     float [S][2][N/2][JG]    per-site gathered couplings, by colour then h = i>>1:
//                                   A_k, k = (+x,-x,+y,-y,+z,-z), with h_x = sum_k A_k s_{nbr k}
//                                   (forward: M_{x,mu}; backward: M_{x-e_mu,mu}^T), 54 floats + 2 pad
//   Jt     float [S][2][L/8][L/8][L][8][4][JG]  (L a multiple of 8 only) the same blocks ordered by
//                                   8 x 8 column tile, plane, row, site: the couplings one CTA of the
//                                   z-marching sweep needs for one plane are 7168 contiguous bytes
// ------------------------------------------------------------------------------------------------
constexpr int G = 32;
constexpr int SITE_FLOATS = 3 * G;
constexpr int JG = 56;

enum : uint32_t { STREAM_HB = 1, STREAM_PT = 2, STREAM_SPINS = 3, STREAM_COUPLINGS = 4 };

// Philox4x32-10 (Salmon et al., SC'11); DESIGN.md section 3.1.
__host__ __device__ inline void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
#ifdef __CUDA_ARCH__
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
#else
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
#endif
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// r = ((w >> 9) + 1/2) 2^-23: exact in fp32
__device__ __forceinline__ float uniform23(uint32_t w) { return ((float)(w >> 9) + 0.5f) * (1.0f / 8388608.0f); }

// Overrelaxation, Eq. (A2): s <- 2 h (h.s)/h^2 - s; h.h < 1e-30 leaves s.
__device__ __forceinline__ void or_update(float hx, float hy, float hz, float& sx, float& sy, float& sz)
{
    const float hh = fmaf(hx, hx, fmaf(hy, hy, hz * hz));
    const float hs = fmaf(hx, sx, fmaf(hy, sy, hz * sz));
    if (hh >= 1e-30f) {
        const float f = __fdividef(2.0f * hs, hh);   // MUFU.RCP + FMUL (2 ulp): the drift it adds to |s| and to s.h is of the order of the fp32 rounding of the reflection itself
        sx = fmaf(f, hx, -sx);
        sy = fmaf(f, hy, -sy);
        sz = fmaf(f, hz, -sz);
    }
}

// Heat bath, Eq. (A1): s drawn from exp(beta s.h).  Exact inverse CDF of the polar
// cosine about n = h/|h|, evaluated hemisphere by hemisphere so that whichever of w = 1-u, w' = 1+u is
// small carries a few-ulp relative error (reading R23); uniform azimuth in the frame of
// Duff et al. (JCGT 2017).
__device__ __forceinline__ void hb_update(float hx, float hy, float hz, float beta, float r1, float r2,
                                          float& sx, float& sy, float& sz)
{
    const float hh = fmaf(hx, hx, fmaf(hy, hy, hz * hz));
    float nx = 0.0f, ny = 0.0f, nz = 1.0f, kappa = 0.0f;
    if (hh >= 1e-30f) {
        const float hn = sqrtf(hh);
        nx = hx / hn; ny = hy / hn; nz = hz / hn;
        kappa = beta * hn;
    }
    float w, wp, u;                    // w = 1 - u (from the north pole), wp = 1 + u (from the south pole)
    if (kappa < 1e-15f) {              // uniform law
        w = 2.0f * r1; wp = 2.0f - w; u = 1.0f - w;
    } else if (r1 <= 1.0f / (1.0f + expf(-kappa))) {      // u >= 0
        const float x = -r1 * expm1f(-2.0f * kappa);       // r1 (1 - e^{-2 kappa}) in [0,1)
        const float lg = (x <= 0.5f) ? log1pf(-x) : logf((1.0f - r1) + r1 * expf(-2.0f * kappa));
        w = -lg / kappa; wp = 2.0f - w; u = 1.0f - w;
    } else {                                               // u < 0; only reachable for kappa < 16.7
        wp = log1pf((1.0f - r1) * expm1f(2.0f * kappa)) / kappa; w = 2.0f - wp; u = wp - 1.0f;
    }
    const float t = sqrtf(fmaxf(w * wp, 0.0f));
    float sp, cp;
    sincospif(2.0f * r2, &sp, &cp);
    const float sg = copysignf(1.0f, nz);
    const float a = -1.0f / (sg + nz);
    const float b = nx * ny * a;
    const float e1x = 1.0f + sg * nx * nx * a, e1y = sg * b, e1z = -sg * nx;
    const float e2x = b, e2y = sg + ny * ny * a, e2z = -ny;
    sx = fmaf(u, nx, t * fmaf(cp, e1x, sp * e2x));
    sy = fmaf(u, ny, t * fmaf(cp, e1y, sp * e2y));
    sz = fmaf(u, nz, t * fmaf(cp, e1z, sp * e2z));
}

// Site coordinates of the h-th site of `colour` (h = i >> 1): x1 = 2*(h mod L/2) + ((x2+x3+colour)&1).
// LOG2L > 0: power-of-two L by shifts (the paper's bitwise coordinates); 0: any even L.
template <int LOG2L>
__device__ __forceinline__ void site_of(int h, int colour, int L, int& x, int& y, int& z)
{
    if constexpr (LOG2L > 0) {
        constexpr int LH = LOG2L - 1;
        const int xh = h & ((1 << LH) - 1);
        y = (h >> LH) & ((1 << LOG2L) - 1);
        z = h >> (LH + LOG2L);
        x = 2 * xh + ((y + z + colour) & 1);
    } else {
        const int Lh = L >> 1;
        const int xh = h % Lh;
        const int r = h / Lh;
        y = r % L;
        z = r / L;
        x = 2 * xh + ((y + z + colour) & 1);
    }
}

// position of site i in the colour-split site order of the spin array (units of one site = SITE_FLOATS floats)
__device__ __forceinline__ size_t site_slot(int i, int L, int Nh)
{
    const int x = i % L, y = (i / L) % L, z = i / (L * L);
    return (size_t)((x + y + z) & 1) * Nh + (size_t)(i >> 1);
}

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }

}  // namespace sg
