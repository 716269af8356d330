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

// Global copy id of local copy c of a sample (it enters the Philox counters of the heat bath and of the initial spins):
// gbase = id of the sample's local copy 0; a context that holds only Tl of the chain's slots per replica (temperature-slot
// sharding, sg_shape.first_slot / n_temps_total) skips Tpad = n_temps_total - Tl ids between its replicas.
__device__ __forceinline__ uint32_t copy_gid(uint32_t gbase, int c, int Tl, int Tpad)
{
    return gbase + (uint32_t)c + (Tpad ? (uint32_t)((c / Tl) * Tpad) : 0u);
}

// h[j] += c * n[j] for the four copies a thread holds: the inner step of every field computation.  Two FFMA2 (fma.rn.f32x2 with
// the coupling as its scalar operand) instead of four FFMA -- the same four fp32 FMAs with round to nearest, bit for bit, in half
// the issue slots (measured on the power-capped cfg-4 loop against the scalar form: OR half-sweep 659.5 -> 649.6 us, heat bath
// -4.4 %; profiles/r2e_whatif.md, profiles/r2_sass_histogram.md).
__device__ __forceinline__ void fma4(float c, const float (&n)[4], float (&h)[4])
{
    const float2 cc = make_float2(c, c);
    const float2 lo = __ffma2_rn(cc, make_float2(n[0], n[1]), make_float2(h[0], h[1]));
    const float2 hi = __ffma2_rn(cc, make_float2(n[2], n[3]), make_float2(h[2], h[3]));
    h[0] = lo.x; h[1] = lo.y; h[2] = hi.x; h[3] = hi.y;
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

// MUFU approximations (1-2 ulp): reciprocal, reciprocal square root, square root, 2^x
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float ex2_approx(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// ln(u), u a normal positive float, to a few ulp RELATIVE also next to u = 1 (MUFU.LG2 is only absolutely
// accurate there): u = m 2^e with m in [sqrt(1/2), sqrt(2)), ln m = 2 atanh(s), s = (m-1)/(m+1), |s| < 0.1716,
// odd series up to s^9 (next term 2 s^11/11 < 7e-10 ln m).
__device__ __forceinline__ float log_rel(float u)
{
    const int iu = __float_as_int(u);
    const int e = (iu - 0x3f3504f3) >> 23;
    const float f = __int_as_float(iu - (e << 23)) - 1.0f;       // exact
    const float s = f * rcp_approx(2.0f + f);
    const float z = s * s;
    const float p = fmaf(z, fmaf(z, fmaf(z, 1.0f / 9.0f, 1.0f / 7.0f), 0.2f), 1.0f / 3.0f);
    const float s2 = s + s;
    return fmaf((float)e, 0.69314718f, fmaf(s2 * z, p, s2));
}

// Heat bath, Eq. (A1): s drawn from exp(beta s.h).  Exact inverse CDF of the polar cosine
// about n = h/|h|, evaluated so that whichever of w = 1-u (distance from the north
// pole) and w' = 1+u (from the south pole) is small carries a few-ulp relative error (reading R23), branch-free:
//   E = e^{-2 kappa}, d = 1 - E, x = r1 d, x' = (1-r1) d / E, y = (1-r1) + r1 E      (1-r1 is exact in fp32)
//   w  = -ln(1 - x)/kappa = -ln(y)/kappa,      w' = ln(1 + x')/kappa,      w + w' = 2
// the smaller of x, x' (if <= 1/2) goes through log1p (= ln of the rounded sum plus the first-order correction
// for that rounding), otherwise ln(y) is well conditioned; uniform azimuth in the frame of Duff et al. (JCGT 2017).
__device__ __forceinline__ void hb_update(float hx, float hy, float hz, float beta, float r1, float r2,
                                          float& sx, float& sy, float& sz)
{
    const float hh = fmaf(hx, hx, fmaf(hy, hy, hz * hz));
    float nx = 0.0f, ny = 0.0f, nz = 1.0f, kappa = 0.0f;
    if (hh >= 1e-30f) {
        const float rs = rsqrt_approx(hh);
        nx = hx * rs; ny = hy * rs; nz = hz * rs;
        kappa = beta * (hh * rs);
    }
    float w, wp, u;                    // w = 1 - u, wp = 1 + u
    if (kappa < 1e-15f) {              // uniform law
        w = 2.0f * r1; wp = 2.0f - w; u = 1.0f - w;
    } else {
        const float a2 = 2.0f * kappa;
        const float E = ex2_approx(-1.44269504f * a2);            // 0 for kappa > 43.6: then x' = inf, y = 1 - r1
        float dp = fmaf(a2, 1.0f / 5040.0f, -1.0f / 720.0f);      // 1 - e^{-a} by its series for a < 0.3 (7 terms: 2e-8)
        dp = fmaf(dp, a2, 1.0f / 120.0f); dp = fmaf(dp, a2, -1.0f / 24.0f); dp = fmaf(dp, a2, 1.0f / 6.0f);
        dp = fmaf(dp, a2, -0.5f); dp = fmaf(dp, a2, 1.0f); dp *= a2;
        const float d = (a2 < 0.3f) ? dp : 1.0f - E;
        const float q1 = 1.0f - r1;
        const float x = r1 * d;
        const float xs = q1 * (d * rcp_approx(E));
        const float y = fmaf(r1, E, q1);
        const bool south = xs < x;
        const bool mid = fminf(x, xs) > 0.5f;
        const float zs = south ? xs : -x;
        const float arg = mid ? y : 1.0f + zs;
        float lg = log_rel(arg);
        lg += mid ? 0.0f : (zs - (arg - 1.0f)) * rcp_approx(arg);  // arg - 1 is exact for arg in [1/2, 2]
        const float v = lg * rcp_approx(kappa);
        if (south && !mid) { wp = v; w = 2.0f - v; u = v - 1.0f; }
        else { w = -v; wp = 2.0f + v; u = 1.0f + v; }
    }
    const float t = sqrt_approx(fmaxf(w * wp, 0.0f));
    // phi = 2 pi r2 reduced exactly to [-pi, pi); MUFU sine / cosine (absolute error 2^-21.4 on that range)
    const float ph = 6.2831853f * (r2 - (r2 >= 0.5f ? 1.0f : 0.0f));
    const float sp = __sinf(ph), cp = __cosf(ph);
    const float sg = copysignf(1.0f, nz);
    const float a = -rcp_approx(sg + nz);
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
