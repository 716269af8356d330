// sg_measure.cuh -- S5 at streaming speed: overlaps q^(0), q^(k_mu) of all replica pairs in ONE read pass of the spins
// (SURVEY.md section 8(a) S5).
//
// Why.  k_measure (sg_kernels.cuh) stages a few sites of all copies in shared memory and lets thread = (pair, temperature)
// gather its two copies from there: 0.17 of the HBM roofline (random banks, fp64 work per site and pair).  Here
// thread = (lattice row (x2, x3), temperature t) and walks along x1.  It reads, straight from global memory, the spin
// of EVERY replica at temperature t (its slot comes from the permutation once per thread) -- 3 R floats per site -- and
// forms all P = R(R-1)/2 pair products from those registers, so every spin is loaded once for all pairs.  The threads of a
// warp are consecutive temperatures of one replica window, i.e. a permutation of <= 2 copy groups: each warp load touches
// one or two full 128-byte lines, and the <= 2 warps that cover a row's temperatures consume the lines completely (L1).
// Row sums (q, q cos 2 pi x1/L, q sin 2 pi x1/L) are fp32 over the <= L sites of a row; they are folded into fp64
// accumulators (in shared memory, one column per thread) with the row's x2, x3 phases; the CTA reduces its rows in a fixed
// order and writes one partial per (chunk, pair, temperature), which k_reduce_measure sums in fixed order: bit-reproducible.
#pragma once
#include "sg_device.cuh"

namespace sg {

constexpr int MROWS_THREADS = 256;

struct MeasureRowsParams {
    const float* spins;        // [S][NG][2][Nh][3][G]
    const int* slot_of_temp;   // [S][R][T]
    const double* phase;       // [L][2] cos, sin of 2 pi x / L
    double* Mpart;             // [S][nchunk][PT][7]
    int L, N, Nh, NG, R, T, P, nchunk, rows_per_cta, Tw, rows_t;
};

inline size_t mrows_smem_bytes(int L, int R)
{
    const int P = R * (R - 1) / 2;
    return (size_t)P * 7 * MROWS_THREADS * sizeof(double) + (size_t)2 * L * sizeof(float);
}

template <int R_>
__global__ void __launch_bounds__(MROWS_THREADS) k_measure_rows(const MeasureRowsParams p)
{
    constexpr int P_ = R_ * (R_ - 1) / 2;
    extern __shared__ __align__(16) unsigned char mr_smem[];
    double* const sacc = reinterpret_cast<double*>(mr_smem);                        // [P_*7][MROWS_THREADS]
    float* const phx = reinterpret_cast<float*>(sacc + (size_t)P_ * 7 * MROWS_THREADS);   // [L][2]
    const int tid = threadIdx.x, L = p.L;
    const int rt = tid / p.Tw, tx = tid - rt * p.Tw;
    const int t = blockIdx.z * p.Tw + tx;
    const int chunk = blockIdx.x, sample = blockIdx.y;
    const bool live = (rt < p.rows_t) && (t < p.T);

    for (int u = tid; u < 2 * L; u += MROWS_THREADS) phx[u] = (float)p.phase[u];
#pragma unroll
    for (int v = 0; v < P_ * 7; ++v) sacc[v * MROWS_THREADS + tid] = 0.0;
    __syncthreads();

    if (live) {
        const float* base[R_];
#pragma unroll
        for (int a = 0; a < R_; ++a) {
            const int c = a * p.T + p.slot_of_temp[((size_t)sample * p.R + a) * p.T + t];
            base[a] = p.spins + ((size_t)(sample * p.NG + c / G) * p.N) * SITE_FLOATS + (c % G);
        }
        const int row_end = min(L * L, (chunk + 1) * p.rows_per_cta);
        const int Lh = L >> 1;
        for (int row = chunk * p.rows_per_cta + rt; row < row_end; row += p.rows_t) {
            const int y = row % L, z = row / L;
            const int c0 = (y + z) & 1;                       // colour of the site x1 = 0 of this row
            // colour-split order: sites x1 = 2m and 2m + 1 sit at (L row)/2 + m of their colour's half
            const size_t pe = ((size_t)c0 * p.Nh + (size_t)Lh * row) * SITE_FLOATS;
            const size_t po = ((size_t)(1 - c0) * p.Nh + (size_t)Lh * row) * SITE_FLOATS;
            float rs[P_], rc[P_], rn[P_];
#pragma unroll
            for (int k = 0; k < P_; ++k) { rs[k] = 0.f; rc[k] = 0.f; rn[k] = 0.f; }
#pragma unroll 2
            for (int m = 0; m < Lh; ++m) {
                float se[R_][3], so[R_][3];
#pragma unroll
                for (int a = 0; a < R_; ++a)
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        se[a][k] = __ldg(base[a] + pe + (size_t)m * SITE_FLOATS + k * G);
                        so[a][k] = __ldg(base[a] + po + (size_t)m * SITE_FLOATS + k * G);
                    }
                const float2 ce = *reinterpret_cast<const float2*>(phx + 4 * m), co = *reinterpret_cast<const float2*>(phx + 4 * m + 2);
                int k = 0;
#pragma unroll
                for (int a = 0; a < R_; ++a)
#pragma unroll
                    for (int b = a + 1; b < R_; ++b, ++k) {
                        const float qe = fmaf(se[a][0], se[b][0], fmaf(se[a][1], se[b][1], se[a][2] * se[b][2]));
                        const float qo = fmaf(so[a][0], so[b][0], fmaf(so[a][1], so[b][1], so[a][2] * so[b][2]));
                        rs[k] += qe; rc[k] = fmaf(qe, ce.x, rc[k]); rn[k] = fmaf(qe, ce.y, rn[k]);
                        rs[k] += qo; rc[k] = fmaf(qo, co.x, rc[k]); rn[k] = fmaf(qo, co.y, rn[k]);
                    }
            }
            const double cy = p.phase[2 * y], sy = p.phase[2 * y + 1], cz = p.phase[2 * z], sz = p.phase[2 * z + 1];
#pragma unroll
            for (int k = 0; k < P_; ++k) {
                double* a7 = sacc + (size_t)(k * 7) * MROWS_THREADS + tid;
                const double q = (double)rs[k];
                a7[0] += q;
                a7[1 * MROWS_THREADS] += (double)rc[k];
                a7[2 * MROWS_THREADS] += (double)rn[k];
                a7[3 * MROWS_THREADS] = fma(q, cy, a7[3 * MROWS_THREADS]);
                a7[4 * MROWS_THREADS] = fma(q, sy, a7[4 * MROWS_THREADS]);
                a7[5 * MROWS_THREADS] = fma(q, cz, a7[5 * MROWS_THREADS]);
                a7[6 * MROWS_THREADS] = fma(q, sz, a7[6 * MROWS_THREADS]);
            }
        }
    }
    __syncthreads();
    // sum over the CTA's row threads in a fixed order; thread (rt = 0, tx) writes the partial of temperature t
    if (rt == 0 && t < p.T) {
        const int PT = p.P * p.T;
#pragma unroll
        for (int k = 0; k < P_; ++k) {
            double* dst = p.Mpart + (((size_t)sample * p.nchunk + chunk) * PT + (size_t)k * p.T + t) * 7;
#pragma unroll
            for (int v = 0; v < 7; ++v) {
                double acc = 0.0;
                for (int r = 0; r < p.rows_t; ++r) acc += sacc[(size_t)(k * 7 + v) * MROWS_THREADS + r * p.Tw + tx];
                dst[v] = acc;
            }
        }
    }
}

}  // namespace sg
