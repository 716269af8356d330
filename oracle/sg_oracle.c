/*
 * sg_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU oracle for the hot path of
 * arXiv:1309.1599 (3d Heisenberg spin glass with random anisotropic couplings).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code with the CUDA library (csrc/), and neither
 * includes the other.  It is never tuned: every function is the paper's definition written out,
 * one site at a time, in the paper's order and notation.  Citations are PAPER.md:<line>.
 *
 * Notation.  N = L^3, even L >= 2, periodic.  Site x = (x1,x2,x3) has the
 * linear index i = x1 + L*(x2 + L*x3) and colour p = (x1+x2+x3) mod 2.  Forward link (x,mu),
 * mu = 0,1,2, joins x and x+e_mu and carries the 3x3 matrix M[mu][i][a][b]: the first index a acts on
 * s_x, the second on s_{x+e_mu}.  The paper's model is M = J*1 + D with D symmetric
 * (Eq. (1)); a general M is the north_star's reading "J_yx = J_xy^T".
 *
 *   H   = - sum_{x,mu} s_x^T M_{x,mu} s_{x+e_mu}                               (Eq. (1))
 *   h_x =   sum_mu [ M_{x,mu} s_{x+e_mu} + M_{x-e_mu,mu}^T s_{x-e_mu} ]         (footnote 64)
 *
 * One lattice copy is s[a*N + i], a = 0,1,2 (doubles).  The couplings of one sample are
 * M[((mu*N + i)*3 + a)*3 + b] (doubles; the parity tests pass fp32-representable values).
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors, energy routes
 * against a dense numpy matrix and the exhaustive L=2 enumeration, ferromagnetic closed forms,
 * gauge / rotation / time-reversal invariance, OR energy conservation and involution, Langevin
 * moments and the KS test of the heat-bath law, Schwinger-Dyson (Eq. (A6)), exact Heisenberg ring
 * energies, Fourier closed forms, PT acceptance frequencies; chirality (Eq. (2)) against orthonormal triads,
 * numpy determinants / FFT, the conical-spiral closed form and its symmetries; Eq. (4) against the lattice
 * Ornstein-Zernike propagator.  What stays "parity unpinned": the
 * literal spin values after a seeded sweep (the paper prints none); the oracle defines them.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SGO_PI 3.14159265358979323846

/* ------------------------------------------------------------------------------------------ */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  north_star: "a counter-based Philox RNG".  */
/* DESIGN.md section 3 fixes the counter/key layout of every stream.                            */
/* ------------------------------------------------------------------------------------------ */
void sgo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* stream ids (counter word c3) */
enum { SGO_STREAM_HB = 1, SGO_STREAM_PT = 2, SGO_STREAM_SPINS = 3, SGO_STREAM_COUPLINGS = 4 };

static void sgo_draw(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t stream, uint32_t w[4])
{
    uint32_t ctr[4] = { c0, c1, c2, stream };
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    sgo_philox4x32_10(ctr, key, w);
}

/* r = ((w >> 9) + 1/2) 2^-23 in (0,1): 23 bits, exactly representable in fp32 and fp64. */
double sgo_uniform23(uint32_t w) { return ((double)(w >> 9) + 0.5) / 8388608.0; }
/* u = (w + 1/2) 2^-32 in (0,1): full word, fp64 only (coupling generator). */
double sgo_uniform32(uint32_t w) { return ((double)w + 0.5) / 4294967296.0; }

/* ------------------------------------------------------------------------------------------ */
/* Lattice                                                                                    */
/* ------------------------------------------------------------------------------------------ */
int sgo_site(int L, int x1, int x2, int x3) { return x1 + L * (x2 + L * x3); }

void sgo_coords(int L, int i, int x[3])
{
    x[0] = i % L;
    x[1] = (i / L) % L;
    x[2] = i / (L * L);
}

int sgo_colour(int L, int i)
{
    int x[3];
    sgo_coords(L, i, x);
    return (x[0] + x[1] + x[2]) & 1;
}

/* site index of x + dir*e_mu, dir = +1 or -1, periodic ("periodic boundary conditions") */
int sgo_neighbour(int L, int i, int mu, int dir)
{
    int x[3];
    sgo_coords(L, i, x);
    x[mu] = (x[mu] + dir + L) % L;
    return sgo_site(L, x[0], x[1], x[2]);
}

/* ------------------------------------------------------------------------------------------ */
/* Generators (S0).  Couplings: PAPER.md:65-73 and BASELINE.json configs; DESIGN.md section 3.  */
/* ------------------------------------------------------------------------------------------ */
enum { SGO_OFFDIAG_SYM = 0, SGO_PAPER_SYM6 = 1, SGO_GENERAL9 = 2, SGO_BIMODAL = 3, SGO_FERRO = 4 };

/* 12 standard normals of link l = 3i+mu of `sample`: three Philox calls j = 0,1,2 with counter
 * (l, sample, j, 4); each call gives two Box-Muller pairs (w0,w1) and (w2,w3). */
static void sgo_link_normals(uint64_t seed, uint32_t link, uint32_t sample, double n[12], uint32_t w0[4])
{
    for (uint32_t j = 0; j < 3; ++j) {
        uint32_t w[4];
        sgo_draw(seed, link, sample, j, SGO_STREAM_COUPLINGS, w);
        if (j == 0) memcpy(w0, w, sizeof(uint32_t) * 4);
        for (int pair = 0; pair < 2; ++pair) {
            double u0 = sgo_uniform32(w[2 * pair]);
            double u1 = sgo_uniform32(w[2 * pair + 1]);
            double rad = sqrt(-2.0 * log(u0));
            n[4 * j + 2 * pair]     = rad * cos(2.0 * SGO_PI * u1);
            n[4 * j + 2 * pair + 1] = rad * sin(2.0 * SGO_PI * u1);
        }
    }
}

/* M[3][N][3][3] of one sample; every entry rounded to the nearest fp32 (couplings are fp32 data
 * common to both sides, reading R20). */
void sgo_gen_couplings(int L, uint64_t seed, uint32_t sample, int mode, double sigma_D, double* M)
{
    int N = L * L * L;
    for (int i = 0; i < N; ++i) {
        for (int mu = 0; mu < 3; ++mu) {
            double n[12];
            uint32_t w0[4];
            double m[3][3] = { { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
            sgo_link_normals(seed, (uint32_t)(3 * i + mu), sample, n, w0);
            if (mode == SGO_OFFDIAG_SYM) {          /* J = a*1 + D, D off-diagonal symmetric (configs) */
                m[0][0] = m[1][1] = m[2][2] = n[0];
                m[0][1] = m[1][0] = sigma_D * n[1];
                m[0][2] = m[2][0] = sigma_D * n[2];
                m[1][2] = m[2][1] = sigma_D * n[3];
            } else if (mode == SGO_PAPER_SYM6) {    /* six independent elements, alpha >= beta */
                m[0][0] = n[0] + sigma_D * n[1];
                m[1][1] = n[0] + sigma_D * n[2];
                m[2][2] = n[0] + sigma_D * n[3];
                m[0][1] = m[1][0] = sigma_D * n[4];
                m[0][2] = m[2][0] = sigma_D * n[5];
                m[1][2] = m[2][1] = sigma_D * n[6];
            } else if (mode == SGO_GENERAL9) {      /* nine independent entries (exercises M^T) */
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) m[a][b] = sigma_D * n[3 * a + b];
            } else if (mode == SGO_BIMODAL) {       /* J = +-1, D^{ab} = +-D from sign bits */
                double J = (w0[0] & 1u) ? 1.0 : -1.0;
                double d[6];
                for (int k = 0; k < 6; ++k) d[k] = ((w0[0] >> (k + 1)) & 1u) ? sigma_D : -sigma_D;
                m[0][0] = J + d[0];
                m[1][1] = J + d[1];
                m[2][2] = J + d[2];
                m[0][1] = m[1][0] = d[3];
                m[0][2] = m[2][0] = d[4];
                m[1][2] = m[2][1] = d[5];
            } else {                                /* SGO_FERRO: M = 1 (PAPER.md:408 cross-check) */
                m[0][0] = m[1][1] = m[2][2] = 1.0;
            }
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b)
                    M[(((size_t)mu * N + i) * 3 + a) * 3 + b] = (double)(float)m[a][b];
        }
    }
}

/* initial spins of global copy g, uniform on S^2, stored as fp32 values: counter (i, g, 0, 3);
 * z = 1 - 2 r1, phi = 2 pi r2, s = (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z). */
void sgo_gen_spins(int L, uint64_t seed, uint32_t g, double* s)
{
    int N = L * L * L;
    for (int i = 0; i < N; ++i) {
        uint32_t w[4];
        sgo_draw(seed, (uint32_t)i, g, 0u, SGO_STREAM_SPINS, w);
        double z = 1.0 - 2.0 * sgo_uniform23(w[0]);
        double phi = 2.0 * SGO_PI * sgo_uniform23(w[1]);
        double rho = sqrt(1.0 - z * z);
        s[0 * N + i] = (double)(float)(rho * cos(phi));
        s[1 * N + i] = (double)(float)(rho * sin(phi));
        s[2 * N + i] = (double)(float)z;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Local field and energy                                                                     */
/* ------------------------------------------------------------------------------------------ */
/* h_x = sum_mu [ M_{x,mu} s_{x+e_mu} + M_{x-e_mu,mu}^T s_{x-e_mu} ]  (fn. 64, PAPER.md:512;
 * the transpose on the backward link follows from s_x^T M s_y = s_y^T M^T s_x, reading R2). */
void sgo_local_field(int L, const double* M, const double* s, int i, double h[3])
{
    int N = L * L * L;
    h[0] = h[1] = h[2] = 0.0;
    for (int mu = 0; mu < 3; ++mu) {
        int jf = sgo_neighbour(L, i, mu, +1);
        int jb = sgo_neighbour(L, i, mu, -1);
        const double* Mf = M + ((size_t)mu * N + i) * 9;   /* link (x, mu)       */
        const double* Mb = M + ((size_t)mu * N + jb) * 9;  /* link (x-e_mu, mu)  */
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                h[a] += Mf[3 * a + b] * s[b * N + jf];
                h[a] += Mb[3 * b + a] * s[b * N + jb];
            }
    }
}

/* H = - sum over the 3N forward links of s_x^T M_{x,mu} s_{x+e_mu}  (Eq. (1)).
 * For L = 2 the +mu and -mu neighbours coincide; both links are still summed (reading R5). */
double sgo_energy(int L, const double* M, const double* s)
{
    int N = L * L * L;
    double H = 0.0;
    for (int i = 0; i < N; ++i)
        for (int mu = 0; mu < 3; ++mu) {
            int j = sgo_neighbour(L, i, mu, +1);
            const double* m = M + ((size_t)mu * N + i) * 9;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) H -= s[a * N + i] * m[3 * a + b] * s[b * N + j];
        }
    return H;
}

/* Second and third routes to H, used only by the pins: -1/2 sum_x s_x.h_x and -sum_{p(x)=c} s_x.h_x */
double sgo_energy_from_fields(int L, const double* M, const double* s, int colour /* -1: all sites, halved */)
{
    int N = L * L * L;
    double acc = 0.0;
    for (int i = 0; i < N; ++i) {
        if (colour >= 0 && sgo_colour(L, i) != colour) continue;
        double h[3];
        sgo_local_field(L, M, s, i, h);
        acc += s[0 * N + i] * h[0] + s[1 * N + i] * h[1] + s[2 * N + i] * h[2];
    }
    return colour < 0 ? -0.5 * acc : -acc;
}

/* ------------------------------------------------------------------------------------------ */
/* Single-spin updates (App. A.1)                                                             */
/* ------------------------------------------------------------------------------------------ */
/* Overrelaxation, Eq. (A2): s_new = 2 h (h.s_old)/h^2 - s_old.
 * h.h < 1e-30: the spin is left unchanged (reading R8).  No renormalisation (R9). */
void sgo_or_update(const double h[3], double s[3])
{
    double hh = h[0] * h[0] + h[1] * h[1] + h[2] * h[2];
    if (hh < 1e-30) return;
    double hs = h[0] * s[0] + h[1] * s[1] + h[2] * s[2];
    double f = 2.0 * hs / hh;
    for (int a = 0; a < 3; ++a) s[a] = f * h[a] - s[a];
}

/* Heat bath, Eq. (A1): draw s from P(s) ~ exp(beta s.h) on the unit sphere.
 * Exact inverse CDF of the polar cosine u = s.n about n = h/|h| (reading R6), kappa = beta |h|:
 *     r1 = P(U >= u) = (e^kappa - e^{kappa u}) / (e^kappa - e^{-kappa})
 *  => w = 1 - u = -log(1 - r1 (1 - e^{-2 kappa})) / kappa      in [0, 2]
 * azimuth phi = 2 pi r2 in the right-handed orthonormal frame (e1, e2, n) of Duff et al. (JCGT 2017,
 * "Building an orthonormal basis, revisited"), reading R7.  h.h < 1e-30 => n = z^, kappa = 0;
 * kappa < 1e-15 => the uniform law w = 2 r1 (reading R8). */
void sgo_hb_update(const double h[3], double beta, double r1, double r2, double s[3])
{
    double hh = h[0] * h[0] + h[1] * h[1] + h[2] * h[2];
    double n[3] = { 0.0, 0.0, 1.0 };
    double kappa = 0.0;
    if (hh >= 1e-30) {
        double hn = sqrt(hh);
        n[0] = h[0] / hn; n[1] = h[1] / hn; n[2] = h[2] / hn;
        kappa = beta * hn;
    }
    double w;
    if (kappa < 1e-15) {
        w = 2.0 * r1;
    } else {
        double c = -expm1(-2.0 * kappa);
        w = -log1p(-r1 * c) / kappa;
    }
    double u = 1.0 - w;
    double t2 = w * (2.0 - w);
    double t = t2 > 0.0 ? sqrt(t2) : 0.0;
    double phi = 2.0 * SGO_PI * r2;
    double sg = copysign(1.0, n[2]);
    double a = -1.0 / (sg + n[2]);
    double b = n[0] * n[1] * a;
    double e1[3] = { 1.0 + sg * n[0] * n[0] * a, sg * b, -sg * n[0] };
    double e2[3] = { b, sg + n[1] * n[1] * a, -n[1] };
    double cp = cos(phi), sp = sin(phi);
    for (int k = 0; k < 3; ++k) s[k] = u * n[k] + t * (cp * e1[k] + sp * e2[k]);
}

/* Ill-conditioning flag of a site for the fp32-vs-fp64 elementwise comparison:
 * bit 0: |h| < 0.1 (direction of h not resolved to 1e-5 by an fp32 field);
 * bit 1: heat bath only, |n_z| < 1e-5 (the frame's one discontinuity, n_z = 0). */
static uint8_t sgo_flag(const double h[3], int kind)
{
    double hn = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
    uint8_t f = 0;
    if (hn < 0.1) f |= 1;
    if (kind == 1 && hn > 0.0 && fabs(h[2] / hn) < 1e-5) f |= 2;
    return f;
}

/* ------------------------------------------------------------------------------------------ */
/* Sweeps (App. A.1: "update all spins in the black sublattice, updating the white */
/* spins only afterwards"; checkerboard is fixed by north_star, colour 0 first, reading R4)     */
/* ------------------------------------------------------------------------------------------ */
/* One half-sweep of one copy.  kind 0 = OR, 1 = HB.  HB uniforms: counter (i, g, hb_counter, 1),
 * r1 = u23(w0), r2 = u23(w1).  store_fp32 != 0 rounds each new spin component to the nearest fp32
 * (the state precision of reading R20); 0 keeps full doubles (used by the invariance pins).
 * flags (may be NULL): per-site ill-conditioning flag of the sites updated, others untouched.
 * hnorm (may be NULL): |h_x| of the sites updated (the tests propagate measured errors with it).
 * sd (may be NULL): accumulates over the updated sites sum s_new.h, sum h.h, sum (s_new.h)^2 (Eq. (A6)). */
void sgo_halfsweep(int L, const double* M, double* s, int kind, int colour, double beta,
                   uint64_t seed, uint32_t g, uint32_t hb_counter, int store_fp32,
                   uint8_t* flags, double* hnorm, double sd[3])
{
    int N = L * L * L;
    for (int i = 0; i < N; ++i) {
        if (sgo_colour(L, i) != colour) continue;
        double h[3], sx[3] = { s[0 * N + i], s[1 * N + i], s[2 * N + i] };
        sgo_local_field(L, M, s, i, h);
        if (kind == 0) {
            sgo_or_update(h, sx);
        } else {
            uint32_t w[4];
            sgo_draw(seed, (uint32_t)i, g, hb_counter, SGO_STREAM_HB, w);
            sgo_hb_update(h, beta, sgo_uniform23(w[0]), sgo_uniform23(w[1]), sx);
        }
        for (int a = 0; a < 3; ++a) s[a * N + i] = store_fp32 ? (double)(float)sx[a] : sx[a];
        if (flags) flags[i] = sgo_flag(h, kind);
        if (hnorm) hnorm[i] = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
        if (sd) {
            double sh = sx[0] * h[0] + sx[1] * h[1] + sx[2] * h[2];
            sd[0] += sh;
            sd[1] += h[0] * h[0] + h[1] * h[1] + h[2] * h[2];
            sd[2] += sh * sh;
        }
    }
}

/* Test diagnostic (no arithmetic of the method): the two uniforms the heat bath of sgo_halfsweep draws at every site of
 * copy g in HB sweep hb_counter (stream 1 of SURVEY.md section 8(c) step 2: counter (i, g, hb_counter, 1), w0 -> r1, w1 -> r2).
 * The tests use it to FIND sweeps in which r1 falls in its extreme tails (2^-24, 1 - 2^-24). */
void sgo_hb_uniforms(int N, uint64_t seed, uint32_t g, uint32_t hb_counter, double* r1, double* r2)
{
    for (int i = 0; i < N; ++i) {
        uint32_t w[4];
        sgo_draw(seed, (uint32_t)i, g, hb_counter, SGO_STREAM_HB, w);
        r1[i] = sgo_uniform23(w[0]);
        r2[i] = sgo_uniform23(w[1]);
    }
}

/* n_sweeps full sweeps (colour 0 then colour 1) of n_copies copies of one sample.
 * spins[n_copies][3][N]; beta_of_copy[n_copies] (ignored for OR); copy c has global id g0 + c;
 * HB sweep k uses hb_counter0 + k.  Copies are independent between PT sweeps, so the
 * loop over copies is the one place OpenMP is used (the arithmetic per copy is untouched). */
void sgo_sweep_copies(int L, const double* M, double* spins, int n_copies, int kind, int n_sweeps,
                      const double* beta_of_copy, uint64_t seed, uint32_t g0, uint32_t hb_counter0,
                      int store_fp32)
{
    size_t stride = (size_t)3 * L * L * L;
#pragma omp parallel for schedule(dynamic, 1) if (n_copies >= 4 && (size_t)n_copies * stride > 20000)
    for (int c = 0; c < n_copies; ++c)
        for (int k = 0; k < n_sweeps; ++k)
            for (int colour = 0; colour < 2; ++colour)
                sgo_halfsweep(L, M, spins + c * stride, kind, colour, kind ? beta_of_copy[c] : 0.0,
                              seed, g0 + (uint32_t)c, hb_counter0 + (uint32_t)k, store_fp32, NULL, NULL, NULL);
}

void sgo_energy_copies(int L, const double* M, const double* spins, int n_copies, double* E)
{
    size_t stride = (size_t)3 * L * L * L;
#pragma omp parallel for schedule(dynamic, 1) if (n_copies >= 4 && (size_t)n_copies * stride > 20000)
    for (int c = 0; c < n_copies; ++c) E[c] = sgo_energy(L, M, spins + c * stride);
}

int sgo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* Parallel tempering (App. A.1): swap neighbouring temperatures, Metropolis       */
/* acceptance, "exchanging configurations is equivalent to exchange temperatures".              */
/* ------------------------------------------------------------------------------------------ */
/* One PT sweep of one chain = (sample, replica): pairs t = 0..T-2 in order on the updated
 * assignment (reading R11).  E_slot[T]: total H of the chain's slots.  slot_of_temp / temp_of_slot:
 * the chain's permutation and its inverse, updated in place.  Uniform: counter (t, chain, pt_counter, 2),
 * r = u23(w0).  Accept iff Delta >= 0 or r < exp(Delta), Delta = (beta_t - beta_{t+1})(E_i - E_j)
 * (north_star check 6, reading R12).  attempts/accepts[T-1] are incremented (may be NULL). */
void sgo_pt_sweep(int T, const double* betas, const double* E_slot, int* slot_of_temp, int* temp_of_slot,
                  uint64_t seed, uint32_t chain, uint32_t pt_counter, uint64_t* attempts, uint64_t* accepts)
{
    for (int t = 0; t + 1 < T; ++t) {
        int i = slot_of_temp[t], j = slot_of_temp[t + 1];
        double delta = (betas[t] - betas[t + 1]) * (E_slot[i] - E_slot[j]);
        uint32_t w[4];
        sgo_draw(seed, (uint32_t)t, chain, pt_counter, SGO_STREAM_PT, w);
        double r = sgo_uniform23(w[0]);
        int accept = (delta >= 0.0) || (r < exp(delta));
        if (attempts) attempts[t] += 1;
        if (accept) {
            slot_of_temp[t] = j; slot_of_temp[t + 1] = i;
            temp_of_slot[j] = t; temp_of_slot[i] = t + 1;
            if (accepts) accepts[t] += 1;
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Overlap observables (Sect. II.B): q_x = s^a_x . s^b_x,                           */
/* q^(k) = sum_x q_x e^{i k.x} / N at k = 0 and k_min = (2 pi/L,0,0) + permutations */
/* ------------------------------------------------------------------------------------------ */
/* out[0] = q^(0); out[1+2mu], out[2+2mu] = Re, Im of q^(k_mu), mu = 0,1,2. */
void sgo_overlap(int L, const double* sa, const double* sb, double out[7])
{
    int N = L * L * L;
    for (int k = 0; k < 7; ++k) out[k] = 0.0;
    for (int i = 0; i < N; ++i) {
        int x[3];
        sgo_coords(L, i, x);
        double q = sa[0 * N + i] * sb[0 * N + i] + sa[1 * N + i] * sb[1 * N + i] + sa[2 * N + i] * sb[2 * N + i];
        out[0] += q;
        for (int mu = 0; mu < 3; ++mu) {
            double ang = 2.0 * SGO_PI * (double)x[mu] / (double)L;
            out[1 + 2 * mu] += q * cos(ang);
            out[2 + 2 * mu] += q * sin(ang);
        }
    }
    for (int k = 0; k < 7; ++k) out[k] /= (double)N;
}

/* ------------------------------------------------------------------------------------------ */
/* Chirality observables (Sect. II.B, Eq. (2)):                                  */
/*   zeta_{x,mu} = s_{x+e_mu} . (s_x x s_{x-e_mu}),  kappa_{x,mu} = zeta^a_{x,mu} zeta^b_{x,mu},  */
/*   q^_CG^mu(k) = sum_x kappa_{x,mu} e^{i k.x} / N   at k = 0 and k_min + permutations.          */
/* ------------------------------------------------------------------------------------------ */
double sgo_chirality(int L, const double* s, int i, int mu)
{
    int N = L * L * L;
    int ip = sgo_neighbour(L, i, mu, +1), im = sgo_neighbour(L, i, mu, -1);
    double a[3], b[3], c[3];          /* a = s_{x+e_mu}, b = s_x, c = s_{x-e_mu} */
    for (int k = 0; k < 3; ++k) { a[k] = s[k * N + ip]; b[k] = s[k * N + i]; c[k] = s[k * N + im]; }
    double cr[3] = { b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0] };
    return a[0] * cr[0] + a[1] * cr[1] + a[2] * cr[2];
}

/* out[mu] = q^_CG^mu(0); out[3 + 2*(3*mu + nu)], out[4 + 2*(3*mu + nu)] = Re, Im of q^_CG^mu(k_nu),
 * k_nu = 2 pi e_nu / L; mu, nu = 0,1,2 (21 numbers). */
void sgo_chiral_overlap(int L, const double* sa, const double* sb, double out[21])
{
    int N = L * L * L;
    for (int k = 0; k < 21; ++k) out[k] = 0.0;
    for (int i = 0; i < N; ++i) {
        int x[3];
        sgo_coords(L, i, x);
        for (int mu = 0; mu < 3; ++mu) {
            double kap = sgo_chirality(L, sa, i, mu) * sgo_chirality(L, sb, i, mu);
            out[mu] += kap;
            for (int nu = 0; nu < 3; ++nu) {
                double ang = 2.0 * SGO_PI * (double)x[nu] / (double)L;
                out[3 + 2 * (3 * mu + nu)] += kap * cos(ang);
                out[4 + 2 * (3 * mu + nu)] += kap * sin(ang);
            }
        }
    }
    for (int k = 0; k < 21; ++k) out[k] /= (double)N;
}

/* Second-moment correlation length, Eq. (4) PAPER.md:93-97:
 *   xi = sqrt(chi(0)/chi(k_min) - 1) / (2 sin(k_min/2)),  k_min = 2 pi / L;
 * chi = N <|q^(k)|^2> (Eq. (3)).  A ratio below 1 (possible for noisy estimates) gives NaN. */
double sgo_xi(int L, double chi0, double chik)
{
    return sqrt(chi0 / chik - 1.0) / (2.0 * sin(SGO_PI / (double)L));
}

/* ------------------------------------------------------------------------------------------ */
/* Schwinger-Dyson monitor (App. A.4, Eq. (A6)): the two site averages of     */
/*   2 T <s_x.h_x> - <(h_x)^2 - (s_x.h_x)^2> = 0,   "averaged over all the sites in the lattice" */
/* ------------------------------------------------------------------------------------------ */
/* out[0] = sum_x s_x.h_x / N,  out[1] = sum_x [ h_x.h_x - (s_x.h_x)^2 ] / N  of one configuration. */
void sgo_sd_terms(int L, const double* M, const double* s, double out[2])
{
    int N = L * L * L;
    out[0] = out[1] = 0.0;
    for (int i = 0; i < N; ++i) {
        double h[3];
        sgo_local_field(L, M, s, i, h);
        double sh = s[0 * N + i] * h[0] + s[1 * N + i] * h[1] + s[2 * N + i] * h[2];
        out[0] += sh;
        out[1] += h[0] * h[0] + h[1] * h[1] + h[2] * h[2] - sh * sh;
    }
    out[0] /= (double)N;
    out[1] /= (double)N;
}

/* ------------------------------------------------------------------------------------------ */
/* Random walk in temperature (Sect. III: "the random walk in temperatures of     */
/* each sample"; "all the replicas stay a significant amount of time at each temperature").     */
/* ------------------------------------------------------------------------------------------ */
/* Bookkeeping after one PT sweep of one chain.  Every configuration (slot) carries a label: 0 = has not
 * touched an end of the ladder yet, 1 = last touched temperature index 0, 2 = last touched index T-1.
 * A ROUND TRIP of a configuration is index 0 -> index T-1 -> index 0; round_trips counts the completions,
 * summed over the chain's T configurations.  visits[slot*T + t] (may be NULL) counts the sweeps after which
 * the configuration in `slot` sat at temperature index t (the histogram of its walk). */
void sgo_pt_walk_update(int T, const int* temp_of_slot, int* label, uint64_t* round_trips, uint64_t* visits)
{
    for (int slot = 0; slot < T; ++slot) {
        int t = temp_of_slot[slot];
        if (t == 0) {
            if (label[slot] == 2) *round_trips += 1;
            label[slot] = 1;
        } else if (t == T - 1) {
            if (label[slot] == 1) label[slot] = 2;        /* a trip starts at index 0 only: label 0 stays 0 */
        }
        if (visits) visits[(size_t)slot * T + t] += 1;
    }
}
