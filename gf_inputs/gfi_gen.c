/*
 * gf_inputs/gfi_gen.c -- seeded synthetic gauge-field generators (INPUTS ONLY).
 *
 * This module produces the lattice configurations that both the CPU oracle (oracle/) and the CUDA
 * library (paper_1209_4008_b200/) are run on.  It holds none of the gauge-fixing method's arithmetic
 * (no K(x), no SU(2) subgroup update, no functional, no theta): it only draws SU(3) matrices.
 * It shares no code with oracle/ or with the CUDA path; its Philox4x32-10 is its own copy.
 *
 * The paper's workloads are Monte-Carlo SU(3) configurations on N_s^3 x N_t lattices (sec. 4.1,
 * PAPER.md:156 sec. 5); those are not available, so seeded stand-ins of the same shape are drawn here
 * (recipe: SURVEY.md sec. 8(d), restated in DESIGN.md "Input recipe"):
 *
 *   normal deviates : Philox4x32-10, key = (seed_lo, seed_hi), counter = (site s, field id f, block b, 0);
 *                     32-bit words x -> u = (x + 0.5) * 2^-32;  Box-Muller pairs
 *                     (z0, z1) = sqrt(-2 ln u_a) (cos 2 pi u_b, sin 2 pi u_b) from (x0,x1) and (x2,x3).
 *   Haar SU(3) g(x) : f = 4; rows 0,1 from 12 normals (complex Gaussian), Gram-Schmidt, row2 = conj(row0 x row1).
 *   smooth link     : f = mu; H Hermitian traceless (diag ~ N(0,1), off-diag (a+ib)/sqrt2), U = exp(i eps H),
 *                     reunitarised, then U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger   (eq. 1.1).
 *   trivial orbit   : U_mu(x) = g(x) g(x+mu)^dagger (a pure gauge; BASELINE.json configs[0]).
 *   hot             : f = 8 + mu; every link an independent Haar SU(3) matrix (used by oracle pins only).
 *
 * Canonical layout: site s = x + Nx (y + Ny (z + Nz t)); double index
 * (((s*4 + mu)*3 + row)*3 + col)*2 + {0: re, 1: im}; mu = 0,1,2,3 <-> x,y,z,t; periodic boundaries.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

typedef double complex cplx;

/* ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), this module's own copy ---- */
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
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
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void gfi_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    philox4x32_10(ctr, key, out);
}

/* four N(0,1) deviates from one Philox block */
static void normals4(uint64_t seed, uint32_t s, uint32_t f, uint32_t b, double z[4])
{
    const double two_pi = 6.283185307179586476925286766559;
    uint32_t ctr[4] = { s, f, b, 0u };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t x[4];
    philox4x32_10(ctr, key, x);
    for (int p = 0; p < 2; ++p) {
        double ua = ((double)x[2 * p] + 0.5) * (1.0 / 4294967296.0);
        double ub = ((double)x[2 * p + 1] + 0.5) * (1.0 / 4294967296.0);
        double r = sqrt(-2.0 * log(ua));
        z[2 * p] = r * cos(two_pi * ub);
        z[2 * p + 1] = r * sin(two_pi * ub);
    }
}

/* rows 0,1 -> orthonormal; row 2 = conj(row0 x row1): a special unitary matrix */
static void gram_schmidt_su3(cplx m[9])
{
    double n0 = 0.0;
    for (int c = 0; c < 3; ++c) n0 += creal(m[c] * conj(m[c]));
    n0 = 1.0 / sqrt(n0);
    for (int c = 0; c < 3; ++c) m[c] *= n0;
    cplx dot = 0.0;
    for (int c = 0; c < 3; ++c) dot += conj(m[c]) * m[3 + c];
    for (int c = 0; c < 3; ++c) m[3 + c] -= dot * m[c];
    double n1 = 0.0;
    for (int c = 0; c < 3; ++c) n1 += creal(m[3 + c] * conj(m[3 + c]));
    n1 = 1.0 / sqrt(n1);
    for (int c = 0; c < 3; ++c) m[3 + c] *= n1;
    m[6] = conj(m[1] * m[5] - m[2] * m[4]);
    m[7] = conj(m[2] * m[3] - m[0] * m[5]);
    m[8] = conj(m[0] * m[4] - m[1] * m[3]);
}

/* Haar-distributed SU(3) matrix from 12 normals of field id f at site s */
static void haar_su3(uint64_t seed, uint32_t s, uint32_t f, cplx g[9])
{
    double z[12];
    for (uint32_t b = 0; b < 3; ++b) normals4(seed, s, f, b, z + 4 * b);
    for (int e = 0; e < 6; ++e) g[e] = z[2 * e] + I * z[2 * e + 1];
    gram_schmidt_su3(g);
}

void gfi_haar_su3(uint64_t seed, uint32_t s, uint32_t f, double *g_out)
{
    cplx g[9];
    haar_su3(seed, s, f, g);
    memcpy(g_out, g, sizeof g);
}

static void mat_mul(const cplx a[9], const cplx b[9], cplx out[9])
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            out[3 * r + c] = a[3 * r] * b[c] + a[3 * r + 1] * b[3 + c] + a[3 * r + 2] * b[6 + c];
}

static void mat_mul_dag(const cplx a[9], const cplx b[9], cplx out[9]) /* a * b^dagger */
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            out[3 * r + c] = a[3 * r] * conj(b[3 * c]) + a[3 * r + 1] * conj(b[3 * c + 1])
                           + a[3 * r + 2] * conj(b[3 * c + 2]);
}

/* exp(i eps H) for traceless Hermitian H by scaling-and-squaring of a Taylor series */
static void exp_i_eps_h(const cplx h[9], double eps, cplx u[9])
{
    double norm = 0.0;
    for (int e = 0; e < 9; ++e) norm += cabs(h[e]);
    norm *= fabs(eps);
    int squarings = 0;
    while (norm > 0.25 && squarings < 40) { norm *= 0.5; ++squarings; }
    double scale = eps / (double)(1ull << squarings);
    cplx a[9], term[9], tmp[9];
    for (int e = 0; e < 9; ++e) a[e] = I * scale * h[e];
    for (int e = 0; e < 9; ++e) { u[e] = (e % 4 == 0) ? 1.0 : 0.0; term[e] = u[e]; }
    for (int n = 1; n <= 20; ++n) {
        mat_mul(term, a, tmp);
        for (int e = 0; e < 9; ++e) { term[e] = tmp[e] / (double)n; u[e] += term[e]; }
    }
    for (int q = 0; q < squarings; ++q) {
        mat_mul(u, u, tmp);
        memcpy(u, tmp, sizeof tmp);
    }
    gram_schmidt_su3(u);
}

static inline long site_of(const int N[4], const int x[4])
{
    return x[0] + (long)N[0] * (x[1] + (long)N[1] * (x[2] + (long)N[2] * x[3]));
}

static inline void coords_of(const int N[4], long s, int x[4])
{
    x[0] = (int)(s % N[0]); s /= N[0];
    x[1] = (int)(s % N[1]); s /= N[1];
    x[2] = (int)(s % N[2]); s /= N[2];
    x[3] = (int)s;
}

static inline long forward_site(const int N[4], long s, int mu)
{
    int x[4];
    coords_of(N, s, x);
    x[mu] = (x[mu] + 1) % N[mu];
    return site_of(N, x);
}

/*
 * kind 0: trivial orbit  U = g(x) g(x+mu)^dagger
 * kind 1: smooth random  U = g(x) exp(i eps H_mu(x)) g(x+mu)^dagger
 * kind 2: hot            U = independent Haar matrix per link (no gauge transformation applied)
 * kind 3: smooth random WITHOUT the random gauge transformation (U = exp(i eps H)); close to the unit field
 * U_out: canonical layout, V*4*9 complex doubles.
 */
int gfi_generate(const int N[4], int kind, double eps, uint64_t seed, double *U_out)
{
    if (kind < 0 || kind > 3) return -1;
    const long V = (long)N[0] * N[1] * N[2] * N[3];
    cplx *U = (cplx *)U_out;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s) {
        cplx gx[9];
        if (kind == 0 || kind == 1) haar_su3(seed, (uint32_t)s, 4u, gx);
        for (int mu = 0; mu < 4; ++mu) {
            cplx *out = U + (s * 4 + mu) * 9;
            if (kind == 2) { haar_su3(seed, (uint32_t)s, 8u + (uint32_t)mu, out); continue; }
            cplx link[9];
            if (kind == 0) {
                for (int e = 0; e < 9; ++e) link[e] = (e % 4 == 0) ? 1.0 : 0.0;
            } else {
                double z[12];
                for (uint32_t b = 0; b < 3; ++b) normals4(seed, (uint32_t)s, (uint32_t)mu, b, z + 4 * b);
                const double r = 0.70710678118654752440;
                cplx h[9];
                h[0] = z[0]; h[4] = z[1]; h[8] = z[2];
                h[1] = (z[3] + I * z[4]) * r;  h[3] = conj(h[1]);
                h[2] = (z[5] + I * z[6]) * r;  h[6] = conj(h[2]);
                h[5] = (z[7] + I * z[8]) * r;  h[7] = conj(h[5]);
                double tr = (z[0] + z[1] + z[2]) / 3.0;
                h[0] -= tr; h[4] -= tr; h[8] -= tr;
                exp_i_eps_h(h, eps, link);
            }
            if (kind == 3) { memcpy(out, link, sizeof link); continue; }
            cplx gy[9], tmp[9];
            haar_su3(seed, (uint32_t)forward_site(N, s, mu), 4u, gy);
            mat_mul(gx, link, tmp);
            mat_mul_dag(tmp, gy, out);
        }
    }
    return 0;
}
