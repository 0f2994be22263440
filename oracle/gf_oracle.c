/*
 * oracle/gf_oracle.c -- plain, slow, fp64 CPU oracle for lattice gauge fixing by checkerboard overrelaxation
 * and SU(2)-heatbath simulated annealing (Schroeck & Vogt, arXiv:1209.4008; text in /root/reference/PAPER.md).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA path
 * (paper_1209_4008_b200/csrc) and neither includes the other.
 *
 * It follows Alg. 1 step by step, in the paper's order and notation, on the canonical
 * layout  U[s][mu][row][col]  (complex double), s = x + Nx (y + Ny (z + Nz t)), mu = 0..3 <-> x,y,z,t,
 * periodic boundaries.  Where the paper is silent, garbled or ambiguous the readings C1..C16 of
 * SURVEY.md sec. 8(c) (restated in DESIGN.md "Readings of the paper") are taken; each is cited where used.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md "Oracle pins".  Unpinned by the paper and
 * therefore "parity unpinned" beyond GPU-vs-oracle agreement: (i) the absolute F / theta trajectory and the
 * Gribov copy reached on the smooth-random configurations; (ii) the annealing temperature convention,
 * schedule shape and the choice of the Kennedy-Pendleton sampler (C13/C14) -- the paper only names
 * "simulated annealing".
 *
 * No blocking, fusion or reordering beyond the algorithm as stated; OpenMP over the sites of one parity is
 * legal because in a half-sweep every link is touched by exactly one active site (C6), and changes no result.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

enum { ORC_LANDAU = 0, ORC_COULOMB = 1 };

/* ------------------------------------------------------------------------------------------------ */
/* lattice indexing: 4D index linearised with divisions and modulo; periodic (C5)   */
/* ------------------------------------------------------------------------------------------------ */
static inline long lat_volume(const int N[4]) { return (long)N[0] * N[1] * N[2] * N[3]; }

static inline void lat_coords(const int N[4], long s, int x[4])
{
    x[0] = (int)(s % N[0]); s /= N[0];
    x[1] = (int)(s % N[1]); s /= N[1];
    x[2] = (int)(s % N[2]); s /= N[2];
    x[3] = (int)s;
}

static inline long lat_site(const int N[4], const int x[4])
{
    return x[0] + (long)N[0] * (x[1] + (long)N[1] * (x[2] + (long)N[2] * x[3]));
}

/* site x + dir*mu_hat, dir = +1 or -1, periodic */
static inline long lat_shift(const int N[4], long s, int mu, int dir)
{
    int x[4];
    lat_coords(N, s, x);
    x[mu] = (x[mu] + dir + N[mu]) % N[mu];
    return lat_site(N, x);
}

/* parity = (x+y+z+t) mod 2; RED = 0 is updated first, then BLACK = 1 (C5) */
static inline int lat_parity(const int N[4], long s)
{
    int x[4];
    lat_coords(N, s, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
}

static inline cplx *link_at(cplx *U, long s, int mu) { return U + (s * 4 + mu) * 9; }
static inline const cplx *clink_at(const cplx *U, long s, int mu) { return U + (s * 4 + mu) * 9; }

/* number of directions entering K, F and theta: 4 for Landau, 3 (mu = x,y,z) for Coulomb (C12) */
static inline int gauge_nd(int gauge) { return gauge == ORC_COULOMB ? 3 : 4; }

/* ------------------------------------------------------------------------------------------------ */
/* 3x3 complex helpers                                                                              */
/* ------------------------------------------------------------------------------------------------ */
static void m_mul(const cplx a[9], const cplx b[9], cplx out[9])
{
    cplx t[9];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            t[3 * r + c] = a[3 * r] * b[c] + a[3 * r + 1] * b[3 + c] + a[3 * r + 2] * b[6 + c];
    memcpy(out, t, sizeof t);
}

static void m_dagger(const cplx a[9], cplx out[9])
{
    cplx t[9];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            t[3 * r + c] = conj(a[3 * c + r]);
    memcpy(out, t, sizeof t);
}

/* ------------------------------------------------------------------------------------------------ */
/* K(x), eq. 2.3 in the in-place formulation (C2): the links already hold U^g, so      */
/*   K(x) = sum_{mu < Nd} [ U_mu(x) + U_mu(x - mu)^dagger ]                                          */
/* ------------------------------------------------------------------------------------------------ */
void orc_build_K(const int N[4], int gauge, const double *U_, long s, double *K_)
{
    const cplx *U = (const cplx *)U_;
    cplx *K = (cplx *)K_;
    for (int e = 0; e < 9; ++e) K[e] = 0.0;
    for (int mu = 0; mu < gauge_nd(gauge); ++mu) {
        const cplx *fwd = clink_at(U, s, mu);
        const cplx *bwd = clink_at(U, lat_shift(N, s, mu, -1), mu);
        cplx bwd_dag[9];
        m_dagger(bwd, bwd_dag);
        for (int e = 0; e < 9; ++e) K[e] += fwd[e] + bwd_dag[e];
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* SU(2) subgroup pieces.  Quaternion q = (q0,q1,q2,q3) <-> 2x2 matrix q0 + i (q1 s1 + q2 s2 + q3 s3): */
/*   a = q0 + i q3, b = q2 + i q1;  G_ii = a, G_ij = b, G_ji = -conj(b), G_jj = conj(a)      (C4)    */
/* ------------------------------------------------------------------------------------------------ */

/* (C7) quaternionic part of the (i,j) block of K -- the only part Re tr[G K] depends on:
 *   Re tr[G K] = const + g0 k0 - g1 k1 - g2 k2 - g3 k3                                              */
void orc_su2_project(const double *K_, int i, int j, double k[4])
{
    const cplx *K = (const cplx *)K_;
    k[0] = creal(K[3 * i + i] + K[3 * j + j]);
    k[1] = cimag(K[3 * i + j] + K[3 * j + i]);
    k[2] = creal(K[3 * i + j] - K[3 * j + i]);
    k[3] = cimag(K[3 * i + i] - K[3 * j + j]);
}

/* eq. 2.4 applied to the projected block (C7): g = K^dagger / sqrt(det K^dagger)
 * = (k0, -k1, -k2, -k3) / |k|.  Degenerate block (|k| < 1e-300): identity (C9 guards).              */
void orc_su2_maximiser(const double k[4], double g[4])
{
    double n = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2] + k[3] * k[3]);
    if (n < 1e-300) { g[0] = 1.0; g[1] = g[2] = g[3] = 0.0; return; }
    g[0] = k[0] / n; g[1] = -k[1] / n; g[2] = -k[2] / n; g[3] = -k[3] / n;
}

/* g -> g^omega "to second order", reading C9: binomial series in (g - 1) cut after n = 2,
 *   g^w ~ 1 + w (g-1) + w(w-1)/2 (g-1)^2,   with (g-1)^2 = (d^2 - |gvec|^2, 2 d gvec), d = g0 - 1,
 *   |gvec|^2 = 1 - g0^2  =>  h0 = 1 + w d (1 + (w-1) g0),  hvec = w (1 + (w-1) d) gvec,
 * then "project to SU(2)" (Alg. 1): h <- h / |h|.  If |h|^2 < 1e-20 take h = g.        */
void orc_su2_overrelax(const double g[4], double omega, double h[4])
{
    double d = g[0] - 1.0;
    double h0 = 1.0 + omega * d * (1.0 + (omega - 1.0) * g[0]);
    double f = omega * (1.0 + (omega - 1.0) * d);
    double h1 = f * g[1], h2 = f * g[2], h3 = f * g[3];
    double n2 = h0 * h0 + h1 * h1 + h2 * h2 + h3 * h3;
    if (n2 < 1e-20) { h[0] = g[0]; h[1] = g[1]; h[2] = g[2]; h[3] = g[3]; return; }
    double n = sqrt(n2);
    h[0] = h0 / n; h[1] = h1 / n; h[2] = h2 / n; h[3] = h3 / n;
}

/* quaternion product consistent with the embedding C4:
 *   (pq)_0 = p0 q0 - p.q ,  (pq)_vec = p0 qvec + q0 pvec - pvec x qvec                              */
void orc_quat_mul(const double p[4], const double q[4], double out[4])
{
    double r0 = p[0] * q[0] - p[1] * q[1] - p[2] * q[2] - p[3] * q[3];
    double r1 = p[0] * q[1] + q[0] * p[1] - (p[2] * q[3] - p[3] * q[2]);
    double r2 = p[0] * q[2] + q[0] * p[2] - (p[3] * q[1] - p[1] * q[3]);
    double r3 = p[0] * q[3] + q[0] * p[3] - (p[1] * q[2] - p[2] * q[1]);
    out[0] = r0; out[1] = r1; out[2] = r2; out[3] = r3;
}

/* embed quaternion q in the (i,j) subgroup of SU(3) (C4) */
void orc_su2_embed(const double q[4], int i, int j, double *G_)
{
    cplx *G = (cplx *)G_;
    for (int e = 0; e < 9; ++e) G[e] = (e % 4 == 0) ? 1.0 : 0.0;
    cplx a = q[0] + I * q[3], b = q[2] + I * q[1];
    G[3 * i + i] = a;
    G[3 * i + j] = b;
    G[3 * j + i] = -conj(b);
    G[3 * j + j] = conj(a);
}

/* Alg. 1 inner "for all mu": U_mu(x) <- G U_mu(x), U_mu(x-mu) <- U_mu(x-mu) G^dagger.
 * All four mu, also in Coulomb gauge: the temporal links must be transformed too (C12).            */
static void apply_G_to_links(const int N[4], cplx *U, long s, const cplx G[9])
{
    cplx Gdag[9];
    m_dagger(G, Gdag);
    for (int mu = 0; mu < 4; ++mu) {
        cplx *fwd = link_at(U, s, mu);
        cplx *bwd = link_at(U, lat_shift(N, s, mu, -1), mu);
        m_mul(G, fwd, fwd);
        m_mul(bwd, Gdag, bwd);
    }
}

static const int SUBGROUP[3][2] = { { 0, 1 }, { 0, 2 }, { 1, 2 } }; /* order of the subgroups (C4) */

/* ------------------------------------------------------------------------------------------------ */
/* one site update of Alg. 1, data flow of C8: build K once; for each subgroup        */
/* maximise, overrelax, apply G to the 8 links at once and set K <- G K.                             */
/* ------------------------------------------------------------------------------------------------ */
void orc_site_overrelax(const int N[4], int gauge, double *U_, long s, double omega)
{
    cplx *U = (cplx *)U_;
    cplx K[9], G[9];
    orc_build_K(N, gauge, U_, s, (double *)K);
    for (int sub = 0; sub < 3; ++sub) {
        const int i = SUBGROUP[sub][0], j = SUBGROUP[sub][1];
        double k[4], g[4], h[4];
        orc_su2_project((const double *)K, i, j, k);
        orc_su2_maximiser(k, g);
        orc_su2_overrelax(g, omega, h);
        orc_su2_embed(h, i, j, (double *)G);
        apply_G_to_links(N, U, s, G);
        m_mul(G, K, K);
    }
}

/* one checkerboard half-sweep over sublattice `parity` (Alg. 1 "for all x of sublattice") */
void orc_overrelax_half(const int N[4], int gauge, double *U, double omega, int parity)
{
    const long V = lat_volume(N);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s)
        if (lat_parity(N, s) == parity) orc_site_overrelax(N, gauge, U, s, omega);
}

/* Alg. 1 with a fixed number of iterations (the stop rule lives in the caller, C11) */
void orc_overrelax(const int N[4], int gauge, double *U, double omega, int nsweeps)
{
    for (int sweep = 0; sweep < nsweeps; ++sweep)
        for (int parity = 0; parity < 2; ++parity) /* RED, BLACK */
            orc_overrelax_half(N, gauge, U, omega, parity);
}

/* ------------------------------------------------------------------------------------------------ */
/* reductions.  Per-site contributions are stored and summed in canonical site order.              */
/* ------------------------------------------------------------------------------------------------ */

/* eq. 2.1, reading C1: F = sum_{x, mu<Nd} Re tr U_mu(x) / (N_c Nd V) on the current links */
double orc_functional(const int N[4], int gauge, const double *U_)
{
    const cplx *U = (const cplx *)U_;
    const long V = lat_volume(N);
    const int nd = gauge_nd(gauge);
    double *per_site = (double *)malloc(sizeof(double) * (size_t)V);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s) {
        double acc = 0.0;
        for (int mu = 0; mu < nd; ++mu) {
            const cplx *u = clink_at(U, s, mu);
            acc += creal(u[0]) + creal(u[4]) + creal(u[8]);
        }
        per_site[s] = acc;
    }
    double sum = 0.0;
    for (long s = 0; s < V; ++s) sum += per_site[s];
    free(per_site);
    return sum / (3.0 * nd * (double)V);
}

/* tr[Delta Delta^dagger] at one site, reading C3:
 *   Delta(x) = [ (K(x) - K(x)^dagger) / (2i) ]_traceless ,  tr[Delta Delta^dagger] = sum_ab |Delta_ab|^2 */
double orc_site_theta(const int N[4], int gauge, const double *U, long s)
{
    cplx K[9], Kdag[9], D[9];
    orc_build_K(N, gauge, U, s, (double *)K);
    m_dagger(K, Kdag);
    for (int e = 0; e < 9; ++e) D[e] = (K[e] - Kdag[e]) / (2.0 * I);
    cplx tr = (D[0] + D[4] + D[8]) / 3.0;
    D[0] -= tr; D[4] -= tr; D[8] -= tr;
    double acc = 0.0;
    for (int e = 0; e < 9; ++e) acc += creal(D[e]) * creal(D[e]) + cimag(D[e]) * cimag(D[e]);
    return acc;
}

/* eq. 2.5: theta = (1 / (V N_c)) sum_x tr[Delta Delta^dagger].
 * theta_slices (may be NULL) receives the Nt per-timeslice values (1/(V_s N_c)) sum_{x in slice} (C12). */
double orc_theta(const int N[4], int gauge, const double *U, double *theta_slices)
{
    const long V = lat_volume(N);
    const long Vs = (long)N[0] * N[1] * N[2];
    double *per_site = (double *)malloc(sizeof(double) * (size_t)V);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s) per_site[s] = orc_site_theta(N, gauge, U, s);
    double sum = 0.0;
    for (int t = 0; t < N[3]; ++t) {
        double slice = 0.0;
        for (long v = 0; v < Vs; ++v) slice += per_site[t * Vs + v];
        if (theta_slices) theta_slices[t] = slice / (3.0 * (double)Vs);
        sum += slice;
    }
    free(per_site);
    return sum / (3.0 * (double)V);
}

/* the value gf_theta reports: Landau eq. 2.5; Coulomb max over timeslices (C12) */
double orc_theta_report(const int N[4], int gauge, const double *U)
{
    if (gauge != ORC_COULOMB) return orc_theta(N, gauge, U, NULL);
    double *sl = (double *)malloc(sizeof(double) * (size_t)N[3]);
    orc_theta(N, gauge, U, sl);
    double m = sl[0];
    for (int t = 1; t < N[3]; ++t) if (sl[t] > m) m = sl[t];
    free(sl);
    return m;
}

/* average plaquette (1/(6 V N_c)) sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]:
 * gauge invariant under eq. 1.1 -- used only as an invariant in the pins (P5)         */
double orc_plaquette(const int N[4], const double *U_)
{
    const cplx *U = (const cplx *)U_;
    const long V = lat_volume(N);
    double *per_site = (double *)malloc(sizeof(double) * (size_t)V);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s) {
        double acc = 0.0;
        for (int mu = 0; mu < 4; ++mu)
            for (int nu = mu + 1; nu < 4; ++nu) {
                cplx a[9], b[9], p[9];
                m_mul(clink_at(U, s, mu), clink_at(U, lat_shift(N, s, mu, +1), nu), p);
                m_dagger(clink_at(U, lat_shift(N, s, nu, +1), mu), a);
                m_dagger(clink_at(U, s, nu), b);
                m_mul(p, a, p);
                m_mul(p, b, p);
                acc += creal(p[0] + p[4] + p[8]);
            }
        per_site[s] = acc;
    }
    double sum = 0.0;
    for (long s = 0; s < V; ++s) sum += per_site[s];
    free(per_site);
    return sum / (6.0 * 3.0 * (double)V);
}

/* max over links of max_ab |(U U^dagger - 1)_ab| and of |det U - 1|  (P6) */
void orc_unitarity_defect(const int N[4], const double *U_, double *max_uudag, double *max_det)
{
    const cplx *U = (const cplx *)U_;
    const long V = lat_volume(N);
    double mu_ = 0.0, md = 0.0;
    for (long l = 0; l < V * 4; ++l) {
        const cplx *u = U + l * 9;
        cplx ud[9], p[9];
        m_dagger(u, ud);
        m_mul(u, ud, p);
        for (int e = 0; e < 9; ++e) {
            double dev = cabs(p[e] - ((e % 4 == 0) ? 1.0 : 0.0));
            if (dev > mu_) mu_ = dev;
        }
        cplx det = u[0] * (u[4] * u[8] - u[5] * u[7]) - u[1] * (u[3] * u[8] - u[5] * u[6])
                 + u[2] * (u[3] * u[7] - u[4] * u[6]);
        double dd = cabs(det - 1.0);
        if (dd > md) md = dd;
    }
    *max_uudag = mu_;
    *max_det = md;
}

/* reunitarise every link: Gram-Schmidt rows 0,1; row 2 = conj(row0 x row1) (C15/C16).  The definition of what the
 * CUDA path's re-orthonormalisation on load computes; not called by the sweeps of the oracle (fp64 needs none). */
void orc_reunitarise(const int N[4], double *U_)
{
    cplx *U = (cplx *)U_;
    const long V = lat_volume(N);
    for (long l = 0; l < V * 4; ++l) {
        cplx *m = U + l * 9;
        double n0 = 0.0;
        for (int c = 0; c < 3; ++c) n0 += creal(m[c] * conj(m[c]));
        n0 = sqrt(n0);
        for (int c = 0; c < 3; ++c) m[c] /= n0;
        cplx dot = 0.0;
        for (int c = 0; c < 3; ++c) dot += conj(m[c]) * m[3 + c];
        for (int c = 0; c < 3; ++c) m[3 + c] -= dot * m[c];
        double n1 = 0.0;
        for (int c = 0; c < 3; ++c) n1 += creal(m[3 + c] * conj(m[3 + c]));
        n1 = sqrt(n1);
        for (int c = 0; c < 3; ++c) m[3 + c] /= n1;
        m[6] = conj(m[1] * m[5] - m[2] * m[4]);
        m[7] = conj(m[2] * m[3] - m[0] * m[5]);
        m[8] = conj(m[0] * m[4] - m[1] * m[3]);
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): the oracle's own copy                          */
/* ------------------------------------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c[4] = { ctr[0], ctr[1], ctr[2], ctr[3] };
    uint32_t k[2] = { key[0], key[1] };
    for (int round = 0; round < 10; ++round) {
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c[0];
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c[2];
        uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        uint32_t next[4] = { hi1 ^ c[1] ^ k[0], lo1, hi0 ^ c[3] ^ k[1], lo0 };
        memcpy(c, next, sizeof next);
        k[0] += 0x9E3779B9u;
        k[1] += 0xBB67AE85u;
    }
    memcpy(out, c, sizeof c);
}

/* uniform in (0,1) from a 32-bit word, exactly representable in fp32 and fp64 (C14) */
static inline double uniform24(uint32_t x) { return (double)(2u * (x >> 9) + 1u) * (1.0 / 16777216.0); }

/* ------------------------------------------------------------------------------------------------ */
/* SU(2) heatbath draw (C13/C14).  Density of h0: sqrt(1 - h0^2) exp(alpha h0); Kennedy-Pendleton:   */
/*   delta = (-ln u1 / alpha) cos^2(2 pi u3) + (-ln u2 / alpha); accept iff u4^2 <= 1 - delta/2;     */
/*   h0 = 1 - delta.  Trial t uses Philox block counter (c0,c1,c2,t); the direction of hvec uses the  */
/*   block (c0,c1,c2,0x80000000).  Cap: 4096 trials, then h = (1,0,0,0).                             */
/* Returns the number of trials used (1-based; 4097 if the cap was hit).                             */
/* ------------------------------------------------------------------------------------------------ */
int orc_kp_draw(double alpha, const uint32_t key[2], uint32_t c0, uint32_t c1, uint32_t c2, double h[4])
{
    const double two_pi = 6.283185307179586476925286766559;
    uint32_t ctr[4] = { c0, c1, c2, 0u }, x[4];
    int trial;
    double h0 = 1.0;
    int accepted = 0;
    for (trial = 0; trial < 4096; ++trial) {
        ctr[3] = (uint32_t)trial;
        orc_philox4x32_10(ctr, key, x);
        double u1 = uniform24(x[0]), u2 = uniform24(x[1]), u3 = uniform24(x[2]), u4 = uniform24(x[3]);
        double c = cos(two_pi * u3);
        double delta = (-log(u1) / alpha) * (c * c) + (-log(u2) / alpha);
        if (u4 * u4 <= 1.0 - 0.5 * delta) { h0 = 1.0 - delta; accepted = 1; break; }
    }
    if (!accepted) { h[0] = 1.0; h[1] = h[2] = h[3] = 0.0; return 4097; }
    ctr[3] = 0x80000000u;
    orc_philox4x32_10(ctr, key, x);
    double cos_t = 1.0 - 2.0 * uniform24(x[0]);
    double phi = two_pi * uniform24(x[1]);
    double r = sqrt(fmax(0.0, 1.0 - h0 * h0));
    double sin_t = sqrt(fmax(0.0, 1.0 - cos_t * cos_t));
    h[0] = h0;
    h[1] = r * sin_t * cos(phi);
    h[2] = r * sin_t * sin(phi);
    h[3] = r * cos_t;
    return trial + 1;
}

/* one heatbath site update at temperature T (C13): Boltzmann weight exp(F_raw / T); for subgroup (i,j)
 * P(g) ~ exp(alpha h0), alpha = |k| / T, h = g (x) khat  =>  draw h, set g = h (x) conj(khat).
 * trials (may be NULL): 3 ints per site, trial count of each subgroup.                              */
void orc_site_heatbath(const int N[4], int gauge, double *U_, long s, double T, uint64_t seed, uint32_t step,
                       int *trials)
{
    cplx *U = (cplx *)U_;
    cplx K[9], G[9];
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    const uint32_t parity = (uint32_t)lat_parity(N, s);
    orc_build_K(N, gauge, U_, s, (double *)K);
    for (int sub = 0; sub < 3; ++sub) {
        const int i = SUBGROUP[sub][0], j = SUBGROUP[sub][1];
        double k[4], h[4], g[4];
        orc_su2_project((const double *)K, i, j, k);
        double n = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2] + k[3] * k[3]);
        int ntr = 0;
        if (n < 1e-300) {
            g[0] = 1.0; g[1] = g[2] = g[3] = 0.0;
        } else {
            double alpha = n / T;
            double khat_conj[4] = { k[0] / n, -k[1] / n, -k[2] / n, -k[3] / n };
            ntr = orc_kp_draw(alpha, key, (uint32_t)s, step, (parity << 2) | (uint32_t)sub, h);
            orc_quat_mul(h, khat_conj, g);
        }
        if (trials) trials[3 * s + sub] = ntr;
        orc_su2_embed(g, i, j, (double *)G);
        apply_G_to_links(N, U, s, G);
        m_mul(G, K, K);
    }
}

/* simulated annealing: step i = one full sweep (RED then BLACK) at T_i = T_start + (T_end - T_start) i/(nsteps-1)
 * (nsteps = 1 -> T_start) (C13).  trials (may be NULL): V*3 ints, overwritten every step (last step survives). */
/* one heatbath half-sweep over sublattice `parity` at temperature T, annealing step `step` (C13/C14) */
void orc_heatbath_half(const int N[4], int gauge, double *U, double T, uint64_t seed, uint32_t step, int parity,
                       int *trials)
{
    const long V = lat_volume(N);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s)
        if (lat_parity(N, s) == parity) orc_site_heatbath(N, gauge, U, s, T, seed, step, trials);
}

void orc_anneal(const int N[4], int gauge, double *U, double T_start, double T_end, int nsteps, uint64_t seed,
                int *trials)
{
    for (int step = 0; step < nsteps; ++step) {
        double T = (nsteps > 1) ? T_start + (T_end - T_start) * (double)step / (double)(nsteps - 1) : T_start;
        for (int parity = 0; parity < 2; ++parity) /* RED, BLACK */
            orc_heatbath_half(N, gauge, U, T, seed, (uint32_t)step, parity, trials);
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* Update variants of the relaxation family ("Besides the standard relaxation algorithm */
/* [3] our program supports overrelaxation [4] and stochastic relaxation [5]"; "the      */
/* exponentiation of the gauge transformation is done to first or second order").  The paper gives   */
/* no formulas; readings C17-C19 of DESIGN.md:                                                       */
/*   C17 first order:  g^w ~ 1 + w (g - 1)  =>  h = (1 + w d, w gvec) / |.|,  d = g0 - 1             */
/*   C18 stochastic relaxation [5]: g -> g^2 with probability p, else g (plain relaxation);          */
/*       g^2 = (2 g0^2 - 1, 2 g0 gvec); decision: u < p with u = uniform24(x0) of the Philox block    */
/*       key = seed, counter = (site, sweep, parity<<2 | subgroup, 0x40000000)                       */
/*   C19 microcanonical sweep: g -> g^2 always (leaves F unchanged), n_micro of them after every     */
/*       heatbath sweep of the annealing                                                             */
/* ------------------------------------------------------------------------------------------------ */
enum { ORC_UPDATE_OVERRELAX2 = 0, ORC_UPDATE_OVERRELAX1 = 1, ORC_UPDATE_STOCHASTIC = 2 };

void orc_su2_overrelax1(const double g[4], double omega, double h[4])
{
    double d = g[0] - 1.0;
    double h0 = 1.0 + omega * d;
    double h1 = omega * g[1], h2 = omega * g[2], h3 = omega * g[3];
    double n2 = h0 * h0 + h1 * h1 + h2 * h2 + h3 * h3;
    if (n2 < 1e-20) { h[0] = g[0]; h[1] = g[1]; h[2] = g[2]; h[3] = g[3]; return; }
    double n = sqrt(n2);
    h[0] = h0 / n; h[1] = h1 / n; h[2] = h2 / n; h[3] = h3 / n;
}

void orc_su2_square(const double g[4], double h[4])
{
    double t = 2.0 * g[0];
    h[0] = t * g[0] - 1.0; h[1] = t * g[1]; h[2] = t * g[2]; h[3] = t * g[3];
}

/* one site update with the chosen variant.  squared (may be NULL): 3 ints per site, 1 where g^2 was taken */
void orc_site_relax(const int N[4], int gauge, double *U_, long s, int update, double param, uint64_t seed,
                    uint32_t sweep, int *squared)
{
    cplx *U = (cplx *)U_;
    cplx K[9], G[9];
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    const uint32_t parity = (uint32_t)lat_parity(N, s);
    orc_build_K(N, gauge, U_, s, (double *)K);
    for (int sub = 0; sub < 3; ++sub) {
        const int i = SUBGROUP[sub][0], j = SUBGROUP[sub][1];
        double k[4], g[4], h[4];
        int sq = 0;
        orc_su2_project((const double *)K, i, j, k);
        orc_su2_maximiser(k, g);
        if (update == ORC_UPDATE_OVERRELAX1) {
            orc_su2_overrelax1(g, param, h);
        } else if (update == ORC_UPDATE_STOCHASTIC) {
            uint32_t ctr[4] = { (uint32_t)s, sweep, (parity << 2) | (uint32_t)sub, 0x40000000u }, x[4];
            orc_philox4x32_10(ctr, key, x);
            sq = uniform24(x[0]) < param;
            if (sq) orc_su2_square(g, h);
            else { h[0] = g[0]; h[1] = g[1]; h[2] = g[2]; h[3] = g[3]; }
        } else {
            orc_su2_overrelax(g, param, h);
        }
        if (squared) squared[3 * s + sub] = sq;
        orc_su2_embed(h, i, j, (double *)G);
        apply_G_to_links(N, U, s, G);
        m_mul(G, K, K);
    }
}

/* nsweeps sweeps (RED then BLACK) with the chosen variant; the sweep counter of the random decisions (C18) starts
 * at sweep0 */
void orc_relax_from(const int N[4], int gauge, double *U, int update, double param, int nsweeps, int sweep0,
                    uint64_t seed, int *squared)
{
    const long V = lat_volume(N);
    for (int sweep = 0; sweep < nsweeps; ++sweep)
        for (int parity = 0; parity < 2; ++parity) {
#pragma omp parallel for schedule(static)
            for (long s = 0; s < V; ++s)
                if (lat_parity(N, s) == parity)
                    orc_site_relax(N, gauge, U, s, update, param, seed, (uint32_t)(sweep0 + sweep), squared);
        }
}

/* one call of the relaxation family: the sweep counter starts at 0 */
void orc_relax(const int N[4], int gauge, double *U, int update, double param, int nsweeps, uint64_t seed,
               int *squared)
{
    orc_relax_from(N, gauge, U, update, param, nsweeps, 0, seed, squared);
}

/* annealing with n_micro microcanonical sweeps after every heatbath sweep (C19) */
void orc_anneal_micro(const int N[4], int gauge, double *U, double T_start, double T_end, int nsteps,
                      int n_micro, uint64_t seed, int *trials)
{
    for (int step = 0; step < nsteps; ++step) {
        double T = (nsteps > 1) ? T_start + (T_end - T_start) * (double)step / (double)(nsteps - 1) : T_start;
        for (int parity = 0; parity < 2; ++parity)
            orc_heatbath_half(N, gauge, U, T, seed, (uint32_t)step, parity, trials);
        orc_relax(N, gauge, U, ORC_UPDATE_STOCHASTIC, 2.0, n_micro, seed, NULL); /* p = 2 > u always: g^2 */
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* Alg. 1 outer loop ("while precision theta not reached"), with the paper's cadence of   */
/* the check (F and theta are evaluated after every `check_every`-th iteration; C11):    */
/* theta (Coulomb: max over timeslices, C12) is evaluated before the first sweep and after every sweep */
/* whose number is a multiple of check_every; the loop ends `lag` sweeps after the first check that    */
/* finds theta < theta_tol, or at max_sweeps.  lag = 0 is the paper's loop; lag = 1 (C21) is the loop   */
/* of an implementation that learns theta of the state after sweep n only while sweep n+1 runs (so a   */
/* check at the last allowed sweep cannot take place).  The sweep counter of the stochastic decisions  */
/* (C18) runs on through the whole loop.  Returns the number of sweeps done; theta and F of the final  */
/* state.                                                                                              */
/* ------------------------------------------------------------------------------------------------ */
int orc_fix_lag(const int N[4], int gauge, double *U, int update, double param, double theta_tol, int check_every,
                int max_sweeps, uint64_t seed, int lag, double *theta_out, double *F_out)
{
    int done = 0, stop_at = -1;
    if (orc_theta_report(N, gauge, U) >= theta_tol) {
        while (done < max_sweeps && done != stop_at) {
            orc_relax_from(N, gauge, U, update, param, 1, done, seed, NULL);
            done += 1;
            if (stop_at < 0 && done % check_every == 0 && (lag == 0 || done < max_sweeps))
                if (orc_theta_report(N, gauge, U) < theta_tol) stop_at = done + lag;
        }
    }
    if (theta_out) *theta_out = orc_theta_report(N, gauge, U);
    if (F_out) *F_out = orc_functional(N, gauge, U);
    return done;
}

int orc_fix(const int N[4], int gauge, double *U, int update, double param, double theta_tol, int check_every,
            int max_sweeps, uint64_t seed, double *theta_out, double *F_out)
{
    return orc_fix_lag(N, gauge, U, update, param, theta_tol, check_every, max_sweeps, seed, 0, theta_out, F_out);
}

/* ------------------------------------------------------------------------------------------------ */
/* Coulomb gauge, "each timeslice fixed independently" (BASELINE.json configs[4]; C12, C20): K, F and  */
/* theta of a site use the spatial links of its own timeslice only, so a timeslice whose theta_t is    */
/* below the tolerance can be frozen: its sites are no longer updated (its theta_t then never changes,  */
/* sweeps of the neighbouring slices only multiply the temporal links between them).                   */
/* orc_relax_slices: as orc_relax, restricted to the sites of the timeslices with active[t] != 0.      */
/* orc_fix_slices: Alg. 1 with the stop rule per timeslice: after every check_every sweeps the slices   */
/* with theta_t < theta_tol are frozen for good; ends when none is active or at max_sweeps.            */
/* sweeps_per_slice (Nt ints, may be NULL) receives the sweeps each slice got; returns their maximum.   */
/* ------------------------------------------------------------------------------------------------ */
void orc_relax_slices(const int N[4], int gauge, double *U, int update, double param, int nsweeps, int sweep0,
                      uint64_t seed, const unsigned char *active)
{
    const long V = lat_volume(N);
    const long Vs = (long)N[0] * N[1] * N[2];
    for (int sweep = 0; sweep < nsweeps; ++sweep)
        for (int parity = 0; parity < 2; ++parity) {
#pragma omp parallel for schedule(static)
            for (long s = 0; s < V; ++s)
                if (active[s / Vs] && lat_parity(N, s) == parity)
                    orc_site_relax(N, gauge, U, s, update, param, seed, (uint32_t)(sweep0 + sweep), NULL);
        }
}

/* lag as in orc_fix_lag: a slice found below the tolerance at the check after sweep n is updated for `lag` more
 * sweeps and frozen from sweep n + lag + 1 on */
int orc_fix_slices_lag(const int N[4], int gauge, double *U, int update, double param, double theta_tol,
                       int check_every, int max_sweeps, uint64_t seed, int lag, int *sweeps_per_slice,
                       double *theta_out, double *F_out)
{
    const int Nt = N[3];
    unsigned char *active = (unsigned char *)malloc((size_t)Nt);
    double *sl = (double *)malloc(sizeof(double) * (size_t)Nt);
    int *count = (int *)calloc((size_t)Nt, sizeof(int));
    int *last = (int *)malloc(sizeof(int) * (size_t)Nt); /* last sweep (1-based) in which the slice is updated; -1: open */
    int done = 0, any = 0;
    orc_theta(N, gauge, U, sl);
    for (int t = 0; t < Nt; ++t) { last[t] = sl[t] >= theta_tol ? -1 : 0; any |= last[t] < 0; }
    while (any && done < max_sweeps) {
        for (int t = 0; t < Nt; ++t) active[t] = last[t] < 0 || done + 1 <= last[t];
        orc_relax_slices(N, gauge, U, update, param, 1, done, seed, active);
        done += 1;
        for (int t = 0; t < Nt; ++t) count[t] += active[t];
        if (done % check_every == 0 && (lag == 0 || done < max_sweeps)) {
            orc_theta(N, gauge, U, sl);
            for (int t = 0; t < Nt; ++t)
                if (last[t] < 0 && sl[t] < theta_tol) last[t] = done + lag; /* frozen slices stay frozen */
        }
        any = 0;
        for (int t = 0; t < Nt; ++t) any |= last[t] < 0 || done < last[t];
    }
    orc_theta(N, gauge, U, sl);
    double m = sl[0];
    for (int t = 1; t < Nt; ++t) if (sl[t] > m) m = sl[t];
    if (theta_out) *theta_out = m;
    if (F_out) *F_out = orc_functional(N, gauge, U);
    if (sweeps_per_slice) memcpy(sweeps_per_slice, count, sizeof(int) * (size_t)Nt);
    free(active); free(sl); free(count); free(last);
    return done;
}

int orc_fix_slices(const int N[4], int gauge, double *U, int update, double param, double theta_tol, int check_every,
                   int max_sweeps, uint64_t seed, int *sweeps_per_slice, double *theta_out, double *F_out)
{
    const int Nt = N[3];
    unsigned char *active = (unsigned char *)malloc((size_t)Nt);
    double *sl = (double *)malloc(sizeof(double) * (size_t)Nt);
    int *count = (int *)calloc((size_t)Nt, sizeof(int));
    int done = 0, any = 0;
    orc_theta(N, gauge, U, sl);
    for (int t = 0; t < Nt; ++t) { active[t] = sl[t] >= theta_tol; any |= active[t]; }
    while (any && done < max_sweeps) {
        int n = check_every < max_sweeps - done ? check_every : max_sweeps - done;
        orc_relax_slices(N, gauge, U, update, param, n, done, seed, active);
        done += n;
        orc_theta(N, gauge, U, sl);
        any = 0;
        for (int t = 0; t < Nt; ++t) {
            if (active[t]) count[t] += n;
            active[t] = active[t] && sl[t] >= theta_tol; /* frozen slices stay frozen */
            any |= active[t];
        }
    }
    double m = sl[0];
    for (int t = 1; t < Nt; ++t) if (sl[t] > m) m = sl[t];
    if (theta_out) *theta_out = m;
    if (F_out) *F_out = orc_functional(N, gauge, U);
    if (sweeps_per_slice) memcpy(sweeps_per_slice, count, sizeof(int) * (size_t)Nt);
    free(active); free(sl); free(count);
    return done;
}
