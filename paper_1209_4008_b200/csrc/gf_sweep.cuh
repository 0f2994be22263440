// gf_sweep.cuh -- the checkerboard half-sweep kernel (overrelaxation and SU(2) heatbath), Alg. 1 of the paper
// (PAPER.md:74-91), for sm_100a.
//
// Granularity (re-decided for sm_100a; the paper's Fermi design used 8 threads per site because of a
// 63-register limit): TPS threads share one site, each holding the forward and the
// backward link of 4/TPS directions in registers (TPS = 1: all 8 links, 144 reals).  Partial sums of K(x)
// are combined with warp shuffles (the sm_100a stand-in for the paper's shared-memory accumulator,
// PAPER.md:146); every thread of a site then runs the same three SU(2) subgroup steps redundantly on the
// full K and applies each g to its own links immediately (literal data flow of Alg. 1, C8).
//
// Memory: every link is read once and written once per half-sweep (C6), each access a coalesced 128-bit
// vector per thread (gf_device.cuh); all loads of a thread are issued before the first use.
#pragma once
#include "gf_device.cuh"

namespace gf {

enum { MODE_OVERRELAX = 0, MODE_HEATBATH = 1, MODE_VARIANT = 2 };
// MODE_VARIANT picks the SU(2) step at run time (SweepParams::variant): the update variants the paper's package
// offers beside second-order overrelaxation (readings C17, C18)
enum { VARIANT_OVERRELAX1 = 1, VARIANT_STOCHASTIC = 2 };
constexpr int MAX_BLOCK = 256;

struct SweepParams {
    void* U;        // native field
    Lattice L;
    int parity;     // sublattice updated by this launch: 0 = RED, 1 = BLACK (C5)
    int nd;         // directions entering K: 4 (Landau) or 3 (Coulomb, C12)
    int reunit;     // re-orthonormalise links on load (C15)
    int reverse;    // traverse blocks back to front (L2 reuse between consecutive half-sweeps)
    int ld_policy;  // L2 policy of the link loads / stores (POLICY_*, gf_device.cuh)
    int st_policy;
    int pdl;        // launched with programmatic stream serialization: wait for the previous grid before loading
    unsigned h_begin, h_count; // half-site range updated by this launch (whole lattice: 0, H; a run of timeslices: C20)
    unsigned prefetch; // L2 prefetch distance in sites along the traversal direction (0 = off)
    double omega;   // overrelaxation parameter; MODE_VARIANT: omega (first order) or probability p
    int variant;    // MODE_VARIANT: VARIANT_*
    double T;       // heatbath temperature (C13)
    uint32_t key0, key1, step; // Philox key = seed, step = annealing step (C14)
    unsigned* trials;          // optional: KP trial counts, index 3*s + subgroup
    void* G;                   // Coulomb reading B (C12): accumulated g(x), 2 parity blocks of 18 reals per site
};

// ---------------------------------------------------------------------------------------------------------
// SU(2) step, overrelaxation: maximiser (eq. 2.4, on the projected block, C7), then g^omega to
// second order and reprojection (reading C9):
//   g = (k0,-k1,-k2,-k3)/|k|;  d = g0 - 1;  h0 = 1 + w d (1 + (w-1) g0);  hvec = w (1 + (w-1) d) gvec;  h /= |h|
// ---------------------------------------------------------------------------------------------------------
// Guards (C9) on the squared norms: |k|^2 below TinySq<T> takes G = 1 (the CPU oracle tests |k| < 1e-300; the
// two differ only for |k| in [1e-300, 1e-150), fp32 [.., 1e-18) -- DESIGN.md "Differences").
template <typename T> struct Tiny;
template <> struct Tiny<float> { static constexpr float sq = 1e-36f; };
template <> struct Tiny<double> { static constexpr double sq = 1e-300; };

template <typename T>
__device__ __forceinline__ void su2_overrelax_step(const T (&k)[4], T w, T (&h)[4])
{
    // branch-free: the guards (C9) are selects at the end, so that the compiler can schedule this dependent chain
    // together with the independent link updates of the previous subgroup
    const T n2k = dot4(k[0], k[0], k[1], k[1], k[2], k[2], k[3], k[3]);
    const bool ok = n2k >= Tiny<T>::sq;
    const T inv = gf_rsqrt<T>(ok ? n2k : T(1));
    const T g0 = k[0] * inv, g1 = -k[1] * inv, g2 = -k[2] * inv, g3 = -k[3] * inv;
    const T d = g0 - T(1);
    const T h0 = T(1) + w * d * (T(1) + (w - T(1)) * g0);
    const T f = w * (T(1) + (w - T(1)) * d);
    const T h1 = f * g1, h2 = f * g2, h3 = f * g3;
    const T n2 = dot4(h0, h0, h1, h1, h2, h2, h3, h3);
    const bool ok2 = n2 >= T(1e-20);
    const T hn = gf_rsqrt<T>(ok2 ? n2 : T(1));
    h[0] = ok ? (ok2 ? h0 * hn : g0) : T(1);
    h[1] = ok ? (ok2 ? h1 * hn : g1) : T(0);
    h[2] = ok ? (ok2 ? h2 * hn : g2) : T(0);
    h[3] = ok ? (ok2 ? h3 * hn : g3) : T(0);
}

// SU(2) step of the variants.  First order (C17): g^w ~ 1 + w (g - 1), reprojected.  Stochastic relaxation (C18):
// g^2 = (2 g0^2 - 1, 2 g0 gvec) with probability p, else g; the decision u < p is taken in double on
// u = (2 (x >> 9) + 1) 2^-24 (exact), x the first word of the Philox block (site, sweep, parity<<2|subgroup,
// 0x40000000), so fp32 and fp64 kernels decide exactly like the oracle.
template <typename T>
__device__ __forceinline__ void su2_variant_step(const T (&k)[4], int variant, double param, uint32_t key0,
                                                 uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2, T (&h)[4])
{
    const T n2k = dot4(k[0], k[0], k[1], k[1], k[2], k[2], k[3], k[3]);
    if (!(n2k >= Tiny<T>::sq)) { h[0] = T(1); h[1] = h[2] = h[3] = T(0); return; }
    const T inv = gf_rsqrt<T>(n2k);
    const T g0 = k[0] * inv, g1 = -k[1] * inv, g2 = -k[2] * inv, g3 = -k[3] * inv;
    if (variant == VARIANT_STOCHASTIC) {
        uint32_t x[4];
        philox4x32_10(c0, c1, c2, 0x40000000u, key0, key1, x);
        const double u = (double)(2u * (x[0] >> 9) + 1u) * (1.0 / 16777216.0);
        if (u < param) {
            const T t = T(2) * g0;
            h[0] = gf_fma(t, g0, T(-1)); h[1] = t * g1; h[2] = t * g2; h[3] = t * g3;
        } else {
            h[0] = g0; h[1] = g1; h[2] = g2; h[3] = g3;
        }
        return;
    }
    const T w = (T)param;
    const T h0 = gf_fma(w, g0 - T(1), T(1));
    const T h1 = w * g1, h2 = w * g2, h3 = w * g3;
    const T n2 = dot4(h0, h0, h1, h1, h2, h2, h3, h3);
    if (n2 < T(1e-20)) { h[0] = g0; h[1] = g1; h[2] = g2; h[3] = g3; return; }
    const T hn = gf_rsqrt<T>(n2);
    h[0] = h0 * hn; h[1] = h1 * hn; h[2] = h2 * hn; h[3] = h3 * hn;
}

// ---------------------------------------------------------------------------------------------------------
// SU(2) step, heatbath (C13/C14): alpha = |k|/T; draw h0 with density sqrt(1-h0^2) exp(alpha h0) by
// Kennedy-Pendleton, hvec uniform on the sphere; g = h (x) conj(khat).
// Uniforms: u = (2 (x >> 9) + 1) 2^-24, exact in fp32 and fp64.
// ---------------------------------------------------------------------------------------------------------
template <typename T> struct KPMath;
// fp64: the draw is evaluated in double like the oracle's, with correctly-rounded-to-1-ulp library functions (log,
// cospi/sinpi) but without IEEE divisions and square roots (1/|k| by rsqrt, delta as one fused expression times
// 1/alpha).  The oracle's alpha already differs from the kernel's by an ulp (summation order of K), so decision
// parity rests on the size of the difference, not on the operation order: a decision flips only when u4^2 falls
// within ~1e-15 of the threshold, i.e. with probability ~1e-15 per trial (tests compare every trial count).
template <> struct KPMath<double> {
    static __device__ __forceinline__ double uni(uint32_t x) { return (double)(2u * (x >> 9) + 1u) * (1.0 / 16777216.0); }
    static __device__ __forceinline__ double cos2pi(double u) { return cospi(2.0 * u); }
    static __device__ __forceinline__ double sin2pi(double u) { return sinpi(2.0 * u); }
    static __device__ __forceinline__ double neglog(double u) { return -log(u); }
    static __device__ __forceinline__ void prep(double n2, double T, double& alpha, double& inv_alpha, double& inv_n)
    {
        inv_n = rsqrt(n2);
        alpha = n2 * inv_n / T;
        inv_alpha = T * inv_n;
    }
    static __device__ __forceinline__ double root(double x) { return x > 0.0 ? x * rsqrt(x) : 0.0; }
    static __device__ __forceinline__ double delta(double l1, double l2, double c, double alpha, double inv_alpha)
    {
        (void)alpha;
        return fma(l1, c * c, l2) * inv_alpha;
    }
    static __device__ __forceinline__ bool accept(double u4, double d) { return u4 * u4 <= fma(-0.5, d, 1.0); }
};
// fp32: decision parity with the fp64 oracle cannot be exact (alpha itself differs at 1e-7, C14), so the draw uses
// the SFU: u from the mantissa trick (exact), -ln u = -ln2 * lg2(u) (MUFU.LG2, abs. error ~4e-7), cos/sin by
// MUFU.COS/SIN (abs. error ~5e-7), one reciprocal of alpha per subgroup instead of two divisions per trial.
// A decision flips when u4^2 falls within ~1e-6/alpha of the threshold: ~1e-6 of the (site, subgroup) draws.
template <> struct KPMath<float> {
    // (2 (x >> 9) + 1) 2^-24 = [1 + (x >> 9) 2^-23] - (1 - 2^-24): both terms and the result are fp32 numbers
    static __device__ __forceinline__ float uni(uint32_t x) { return __uint_as_float(0x3F800000u | (x >> 9)) - 0.99999994039535522461f; }
    static __device__ __forceinline__ float cos2pi(float u) { return __cosf(6.283185307179586f * u); }
    static __device__ __forceinline__ float sin2pi(float u) { return __sinf(6.283185307179586f * u); }
    static __device__ __forceinline__ float neglog(float u) { return -0.693147180559945f * __log2f(u); }
    // no division, no IEEE square root: 1/|k| by MUFU.RSQ + one Newton step, alpha and 1/alpha from it
    static __device__ __forceinline__ void prep(float n2, float T, float& alpha, float& inv_alpha, float& inv_n)
    {
        inv_n = gf_rsqrt<float>(n2);
        alpha = n2 * inv_n * __frcp_rn(T);
        inv_alpha = T * inv_n;
    }
    static __device__ __forceinline__ float root(float x) { return x > 0.0f ? x * rsqrtf(x) : 0.0f; }
    static __device__ __forceinline__ float delta(float l1, float l2, float c, float alpha, float inv_alpha)
    {
        (void)alpha;
        return fmaf(l1, c * c, l2) * inv_alpha;
    }
    static __device__ __forceinline__ bool accept(float u4, float d) { return u4 * u4 <= fmaf(-0.5f, d, 1.0f); }
};

// The Philox counters of a draw hold (site, step, parity, subgroup, trial) and no data, so the block of trial 0
// and the direction block of each subgroup are generated up front, as six independent chains, while the thread's
// link loads are in flight (EarlyRandom); only rejected trials call the generator inside the data-dependent loop.
struct EarlyRandom {
    uint32_t trial0[4]; // Philox block of trial 0: u1, u2, u3, u4
    uint32_t dir[2];    // first two words of the direction block (counter word 3 = 0x80000000)
};

__device__ __forceinline__ void early_random(uint32_t key0, uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2,
                                             EarlyRandom& e)
{
    uint32_t x[4];
    philox4x32_10(c0, c1, c2, 0u, key0, key1, e.trial0);
    philox4x32_10(c0, c1, c2, 0x80000000u, key0, key1, x);
    e.dir[0] = x[0];
    e.dir[1] = x[1];
}

// returns the number of trials used (0: degenerate block, identity taken; 4097: cap hit)
template <typename T>
__device__ __forceinline__ unsigned su2_heatbath_step(const T (&k)[4], T temperature, uint32_t key0,
                                                      uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2,
                                                      const EarlyRandom& early, T (&g)[4])
{
    using M = KPMath<T>;
    const T n2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2] + k[3] * k[3];
    if (!(n2 >= Tiny<T>::sq)) { g[0] = T(1); g[1] = g[2] = g[3] = T(0); return 0u; }
    T alpha, inv_alpha, inv_n;
    M::prep(n2, temperature, alpha, inv_alpha, inv_n);
    const T kc0 = k[0] * inv_n, kc1 = -k[1] * inv_n, kc2 = -k[2] * inv_n, kc3 = -k[3] * inv_n; // conj(khat)
    // unit vector of the direction of hvec: data independent, computed ahead of the draw
    const T cos_t = T(1) - T(2) * M::uni(early.dir[0]);
    const T up = M::uni(early.dir[1]);
    const T sin_t = M::root(T(1) - cos_t * cos_t);
    const T e1 = sin_t * M::cos2pi(up), e2 = sin_t * M::sin2pi(up), e3 = cos_t;
    // trial 0 from the words generated up front: straight-line code, so that it can be scheduled together with the
    // link updates of the previous subgroup; only rejected lanes enter the loop
    T h0;
    unsigned trial = 0;
    bool accepted;
    {
        const T u1 = M::uni(early.trial0[0]), u2 = M::uni(early.trial0[1]), u3 = M::uni(early.trial0[2]),
                u4 = M::uni(early.trial0[3]);
        const T c = M::cos2pi(u3);
        const T d = M::delta(M::neglog(u1), M::neglog(u2), c, alpha, inv_alpha);
        accepted = M::accept(u4, d);
        h0 = T(1) - d;
    }
    if (!accepted) {
        uint32_t x[4];
        for (trial = 1; trial < 4096u; ++trial) {
            philox4x32_10(c0, c1, c2, trial, key0, key1, x);
            const T u1 = M::uni(x[0]), u2 = M::uni(x[1]), u3 = M::uni(x[2]), u4 = M::uni(x[3]);
            const T c = M::cos2pi(u3);
            const T d = M::delta(M::neglog(u1), M::neglog(u2), c, alpha, inv_alpha);
            if (M::accept(u4, d)) { h0 = T(1) - d; accepted = true; break; }
        }
    }
    if (!accepted) {
        // h = identity  =>  g = conj(khat)
        g[0] = kc0; g[1] = kc1; g[2] = kc2; g[3] = kc3;
        return 4097u;
    }
    const T r = M::root(T(1) - h0 * h0);
    const T h1 = r * e1, h2 = r * e2, h3 = r * e3;
    // g = h (x) conj(khat):  (pq)_0 = p0 q0 - p.q,  (pq)_vec = p0 qvec + q0 pvec - pvec x qvec   (C13)
    g[0] = h0 * kc0 - h1 * kc1 - h2 * kc2 - h3 * kc3;
    g[1] = h0 * kc1 + kc0 * h1 - (h2 * kc3 - h3 * kc2);
    g[2] = h0 * kc2 + kc0 * h2 - (h3 * kc1 - h1 * kc3);
    g[3] = h0 * kc3 + kc0 * h3 - (h1 * kc2 - h2 * kc1);
    return trial + 1u;
}

// ---------------------------------------------------------------------------------------------------------
// the half-sweep kernel
// ---------------------------------------------------------------------------------------------------------
// CB = Coulomb reading B (C12): the temporal links enter neither K nor F nor theta, they are only multiplied by
// g(x).  Instead of moving them through every half-sweep, the thread that would own them accumulates
// G(x) <- g(x) G(x) in a site field (18 reals, one link's worth instead of two) and the temporal links are
// transformed once at the end of the call, U_t(x) <- G(x) U_t(x) G(x+t)^dagger (coulomb_finish_kernel): 14/16 of the
// bytes of reading A, same result up to rounding.
template <typename T, int R, int TPS, int MODE, bool CB = false>
struct SweepKernel {
    static constexpr int NMU = 4 / TPS;
    using IO = LinkIO<T, R>;
    using GIO = LinkIO<T, 18>;

    template <int I, int J, int SUB>
    static __device__ __forceinline__ void subgroup(const SweepParams& p, cx<T> (&K)[9], cx<T> (&F)[NMU][9],
                                                    cx<T> (&B)[NMU][9], uint32_t site_canon, bool record,
                                                    const EarlyRandom& early, int lane_mu0, cx<T> (&Gt)[9])
    {
        T k[4], h[4];
        su2_project<I, J>(K, k);
        if (MODE == MODE_OVERRELAX) {
            su2_overrelax_step<T>(k, (T)p.omega, h);
        } else if (MODE == MODE_VARIANT) {
            su2_variant_step<T>(k, p.variant, p.omega, p.key0, p.key1, site_canon, p.step,
                                ((uint32_t)p.parity << 2) | (uint32_t)SUB, h);
            (void)early;
        } else {
            unsigned ntr = su2_heatbath_step<T>(k, (T)p.T, p.key0, p.key1, site_canon, p.step,
                                                ((uint32_t)p.parity << 2) | (uint32_t)SUB, early, h);
            if (record && p.trials != nullptr) p.trials[3u * (size_t)site_canon + SUB] = ntr;
        }
        const cx<T> a = {h[0], h[3]}, b = {h[2], h[1]}; // C4
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
            if (CB && lane_mu0 + m == 3) {
                su2_left<I, J>(a, b, Gt);               // G(x) <- g G(x): the temporal links wait (reading B)
            } else {
                su2_left<I, J>(a, b, F[m]);             // U_mu(x)     <- G U_mu(x)
                su2_right_dagger<I, J, 3>(a, b, B[m]);  // U_mu(x-mu)  <- U_mu(x-mu) G^dagger
            }
        }
        su2_left<I, J>(a, b, K);                        // K <- G K  (C8)
    }

    // L2 prefetch for the block that runs `prefetch` sites further along the traversal: the few fat warps of
    // an SM cannot keep enough bytes in flight while they compute, prefetches hold no register and no
    // scoreboard entry, and the 126 MB L2 is the staging buffer.  Addresses are those of this thread shifted
    // by the distance (exact for forward links, exact up to the periodic wrap for backward links: a hint).
    static __device__ __forceinline__ void issue_prefetch(const SweepParams& p, const Site& s, const unsigned (&hb)[NMU],
                                                          int lane_mu0, T* base, size_t H)
    {
        if (p.prefetch) {
            const long long d = p.reverse ? -(long long)p.prefetch : (long long)p.prefetch;
            const long long hf = (long long)s.h + d;
            if (hf >= 0 && hf < (long long)H) {
#pragma unroll
                for (int m = 0; m < NMU; ++m) {
                    const int mu = lane_mu0 + m;
                    const long long hbd = (long long)hb[m] + d;
                    if (CB && mu == 3) continue;
                    IO::prefetch(base + (size_t)(p.parity * 4 + mu) * R * H, H, (size_t)hf);
                    if (hbd >= 0 && hbd < (long long)H) IO::prefetch(base + (size_t)((1 - p.parity) * 4 + mu) * R * H, H, (size_t)hbd);
                }
            }
        }
    }

    static __device__ __forceinline__ void run(const SweepParams& p)
    {
        const unsigned blk = p.reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
        const unsigned gtid = blk * blockDim.x + threadIdx.x;
        const unsigned slot = p.h_begin + gtid / TPS;
        const int lane_mu0 = (int)(gtid % TPS) * NMU; // first direction this thread owns
        const bool active = gtid / TPS < p.h_count;        // inactive threads shadow site 0 and store nothing,
        const Site s = decode_site(p.L, active ? slot : 0u, p.parity); // so warp shuffles stay converged
        const size_t H = p.L.H;
        T* const base = reinterpret_cast<T*>(p.U);

        const MemPolicy pol = {make_l2_policy(p.ld_policy), make_l2_policy(p.st_policy)};
        cx<T> F[NMU][9], B[NMU][9];
        unsigned hb[NMU];
#pragma unroll
        for (int m = 0; m < NMU; ++m) hb[m] = backward_neighbour(p.L, s, lane_mu0 + m);
        // Programmatic dependent launch: this grid may become resident while the previous half-sweep drains
        // (its index arithmetic above overlaps that tail); links are touched only after the previous grid
        // has completed and flushed.  Letting the next grid launch early is always safe for the same reason.
        if (p.pdl) {
            cudaTriggerProgrammaticLaunchCompletion();
            cudaGridDependencySynchronize();
        }
        // the relaxation kernels prefetch before their loads (placed after them the fp64 kernel spills twice as
        // much); the heatbath kernel issues its loads first and hides the prefetch and the generator behind them
        if (MODE != MODE_HEATBATH) issue_prefetch(p, s, hb, lane_mu0, base, H);
        // issue every load before the first use
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
            const int mu = lane_mu0 + m;
            if (CB && mu == 3) continue;
            IO::load(base + (size_t)(p.parity * 4 + mu) * R * H, H, s.h, F[m], pol.ld);
            IO::load(base + (size_t)((1 - p.parity) * 4 + mu) * R * H, H, hb[m], B[m], pol.ld);
        }
        cx<T> Gt[9];
        const bool owns_t = CB && (lane_mu0 + NMU - 1 == 3); // the thread that would hold the temporal links
        if (owns_t) GIO::load(reinterpret_cast<const T*>(p.G) + (size_t)p.parity * 18 * H, H, s.h, Gt, pol.ld);
        if (MODE == MODE_HEATBATH) issue_prefetch(p, s, hb, lane_mu0, base, H);
        // heatbath: random numbers of trial 0 and of the direction, generated under the shadow of the loads
        const uint32_t sc = canonical_index(s);
        EarlyRandom early[3];
        if (MODE == MODE_HEATBATH) {
#pragma unroll
            for (int sub = 0; sub < 3; ++sub)
                early_random(p.key0, p.key1, sc, p.step, ((uint32_t)p.parity << 2) | (uint32_t)sub, early[sub]);
            // pin the 18 words here, before the first use of a loaded link: volatile asm statements keep their
            // order, so the generator runs between the issue of the loads and their consumption
#pragma unroll
            for (int sub = 0; sub < 3; ++sub)
                asm volatile("" :: "r"(early[sub].trial0[0]), "r"(early[sub].trial0[1]), "r"(early[sub].trial0[2]),
                             "r"(early[sub].trial0[3]), "r"(early[sub].dir[0]), "r"(early[sub].dir[1]));
        }
        if (p.reunit) {
#pragma unroll
            for (int m = 0; m < NMU; ++m) {
                if (CB && lane_mu0 + m == 3) continue;
                reunitarise(F[m]);
                reunitarise(B[m]);
            }
            if (owns_t) reunitarise(Gt);
        }

        // K(x) = sum_{mu < nd} [ U_mu(x) + U_mu(x-mu)^dagger ]   (eq. 2.3; C2)
        cx<T> K[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) K[e] = {T(0), T(0)};
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
            if (lane_mu0 + m < p.nd && !(CB && lane_mu0 + m == 3)) {
#pragma unroll
                for (int r = 0; r < 3; ++r)
#pragma unroll
                    for (int c = 0; c < 3; ++c) K[3 * r + c] = K[3 * r + c] + F[m][3 * r + c] + conj(B[m][3 * c + r]);
            }
        }
        if (TPS > 1) {
#pragma unroll
            for (int e = 0; e < 9; ++e) {
#pragma unroll
                for (int off = 1; off < TPS; off <<= 1) {
                    K[e].re += __shfl_xor_sync(0xffffffffu, K[e].re, off);
                    K[e].im += __shfl_xor_sync(0xffffffffu, K[e].im, off);
                }
            }
        }

        const bool record = active && (lane_mu0 == 0);
        subgroup<0, 1, 0>(p, K, F, B, sc, record, early[0], lane_mu0, Gt); // Cabibbo-Marinari subgroups, order of C4
        subgroup<0, 2, 1>(p, K, F, B, sc, record, early[1], lane_mu0, Gt);
        subgroup<1, 2, 2>(p, K, F, B, sc, record, early[2], lane_mu0, Gt);

        if (active) {
#pragma unroll
            for (int m = 0; m < NMU; ++m) {
                const int mu = lane_mu0 + m;
                if (CB && mu == 3) continue;
                IO::store(base + (size_t)(p.parity * 4 + mu) * R * H, H, s.h, F[m], pol.st);
                IO::store(base + (size_t)((1 - p.parity) * 4 + mu) * R * H, H, hb[m], B[m], pol.st);
            }
            if (owns_t) GIO::store(reinterpret_cast<T*>(p.G) + (size_t)p.parity * 18 * H, H, s.h, Gt, pol.st);
        }
    }
};

template <typename T, int R, int TPS, int MODE, bool CB = false>
__global__ void __launch_bounds__(MAX_BLOCK) gf_half_sweep_kernel(const SweepParams p)
{
    SweepKernel<T, R, TPS, MODE, CB>::run(p);
}

} // namespace gf
