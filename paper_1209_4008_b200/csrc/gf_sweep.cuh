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
#include <climits>
#include <type_traits>

#include "gf_device.cuh"

namespace gf {

enum { MODE_OVERRELAX = 0, MODE_HEATBATH = 1, MODE_VARIANT = 2 };
// MODE_VARIANT picks the SU(2) step at run time (SweepParams::variant): the update variants the paper's package
// offers beside second-order overrelaxation (readings C17, C18)
enum { VARIANT_OVERRELAX1 = 1, VARIANT_STOCHASTIC = 2 };
constexpr int MAX_BLOCK = 256;

// what changes from one half-sweep to the next
struct SweepPhase {
    int parity;      // sublattice updated: 0 = RED, 1 = BLACK (C5)
    int reunit;      // re-orthonormalise links on load (C15)
    int reverse;     // traverse blocks back to front (L2 reuse between consecutive half-sweeps)
    uint32_t step;   // Philox counter word 1: annealing step / sweep index within the call (C14, C18)
    double T;        // heatbath temperature (C13)
    int rough_slot;  // hybrid chain: position of this half-sweep in the ring of roughness flags
    int rough_force; // hybrid chain: take the double chain regardless of the flags (first sweep of a call)
};

enum { CHAIN_FP32 = 0, CHAIN_DOUBLE = 1, CHAIN_HYBRID = 2 };
constexpr int ROUGH_RING = 4;

// Device-resident state of the fused F / theta monitor (gf_fix, gf_fix_slices): written by the reduction duty of a BLACK
// half-sweep, read by every later launch (stop, frozen) and, at batch boundaries, by the host.
struct MonitorState {
    unsigned ticket;      // duty blocks that have delivered their group partial
    int stop_from;        // every half-sweep of a sweep >= stop_from returns at once (INT_MAX: none).  Stamped with the
                          // sweep it takes effect from: the duty that decides runs inside a BLACK half-sweep whose
                          // later blocks must still do their work
    int stop_sweep;       // sweep index n whose check decided the stop (stop_from = n + 2), -1: none
    int checks;           // checks completed
    int check_sweep;      // sweep index of the last completed check
    int any_active;       // slices mode: slices still active after the last check
    double theta, F;      // of the last check: theta of eq. 2.5 (Coulomb: max over the timeslices), F of eq. 2.1
};

// Fused monitor of a launch (MON kernels).  The state S_n after sweep n is covered by two kernels: the BLACK half-sweep
// of sweep n ends with K(x) of the updated links in the registers of its (BLACK) sites, and the RED half-sweep of
// sweep n + 1 builds K(x) of its (RED) sites from the links of S_n before it updates them.  Both write one partial of
// sum_x tr[Delta Delta^dagger] per block (post / pre); every link passes through registers once per half-sweep (C6),
// so BLACK_n also writes the partials of F(S_n).  The first blocks of BLACK_{n+1} then reduce these partials in a
// fixed order (no atomics on data: deterministic) and the last of them to finish forms theta(S_n), F(S_n), compares
// with the tolerance and raises `stop` / freezes timeslices, which takes effect from RED_{n+2}: the fixing loop ends
// one sweep after the sweep that met the tolerance, without a separate pass over the field and without a host sync.
struct SweepMonitor {
    double* F_part;           // [blocks] this launch writes: sum of Re tr of the links it stores, mu < nd (NULL: not)
    double* post_part;        // [blocks] this launch writes: sum tr[Delta Delta^dagger] from the final K (NULL: not)
    double* pre_part;         // [blocks] this launch writes: the same from the initial K (NULL: not)
    const double* red_F;      // reduction duty (all three NULL: none): partials of F(S_n), written by BLACK_n
    const double* red_post;   //   of the BLACK sites of S_n, written by BLACK_n
    const double* red_pre;    //   of the RED sites of S_n, written by RED_{n+1}
    double* group;            // [3][Nt][groups] scratch of the duty
    double* theta_t;          // [Nt] per-timeslice theta of the last check (Coulomb)
    int* frozen_from;         // [Nt] slices mode: first sweep (1-based) in which the slice is not updated (INT_MAX: open)
    MonitorState* state;
    int sweep;                // 1-based index of the sweep this launch belongs to
    int check_sweep;          // n of the duty
    int groups;               // duty blocks per timeslice
    int blocks_per_slice;     // partials per timeslice
    int slices;               // != 0: freeze single timeslices (gf_fix_slices), else one stop word
    int coulomb;              // theta = max over timeslices
    int zero;                 // 0 (a value the compiler cannot know: ties the stop test to the link loads)
    double tol;
    double scale_theta_t, scale_theta, scale_F; // 1/(3 Vs), 1/(3 V), 1/(3 nd V)
};

struct SweepParams {
    void* U;        // native field
    Lattice L;
    int nd;         // directions entering K: 4 (Landau) or 3 (Coulomb, C12)
    int ld_policy;  // L2 policy of the link loads / stores (POLICY_*, gf_device.cuh)
    int st_policy;
    int pdl;        // launched with programmatic stream serialization: wait for the previous grid before loading
    unsigned h_begin, h_count; // half-site range updated by this launch (whole lattice: 0, H; a run of timeslices: C20)
    unsigned prefetch; // L2 prefetch distance in sites along the traversal direction (0 = off)
    double omega;   // overrelaxation parameter; MODE_VARIANT: omega (first order) or probability p
    int variant;    // MODE_VARIANT: VARIANT_*
    uint32_t key0, key1;       // Philox key = seed (C14)
    uint32_t site_offset;      // canonical index of local site 0 in the whole lattice (t-slab contexts; else 0): the Philox
                               // counters carry the site of the whole lattice, so a sharded run draws the same numbers
    unsigned* trials;          // optional: KP trial counts, index 3*s + subgroup
    void* G;                   // Coulomb reading B (C12): accumulated g(x), 2 parity blocks of 18 reals per site
    // fp32 kernels: precision of the site chain (K(x), the three SU(2) steps, K <- G K), DESIGN.md sec. 4
    int chain;                 // CHAIN_*
    float watch_thr2;          // relaxation, CHAIN_HYBRID: a step whose conditioning number (squared) is below this marks
                               // the half-sweep rough; heatbath: a site with |k|^2 below it is redone in double
    int* rough;                // CHAIN_HYBRID: ring of ROUGH_RING flags, one per half-sweep
    unsigned long long* dc_count; // diagnostic: [0] launches that ran the double chain, [1] sites redone in double
    SweepPhase ph;
    SweepMonitor mon;          // MON kernels only
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

// cond: the conditioning number of the step, |k|^2 |h|^2 (h before its normalisation).  g = k/|k| turns an absolute
// rounding error e of K into e/|k|, the reprojection h/|h| into e/(|k||h|) (|h| falls to 0.02 at g0 = -1 for
// omega = 1.7, C9): the fp32 kernels redo a site in double where cond is small (fixup_site_f64 below).
template <typename T>
__device__ __forceinline__ void su2_overrelax_step(const T (&k)[4], T w, T (&h)[4], T& cond)
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
    cond = n2k * n2;
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
                                                 uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2, T (&h)[4],
                                                 T& cond)
{
    const T n2k = dot4(k[0], k[0], k[1], k[1], k[2], k[2], k[3], k[3]);
    cond = n2k; // first order: |h|^2 = 1 - 2 w (w-1) (g0-1) >= 1; g^2 is not normalised
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
// One Kennedy-Pendleton trial (C14) splits into a part that depends on the random numbers alone,
//     s = -ln u1 cos^2(2 pi u3) - ln u2,   u4,
// and the part that needs K:  delta = s / alpha,  accept iff u4^2 <= 1 - delta/2.  The first part of trial 0 and the unit
// vector of the direction of hvec are computed up front, while the link loads are in flight (EarlyDraw), for the three
// subgroups at once -- independent chains the scheduler can interleave; behind K only two multiplications and a
// compare are left on the critical path of a subgroup step.
template <typename DT> struct TrialPre {
    DT s;     // l1 c^2 + l2, l = -ln u
    DT lsum;  // 1 + l1 + l2: scale of the absolute error of the SFU value of s (fp32 draw only)
    float u4; // a 24-bit number: exact as a float also in the fp64 draw (one register instead of two)
};
template <typename DT> struct EarlyDraw {
    TrialPre<DT> t0;  // trial 0
    DT e1, e2;        // direction of hvec, from the Philox block with counter word 3 = 0x80000000
    float e3;         // = cos(polar angle) = 1 - 2u, a 24-bit number
};

template <typename T> struct KPMath;
// fp64: the draw is evaluated in double like the oracle's, with correctly-rounded-to-1-ulp library functions (log,
// cospi/sinpi) but without IEEE divisions and square roots (1/|k| by rsqrt, delta as one fused expression times
// 1/alpha).  The oracle's alpha already differs from the kernel's by an ulp (summation order of K), so decision
// parity rests on the size of the difference, not on the operation order: a decision flips only when u4^2 falls
// within ~1e-15 of the threshold, i.e. with probability ~1e-15 per trial (tests compare every trial count).
template <> struct KPMath<double> {
    static __device__ __forceinline__ double uni(uint32_t x) { return (double)(2u * (x >> 9) + 1u) * (1.0 / 16777216.0); }
    static __device__ __forceinline__ double neglog_w(uint32_t x) { return kp_neglog_word(x); } // -ln uni(x), gf_device.cuh
    static __device__ __forceinline__ double root(double x) { return x > 0.0 ? x * rsqrt(x) : 0.0; }
    // the angle of a trial (u3) as it enters sincos2pi; cos^2 of it from the cosine
    static __device__ __forceinline__ double trial_angle(double u3) { return u3; }
    static __device__ __forceinline__ double cos_squared(double c) { return c * c; }
    // sine and cosine of 2 pi uni(x): of the trial's angle (pair = false) and of the direction's (pair = true) alike
    static __device__ __forceinline__ void sincos_w(uint32_t x, bool dir, double& sn, double& cs) { (void)dir; kp_sincos2pi_word(x, sn, cs); }
    static __device__ __forceinline__ bool decide(const TrialPre<double>& t, double inv_alpha, double& d, double& est, bool& border)
    {
        (void)border;
        est = 0.0; // never refined
        d = t.s * inv_alpha;
        const double u4 = (double)t.u4;
        return u4 * u4 <= fma(-0.5, d, 1.0);
    }
};

// fp32: the draw runs on the SFU: u from the mantissa trick (exact), -ln u = -ln2 * lg2(u) (MUFU.LG2), cos / sin by
// MUFU.COS / SIN, one reciprocal of alpha per subgroup instead of two divisions per trial.  The SFU value of delta
// carries an absolute error of up to ~1e-6 (1 + l1 + l2)/alpha (lg2: 2 ulp, 2^-22 near 1; cos: ~4e-7), which would flip
// ~1e-6 of the accept decisions against the fp64 oracle.  Two-tier test: a trial whose u4^2 falls inside that error
// band of the threshold is BORDERLINE: the thread goes on with the fp32 decision, but its site is redone in double at
// the end (fixup_site_f64: K, the draw with 1-ulp log / cospi and the link products in double, from the stored links,
// which nobody else touches in this half-sweep, C6).  The hot path holds no double-precision code and no call; what is
// left are the flips caused by the fp32 rounding of K itself at the sites that are not redone (alpha differs at ~1e-7).
template <> struct KPMath<float> {
    // (2 (x >> 9) + 1) 2^-24 = [1 + (x >> 9) 2^-23] - (1 - 2^-24): both terms and the result are fp32 numbers
    static __device__ __forceinline__ float uni(uint32_t x) { return __uint_as_float(0x3F800000u | (x >> 9)) - 0.99999994039535522461f; }
    static __device__ __forceinline__ float neglog(float u) { return -0.693147180559945f * __log2f(u); }
    static __device__ __forceinline__ float neglog_w(uint32_t x) { return neglog(uni(x)); }
    static __device__ __forceinline__ float root(float x) { return x > 0.0f ? x * rsqrtf(x) : 0.0f; }
    // cos^2(2 pi u3) = (1 + cos(4 pi u3)) / 2, the argument folded exactly into [-pi, pi] (MUFU.COS is specified
    // there): the absolute error of c^2 is half that of the SFU cosine instead of 2 |c| times it
    static __device__ __forceinline__ float trial_angle(float u3) { const float v = 2.0f * u3; return v - rintf(v); }
    static __device__ __forceinline__ float cos_squared(float c) { return fmaf(0.5f, c, 0.5f); }
    static __device__ __forceinline__ void sincos2pi(float a, float& sn, float& cs)
    {
        const float x = 6.283185307179586f * a;
        sn = __sinf(x);
        cs = __cosf(x);
    }
    // sine and cosine of the direction's angle 2 pi uni(x) (dir) or of the trial's folded angle (cos_squared takes that cosine)
    static __device__ __forceinline__ void sincos_w(uint32_t x, bool dir, float& sn, float& cs)
    {
        const float u = uni(x);
        sincos2pi(dir ? u : trial_angle(u), sn, cs);
    }
    // delta of a trial from its uniforms with the 1-ulp library functions instead of the SFU
    static __device__ __forceinline__ float accurate_delta(const uint32_t (&x)[4], float inv_alpha)
    {
        const float l1 = -logf(uni(x[0])), l2 = -logf(uni(x[1]));
        const float c = cospif(2.0f * uni(x[2]));
        return fmaf(l1, c * c, l2) * inv_alpha;
    }
    // est: inv_alpha (1 + l1 + l2), the scale of the absolute error of the SFU value of delta (in units of ~5e-7)
    static __device__ __forceinline__ bool decide(const TrialPre<float>& t, float inv_alpha, float& d, float& est, bool& border)
    {
        d = t.s * inv_alpha;
        const float diff = fmaf(t.u4, t.u4, fmaf(0.5f, d, -1.0f)); // u4^2 - (1 - delta/2)
        est = inv_alpha * t.lsum;
        border = border || fabsf(diff) < fmaf(2e-6f, est, 3e-7f);
        return diff <= 0.0f;
    }
};

// the K-independent part of one trial from its Philox block (u1, u2, u3, u4)
template <typename DT>
__device__ __forceinline__ TrialPre<DT> kp_trial_pre(const uint32_t (&x)[4])
{
    using M = KPMath<DT>;
    DT sn, cs;
    M::sincos_w(x[2], false, sn, cs);
    (void)sn;
    const DT l1 = M::neglog_w(x[0]), l2 = M::neglog_w(x[1]);
    TrialPre<DT> t;
    t.s = gf_fma(l1, M::cos_squared(cs), l2);
    t.lsum = DT(1) + l1 + l2;
    t.u4 = KPMath<float>::uni(x[3]);
    return t;
}

// The Philox counters of a draw hold (site, step, parity, subgroup, trial) and no data, so trial 0 and the direction
// of each subgroup are prepared up front, as independent chains, while the thread's link loads are in flight; only
// rejected trials call the generator inside the data-dependent loop.
template <typename DT>
__device__ __forceinline__ void early_draw(uint32_t key0, uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2, EarlyDraw<DT>& e)
{
    using M = KPMath<DT>;
    uint32_t x[4];
    philox4x32_10(c0, c1, c2, 0u, key0, key1, x);
    e.t0 = kp_trial_pre<DT>(x);
    philox4x32_10(c0, c1, c2, 0x80000000u, key0, key1, x);
    const DT cos_t = DT(1) - DT(2) * M::uni(x[0]);
    const DT sin_t = M::root(DT(1) - cos_t * cos_t);
    DT sn, cs;
    M::sincos_w(x[1], true, sn, cs);
    e.e1 = sin_t * cs;
    e.e2 = sin_t * sn;
    e.e3 = (float)cos_t;
}

// The same for kernels in which two (or four) threads share a site: the two lanes of a pair (lane, lane ^ 1) run ONE
// instruction stream on different data and exchange the results -- role 0 generates the Philox block of trial 0, takes
// -ln u1 and the cosine of the trial; role 1 generates the direction block, takes -ln u2 and sine / cosine of the
// direction: one generator call, one logarithm and one sincos per thread instead of two, two and two.
template <typename DT> struct Shfl;
template <> struct Shfl<float> {
    static __device__ __forceinline__ float get(unsigned mask, float v, int src) { return __shfl_sync(mask, v, src); }
};
template <> struct Shfl<double> {
    static __device__ __forceinline__ double get(unsigned mask, double v, int src) { return __shfl_sync(mask, v, src); }
};

template <typename DT>
__device__ __forceinline__ void early_draw_pair(uint32_t key0, uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2, unsigned mask,
                                                EarlyDraw<DT>& e)
{
    using M = KPMath<DT>;
    const int lane = (int)(threadIdx.x & 31u), src0 = lane & ~1, src1 = lane | 1;
    const bool role = (lane & 1) != 0;
    uint32_t y[4];
    philox4x32_10(c0, c1, c2, role ? 0x80000000u : 0u, key0, key1, y);
    const uint32_t x1 = __shfl_sync(mask, y[1], src0); // u2 and u4 of the trial, generated by role 0
    const uint32_t x3 = __shfl_sync(mask, y[3], src0);
    const DT l = M::neglog_w(role ? x1 : y[0]);
    DT sn, cs;
    M::sincos_w(role ? y[1] : y[2], role, sn, cs);
    const DT cos_t = DT(1) - DT(2) * M::uni(y[0]); // meaningful on role 1
    const DT sin_t = M::root(DT(1) - cos_t * cos_t);
    const DT l1 = Shfl<DT>::get(mask, l, src0), l2 = Shfl<DT>::get(mask, l, src1);
    e.t0.s = gf_fma(l1, M::cos_squared(Shfl<DT>::get(mask, cs, src0)), l2);
    e.t0.lsum = DT(1) + l1 + l2;
    e.t0.u4 = KPMath<float>::uni(x3);
    e.e1 = Shfl<DT>::get(mask, sin_t * cs, src1);
    e.e2 = Shfl<DT>::get(mask, sin_t * sn, src1);
    e.e3 = Shfl<float>::get(mask, (float)cos_t, src1);
}

// returns the number of trials used (0: degenerate block, identity taken; 4097: cap hit); cond = |k|^2 (the
// conditioning number of g = h (x) conj(khat), see su2_overrelax_step).
// CT: type of the site chain (k, khat = k/|k|, g -- the ill-conditioned part); DT: type of the draw (alpha, the
// Kennedy-Pendleton trials, h).  (double, float): fp32 kernels with the chain in double, the draw on the SFU.
// redo (fp32 draw): set where the SFU draw is not good enough for this site -- a borderline accept test (KPMath<float>)
// or an accepted delta whose SFU error would move the links by more than ~1e-5 -- and the site is to be redone in double.
// PAIR: the lanes (lane, lane ^ 1) hold the same site (identical K, bit for bit, so identical decisions): the retry
// loop evaluates two trials per pass, trial t on the even lane and t + 1 on the odd one, and takes the first accepted.
template <typename CT, typename DT, bool PAIR>
__device__ __forceinline__ unsigned su2_heatbath_step(const CT (&k)[4], double Td, uint32_t key0,
                                                      uint32_t key1, uint32_t c0, uint32_t c1, uint32_t c2,
                                                      const EarlyDraw<DT>& early, CT (&g)[4], CT& cond, bool& redo)
{
    using M = KPMath<DT>;
    const CT n2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2] + k[3] * k[3];
    cond = n2;
    if (!(n2 >= Tiny<CT>::sq)) { g[0] = CT(1); g[1] = g[2] = g[3] = CT(0); return 0u; }
    // no division, no IEEE square root: 1/|k| by rsqrt (fp32: MUFU.RSQ + one Newton step), 1/alpha = T/|k| from it
    const CT inv_n = gf_rsqrt<CT>(n2);
    const DT inv_alpha = (DT)((CT)Td * inv_n);
    const CT kc0 = k[0] * inv_n, kc1 = -k[1] * inv_n, kc2 = -k[2] * inv_n, kc3 = -k[3] * inv_n; // conj(khat)
    // trial 0 from the values prepared up front: straight-line code, so that it can be scheduled together with the
    // link updates of the previous subgroup; only rejected lanes enter the loop
    DT d, est;
    unsigned trial = 0;
    bool accepted = M::decide(early.t0, inv_alpha, d, est, redo);
    if (!accepted) {
        if (PAIR) {
            const int lane = (int)(threadIdx.x & 31u), src0 = lane & ~1, src1 = lane | 1;
            const unsigned pair = 3u << src0;
            const unsigned role = (unsigned)(lane & 1);
            for (unsigned t = 1; t < 4096u; t += 2) {
                uint32_t x[4];
                philox4x32_10(c0, c1, c2, t + role, key0, key1, x);
                DT dm, em;
                bool bm = false;
                const bool am = M::decide(kp_trial_pre<DT>(x), inv_alpha, dm, em, bm) && (t + role < 4096u);
                const unsigned acc = __ballot_sync(pair, am) >> src0;      // bit 0: trial t, bit 1: trial t + 1
                const unsigned bor = __ballot_sync(pair, bm) >> src0;
                if (bor & (1u | ((acc & 1u) ? 0u : 2u))) redo = true;      // trial t + 1 counts only if trial t was rejected
                if (acc & 3u) {
                    const int from = (acc & 1u) ? src0 : src1;
                    d = Shfl<DT>::get(pair, dm, from);
                    est = Shfl<DT>::get(pair, em, from);
                    trial = t + ((acc & 1u) ? 0u : 1u);
                    accepted = true;
                    break;
                }
            }
        } else {
            uint32_t x[4];
            for (trial = 1; trial < 4096u; ++trial) {
                philox4x32_10(c0, c1, c2, trial, key0, key1, x);
                if (M::decide(kp_trial_pre<DT>(x), inv_alpha, d, est, redo)) { accepted = true; break; }
            }
        }
    }
    if (!accepted) {
        // h = identity  =>  g = conj(khat)
        g[0] = kc0; g[1] = kc1; g[2] = kc2; g[3] = kc3;
        return 4097u;
    }
    // fp32 draw: the SFU value of the accepted delta is off by ~5e-7 est, which moves h0 by as much and hvec, of
    // length r = sqrt(delta (2 - delta)), by that over r.  Where this is too much for the links (est > 16 r: more than
    // ~8e-6; small alpha, large -ln u, h0 near +-1: 6e-4 of the draws at T = 1.4, none once alpha > 10) delta is taken
    // again from the uniforms of the accepted trial with the 1-ulp functions (logf, cospif: ~1.5e-7 est), a few dozen
    // instructions inline; only where even that is too coarse (est > 64 r, 1e-5 of the draws) the site is redone in double
    if constexpr (sizeof(DT) == 4) {
        if (est * est > DT(256) * fmin(d * (DT(2) - d), DT(1))) {
            uint32_t x[4];
            philox4x32_10(c0, c1, c2, trial, key0, key1, x);
            d = M::accurate_delta(x, inv_alpha);
            redo = redo || est * est > DT(4096) * fmin(d * (DT(2) - d), DT(1));
        }
    }
    const DT h0d = DT(1) - d;
    const DT r = M::root(d * (DT(2) - d)); // = sqrt(1 - h0^2) without the cancellation at small delta
    const CT h0 = (CT)h0d, h1 = (CT)(r * early.e1), h2 = (CT)(r * early.e2), h3 = (CT)(r * (DT)early.e3);
    // g = h (x) conj(khat):  (pq)_0 = p0 q0 - p.q,  (pq)_vec = p0 qvec + q0 pvec - pvec x qvec   (C13)
    g[0] = h0 * kc0 - h1 * kc1 - h2 * kc2 - h3 * kc3;
    g[1] = h0 * kc1 + kc0 * h1 - (h2 * kc3 - h3 * kc2);
    g[2] = h0 * kc2 + kc0 * h2 - (h3 * kc1 - h1 * kc3);
    g[3] = h0 * kc3 + kc0 * h3 - (h1 * kc2 - h2 * kc1);
    return trial + 1u;
}

// ---------------------------------------------------------------------------------------------------------
// fp32 heatbath kernels, rare path: the whole site update in double.
// g = h (x) conj(khat) with khat = k/|k| is ill-conditioned where the projected block is small: the fp32 rounding of K
// (~1e-6) then moves the links by ~1e-6/|k|.  (For the heatbath there is no second small factor, and a BLACK site
// inherits only ~1e-6 from its RED neighbours, so unlike the relaxation sweeps a per-site repair is enough here.)  A
// thread whose |k|^2 fell below SweepParams::watch_thr2 in one of its three subgroup steps, or whose SFU draw was not
// good enough (KPMath<float>), drops its fp32 result and redoes the site here from the stored fp32 links (untouched so
// far: within a half-sweep only this site writes them, C6): K, the three SU(2) steps with the draw in double (same
// arithmetic as the fp64 kernel's), K <- G K and the link products all in double, one rounding to fp32 at the store.
// Every thread of a site takes the same decision (K is bit-identical on them) and redoes its own links; no shuffles
// on this divergent path: each thread builds K for itself.  DESIGN.md sec. 4.
//
// This code runs at ~1e-5 of the sites, i.e. a few dozen times per launch of a 7 M-site lattice, and each time it is COLD:
// its instructions come from L2 or DRAM, ~1 us per 128-byte line (8 instructions), and the block that runs it holds up
// the end of its launch.  So it is written for size, not speed: rolled loops, run-time subgroup indices on arrays in
// local memory, one copy of the trial code (trial 0 is the first pass of the loop), the three SU(2) factors accumulated
// into one 3x3 matrix G = G3 G2 G1 that is applied to the links in a rolled loop (C8: equal to applying them one after
// the other up to rounding, here in double).  Unrolled like the hot path it was 4600 instructions (74 KB) and cost
// 48^3x64 fp32 annealing 13 % through launch tails; profiles/r2_heatbath.md.
// ---------------------------------------------------------------------------------------------------------
// one SU(2) heatbath step in double on the projected block k: the arithmetic of su2_heatbath_step<double, double, false>
// with trial 0 taken inside the loop (one copy of the generator and of the logarithms)
static __device__ __noinline__ unsigned fix_heatbath_step(const double (&k)[4], double Td, uint32_t key0, uint32_t key1, uint32_t c0,
                                                   uint32_t c1, uint32_t c2, double (&g)[4])
{
    using M = KPMath<double>;
    const double n2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2] + k[3] * k[3];
    if (!(n2 >= Tiny<double>::sq)) { g[0] = 1.0; g[1] = g[2] = g[3] = 0.0; return 0u; }
    const double inv_n = gf_rsqrt<double>(n2);
    const double inv_alpha = Td * inv_n;
    const double kc0 = k[0] * inv_n, kc1 = -k[1] * inv_n, kc2 = -k[2] * inv_n, kc3 = -k[3] * inv_n; // conj(khat)
    uint32_t x[4];
    double d = 0.0, est;
    bool accepted = false, border = false;
    unsigned trial = 0;
#pragma unroll 1
    for (; trial < 4096u; ++trial) {
        philox4x32_10(c0, c1, c2, trial, key0, key1, x);
        if (M::decide(kp_trial_pre<double>(x), inv_alpha, d, est, border)) { accepted = true; break; }
    }
    if (!accepted) { g[0] = kc0; g[1] = kc1; g[2] = kc2; g[3] = kc3; return 4097u; } // h = identity
    philox4x32_10(c0, c1, c2, 0x80000000u, key0, key1, x);
    const double cos_t = 1.0 - 2.0 * M::uni(x[0]);
    const double sin_t = M::root(1.0 - cos_t * cos_t);
    double sn, cs;
    M::sincos_w(x[1], true, sn, cs);
    const double r = M::root(d * (2.0 - d));
    const double h0 = 1.0 - d, h1 = r * (sin_t * cs), h2 = r * (sin_t * sn), h3 = r * cos_t;
    g[0] = h0 * kc0 - h1 * kc1 - h2 * kc2 - h3 * kc3; // g = h (x) conj(khat)  (C13)
    g[1] = h0 * kc1 + kc0 * h1 - (h2 * kc3 - h3 * kc2);
    g[2] = h0 * kc2 + kc0 * h2 - (h3 * kc1 - h1 * kc3);
    g[3] = h0 * kc3 + kc0 * h3 - (h1 * kc2 - h2 * kc1);
    return trial + 1u;
}

static __device__ __noinline__ void fix_reunit(cx<double> (&u)[9]) { reunitarise(u); }

// stored fp32 entries -> double, third row rebuilt (R = 12), rows re-orthonormalised on a reunitarisation sweep
template <int R>
__device__ __forceinline__ void fix_widen(const cx<float> (&v)[9], int reunit, cx<double> (&u)[9])
{
#pragma unroll
    for (int e = 0; e < R / 2; ++e) u[e] = {(double)v[e].re, (double)v[e].im};
    if (R == 12) rebuild_row2(u);
    if (reunit) fix_reunit(u);
}

// w = G u (dagger = false) or w = u G^dagger (dagger = true)
template <bool DAGGER>
__device__ __forceinline__ void fix_mul(const cx<double> (&G)[9], const cx<double> (&u)[9], cx<double> (&w)[9])
{
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            cx<double> acc = {0.0, 0.0};
#pragma unroll
            for (int k = 0; k < 3; ++k) acc = acc + (DAGGER ? cmul_cb(u[3 * r + k], G[3 * c + k]) : G[3 * r + k] * u[3 * k + c]);
            w[3 * r + c] = acc;
        }
}

template <int I, int J, int SUB>
__device__ __forceinline__ void fix_subgroup(const SweepParams& p, const SweepPhase& ph, uint32_t sc, bool record, cx<double> (&K)[9],
                                             cx<double> (&G)[9])
{
    double k[4], g[4];
    su2_project<I, J>(K, k);
    const unsigned ntr = fix_heatbath_step(k, ph.T, p.key0, p.key1, sc, ph.step, ((uint32_t)ph.parity << 2) | (uint32_t)SUB, g);
    if (record && p.trials != nullptr) p.trials[3u * (size_t)(sc - p.site_offset) + SUB] = ntr;
    const cx<double> a = {g[0], g[3]}, b = {g[2], g[1]}; // C4
    su2_left<I, J>(a, b, K); // K <- g K  (C8)
    su2_left<I, J>(a, b, G); // G <- g G
}

// The links of the site are fetched ONCE, all together (the block runs in a saturated memory system: every dependent
// round trip costs microseconds), kept as the stored floats, and widened where they are used: for K, then again for the
// products G U, U G^dagger with the accumulated G = g3 g2 g1.
template <int R, int TPS, bool CB>
__device__ __noinline__ void fixup_site_f64(const SweepParams& p, const SweepPhase& ph, unsigned h, int lane_mu0)
{
    constexpr int NMU = 4 / TPS;
    using IO = LinkIO<float, R>;
    using GIO = LinkIO<float, 18>;
    const Site s = decode_site(p.L, h, ph.parity);
    const size_t Hp = p.L.Hp;
    float* const base = reinterpret_cast<float*>(p.U);
    const uint64_t ld = make_l2_policy(POLICY_NORMAL), st = make_l2_policy(p.st_policy);
    cx<float> F[4][9], B[4][9], Gs[9];
    unsigned hb[4];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        hb[mu] = backward_neighbour(p.L, s, mu);
        if (CB && mu == 3) continue;
        IO::load_stored(base + (size_t)(ph.parity * 4 + mu) * R * Hp, Hp, s.h, F[mu], ld);
        IO::load_stored(base + (size_t)((1 - ph.parity) * 4 + mu) * R * Hp, Hp, hb[mu], B[mu], ld);
    }
    const bool owns_t = CB && lane_mu0 + NMU - 1 == 3;
    float* const gb = reinterpret_cast<float*>(p.G) + (size_t)ph.parity * 18 * Hp;
    if (owns_t) GIO::load_stored(gb, Hp, s.h, Gs, ld);
    cx<double> K[9], G[9], u[9], w[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) { K[e] = {0.0, 0.0}; G[e] = {(e & 3) == 0 ? 1.0 : 0.0, 0.0}; }
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) { // eq. 2.3 (C2), every direction entering K
        if (mu >= p.nd || (CB && mu == 3)) continue;
        fix_widen<R>(F[mu], ph.reunit, u);
#pragma unroll
        for (int e = 0; e < 9; ++e) K[e] = K[e] + u[e];
        fix_widen<R>(B[mu], ph.reunit, u);
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) K[3 * r + c] = K[3 * r + c] + conj(u[3 * c + r]);
    }
    const uint32_t sc = canonical_index(s) + p.site_offset;
    const bool record = lane_mu0 == 0;
    fix_subgroup<0, 1, 0>(p, ph, sc, record, K, G); // Cabibbo-Marinari subgroups, order of C4
    fix_subgroup<0, 2, 1>(p, ph, sc, record, K, G);
    fix_subgroup<1, 2, 2>(p, ph, sc, record, K, G);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        if (mu < lane_mu0 || mu >= lane_mu0 + NMU || (CB && mu == 3)) continue;
        fix_widen<R>(F[mu], ph.reunit, u);
        fix_mul<false>(G, u, w); // U_mu(x) <- G U_mu(x)
        IO::store(base + (size_t)(ph.parity * 4 + mu) * R * Hp, Hp, s.h, w, st);
        fix_widen<R>(B[mu], ph.reunit, u);
        fix_mul<true>(G, u, w);  // U_mu(x-mu) <- U_mu(x-mu) G^dagger
        IO::store(base + (size_t)((1 - ph.parity) * 4 + mu) * R * Hp, Hp, hb[mu], w, st);
    }
    if (owns_t) { // reading B: G(x) <- g G(x)
        fix_widen<18>(Gs, ph.reunit, u);
        fix_mul<false>(G, u, w);
        GIO::store(gb, Hp, s.h, w, st);
    }
    if (p.dc_count != nullptr && lane_mu0 == 0) atomicAdd(p.dc_count + 1, 1ull);
}
__device__ __forceinline__ void pin_early(const EarlyDraw<float>& e)
{
    asm volatile("" :: "f"(e.t0.s), "f"(e.t0.lsum), "f"(e.t0.u4), "f"(e.e1), "f"(e.e2), "f"(e.e3));
}
__device__ __forceinline__ void pin_early(const EarlyDraw<double>& e)
{
    asm volatile("" :: "d"(e.t0.s), "f"(e.t0.u4), "d"(e.e1), "d"(e.e2), "f"(e.e3));
}

__device__ __forceinline__ int tie_bits(float x) { return __float_as_int(x); }
__device__ __forceinline__ int tie_bits(double x) { return __double2hiint(x); }

// ---------------------------------------------------------------------------------------------------------
// the half-sweep kernel
// ---------------------------------------------------------------------------------------------------------
// CB = Coulomb reading B (C12): the temporal links enter neither K nor F nor theta, they are only multiplied by
// g(x).  Instead of moving them through every half-sweep, the thread that would own them accumulates
// G(x) <- g(x) G(x) in a site field (18 reals, one link's worth instead of two) and the temporal links are
// transformed once at the end of the call, U_t(x) <- G(x) U_t(x) G(x+t)^dagger (coulomb_finish_kernel): 14/16 of the
// bytes of reading A, same result up to rounding.
//
// fp32 kernels, precision of the site chain.  The links are fp32 in memory and in the link
// products; the site chain -- K(x), the three SU(2) steps, K <- G K -- is ill-conditioned where the projected block
// k or the expanded g^omega is small (g = k/|k|, h/|h|): in fp32 its rounding (~1e-6 on K) moves the links by ~1e-6
// / (|k||h|), and the BLACK half-sweep inherits the errors of the RED one through its own K.  On a random-gauge
// start that breaks north_star's 5e-5 per link at ~1e-5 of the sites; a per-site repair cannot help the BLACK sites
// (their error is in their input).  So the chain runs in double (CT = double: K accumulated exactly from the fp32
// links, G rounded to fp32 once) while the field is rough, and in fp32 once it is smooth: every half-sweep records
// whether any of its steps had a conditioning number |k|^2 |h|^2 below watch_thr2, and a half-sweep takes the
// double chain iff one of the two half-sweeps before it was rough (or the host forces it: the first sweep of every
// call).  The decision is a deterministic function of the field; on a nearly fixed field (|k| ~ 10, |h| ~ 1)
// no launch takes the double chain.  The heatbath kernels keep the fp32 chain and repair single sites instead
// (fixup_site_f64 above).
// DC (fp32 heatbath kernels only): the double chain at every site, for annealing runs in which every link has to meet
// the per-link bound (gf_set_chain(ctx, 1, ..)); the default heatbath kernel keeps the fp32 chain.
// MON (relaxation kernels only): fused F / theta monitor, SweepMonitor above.  0: none; 1: the launch only honours the
// stop / the frozen timeslices (the sweeps between two checks); 2: it also writes partials and / or has the duty.
template <typename T, int R, int TPS, int MODE, bool CB = false, bool DC = false, int MON = 0>
struct SweepKernel {
    static constexpr int NMU = 4 / TPS;
    static constexpr bool FP32 = sizeof(T) == 4;
    static constexpr bool HYB = FP32 && MODE != MODE_HEATBATH;        // relaxation sweeps: chain type chosen per launch
    static constexpr bool FIX = FP32 && MODE == MODE_HEATBATH;        // heatbath: weak sites and weak draws redone in double
    // ACC: the three SU(2) factors of a site are accumulated into G = g3 g2 g1 and applied to the links once (C8): 108
    // multiply-adds per link instead of 144, but nothing independent is left to schedule beside the serial chain of the
    // next subgroup step.  Measured (profiles/r2_variants.md E): pays for the relaxation kernels (+2..5 %) and the fp32
    // 12-real heatbath kernel, costs the other heatbath kernels 4..6 %, whose chain is longer.
#ifdef GF_ACCG
    static constexpr bool ACC = ((GF_ACCG & 1) && R == 12) || ((GF_ACCG & 2) && MODE == MODE_HEATBATH) || (GF_ACCG & 4);
#else
    static constexpr bool ACC = MODE != MODE_HEATBATH || (sizeof(T) == 4 && R == 12);
#endif
    static constexpr int OUT_ROWS = (R == 12 && MON == 0) ? 2 : 3; // rows of an updated link that anybody reads
    static constexpr bool PAIR = MODE == MODE_HEATBATH && TPS >= 2;   // heatbath: two lanes of a site share the work of the draw
    static_assert(!DC || (FP32 && MODE == MODE_HEATBATH), "DC is a variant of the fp32 heatbath kernel");
    static_assert(MON == 0 || MODE != MODE_HEATBATH, "the monitor belongs to the relaxation sweeps");
    using IO = LinkIO<T, R>;
    using GIO = LinkIO<T, 18>;

    // one SU(2) subgroup step on the chain type CT
    template <typename CT, int I, int J, int SUB>
    static __device__ __forceinline__ void subgroup(const SweepParams& p, const SweepPhase& ph, cx<CT> (&K)[9],
                                                    cx<T> (&F)[NMU][9], cx<T> (&B)[NMU][9], uint32_t site_canon,
                                                    bool record, const EarlyDraw<T>& early, int lane_mu0,
                                                    cx<T> (&Gt)[9], bool& watch, cx<CT> (&Gacc)[9])
    {
        CT k[4], h[4], cond;
        su2_project<I, J>(K, k);
        const uint32_t c2 = ((uint32_t)ph.parity << 2) | (uint32_t)SUB;
        if (MODE == MODE_OVERRELAX) {
            su2_overrelax_step<CT>(k, (CT)p.omega, h, cond);
        } else if (MODE == MODE_VARIANT) {
            su2_variant_step<CT>(k, p.variant, p.omega, p.key0, p.key1, site_canon, ph.step, c2, h, cond);
            (void)early;
        } else {
            bool redo = false;
            unsigned ntr = su2_heatbath_step<CT, T, PAIR>(k, ph.T, p.key0, p.key1, site_canon, ph.step, c2, early, h, cond, redo);
            if (record && p.trials != nullptr) p.trials[3u * (size_t)(site_canon - p.site_offset) + SUB] = ntr;
            if (FP32) watch = watch || (redo && p.watch_thr2 >= 0.0f); // a negative threshold: no repairs at all (CHAIN_FP32)
        }
        if (FP32 && !DC) watch = watch || ((float)cond < p.watch_thr2);
        const cx<CT> ac = {h[0], h[3]}, bc = {h[2], h[1]}; // C4
        const cx<T> a = {(T)h[0], (T)h[3]}, b = {(T)h[2], (T)h[1]};
        if (ACC) {
            su2_left<I, J>(ac, bc, Gacc);               // G <- g G: applied to the links after the third step
        } else {
#pragma unroll
            for (int m = 0; m < NMU; ++m) {
                if (CB && lane_mu0 + m == 3) {
                    su2_left<I, J>(a, b, Gt);               // G(x) <- g G(x): the temporal links wait (reading B)
                } else {
                    su2_left<I, J>(a, b, F[m]);             // U_mu(x)     <- G U_mu(x)
                    su2_right_dagger<I, J, 3>(a, b, B[m]);  // U_mu(x-mu)  <- U_mu(x-mu) G^dagger
                }
            }
        }
        su2_left<I, J>(ac, bc, K);                      // K <- G K  (C8)
    }

    // the site chain on the type CT: K(x) from the loaded links, then the three subgroup steps (each applies its G to
    // the links at once, Alg. 1's data flow, C8)
    // mon_skip (MON): the launch is past its stop or the timeslice is frozen; returns false if nothing was updated
    template <typename CT>
    static __device__ __forceinline__ bool chain(const SweepParams& p, const SweepPhase& ph, cx<T> (&F)[NMU][9],
                                                 cx<T> (&B)[NMU][9], cx<T> (&Gt)[9], uint32_t sc,
                                                 const EarlyDraw<T> (&early)[3], int lane_mu0, unsigned mask, bool& watch,
                                                 double& th_pre, double& th_post, int mon_skip)
    {
        // K(x) = sum_{mu < nd} [ U_mu(x) + U_mu(x-mu)^dagger ]   (eq. 2.3; C2)
        cx<CT> K[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) K[e] = {CT(0), CT(0)};
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
            if (lane_mu0 + m < p.nd && !(CB && lane_mu0 + m == 3)) {
#pragma unroll
                for (int r = 0; r < 3; ++r)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        K[3 * r + c].re = (K[3 * r + c].re + (CT)F[m][3 * r + c].re) + (CT)B[m][3 * c + r].re;
                        K[3 * r + c].im = (K[3 * r + c].im + (CT)F[m][3 * r + c].im) - (CT)B[m][3 * c + r].im;
                    }
            }
        }
        if (TPS > 1) {
#pragma unroll
            for (int e = 0; e < 9; ++e) {
#pragma unroll
                for (int off = 1; off < TPS; off <<= 1) {
                    K[e].re += __shfl_xor_sync(mask, K[e].re, off);
                    K[e].im += __shfl_xor_sync(mask, K[e].im, off);
                }
            }
        }
        if (MON) {
            // The test is tied to K (zero is 0, but only the host knows), i.e. to every link load having been issued and
            // answered -- which the first subgroup step needs anyway.  A test on the flag alone is moved ahead of the link
            // loads by ptxas (it sinks them below the branch), and every block then waits for the flag before it asks
            // for its links: +15 % on the whole sweep.
            mon_skip |= tie_bits(K[0].re) & p.mon.zero;
            if (mon_skip) return false;
        }
        const bool record = lane_mu0 == 0;
        if (MON == 2 && p.mon.pre_part != nullptr) th_pre = record ? site_theta(K) : 0.0;
        cx<CT> Gacc[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) Gacc[e] = {(e & 3) == 0 ? CT(1) : CT(0), CT(0)};
        subgroup<CT, 0, 1, 0>(p, ph, K, F, B, sc, record, early[0], lane_mu0, Gt, watch, Gacc); // Cabibbo-Marinari subgroups, order of C4
        subgroup<CT, 0, 2, 1>(p, ph, K, F, B, sc, record, early[1], lane_mu0, Gt, watch, Gacc);
        subgroup<CT, 1, 2, 2>(p, ph, K, F, B, sc, record, early[2], lane_mu0, Gt, watch, Gacc);
        if (ACC) {
            cx<T> G[9]; // rounded to the type of the links once
#pragma unroll
            for (int e = 0; e < 9; ++e) G[e] = {(T)Gacc[e].re, (T)Gacc[e].im};
#pragma unroll
            for (int m = 0; m < NMU; ++m) {
                if (CB && lane_mu0 + m == 3) {
                    mat_left<3>(G, Gt);                       // G(x) <- G G(x)  (reading B)
                } else {
                    mat_left<OUT_ROWS>(G, F[m]);              // U_mu(x)     <- G U_mu(x)
                    mat_right_dagger<OUT_ROWS>(G, B[m]);      // U_mu(x-mu)  <- U_mu(x-mu) G^dagger
                }
            }
        }
        if (MON == 2 && p.mon.post_part != nullptr) th_post = record ? site_theta(K) : 0.0;
        return true;
    }

    // tr[Delta Delta^dagger] at one site from its K (eq. 2.5; C3): Delta = traceless part of (K - K^dagger)/(2i)
    template <typename CT>
    static __device__ __forceinline__ double site_theta(const cx<CT> (&K)[9])
    {
        const CT tr3 = (K[0].im + K[4].im + K[8].im) * CT(1.0 / 3.0);
        CT acc = CT(0);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const CT d = K[4 * a].im - tr3;
            acc += d * d;
        }
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = a + 1; b < 3; ++b) {
                const CT dr = CT(0.5) * (K[3 * a + b].im + K[3 * b + a].im);
                const CT di = CT(0.5) * (K[3 * a + b].re - K[3 * b + a].re);
                acc += CT(2) * (dr * dr + di * di); // Delta is Hermitian: |D_ab|^2 = |D_ba|^2
            }
        return (double)acc;
    }

    // sum over the block; the result is valid in thread 0.  Fixed tree: deterministic.
    static __device__ __forceinline__ double block_sum(double v, double* smem)
    {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
        if (blockDim.x <= 32) return v;
        __syncthreads();
        if ((threadIdx.x & 31) == 0) smem[threadIdx.x >> 5] = v;
        __syncthreads();
        double acc = 0.0;
        if (threadIdx.x == 0)
            for (unsigned w = 0; w < (blockDim.x + 31) / 32; ++w) acc += smem[w];
        return acc;
    }

    // The reduction duty of a BLACK half-sweep (SweepMonitor): duty block j = (t, g) adds its share of the partials
    // of timeslice t, the last block to deliver adds the groups, forms theta and F of S_n and decides.
    static __device__ __noinline__ void monitor_duty(const SweepMonitor& m, int Nt, unsigned j)
    {
        __shared__ double smem[3][MAX_BLOCK / 32];
        __shared__ unsigned last;
        const int t = (int)j / m.groups, g = (int)j % m.groups;
        const int chunk = (m.blocks_per_slice + m.groups - 1) / m.groups;
        const int i0 = g * chunk, i1 = min(i0 + chunk, m.blocks_per_slice);
        double f = 0.0, po = 0.0, pr = 0.0;
        if (!(m.slices && m.frozen_from[t] <= m.check_sweep + 1)) { // the slice was still updated in sweep n + 1
            const size_t base = (size_t)t * m.blocks_per_slice;
            for (int i = i0 + (int)threadIdx.x; i < i1; i += (int)blockDim.x) {
                f += m.red_F[base + i];
                po += m.red_post[base + i];
                pr += m.red_pre[base + i];
            }
        }
        f = block_sum(f, smem[0]);
        po = block_sum(po, smem[1]);
        pr = block_sum(pr, smem[2]);
        if (threadIdx.x == 0) {
            double* grp = m.group + ((size_t)t * m.groups + g) * 3;
            grp[0] = f; grp[1] = po; grp[2] = pr;
            __threadfence();
            last = atomicAdd(&m.state->ticket, 1u) == (unsigned)(Nt * m.groups) - 1u;
        }
        __syncthreads();
        if (!last) return;
        __threadfence();
        // per-timeslice sums in a fixed order (thread t', t' + blockDim, ...), kept in theta_t / group[..][0]
        for (int tt = (int)threadIdx.x; tt < Nt; tt += (int)blockDim.x) {
            if (m.slices && m.frozen_from[tt] <= m.check_sweep + 1) continue; // a frozen slice keeps its last values
            const volatile double* grp = m.group + (size_t)tt * m.groups * 3;
            double ft = 0.0, tht = 0.0;
            for (int gg = 0; gg < m.groups; ++gg) { ft += grp[3 * gg]; tht += grp[3 * gg + 1] + grp[3 * gg + 2]; }
            m.theta_t[tt] = tht * m.scale_theta_t;
            m.theta_t[Nt + tt] = ft; // raw F of the slice
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double sum_th = 0.0, max_th = 0.0, sum_F = 0.0;
            int active = 0;
            for (int tt = 0; tt < Nt; ++tt) {
                const double th = m.theta_t[tt];
                sum_th += th;
                if (tt == 0 || th > max_th) max_th = th;
                sum_F += m.theta_t[Nt + tt];
                if (m.slices) {
                    if (m.frozen_from[tt] == INT_MAX && th < m.tol) m.frozen_from[tt] = m.check_sweep + 2;
                    active += m.frozen_from[tt] == INT_MAX ? 1 : 0;
                }
            }
            MonitorState* st = m.state;
            st->theta = m.coulomb ? max_th : sum_th / (double)Nt; // slices of equal volume: the mean of theta_t is theta
            st->F = sum_F * m.scale_F;
            st->check_sweep = m.check_sweep;
            st->checks += 1;
            st->any_active = active;
            const bool done = m.slices ? active == 0 : st->theta < m.tol;
            if (done && st->stop_from == INT_MAX) { st->stop_sweep = m.check_sweep; st->stop_from = m.check_sweep + 2; }
            st->ticket = 0u;
            __threadfence();
        }
    }

    // L2 prefetch for the block that runs `prefetch` sites further along the traversal: the few fat warps of
    // an SM cannot keep enough bytes in flight while they compute, prefetches hold no register and no
    // scoreboard entry, and the 126 MB L2 is the staging buffer.  Addresses are those of this thread shifted
    // by the distance (exact for forward links, exact up to the periodic wrap for backward links: a hint).
    static __device__ __forceinline__ void issue_prefetch(const SweepParams& p, const SweepPhase& ph, const Site& s,
                                                          const unsigned (&hb)[NMU], int lane_mu0, T* base, size_t H)
    {
        const size_t Hp = p.L.Hp;
        if (p.prefetch) {
            const long long d = ph.reverse ? -(long long)p.prefetch : (long long)p.prefetch;
            const long long hf = (long long)s.h + d;
            if (hf >= 0 && hf < (long long)H) {
#pragma unroll
                for (int m = 0; m < NMU; ++m) {
                    const int mu = lane_mu0 + m;
                    const long long hbd = (long long)hb[m] + d;
                    if (CB && mu == 3) continue;
                    IO::prefetch(base + (size_t)(ph.parity * 4 + mu) * R * Hp, Hp, (size_t)hf);
                    if (hbd >= 0 && hbd < (long long)H) IO::prefetch(base + (size_t)((1 - ph.parity) * 4 + mu) * R * Hp, Hp, (size_t)hbd);
                }
            }
        }
    }

    // the update of the site in half-site slot `slot` (Alg. 1 inner loop) by the TPS threads that
    // share it; this thread owns the directions lane_mu0 .. lane_mu0 + NMU - 1.  `mask`: the lanes of the warp that
    // run this call together (whole sites: TPS divides 32).  `first`: first site update of this thread in the launch
    // (the one-shot kernel: always; it waits for the previous grid there)
    // mon_skip (MON): the launch is past its stop, or the site's timeslice is frozen: nothing is updated.  The words
    // are read by the caller ahead of the link loads and tested behind them, so that the test costs no latency.
    static __device__ __forceinline__ void site_update(const SweepParams& p, const SweepPhase& ph, unsigned slot,
                                                       int lane_mu0, unsigned mask, bool first, const int* mon_stop,
                                                       const int* mon_frozen, double (&mon_out)[3])
    {
        const Site s = decode_site(p.L, slot, ph.parity);
        const size_t H = p.L.H, Hp = p.L.Hp;
        T* const base = reinterpret_cast<T*>(p.U);

        const MemPolicy pol = {make_l2_policy(p.ld_policy), make_l2_policy(p.st_policy)};
        cx<T> F[NMU][9], B[NMU][9];
        unsigned hb[NMU];
#pragma unroll
        for (int m = 0; m < NMU; ++m) hb[m] = backward_neighbour(p.L, s, lane_mu0 + m);
        // Programmatic dependent launch: this grid may become resident while the previous half-sweep drains
        // (its index arithmetic above overlaps that tail); links are touched only after the previous grid
        // has completed and flushed.  Letting the next grid launch early is always safe for the same reason.
        if (p.pdl && first) {
            cudaTriggerProgrammaticLaunchCompletion();
            cudaGridDependencySynchronize();
        }
        // fp32 relaxation sweeps, hybrid chain: were the two half-sweeps before this one rough?  Two L2 hits, issued
        // ahead of the link loads so that the choice is there when the first link arrives
        int rough_now = 0;
        if (HYB && p.chain == CHAIN_HYBRID && !ph.rough_force) rough_now = *((const volatile int*)p.rough + ph.rough_slot);
        int mon_skip = 0;
#ifndef GF_EXP_MON_NOFLAG
        if (MON) { // written by earlier launches only (stamped): plain L2 loads
            mon_skip = p.mon.sweep >= __ldcg(mon_stop);
            if (mon_frozen != nullptr) mon_skip |= p.mon.sweep >= __ldcg(mon_frozen);
        }
#endif
        // the relaxation kernels prefetch before their loads (placed after them the fp64 kernel spills twice as
        // much); the heatbath kernel issues its loads first and hides the prefetch and the generator behind them
        if (MODE != MODE_HEATBATH) issue_prefetch(p, ph, s, hb, lane_mu0, base, H);
        // issue every load before the first use
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
            const int mu = lane_mu0 + m;
            if (CB && mu == 3) continue;
            IO::load(base + (size_t)(ph.parity * 4 + mu) * R * Hp, Hp, s.h, F[m], pol.ld);
            IO::load(base + (size_t)((1 - ph.parity) * 4 + mu) * R * Hp, Hp, hb[m], B[m], pol.ld);
        }
        cx<T> Gt[9];
        const bool owns_t = CB && (lane_mu0 + NMU - 1 == 3); // the thread that would hold the temporal links
        if (owns_t) GIO::load(reinterpret_cast<const T*>(p.G) + (size_t)ph.parity * 18 * Hp, Hp, s.h, Gt, pol.ld);
        if (MODE == MODE_HEATBATH) issue_prefetch(p, ph, s, hb, lane_mu0, base, H);
        // heatbath: random numbers of trial 0 and of the direction, generated under the shadow of the loads
        const uint32_t sc = canonical_index(s) + p.site_offset;
        EarlyDraw<T> early[3];
        if (MODE == MODE_HEATBATH) {
#pragma unroll
            for (int sub = 0; sub < 3; ++sub) {
                const uint32_t c2 = ((uint32_t)ph.parity << 2) | (uint32_t)sub;
                if (PAIR) early_draw_pair<T>(p.key0, p.key1, sc, ph.step, c2, mask, early[sub]);
                else early_draw<T>(p.key0, p.key1, sc, ph.step, c2, early[sub]);
            }
            // pin the values here, before the first use of a loaded link: volatile asm statements keep their order, so
            // the generator and the logarithms run between the issue of the loads and their consumption
#pragma unroll
            for (int sub = 0; sub < 3; ++sub) pin_early(early[sub]);
        }
        if (ph.reunit) {
#pragma unroll
            for (int m = 0; m < NMU; ++m) {
                if (CB && lane_mu0 + m == 3) continue;
                reunitarise(F[m]);
                reunitarise(B[m]);
            }
            if (owns_t) reunitarise(Gt);
        }

        double th_pre = 0.0, th_post = 0.0;
        bool watch = false; // fp32: some step of this site had a small conditioning number
        if constexpr (HYB) {
            const bool dchain = p.chain == CHAIN_DOUBLE || (p.chain == CHAIN_HYBRID && (ph.rough_force | rough_now) != 0);
            const bool updated = dchain ? chain<double>(p, ph, F, B, Gt, sc, early, lane_mu0, mask, watch, th_pre, th_post, mon_skip)
                                        : chain<float>(p, ph, F, B, Gt, sc, early, lane_mu0, mask, watch, th_pre, th_post, mon_skip);
            if (MON && !updated) return;
            if (p.chain == CHAIN_HYBRID) {
                // ring of flags, rough[s] = "half-sweep s runs the double chain": a rough half-sweep marks the next two;
                // the slot three ahead was read by the previous half-sweep and is written by the next two: clear it
                if (watch) { // same value from every writer
                    p.rough[(ph.rough_slot + 1) % ROUGH_RING] = 1;
                    p.rough[(ph.rough_slot + 2) % ROUGH_RING] = 1;
                }
                if (slot == p.h_begin && lane_mu0 == 0) {
                    p.rough[(ph.rough_slot + 3) % ROUGH_RING] = 0;
                    if (dchain && p.dc_count != nullptr) atomicAdd(p.dc_count, 1ull);
                }
            }
        } else {
            (void)rough_now;
            const bool updated = chain<typename std::conditional<DC, double, T>::type>(p, ph, F, B, Gt, sc, early, lane_mu0, mask, watch,
                                                                                        th_pre, th_post, mon_skip);
            if (MON && !updated) return;
            if constexpr (FIX) {
                if (watch) {
                    fixup_site_f64<R, TPS, CB>(p, ph, slot, lane_mu0); // stores the links itself
                    return;
                }
            }
        }

        if (MON == 2) {
            mon_out[1] = th_post;
            mon_out[2] = th_pre;
            if (p.mon.F_part != nullptr) { // eq. 2.1 (C1) on the links this thread stores
                T f = T(0);
#pragma unroll
                for (int m = 0; m < NMU; ++m)
                    if (lane_mu0 + m < p.nd && !(CB && lane_mu0 + m == 3))
                        f += (F[m][0].re + F[m][4].re + F[m][8].re) + (B[m][0].re + B[m][4].re + B[m][8].re);
                mon_out[0] = (double)f;
            }
        }
#pragma unroll
        for (int m = 0; m < NMU; ++m) {
            const int mu = lane_mu0 + m;
            if (CB && mu == 3) continue;
            IO::store(base + (size_t)(ph.parity * 4 + mu) * R * Hp, Hp, s.h, F[m], pol.st);
            IO::store(base + (size_t)((1 - ph.parity) * 4 + mu) * R * Hp, Hp, hb[m], B[m], pol.st);
        }
        if (owns_t) GIO::store(reinterpret_cast<T*>(p.G) + (size_t)ph.parity * 18 * Hp, Hp, s.h, Gt, pol.st);
    }

    static __device__ __forceinline__ void run(const SweepParams& p)
    {
        const unsigned blk = p.ph.reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
        const unsigned gtid = blk * blockDim.x + threadIdx.x;
        double mon_out[3] = {0.0, 0.0, 0.0};
        if (!MON) {
            // threads past the range leave at once: they come in whole sites (TPS divides 32), and exited threads may be
            // named in the mask of the shuffles that combine K
            if (gtid / TPS >= p.h_count) return;
            site_update(p, p.ph, p.h_begin + gtid / TPS, (int)(gtid % TPS) * NMU, 0xffffffffu, true, nullptr, nullptr, mon_out);
            return;
        }
        // monitored launch: the host launches it only where the threads of a timeslice fill whole blocks, so every
        // thread has a site and a block lies inside one timeslice -- no range test, the control flow stays uniform
        const unsigned slot = p.h_begin + gtid / TPS;
        const int* fr = nullptr;
        if (p.mon.slices) fr = p.mon.frozen_from + slot / (p.L.H / (unsigned)p.L.Nt);
        site_update(p, p.ph, slot, (int)(gtid % TPS) * NMU, 0xffffffffu, true, &p.mon.state->stop_from, fr, mon_out);
        if (MON < 2) return;
        if (p.mon.F_part != nullptr || p.mon.post_part != nullptr || p.mon.pre_part != nullptr) {
            __shared__ double smem[3][MAX_BLOCK / 32];
            const unsigned part = (p.h_begin * TPS) / blockDim.x + blk; // index of this block's partials: its place in the lattice
            if (p.mon.F_part != nullptr) {
                const double v = block_sum(mon_out[0], smem[0]);
                if (threadIdx.x == 0) p.mon.F_part[part] = v;
            }
            if (p.mon.post_part != nullptr) {
                const double v = block_sum(mon_out[1], smem[1]);
                if (threadIdx.x == 0) p.mon.post_part[part] = v;
            }
            if (p.mon.pre_part != nullptr) {
                const double v = block_sum(mon_out[2], smem[2]);
                if (threadIdx.x == 0) p.mon.pre_part[part] = v;
            }
        }
#ifndef GF_EXP_MON_NODUTY
        if (p.mon.red_post != nullptr && blockIdx.x < (unsigned)(p.L.Nt * p.mon.groups) && p.mon.sweep < __ldcg(&p.mon.state->stop_from))
            monitor_duty(p.mon, p.L.Nt, blockIdx.x);
#endif
    }
};

// Register budget.  The fp32 relaxation kernels hold two chains (fp32 and double, chosen per launch); the double one
// needs more registers, but it runs on rough fields only, so the kernel is held to what the fp32 chain alone needs
// (the double chain spills instead) -- otherwise the steady state pays for the rare path with occupancy (fp32 R12,
// two threads per site: 128 -> 174 registers cost 18 %).  Blocks of up to MAX_BLOCK threads must stay launchable.
template <typename T, int R, int TPS, int MODE, bool CB>
constexpr int sweep_max_registers()
{
    if (sizeof(T) == 4 && MODE != MODE_HEATBATH) { // what ptxas gives the same kernel with the fp32 chain alone, rounded up to 8
        const bool var = MODE == MODE_VARIANT;
        if (R == 12) {
            if (TPS == 1) return CB ? (var ? 184 : 200) : 255;
            if (TPS == 2) return 128;
            return CB ? 96 : (var ? 104 : 80);
        }
        if (TPS == 2) return CB ? (var ? 136 : 144) : (var ? 136 : 184);
        if (TPS == 4) return CB ? 104 : (var ? 104 : 120);
    }
    return 255;
}

template <typename T, int R, int TPS, int MODE, bool CB = false, bool DC = false, int MON = 0>
__global__ void __maxnreg__((sweep_max_registers<T, R, TPS, MODE, CB>())) gf_half_sweep_kernel(const __grid_constant__ SweepParams p)
{
    SweepKernel<T, R, TPS, MODE, CB, DC, MON>::run(p);
}

} // namespace gf
