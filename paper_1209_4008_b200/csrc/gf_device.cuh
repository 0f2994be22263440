// gf_device.cuh -- device-side building blocks of libgf.so (sm_100a): complex / SU(3) register arithmetic,
// the native link layout, checkerboard site indexing, Philox4x32-10.
//
// Native layout ("Data layout in HBM").  H = V/2 sites per parity.  Half-site index of a site
// (x,y,z,t) of parity p = (x+y+z+t)&1:   h = (x>>1) + (Nx/2) * (y + Ny * (z + Nz * t)).
// Link U_mu(x) lives in link block  l = p*4 + mu  (parity-split: PAPER.md:124), which holds R*Hp reals, Hp = H rounded
// up to a multiple of 32.  Inside a block the sites are grouped in TILES of 32 consecutive half-sites (one warp's worth);
// inside a tile the complex entries e = 3*row + col (e < R/2; R = 12 stores rows 0,1 only) are
// component-major with the site index fastest, in 128-bit vectors:
//   fp64: tile = R/2 planes of 32 double2 (re,im)                      -> real offset  (h>>5)*R*32 + e*64 + 2*(h&31)
//   fp32: tile = R/4 planes of 32 float4 (re,im of e=2q; re,im of e=2q+1) -> real offset  (h>>5)*R*32 + q*128 + 4*(h&31)
//         R = 18: the ninth entry (e = 8) is a trailing plane of 32 float2 at  (h>>5)*R*32 + 512 + 2*(h&31)
// so a warp's load of one plane is one contiguous 512-byte (fp32 tail: 256-byte) run, as with whole-lattice planes, but
// all planes of a link sit at CONSTANT offsets from one address per thread: one address computation per link instead
// of one per plane (the half-sweep spent 15 % of its instructions on 64-bit address arithmetic), and a site's link is
// one 2.3 KB (fp32 R18) stretch of a DRAM page instead of five pages.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gf {

// ---------------------------------------------------------------------------------------------------------
// complex numbers in registers
// ---------------------------------------------------------------------------------------------------------
template <typename T>
struct cx {
    T re, im;
};

template <typename T>
__device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return {a.re + b.re, a.im + b.im}; }
template <typename T>
__device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return {a.re - b.re, a.im - b.im}; }
template <typename T>
__device__ __forceinline__ cx<T> operator*(cx<T> a, cx<T> b)
{
    return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
template <typename T>
__device__ __forceinline__ cx<T> conj(cx<T> a) { return {a.re, -a.im}; }
// conj(a) * b
template <typename T>
__device__ __forceinline__ cx<T> cmul_ca(cx<T> a, cx<T> b)
{
    return {a.re * b.re + a.im * b.im, a.re * b.im - a.im * b.re};
}
// a * conj(b)
template <typename T>
__device__ __forceinline__ cx<T> cmul_cb(cx<T> a, cx<T> b)
{
    return {a.re * b.re + a.im * b.im, a.im * b.re - a.re * b.im};
}

template <typename T> __device__ __forceinline__ T gf_rsqrt(T x);
// MUFU.RSQ (<= 2 ulp, slightly biased) plus one Newton step: without the step the bias of the normalisation of
// every SU(2) element accumulates into a unitarity drift of the fp32 links (C15); no division, no slow path
template <> __device__ __forceinline__ float gf_rsqrt<float>(float x)
{
    const float y = rsqrtf(x);
    return y * fmaf(-0.5f * x * y, y, 1.5f);
}
template <> __device__ __forceinline__ double gf_rsqrt<double>(double x) { return rsqrt(x); } // <= 1 ulp
template <typename T> __device__ __forceinline__ T gf_sqrt(T x);
template <> __device__ __forceinline__ float gf_sqrt<float>(float x) { return sqrtf(x); }
template <> __device__ __forceinline__ double gf_sqrt<double>(double x) { return sqrt(x); }
__device__ __forceinline__ float gf_fma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double gf_fma(double a, double b, double c) { return fma(a, b, c); }

// x0 y0 + x1 y1 + x2 y2 + x3 y3 as one multiply and three fused multiply-adds.  The complex products of the
// link updates are written with it explicitly: left to itself the compiler keeps the two complex products of
// a*u + b*v apart (4 FMUL + 4 FFMA + 2 FADD per entry instead of 2 FMUL + 6 FFMA), which costs issue slots
// and, at the 1 kW power cap, clock.
template <typename T>
__device__ __forceinline__ T dot4(T x0, T y0, T x1, T y1, T x2, T y2, T x3, T y3)
{
    return gf_fma(x0, y0, gf_fma(x1, y1, gf_fma(x2, y2, x3 * y3)));
}

// ---------------------------------------------------------------------------------------------------------
// SU(3) links: 9 complex entries, row-major, always fully unrolled so they stay in registers
// ---------------------------------------------------------------------------------------------------------

// conj(p q - r s)
template <typename T>
__device__ __forceinline__ cx<T> cross_entry(cx<T> p, cx<T> q, cx<T> r, cx<T> s)
{
    return {dot4(p.re, q.re, -p.im, q.im, -r.re, s.re, r.im, s.im),
            dot4(-p.re, q.im, -p.im, q.re, r.re, s.im, r.im, s.re)};
}

// row 2 = conj(row0 x row1)  (C16; "reconstruct the third line")
template <typename T>
__device__ __forceinline__ void rebuild_row2(cx<T> (&u)[9])
{
    u[6] = cross_entry(u[1], u[5], u[2], u[4]);
    u[7] = cross_entry(u[2], u[3], u[0], u[5]);
    u[8] = cross_entry(u[0], u[4], u[1], u[3]);
}

// Gram-Schmidt on rows 0,1 then row 2 rebuilt: the fp32 unitarity policy (C15)
template <typename T>
__device__ __forceinline__ void reunitarise(cx<T> (&u)[9])
{
    T n0 = gf_rsqrt<T>(u[0].re * u[0].re + u[0].im * u[0].im + u[1].re * u[1].re + u[1].im * u[1].im +
                       u[2].re * u[2].re + u[2].im * u[2].im);
#pragma unroll
    for (int c = 0; c < 3; ++c) { u[c].re *= n0; u[c].im *= n0; }
    cx<T> dot = cmul_ca(u[0], u[3]) + cmul_ca(u[1], u[4]) + cmul_ca(u[2], u[5]);
#pragma unroll
    for (int c = 0; c < 3; ++c) u[3 + c] = u[3 + c] - dot * u[c];
    T n1 = gf_rsqrt<T>(u[3].re * u[3].re + u[3].im * u[3].im + u[4].re * u[4].re + u[4].im * u[4].im +
                       u[5].re * u[5].re + u[5].im * u[5].im);
#pragma unroll
    for (int c = 0; c < 3; ++c) { u[3 + c].re *= n1; u[3 + c].im *= n1; }
    rebuild_row2(u);
}

// SU(2) element embedded in the (I,J) subgroup (C4): quaternion q -> a = q0 + i q3, b = q2 + i q1;
// G_II = a, G_IJ = b, G_JI = -conj(b), G_JJ = conj(a).
// Left multiplication  M <- G M  touches rows I,J   (Alg. 1; 84 flop per link):
//   m_I <- a m_I + b m_J ,   m_J <- conj(a) m_J - conj(b) m_I
template <int I, int J, typename T>
__device__ __forceinline__ void su2_left(cx<T> a, cx<T> b, cx<T> (&m)[9])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cx<T> ui = m[3 * I + c], uj = m[3 * J + c];
        m[3 * I + c] = {dot4(a.re, ui.re, -a.im, ui.im, b.re, uj.re, -b.im, uj.im),
                        dot4(a.re, ui.im, a.im, ui.re, b.re, uj.im, b.im, uj.re)};
        m[3 * J + c] = {dot4(a.re, uj.re, a.im, uj.im, -b.re, ui.re, -b.im, ui.im),
                        dot4(a.re, uj.im, -a.im, uj.re, -b.re, ui.im, b.im, ui.re)};
    }
}
// Right multiplication  M <- M G^dagger  touches columns I,J   (Alg. 1; 84 flop per link).
// (G^dagger)_II = conj(a), (G^dagger)_IJ = -b, (G^dagger)_JI = conj(b), (G^dagger)_JJ = a:
//   m_I <- m_I conj(a) + m_J conj(b) ,   m_J <- m_J a - m_I b
template <int I, int J, int ROWS, typename T>
__device__ __forceinline__ void su2_right_dagger(cx<T> a, cx<T> b, cx<T> (&m)[9])
{
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        const cx<T> ui = m[3 * r + I], uj = m[3 * r + J];
        m[3 * r + I] = {dot4(ui.re, a.re, ui.im, a.im, uj.re, b.re, uj.im, b.im),
                        dot4(ui.im, a.re, -ui.re, a.im, uj.im, b.re, -uj.re, b.im)};
        m[3 * r + J] = {dot4(uj.re, a.re, -uj.im, a.im, -ui.re, b.re, ui.im, b.im),
                        dot4(uj.re, a.im, uj.im, a.re, -ui.re, b.im, -ui.im, b.re)};
    }
}

// Full 3x3 products with an accumulated G = g3 g2 g1 (C8: applying the three SU(2) factors one after the other or their
// product once is the same up to rounding): 108 multiply-adds per link instead of 3 x 48.  ROWS: rows of the result
// that are needed (R = 12 stores rows 0,1 only).  Six-term dot products as one multiply and five fused multiply-adds.
template <typename T>
__device__ __forceinline__ T dot6(T x0, T y0, T x1, T y1, T x2, T y2, T x3, T y3, T x4, T y4, T x5, T y5)
{
    return gf_fma(x0, y0, gf_fma(x1, y1, gf_fma(x2, y2, gf_fma(x3, y3, gf_fma(x4, y4, x5 * y5)))));
}
// u <- G u, rows 0 .. ROWS-1 of the result (the others are left as they were)
template <int ROWS, typename T>
__device__ __forceinline__ void mat_left(const cx<T> (&G)[9], cx<T> (&u)[9])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cx<T> u0 = u[c], u1 = u[3 + c], u2 = u[6 + c];
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
            const cx<T> g0 = G[3 * r], g1 = G[3 * r + 1], g2 = G[3 * r + 2];
            u[3 * r + c] = {dot6(g0.re, u0.re, -g0.im, u0.im, g1.re, u1.re, -g1.im, u1.im, g2.re, u2.re, -g2.im, u2.im),
                            dot6(g0.re, u0.im, g0.im, u0.re, g1.re, u1.im, g1.im, u1.re, g2.re, u2.im, g2.im, u2.re)};
        }
    }
}
// u <- u G^dagger, rows 0 .. ROWS-1:  (u G^dagger)_rc = sum_k u_rk conj(G_ck)
template <int ROWS, typename T>
__device__ __forceinline__ void mat_right_dagger(const cx<T> (&G)[9], cx<T> (&u)[9])
{
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        const cx<T> u0 = u[3 * r], u1 = u[3 * r + 1], u2 = u[3 * r + 2];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const cx<T> g0 = G[3 * c], g1 = G[3 * c + 1], g2 = G[3 * c + 2];
            u[3 * r + c] = {dot6(u0.re, g0.re, u0.im, g0.im, u1.re, g1.re, u1.im, g1.im, u2.re, g2.re, u2.im, g2.im),
                            dot6(u0.im, g0.re, -u0.re, g0.im, u1.im, g1.re, -u1.re, g1.im, u2.im, g2.re, -u2.re, g2.im)};
        }
    }
}

// quaternionic part of the (I,J) block of K (C7):  Re tr[G K] = const + g0 k0 - g1 k1 - g2 k2 - g3 k3
template <int I, int J, typename T>
__device__ __forceinline__ void su2_project(const cx<T> (&K)[9], T (&k)[4])
{
    k[0] = K[3 * I + I].re + K[3 * J + J].re;
    k[1] = K[3 * I + J].im + K[3 * J + I].im;
    k[2] = K[3 * I + J].re - K[3 * J + I].re;
    k[3] = K[3 * I + I].im - K[3 * J + J].im;
}

// ---------------------------------------------------------------------------------------------------------
// native layout access.  Every access is one 128-bit (fp32 R18 tail plane: 64-bit) vector per thread with an
// explicit L2 cache policy (createpolicy + .L2::cache_hint): within a half-sweep every link is read exactly
// once and written exactly once (C6), so loads are streaming (L1 no-allocate, L2 evict-first by default) while
// stores may ask L2 to keep the line (evict-last) for the next half-sweep, which starts where this one ended
// (gf_set_l2_reversal).  DESIGN.md "Kernels / L2 policy".
// ---------------------------------------------------------------------------------------------------------
enum { POLICY_NORMAL = 0, POLICY_EVICT_FIRST = 1, POLICY_EVICT_LAST = 2 };

__device__ __forceinline__ uint64_t make_l2_policy(int kind)
{
    uint64_t p;
    if (kind == POLICY_EVICT_FIRST) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else if (kind == POLICY_EVICT_LAST) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}

struct MemPolicy {
    uint64_t ld, st;
};

__device__ __forceinline__ float4 ldg(const float4* p, uint64_t pol)
{
    float4 v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ldg(const float2* p, uint64_t pol)
{
    float2 v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 ldg(const double2* p, uint64_t pol)
{
    double2 v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ void stg(float4* p, float4 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void stg(float2* p, float2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1,%2}, %3;" :: "l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void stg(double2* p, double2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" :: "l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

// L2 prefetch of the 128-byte line holding p (a hint: no register, no scoreboard)
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

template <typename T, int R> struct LinkIO;

constexpr int TILE = 32; // sites per tile of the native layout

template <int R>
struct LinkIO<double, R> {
    static constexpr int NE = R / 2;
    // blk: first real of the link block; Hp: padded sites per block (unused: the tiles carry the layout); h: half-site index
    static __device__ __forceinline__ const double2* at(const double* blk, size_t h)
    {
        return reinterpret_cast<const double2*>(blk) + (h >> 5) * (size_t)(NE * TILE) + (h & 31);
    }
    static __device__ __forceinline__ void load(const double* blk, size_t, size_t h, cx<double> (&u)[9], uint64_t pol)
    {
        const double2* p = at(blk, h);
#pragma unroll
        for (int e = 0; e < NE; ++e) {
            double2 v = ldg(p + e * TILE, pol);
            u[e] = {v.x, v.y};
        }
        if (R == 12) rebuild_row2(u);
    }
    // Re tr U from the diagonal planes alone (R = 12: rows 0,1 in full, entry (2,2) rebuilt)
    static __device__ __forceinline__ double trace_re(const double* blk, size_t Hp, size_t h, uint64_t pol)
    {
        const double2* p = at(blk, h);
        if (R == 18) return ldg(p, pol).x + ldg(p + 4 * TILE, pol).x + ldg(p + 8 * TILE, pol).x;
        cx<double> u[9];
        load(blk, Hp, h, u, pol);
        return u[0].re + u[4].re + u[8].re;
    }
    static __device__ __forceinline__ void prefetch(const double* blk, size_t, size_t h)
    {
        const double2* p = at(blk, h);
#pragma unroll
        for (int e = 0; e < NE; ++e) prefetch_l2(p + e * TILE);
    }
    static __device__ __forceinline__ void store(double* blk, size_t, size_t h, const cx<double> (&u)[9], uint64_t pol)
    {
        double2* p = const_cast<double2*>(at(blk, h));
#pragma unroll
        for (int e = 0; e < NE; ++e) stg(p + e * TILE, make_double2(u[e].re, u[e].im), pol);
    }
};

template <int R>
struct LinkIO<float, R> {
    static constexpr int NQ = R / 4; // float4 planes: 4 (R18) or 3 (R12)
    static __device__ __forceinline__ const float* tile(const float* blk, size_t h) { return blk + (h >> 5) * (size_t)(R * TILE); }
    // the stored entries only (R = 12: u[6..8] untouched)
    static __device__ __forceinline__ void load_stored(const float* blk, size_t, size_t h, cx<float> (&u)[9], uint64_t pol)
    {
        const float* t = tile(blk, h);
        const float4* p = reinterpret_cast<const float4*>(t) + (h & 31);
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            float4 v = ldg(p + q * TILE, pol);
            u[2 * q] = {v.x, v.y};
            u[2 * q + 1] = {v.z, v.w};
        }
        if (R == 18) {
            float2 v = ldg(reinterpret_cast<const float2*>(t + 16 * TILE) + (h & 31), pol);
            u[8] = {v.x, v.y};
        }
    }
    static __device__ __forceinline__ void load(const float* blk, size_t Hp, size_t h, cx<float> (&u)[9], uint64_t pol)
    {
        load_stored(blk, Hp, h, u, pol);
        if (R == 12) rebuild_row2(u);
    }
    // float storage, double arithmetic (the rare-path fix-up of the fp32 sweep, gf_sweep.cuh): the stored floats are
    // widened exactly; R = 12: row 2 is rebuilt in double
    static __device__ __forceinline__ void load(const float* blk, size_t Hp, size_t h, cx<double> (&u)[9], uint64_t pol)
    {
        cx<float> v[9];
        load_stored(blk, Hp, h, v, pol);
#pragma unroll
        for (int e = 0; e < R / 2; ++e) u[e] = {(double)v[e].re, (double)v[e].im};
        if (R == 12) rebuild_row2(u);
    }
    static __device__ __forceinline__ void store(float* blk, size_t Hp, size_t h, const cx<double> (&u)[9], uint64_t pol)
    {
        cx<float> v[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) v[e] = {(float)u[e].re, (float)u[e].im};
        store(blk, Hp, h, v, pol);
    }
    static __device__ __forceinline__ double trace_re(const float* blk, size_t Hp, size_t h, uint64_t pol)
    {
        if (R == 18) {
            const float* t = tile(blk, h);
            const float4* p = reinterpret_cast<const float4*>(t) + (h & 31);
            return (double)ldg(p, pol).x + (double)ldg(p + 2 * TILE, pol).x +
                   (double)ldg(reinterpret_cast<const float2*>(t + 16 * TILE) + (h & 31), pol).x;
        }
        cx<float> u[9];
        load(blk, Hp, h, u, pol);
        return (double)u[0].re + (double)u[4].re + (double)u[8].re;
    }
    static __device__ __forceinline__ void prefetch(const float* blk, size_t, size_t h)
    {
        const float* t = tile(blk, h);
        const float4* p = reinterpret_cast<const float4*>(t) + (h & 31);
#pragma unroll
        for (int q = 0; q < NQ; ++q) prefetch_l2(p + q * TILE);
        if (R == 18) prefetch_l2(reinterpret_cast<const float2*>(t + 16 * TILE) + (h & 31));
    }
    static __device__ __forceinline__ void store(float* blk, size_t, size_t h, const cx<float> (&u)[9], uint64_t pol)
    {
        float* t = const_cast<float*>(tile(blk, h));
        float4* p = reinterpret_cast<float4*>(t) + (h & 31);
#pragma unroll
        for (int q = 0; q < NQ; ++q)
            stg(p + q * TILE, make_float4(u[2 * q].re, u[2 * q].im, u[2 * q + 1].re, u[2 * q + 1].im), pol);
        if (R == 18) stg(reinterpret_cast<float2*>(t + 16 * TILE) + (h & 31), make_float2(u[8].re, u[8].im), pol);
    }
};

// ---------------------------------------------------------------------------------------------------------
// checkerboard site indexing ("divisions and modulo conversions"; C5: periodic, parity =
// (x+y+z+t)&1)
// ---------------------------------------------------------------------------------------------------------
struct Lattice {
    int Nxh, Ny, Nz, Nt; // Nxh = Nx/2
    unsigned H;          // V/2
    unsigned Hp;         // H rounded up to whole tiles of 32 sites: sites per link block in memory
};

struct Site {
    unsigned h;      // half-site index inside its parity block
    int xh, y, z, t; // x = 2*xh + q
    int q;           // (y + z + t + parity) & 1
};

__device__ __forceinline__ Site decode_site(const Lattice& L, unsigned h, int parity)
{
    Site s;
    s.h = h;
    unsigned r = h / (unsigned)L.Nxh;
    s.xh = (int)(h - r * (unsigned)L.Nxh);
    unsigned r2 = r / (unsigned)L.Ny;
    s.y = (int)(r - r2 * (unsigned)L.Ny);
    unsigned r3 = r2 / (unsigned)L.Nz;
    s.z = (int)(r2 - r3 * (unsigned)L.Nz);
    s.t = (int)r3;
    s.q = (s.y + s.z + s.t + parity) & 1;
    return s;
}

// canonical site index s = x + Nx (y + Ny (z + Nz t)) = 2h + q
__device__ __forceinline__ unsigned canonical_index(const Site& s) { return 2u * s.h + (unsigned)s.q; }

// half-site index (in the OTHER parity block) of the neighbour x - mu_hat
__device__ __forceinline__ unsigned backward_neighbour(const Lattice& L, const Site& s, int mu)
{
    if (mu == 0) {
        // x - 1 = 2 xh + q - 1: same xh when q = 1, xh - 1 (periodic) when q = 0
        if (s.q) return s.h;
        return s.xh == 0 ? s.h + (unsigned)(L.Nxh - 1) : s.h - 1u;
    }
    if (mu == 1) {
        unsigned st = (unsigned)L.Nxh;
        return s.y == 0 ? s.h + st * (unsigned)(L.Ny - 1) : s.h - st;
    }
    if (mu == 2) {
        unsigned st = (unsigned)L.Nxh * (unsigned)L.Ny;
        return s.z == 0 ? s.h + st * (unsigned)(L.Nz - 1) : s.h - st;
    }
    unsigned st = (unsigned)L.Nxh * (unsigned)L.Ny * (unsigned)L.Nz;
    return s.t == 0 ? s.h + st * (unsigned)(L.Nt - 1) : s.h - st;
}

// ---------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) -- the CUDA path's own copy
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0; // one IMAD.WIDE.U32 gives hi and lo
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c3 = (uint32_t)p0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ---------------------------------------------------------------------------------------------------------
// Double-precision functions of the Kennedy-Pendleton draw (C14), written for their actual arguments: the
// uniforms are u = (2 (x >> 9) + 1) 2^-24, 24-bit numbers.  The library's log / sincospi are general (special
// cases behind branches, 64-bit immediates moved through uniform registers: ~80 / ~75 instructions each),
// and the fp64 annealing kernel is bound by instruction issue and instruction fetch, not by memory
// (profiles/r2_ncu_heatbath.md).  Here: branch-free, ~35 instructions each, errors of a few 1e-16 (checked over
// all 2^23 arguments by tests/test_gpu_variants.py through gf_debug_kp_math).  Tables: gf_kp_tables.inc, written
// by gen_kp_tables.py.  (The coefficients stay literals: read from a __constant__ array instead, ptxas keeps
// them in registers across the three subgroup steps and the kernel spills 248 bytes -- 219 -> 247 us.)
// ---------------------------------------------------------------------------------------------------------
#include "gf_kp_tables.inc"

// -ln u, u the uniform of the Philox word x.  u = m 2^(e-24), m in [1,2) from the leading one of w = 2 (x >> 9) + 1;
// bin j = top 7 bits of m; f = m r_j - 1 (exact), ln m = T_j + log1p(f); for j >= 64 the table holds T_j - ln 2 and the
// exponent counts one more, so that nothing cancels as u -> 1.
__device__ __forceinline__ double kp_neglog_word(uint32_t x)
{
    const uint32_t w = 2u * (x >> 9) + 1u; // odd, < 2^24
    const int lz = __clz((int)w);          // >= 8
    const uint32_t mi = w << (lz - 8);     // 24 bits, leading one at bit 23: m = mi 2^-23
    const int j = (int)((mi >> 16) & 127u);
    const double2 t = GF_KP_LOG_TAB[j];
    const double m = __hiloint2double((int)(0x3FF00000u | ((mi >> 3) & 0xFFFFFu)), (int)(mi << 29));
    const double f = fma(m, t.x, -1.0);
    double p = 1.0 / 7.0;
    p = fma(p, f, -1.0 / 6.0);
    p = fma(p, f, 1.0 / 5.0);
    p = fma(p, f, -1.0 / 4.0);
    p = fma(p, f, 1.0 / 3.0);
    p = fma(p, f, -1.0 / 2.0);
    p = fma(p, f, 1.0);
    p *= f; // log1p(f), |f| < 0.006
    const double n = (double)(lz - (j < 64 ? 7 : 8)); // 24 - e, e = 31 - lz; one less where the table took ln 2
    return fma(n, GF_KP_LN2_HI, fma(n, GF_KP_LN2_LO, -p) - t.y);
}

// sin(2 pi u), cos(2 pi u), u the uniform of the Philox word x: 4u = q + r exactly, q = 0..4, |r| <= 1/2;
// sin / cos(pi r / 2) by their series in r^2, then the quadrant
__device__ __forceinline__ void kp_sincos2pi_word(uint32_t x, double& sn, double& cs)
{
    const uint32_t w = 2u * (x >> 9) + 1u;             // 4u = w 2^-22
    const uint32_t q = (w + (1u << 21)) >> 22;         // nearest integer (w is odd: no ties)
    const double r = (double)((int)w - (int)(q << 22)) * (1.0 / 4194304.0);
    const double z = r * r;
    double s = GF_KP_S7;
    s = fma(s, z, GF_KP_S6); s = fma(s, z, GF_KP_S5); s = fma(s, z, GF_KP_S4); s = fma(s, z, GF_KP_S3);
    s = fma(s, z, GF_KP_S2); s = fma(s, z, GF_KP_S1); s = fma(s, z, GF_KP_S0);
    s *= r;
    double c = GF_KP_C8;
    c = fma(c, z, GF_KP_C7); c = fma(c, z, GF_KP_C6); c = fma(c, z, GF_KP_C5); c = fma(c, z, GF_KP_C4);
    c = fma(c, z, GF_KP_C3); c = fma(c, z, GF_KP_C2); c = fma(c, z, GF_KP_C1); c = fma(c, z, GF_KP_C0);
    // angle = (pi/2)(q + r): q = 0: (s, c); 1: (c, -s); 2: (-s, -c); 3: (-c, s); 4 = 0
    const bool swap = (q & 1u) != 0u;
    const double a = swap ? c : s, b = swap ? s : c;
    sn = (q & 2u) ? -a : a;
    cs = (((q + 1u) & 2u) != 0u) ? -b : b;
}

} // namespace gf
