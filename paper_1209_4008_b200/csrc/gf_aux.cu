// gf_aux.cu -- layout conversion (canonical fp64 <-> native) and the F_g / theta reductions (the paper's second
// kernel: "checks the current value of the gauge fixing functional F_g[U] and the gauge precision
// theta").  Reductions: fp64 arithmetic on the stored links, warp shuffles inside a block, one partial per block,
// then a single-block final pass that adds the partials in a fixed order (deterministic, no atomics).
#include <cstdarg>
#include <cstdio>

#include "gf_internal.h"
#include "gf_device.cuh"

namespace gf {

constexpr int AUX_BLOCK = 256;

// ---------------------------------------------------------------------------------------------------------
// pack / unpack.  One thread per (half-site h, link block l = parity*4 + mu).
// ---------------------------------------------------------------------------------------------------------
template <typename T, int R, typename S>
__global__ void __launch_bounds__(AUX_BLOCK) pack_kernel(Lattice L, unsigned H_own, const S* __restrict__ canon, T* __restrict__ native)
{
    // H_own < L.H on a slab context: the ghost slice (the last one) has no canonical counterpart
    const unsigned long long gid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (unsigned long long)H_own * 8ull) return;
    const unsigned h = (unsigned)(gid % H_own);
    const int l = (int)(gid / H_own), parity = l >> 2, mu = l & 3;
    const Site s = decode_site(L, h, parity);
    const S* src = canon + ((size_t)canonical_index(s) * 4 + mu) * 18;
    cx<T> u[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) u[e] = {(T)src[2 * e], (T)src[2 * e + 1]};
    LinkIO<T, R>::store(native + (size_t)l * R * L.Hp, L.Hp, h, u, make_l2_policy(POLICY_NORMAL));
}

template <typename T, int R, typename S>
__global__ void __launch_bounds__(AUX_BLOCK) unpack_kernel(Lattice L, unsigned H_own, const T* __restrict__ native, S* __restrict__ canon)
{
    const unsigned long long gid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (unsigned long long)H_own * 8ull) return;
    const unsigned h = (unsigned)(gid % H_own);
    const int l = (int)(gid / H_own), parity = l >> 2, mu = l & 3;
    const Site s = decode_site(L, h, parity);
    cx<T> u[9];
    LinkIO<T, R>::load(native + (size_t)l * R * L.Hp, L.Hp, h, u, make_l2_policy(POLICY_NORMAL));
    S* dst = canon + ((size_t)canonical_index(s) * 4 + mu) * 18;
#pragma unroll
    for (int e = 0; e < 9; ++e) { dst[2 * e] = (S)u[e].re; dst[2 * e + 1] = (S)u[e].im; }
}

// canon_f32: the canonical field holds float instead of double (host-buffer path of fp32 contexts)
template <typename S>
static cudaError_t launch_pack_t(int prec, int R, const Lattice& L, unsigned H_own, const S* canon, void* native, cudaStream_t st)
{
    const unsigned long long n = (unsigned long long)H_own * 8ull;
    const unsigned grid = (unsigned)((n + AUX_BLOCK - 1) / AUX_BLOCK);
    if (prec == 0 && R == 18) pack_kernel<float, 18, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, canon, (float*)native);
    else if (prec == 0 && R == 12) pack_kernel<float, 12, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, canon, (float*)native);
    else if (prec == 1 && R == 18) pack_kernel<double, 18, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, canon, (double*)native);
    else if (prec == 1 && R == 12) pack_kernel<double, 12, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, canon, (double*)native);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

template <typename S>
static cudaError_t launch_unpack_t(int prec, int R, const Lattice& L, unsigned H_own, const void* native, S* canon, cudaStream_t st)
{
    const unsigned long long n = (unsigned long long)H_own * 8ull;
    const unsigned grid = (unsigned)((n + AUX_BLOCK - 1) / AUX_BLOCK);
    if (prec == 0 && R == 18) unpack_kernel<float, 18, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, (const float*)native, canon);
    else if (prec == 0 && R == 12) unpack_kernel<float, 12, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, (const float*)native, canon);
    else if (prec == 1 && R == 18) unpack_kernel<double, 18, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, (const double*)native, canon);
    else if (prec == 1 && R == 12) unpack_kernel<double, 12, S><<<grid, AUX_BLOCK, 0, st>>>(L, H_own, (const double*)native, canon);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

cudaError_t launch_pack(int prec, int R, const Lattice& L, unsigned H_own, const double* canon, void* native, cudaStream_t st)
{
    return launch_pack_t<double>(prec, R, L, H_own, canon, native, st);
}
cudaError_t launch_unpack(int prec, int R, const Lattice& L, unsigned H_own, const void* native, double* canon, cudaStream_t st)
{
    return launch_unpack_t<double>(prec, R, L, H_own, native, canon, st);
}
cudaError_t launch_pack_f32(int prec, int R, const Lattice& L, unsigned H_own, const float* canon, void* native, cudaStream_t st)
{
    return launch_pack_t<float>(prec, R, L, H_own, canon, native, st);
}
cudaError_t launch_unpack_f32(int prec, int R, const Lattice& L, unsigned H_own, const void* native, float* canon, cudaStream_t st)
{
    return launch_unpack_t<float>(prec, R, L, H_own, native, canon, st);
}

// t-slab faces (NEXT-4): the temporal links of one parity block of one timeslice, gathered into a contiguous message
// (plane-major: real k of site i at k/VEC * Hs * VEC + i * VEC + k % VEC, fp32 R18 tail plane behind the float4 planes)
// / scattered back.  One thread per site of the face.
template <typename T, int R, bool PACK>
__global__ void __launch_bounds__(AUX_BLOCK) face_kernel(Lattice L, unsigned Hs, int t, int block_parity, T* __restrict__ native,
                                                         T* __restrict__ buf)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Hs) return;
    constexpr int VEC = 16 / sizeof(T), NV = R / VEC; // whole 128-bit vectors per link; fp32 R18: plus two reals
    T* blk = native + (size_t)(block_parity * 4 + 3) * R * L.Hp;
    const size_t h = (size_t)t * Hs + i;
    T* a = blk + (h >> 5) * (size_t)(R * TILE) + (h & 31) * VEC; // plane 0 of this site inside its tile
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        T* b = buf + ((size_t)v * Hs + i) * VEC;
#pragma unroll
        for (int k = 0; k < VEC; ++k) { if (PACK) b[k] = a[v * TILE * VEC + k]; else a[v * TILE * VEC + k] = b[k]; }
    }
    if (sizeof(T) == 4 && R == 18) {
        T* a2 = blk + (h >> 5) * (size_t)(R * TILE) + 16 * TILE + (h & 31) * 2;
        T* b = buf + (size_t)16 * Hs + (size_t)i * 2;
        if (PACK) { b[0] = a2[0]; b[1] = a2[1]; } else { a2[0] = b[0]; a2[1] = b[1]; }
    }
}

cudaError_t launch_face(int prec, int R, const Lattice& L, unsigned Hs, int t, int block_parity, bool pack, void* native,
                        void* buf, cudaStream_t st)
{
    const unsigned grid = (Hs + AUX_BLOCK - 1) / AUX_BLOCK;
#define GF_FACE(T, RR)                                                                                              \
    do {                                                                                                            \
        if (pack) face_kernel<T, RR, true><<<grid, AUX_BLOCK, 0, st>>>(L, Hs, t, block_parity, (T*)native, (T*)buf);  \
        else face_kernel<T, RR, false><<<grid, AUX_BLOCK, 0, st>>>(L, Hs, t, block_parity, (T*)native, (T*)buf);      \
    } while (0)
    if (prec == 0 && R == 18) GF_FACE(float, 18);
    else if (prec == 0 && R == 12) GF_FACE(float, 12);
    else if (prec == 1 && R == 18) GF_FACE(double, 18);
    else if (prec == 1 && R == 12) GF_FACE(double, 12);
    else return cudaErrorInvalidValue;
#undef GF_FACE
    return cudaGetLastError();
}

// native -> native between precisions / storage formats (mixed-precision fixing: fp32 sweeps, fp64 polish)
template <typename TS, int RS, typename TD, int RD>
__global__ void __launch_bounds__(AUX_BLOCK) convert_kernel(Lattice L, const TS* __restrict__ src, TD* __restrict__ dst)
{
    const unsigned long long gid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (unsigned long long)L.H * 8ull) return;
    const unsigned h = (unsigned)(gid % L.H);
    const int l = (int)(gid / L.H);
    const uint64_t pol = make_l2_policy(POLICY_NORMAL);
    cx<TS> u[9];
    LinkIO<TS, RS>::load(src + (size_t)l * RS * L.Hp, L.Hp, h, u, pol);
    cx<TD> v[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) v[e] = {(TD)u[e].re, (TD)u[e].im};
    // widening: the fp32 links are unitary to 1e-7 only; Gram-Schmidt in the wider type makes the fp64 field an
    // SU(3) field to rounding, so that the polish starts from a proper configuration (C15)
    if (sizeof(TD) > sizeof(TS)) reunitarise(v);
    LinkIO<TD, RD>::store(dst + (size_t)l * RD * L.Hp, L.Hp, h, v, pol);
}

template <typename TS, int RS>
static cudaError_t launch_convert_from(int dprec, int dR, const Lattice& L, const void* src, void* dst, cudaStream_t st)
{
    const unsigned long long n = (unsigned long long)L.H * 8ull;
    const unsigned grid = (unsigned)((n + AUX_BLOCK - 1) / AUX_BLOCK);
    if (dprec == 0 && dR == 18) convert_kernel<TS, RS, float, 18><<<grid, AUX_BLOCK, 0, st>>>(L, (const TS*)src, (float*)dst);
    else if (dprec == 0 && dR == 12) convert_kernel<TS, RS, float, 12><<<grid, AUX_BLOCK, 0, st>>>(L, (const TS*)src, (float*)dst);
    else if (dprec == 1 && dR == 18) convert_kernel<TS, RS, double, 18><<<grid, AUX_BLOCK, 0, st>>>(L, (const TS*)src, (double*)dst);
    else if (dprec == 1 && dR == 12) convert_kernel<TS, RS, double, 12><<<grid, AUX_BLOCK, 0, st>>>(L, (const TS*)src, (double*)dst);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

cudaError_t launch_convert(int sprec, int sR, int dprec, int dR, const Lattice& L, const void* src, void* dst, cudaStream_t st)
{
    if (sprec == 0 && sR == 18) return launch_convert_from<float, 18>(dprec, dR, L, src, dst, st);
    if (sprec == 0 && sR == 12) return launch_convert_from<float, 12>(dprec, dR, L, src, dst, st);
    if (sprec == 1 && sR == 18) return launch_convert_from<double, 18>(dprec, dR, L, src, dst, st);
    if (sprec == 1 && sR == 12) return launch_convert_from<double, 12>(dprec, dR, L, src, dst, st);
    return cudaErrorInvalidValue;
}

// Coulomb reading B (C12): G(x) = 1 before the sweeps; afterwards U_t(x) <- G(x) U_t(x) G(x+t)^dagger for every site.
// G: 2 parity blocks of H links in the 18-real layout.
template <typename T>
__global__ void __launch_bounds__(AUX_BLOCK) coulomb_init_kernel(Lattice L, T* __restrict__ G)
{
    const unsigned long long gid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (unsigned long long)L.H * 2ull) return;
    const unsigned h = (unsigned)(gid % L.H);
    const int parity = (int)(gid / L.H);
    cx<T> u[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) u[e] = {(e % 4 == 0) ? T(1) : T(0), T(0)};
    LinkIO<T, 18>::store(G + (size_t)parity * 18 * L.Hp, L.Hp, h, u, make_l2_policy(POLICY_NORMAL));
}

template <typename T, int R>
__global__ void __launch_bounds__(AUX_BLOCK) coulomb_finish_kernel(Lattice L, T* __restrict__ native, const T* __restrict__ G)
{
    const unsigned long long gid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (unsigned long long)L.H * 2ull) return;
    const unsigned h = (unsigned)(gid % L.H);
    const int parity = (int)(gid / L.H);
    const uint64_t pol = make_l2_policy(POLICY_NORMAL);
    const Site s = decode_site(L, h, parity);
    // x + t_hat: other parity block, one timeslice up (periodic)
    const unsigned st = (unsigned)L.Nxh * (unsigned)L.Ny * (unsigned)L.Nz;
    const unsigned hf = s.t == L.Nt - 1 ? h - st * (unsigned)(L.Nt - 1) : h + st;
    cx<T> u[9], g[9], gn[9], t[9];
    T* blk = native + (size_t)(parity * 4 + 3) * R * L.Hp;
    LinkIO<T, R>::load(blk, L.Hp, h, u, pol);
    LinkIO<T, 18>::load(G + (size_t)parity * 18 * L.Hp, L.Hp, h, g, pol);
    LinkIO<T, 18>::load(G + (size_t)(1 - parity) * 18 * L.Hp, L.Hp, hf, gn, pol);
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) t[3 * r + c] = g[3 * r] * u[c] + g[3 * r + 1] * u[3 + c] + g[3 * r + 2] * u[6 + c];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c)
            u[3 * r + c] = cmul_cb(t[3 * r], gn[3 * c]) + cmul_cb(t[3 * r + 1], gn[3 * c + 1]) + cmul_cb(t[3 * r + 2], gn[3 * c + 2]);
    LinkIO<T, R>::store(blk, L.Hp, h, u, pol);
}

cudaError_t launch_coulomb_init(int prec, const Lattice& L, void* G, cudaStream_t st)
{
    const unsigned long long n = (unsigned long long)L.H * 2ull;
    const unsigned grid = (unsigned)((n + AUX_BLOCK - 1) / AUX_BLOCK);
    if (prec == 0) coulomb_init_kernel<float><<<grid, AUX_BLOCK, 0, st>>>(L, (float*)G);
    else coulomb_init_kernel<double><<<grid, AUX_BLOCK, 0, st>>>(L, (double*)G);
    return cudaGetLastError();
}

cudaError_t launch_coulomb_finish(int prec, int R, const Lattice& L, void* native, const void* G, cudaStream_t st)
{
    const unsigned long long n = (unsigned long long)L.H * 2ull;
    const unsigned grid = (unsigned)((n + AUX_BLOCK - 1) / AUX_BLOCK);
    if (prec == 0 && R == 18) coulomb_finish_kernel<float, 18><<<grid, AUX_BLOCK, 0, st>>>(L, (float*)native, (const float*)G);
    else if (prec == 0 && R == 12) coulomb_finish_kernel<float, 12><<<grid, AUX_BLOCK, 0, st>>>(L, (float*)native, (const float*)G);
    else if (prec == 1 && R == 18) coulomb_finish_kernel<double, 18><<<grid, AUX_BLOCK, 0, st>>>(L, (double*)native, (const double*)G);
    else if (prec == 1 && R == 12) coulomb_finish_kernel<double, 12><<<grid, AUX_BLOCK, 0, st>>>(L, (double*)native, (const double*)G);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// reductions.  Grid (bx, 2*Nt): blockIdx.y = 2*t + parity, so every block lies inside one timeslice and the
// Coulomb per-timeslice theta (C12) falls out of the same partials.
// ---------------------------------------------------------------------------------------------------------
int reduce_blocks_per_slice(const Lattice& L)
{
    const unsigned Hs = (unsigned)L.Nxh * L.Ny * L.Nz;
    return (int)((Hs + AUX_BLOCK - 1) / AUX_BLOCK);
}

__device__ __forceinline__ void block_sum_to(double v, double* dst)
{
    __shared__ double warp_sums[AUX_BLOCK / 32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if ((threadIdx.x & 31) == 0) warp_sums[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double acc = 0.0;
#pragma unroll
        for (int w = 0; w < AUX_BLOCK / 32; ++w) acc += warp_sums[w];
        *dst = acc;
    }
}

// eq. 2.1, reading C1: sum over x, mu < nd of Re tr U_mu(x) on the current links
template <typename T, int R>
__global__ void __launch_bounds__(AUX_BLOCK) functional_kernel(Lattice L, int nd, const T* __restrict__ native,
                                                               double* __restrict__ partials)
{
    const unsigned Hs = (unsigned)L.Nxh * L.Ny * L.Nz;
    const unsigned local = blockIdx.x * blockDim.x + threadIdx.x;
    const int t = blockIdx.y >> 1, parity = blockIdx.y & 1;
    double acc = 0.0;
    const uint64_t pol = make_l2_policy(POLICY_NORMAL);
    if (local < Hs) {
        const unsigned h = (unsigned)t * Hs + local;
        for (int mu = 0; mu < nd; ++mu)
            acc += (double)LinkIO<T, R>::trace_re(native + (size_t)(parity * 4 + mu) * R * L.Hp, L.Hp, h, pol);
    }
    block_sum_to(acc, partials + (size_t)blockIdx.y * gridDim.x + blockIdx.x);
}

// eq. 2.5, reading C3: Delta(x) = traceless part of (K - K^dagger)/(2i),
// tr[Delta Delta^dagger] = sum_ab |Delta_ab|^2.  K from eq. 2.3 in the in-place form (C2).
template <typename T, int R>
__global__ void __launch_bounds__(AUX_BLOCK) theta_kernel(Lattice L, int nd, const T* __restrict__ native,
                                                          double* __restrict__ partials)
{
    const unsigned Hs = (unsigned)L.Nxh * L.Ny * L.Nz;
    const unsigned local = blockIdx.x * blockDim.x + threadIdx.x;
    const int t = blockIdx.y >> 1, parity = blockIdx.y & 1;
    double acc = 0.0;
    const uint64_t pol = make_l2_policy(POLICY_NORMAL);
    if (local < Hs) {
        const Site s = decode_site(L, (unsigned)t * Hs + local, parity);
        cx<double> K[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) K[e] = {0.0, 0.0};
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) { // unrolled: the loads of all directions are in flight together
            if (mu >= nd) break;
            cx<T> f[9], b[9];
            LinkIO<T, R>::load(native + (size_t)(parity * 4 + mu) * R * L.Hp, L.Hp, s.h, f, pol);
            LinkIO<T, R>::load(native + (size_t)((1 - parity) * 4 + mu) * R * L.Hp, L.Hp, backward_neighbour(L, s, mu), b, pol);
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    K[3 * r + c].re += (double)f[3 * r + c].re + (double)b[3 * c + r].re;
                    K[3 * r + c].im += (double)f[3 * r + c].im - (double)b[3 * c + r].im;
                }
        }
        // D_ab = (K_ab - conj(K_ba)) / (2i) = [ (Im K_ab + Im K_ba) - i (Re K_ab - Re K_ba) ] / 2
        const double tr3 = (K[0].im + K[4].im + K[8].im) / 3.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double d = K[4 * a].im - tr3;
            acc += d * d;
        }
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b2 = a + 1; b2 < 3; ++b2) {
                const double dr = 0.5 * (K[3 * a + b2].im + K[3 * b2 + a].im);
                const double di = 0.5 * (K[3 * a + b2].re - K[3 * b2 + a].re);
                acc += 2.0 * (dr * dr + di * di); // D is Hermitian: |D_ab|^2 = |D_ba|^2
            }
    }
    block_sum_to(acc, partials + (size_t)blockIdx.y * gridDim.x + blockIdx.x);
}

// final pass: one block; thread i adds the partials of timeslices i, i+blockDim, ... in index order; thread 0 then
// combines the slices in order.  scale_total multiplies the lattice sum; scale_slice the per-slice sums.
__global__ void __launch_bounds__(AUX_BLOCK) final_kernel(int Nt, int per_slice, const double* __restrict__ partials,
                                                          double scale_total, double scale_slice, double* __restrict__ out)
{
    for (int t = threadIdx.x; t < Nt; t += blockDim.x) {
        double acc = 0.0;
        const double* p = partials + (size_t)t * per_slice;
        for (int i = 0; i < per_slice; ++i) acc += p[i];
        out[2 + t] = acc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double total = 0.0, mx = 0.0;
        for (int t = 0; t < Nt; ++t) {
            const double v = out[2 + t];
            total += v;
            const double sv = v * scale_slice;
            if (t == 0 || sv > mx) mx = sv;
            out[2 + t] = sv;
        }
        out[0] = total * scale_total;
        out[1] = mx;
    }
}

// nt: timeslices reduced (L.Nt, or the owned slices of a slab context: its ghost slice is left out)
template <bool THETA>
static cudaError_t launch_reduction(int prec, int R, const Lattice& L, int nt, int nd, const void* native, double* partials,
                                    double* out, cudaStream_t st)
{
    const int bx = reduce_blocks_per_slice(L);
    const dim3 grid((unsigned)bx, (unsigned)(2 * nt));
#define GF_RED(T, RR)                                                                                   \
    do {                                                                                                \
        if (THETA) theta_kernel<T, RR><<<grid, AUX_BLOCK, 0, st>>>(L, nd, (const T*)native, partials);   \
        else functional_kernel<T, RR><<<grid, AUX_BLOCK, 0, st>>>(L, nd, (const T*)native, partials);    \
    } while (0)
    if (prec == 0 && R == 18) GF_RED(float, 18);
    else if (prec == 0 && R == 12) GF_RED(float, 12);
    else if (prec == 1 && R == 18) GF_RED(double, 18);
    else if (prec == 1 && R == 12) GF_RED(double, 12);
    else return cudaErrorInvalidValue;
#undef GF_RED
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double Vs = 2.0 * (double)L.H / (double)L.Nt, V = Vs * (double)nt;
    const double scale_total = THETA ? 1.0 / (3.0 * V) : 1.0 / (3.0 * nd * V);
    const double scale_slice = THETA ? 1.0 / (3.0 * Vs) : 1.0 / (3.0 * nd * Vs);
    final_kernel<<<1, AUX_BLOCK, 0, st>>>(nt, 2 * bx, partials, scale_total, scale_slice, out);
    return cudaGetLastError();
}

cudaError_t launch_functional(int prec, int R, const Lattice& L, int nt, int nd, const void* native, double* partials,
                              double* out, cudaStream_t st)
{
    return launch_reduction<false>(prec, R, L, nt, nd, native, partials, out, st);
}

cudaError_t launch_theta(int prec, int R, const Lattice& L, int nt, int nd, const void* native, double* partials,
                         double* out, cudaStream_t st)
{
    return launch_reduction<true>(prec, R, L, nt, nd, native, partials, out, st);
}

} // namespace gf

// ---------------------------------------------------------------------------------------------------------
// gf_debug_kp_math: the double-precision functions of the Kennedy-Pendleton draw (kp_neglog_word, kp_sincos2pi_word,
// gf_device.cuh) on given Philox words, so that a test can check them over their whole domain (2^23 uniforms)
// ---------------------------------------------------------------------------------------------------------
__global__ void kp_math_kernel(const unsigned* __restrict__ words, int n, double* __restrict__ nl, double* __restrict__ sn,
                               double* __restrict__ cs)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t x = words[i];
    if (nl != nullptr) nl[i] = gf::kp_neglog_word(x);
    if (sn != nullptr || cs != nullptr) {
        double s, c;
        gf::kp_sincos2pi_word(x, s, c);
        if (sn != nullptr) sn[i] = s;
        if (cs != nullptr) cs[i] = c;
    }
}

extern "C" int gf_debug_kp_math(const unsigned* words_dev, int n, double* neglog_dev, double* sin_dev, double* cos_dev, void* stream)
{
    if (words_dev == nullptr || n < 0) return -1; // GF_EINVAL
    if (n == 0) return 0;
    kp_math_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(words_dev, n, neglog_dev, sin_dev, cos_dev);
    return cudaGetLastError() == cudaSuccess ? 0 : -2; // GF_ECUDA
}


// ---------------------------------------------------------------------------------------------------------
// gf_theta_static (include/gf.h): the theta reduction for callers that must not allocate.
//
// Who that is.  A gauge-fixing step usually sits inside somebody else's program: a Monte Carlo or measurement code that
// took (nearly) all of the GPU's memory into its own pool when it started, or a job that shares the GPU under a fixed
// memory budget.  From there a cudaMalloc inside this library either fails outright or takes memory the host program
// has already promised elsewhere; and every cudaMalloc / cudaFree stalls the whole device while the driver maps memory,
// which is poison for a loop that checks theta every few sweeps.  gf_theta goes through a gf_ctx, and gf_create
// allocates.  This entry point needs no context and asks the driver for nothing: its inputs and outputs are the
// caller's, and the one piece of scratch the reduction needs -- one partial sum per thread block -- is the fixed array
// below, which is part of the library image itself.
//
// What it costs.  kStaticPartials doubles (1 MiB) of device memory on every GPU on which a process has loaded
// libgf.so, from the load until the process exits, whether or not this call is ever used.  A lattice that needs more
// block partials than that is refused (GF_EINVAL), not truncated.
//
// Sharing.  There is one array per GPU and every call on that GPU uses it.  Nothing in it has to start at zero: a launch
// writes every slot it later reads (one per block of the grid) before the final pass reads them, so the values a
// previous call left behind are never seen and no clearing pass is launched.  Two calls that are on the GPU at the
// same time (different streams, different host threads) write the same slots and read each other's sums: the caller
// must order them (same stream, or an event between them).
// ---------------------------------------------------------------------------------------------------------
namespace gf {

constexpr size_t kStaticPartials = 131072; // 64^4 needs 65536, 48^3 x 64 needs 27648, 64^3 x 128 exactly this many
constexpr int kStaticMaxDevices = 64;

// In device code this name IS the array.  In host code it is only a handle for the runtime's symbol calls -- never a
// device address: handing `static_partials` itself to a kernel from the host would give it a host address.
static __device__ __align__(256) double static_partials[kStaticPartials];

static double* g_static_partials_addr[kStaticMaxDevices]; // device address of the array on device i, once resolved
static int g_static_lock;                                  // spin flag guarding the table (no mutex header needed)

// Resolve, once per device and with that device current, where the array lives on it.
static cudaError_t static_partials_address(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    while (__atomic_exchange_n(&g_static_lock, 1, __ATOMIC_ACQUIRE)) { }
    double* p = g_static_partials_addr[dev];
    if (p == nullptr) {
        e = cudaGetSymbolAddress((void**)&p, static_partials);
        if (e == cudaSuccess && p == nullptr) e = cudaErrorInvalidSymbol;
        if (e == cudaSuccess) g_static_partials_addr[dev] = p;
    }
    __atomic_store_n(&g_static_lock, 0, __ATOMIC_RELEASE);
    if (e == cudaSuccess) *out = p;
    return e;
}

static int static_fail(char* err, size_t err_len, int code, const char* fmt, ...)
{
    if (err != nullptr && err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

} // namespace gf

extern "C" size_t gf_theta_static_max_partials(void) { return gf::kStaticPartials; }

extern "C" int gf_theta_static(int Nx, int Ny, int Nz, int Nt, int precision, int gauge, int reals_per_link,
                               const void* U_native_dev, double* out_dev, void* stream, char* err, size_t err_len)
{
    using namespace gf;
    const char* who = "gf_theta_static";
    if (err != nullptr && err_len > 0) err[0] = 0;
    const int N[4] = {Nx, Ny, Nz, Nt};
    for (int d = 0; d < 4; ++d)
        if (N[d] < 2 || (N[d] & 1))
            return static_fail(err, err_len, -1, "%s: extent %d is %d; every extent must be even and >= 2", who, d, N[d]);
    const unsigned long long V = (unsigned long long)Nx * Ny * Nz * Nt;
    if (V >= (1ull << 31)) return static_fail(err, err_len, -1, "%s: volume %llu >= 2^31", who, V);
    if (precision != 0 && precision != 1) return static_fail(err, err_len, -1, "%s: unknown precision %d", who, precision);
    if (gauge != 0 && gauge != 1) return static_fail(err, err_len, -1, "%s: unknown gauge %d", who, gauge);
    if (reals_per_link != 12 && reals_per_link != 18)
        return static_fail(err, err_len, -1, "%s: reals_per_link must be 12 or 18, got %d", who, reals_per_link);
    if (U_native_dev == nullptr || out_dev == nullptr) return static_fail(err, err_len, -1, "%s: NULL field or output", who);

    Lattice L;
    L.Nxh = Nx / 2; L.Ny = Ny; L.Nz = Nz; L.Nt = Nt; L.H = (unsigned)(V / 2);
    L.Hp = (L.H + 31u) & ~31u;
    const unsigned long long need = (unsigned long long)reduce_blocks_per_slice(L) * 2ull * (unsigned long long)Nt;
    if (need > kStaticPartials)
        return static_fail(err, err_len, -1,
                           "%s: a %dx%dx%dx%d lattice needs %llu block partials, the built-in scratch holds %zu (%zu KiB); "
                           "use gf_theta on a context for lattices this large",
                           who, Nx, Ny, Nz, Nt, need, (size_t)kStaticPartials, (size_t)(kStaticPartials * sizeof(double) / 1024));

    double* partials = nullptr;
    cudaError_t e = static_partials_address(&partials);
    if (e != cudaSuccess)
        return static_fail(err, err_len, -2, "%s: address of the built-in scratch: %s", who, cudaGetErrorString(e));
    e = launch_theta(precision, reals_per_link, L, Nt, gauge == 1 ? 3 : 4, U_native_dev, partials, out_dev, (cudaStream_t)stream);
    if (e != cudaSuccess) return static_fail(err, err_len, -2, "%s: launch: %s", who, cudaGetErrorString(e));
    return 0;
}
