// gf_internal.h -- declarations shared by the translation units of libgf.so (host side)
#pragma once
#include <cuda_runtime.h>

namespace gf {

struct SweepParams;
struct Lattice;

// gf_sweep_inst.cu, one pair per (precision, reals-per-link)
#define GF_DECLARE_SWEEP(sfx)                                                                                 \
    cudaError_t launch_sweep_##sfx(int tps, int mode, int block, const SweepParams& p, cudaStream_t stream); \
    cudaError_t sweep_attributes_##sfx(int tps, int mode, bool reading_b, bool dc, cudaFuncAttributes* attr);
GF_DECLARE_SWEEP(f32_r12)
GF_DECLARE_SWEEP(f32_r18)
GF_DECLARE_SWEEP(f64_r12)
GF_DECLARE_SWEEP(f64_r18)
#undef GF_DECLARE_SWEEP

// gf_aux.cu: layout conversion and reductions.  prec: 0 fp32, 1 fp64; R: 12 or 18.
// H_own: half-sites with a canonical counterpart (L.H, or less on a slab context whose last slice is a ghost)
cudaError_t launch_pack(int prec, int R, const Lattice& L, unsigned H_own, const double* canon, void* native,
                        cudaStream_t stream);
cudaError_t launch_unpack(int prec, int R, const Lattice& L, unsigned H_own, const void* native, double* canon,
                          cudaStream_t stream);

cudaError_t launch_pack_f32(int prec, int R, const Lattice& L, unsigned H_own, const float* canon, void* native, cudaStream_t stream);
cudaError_t launch_unpack_f32(int prec, int R, const Lattice& L, unsigned H_own, const void* native, float* canon, cudaStream_t stream);

// t-slab faces: temporal links of parity block `block_parity` of local timeslice t <-> contiguous buffer
cudaError_t launch_face(int prec, int R, const Lattice& L, unsigned Hs, int t, int block_parity, bool pack, void* native,
                        void* buf, cudaStream_t stream);

cudaError_t launch_convert(int sprec, int sR, int dprec, int dR, const Lattice& L, const void* src, void* dst,
                           cudaStream_t stream);

// Coulomb reading B: G(x) = 1; U_t(x) <- G(x) U_t(x) G(x+t)^dagger
cudaError_t launch_coulomb_init(int prec, const Lattice& L, void* G, cudaStream_t stream);
cudaError_t launch_coulomb_finish(int prec, int R, const Lattice& L, void* native, const void* G, cudaStream_t stream);

// Reduction scratch (device): partial sums per block, then a deterministic fixed-order final pass.
//   functional: out[0] = sum_{x, mu<nd} Re tr U_mu(x) / (3 nd V)
//   theta:      out[0] = theta over the whole lattice (eq. 2.5); out[1] = max_t theta_t; out[2+t] = theta_t
int reduce_blocks_per_slice(const Lattice& L);
cudaError_t launch_functional(int prec, int R, const Lattice& L, int nt, int nd, const void* native, double* partials,
                              double* out, cudaStream_t stream);
cudaError_t launch_theta(int prec, int R, const Lattice& L, int nt, int nd, const void* native, double* partials,
                         double* out, cudaStream_t stream);

} // namespace gf
