// gf_sweep_inst.cu -- one translation unit per (precision, reals-per-link): compiled four times by build.py with
//   -DGF_INST_FP64={0,1} -DGF_INST_R={12,18}
// so the seventy-two half-sweep kernels build in parallel.  Each unit exports one launcher and one
// attribute query, declared in gf_internal.h.
#include "gf_internal.h"
#include "gf_sweep.cuh"

#if GF_INST_FP64
typedef double real_t;
#else
typedef float real_t;
#endif

#define GF_CAT3_(a, b, c) a##b##c
#define GF_CAT3(a, b, c) GF_CAT3_(a, b, c)
#if GF_INST_FP64
#define GF_SUFFIX GF_CAT3(f64, _r, GF_INST_R)
#else
#define GF_SUFFIX GF_CAT3(f32, _r, GF_INST_R)
#endif
#define GF_NAME(stem) GF_CAT3(stem, _, GF_SUFFIX)

namespace gf {

typedef void (*sweep_fn)(const SweepParams);

template <int MODE, bool CB, bool DC, int MON>
static sweep_fn pick_tps(int tps)
{
    constexpr int R = GF_INST_R;
    if (tps == 1) return gf_half_sweep_kernel<real_t, R, 1, MODE, CB, DC, MON>;
    if (tps == 2) return gf_half_sweep_kernel<real_t, R, 2, MODE, CB, DC, MON>;
    if (tps == 4) return gf_half_sweep_kernel<real_t, R, 4, MODE, CB, DC, MON>;
    return nullptr;
}

// dc: fp32 heatbath kernel with the double chain at every site (the relaxation kernels pick their chain at run time)
// mon: relaxation kernel with the fused F / theta monitor (1: stop test only, 2: partials and duty)
template <int MODE, bool CB>
static sweep_fn pick_mon(int tps, int mon)
{
    if (mon == 2) return pick_tps<MODE, CB, false, 2>(tps);
    if (mon == 1) return pick_tps<MODE, CB, false, 1>(tps);
    return pick_tps<MODE, CB, false, 0>(tps);
}

template <bool CB>
static sweep_fn pick_mode(int tps, int mode, bool dc, int mon)
{
    if (mode == MODE_OVERRELAX) return pick_mon<MODE_OVERRELAX, CB>(tps, mon);
    if (mode == MODE_VARIANT) return pick_mon<MODE_VARIANT, CB>(tps, mon);
    if (mode == MODE_HEATBATH && mon == 0) {
#if !GF_INST_FP64
        if (dc) return pick_tps<MODE_HEATBATH, CB, true, 0>(tps);
#endif
        (void)dc;
        return pick_tps<MODE_HEATBATH, CB, false, 0>(tps);
    }
    return nullptr;
}

// cb: Coulomb reading B
static sweep_fn pick(int tps, int mode, bool cb, bool dc, int mon)
{
    return cb ? pick_mode<true>(tps, mode, dc, mon) : pick_mode<false>(tps, mode, dc, mon);
}

cudaError_t GF_NAME(launch_sweep)(int tps, int mode, int block, const SweepParams& p, cudaStream_t stream)
{
    const bool check = p.mon.F_part || p.mon.post_part || p.mon.pre_part || p.mon.red_post;
    sweep_fn fn = pick(tps, mode, p.G != nullptr, p.chain == CHAIN_DOUBLE, p.mon.state == nullptr ? 0 : (check ? 2 : 1));
    if (fn == nullptr || block <= 0 || block > MAX_BLOCK || (block % 32) != 0) return cudaErrorInvalidValue;
    const unsigned long long threads = (unsigned long long)p.h_count * (unsigned long long)tps;
    if (p.h_count == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((threads + (unsigned)block - 1ull) / (unsigned)block);
    if (!p.pdl) {
        fn<<<grid, block, 0, stream>>>(p);
        return cudaGetLastError();
    }
    // programmatic dependent launch: the grid may start while the previous kernel on the stream drains; the
    // kernel itself waits (cudaGridDependencySynchronize) before it touches the field
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, fn, p);
}

cudaError_t GF_NAME(sweep_attributes)(int tps, int mode, bool reading_b, bool dc, cudaFuncAttributes* attr)
{
    sweep_fn fn = pick(tps, mode, reading_b, dc, 0);
    if (fn == nullptr) return cudaErrorInvalidValue;
    return cudaFuncGetAttributes(attr, fn);
}

} // namespace gf
