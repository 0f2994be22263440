// gf_sweep_inst.cu -- the half-sweep kernels of one (precision, reals-per-link), compiled by build.py as three translation
// units per pair so that the instantiations build in parallel:
//   -DGF_INST_FP64={0,1} -DGF_INST_R={12,18} -DGF_INST_PART={0,1,2}
//   part 0: relaxation kernels (overrelaxation, variants) and the launcher / attribute query (declared in gf_internal.h)
//   part 1: relaxation kernels with the fused F / theta monitor
//   part 2: heatbath kernels
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

// the kernels of the other parts, by their selectors (NULL: no such kernel)
sweep_fn GF_NAME(pick_monitor)(int tps, int mode, bool cb, int mon);
sweep_fn GF_NAME(pick_heatbath)(int tps, bool cb, bool dc);

template <int MODE, bool CB, bool DC, int MON>
static sweep_fn pick_tps(int tps)
{
    constexpr int R = GF_INST_R;
    if (tps == 1) return gf_half_sweep_kernel<real_t, R, 1, MODE, CB, DC, MON>;
    if (tps == 2) return gf_half_sweep_kernel<real_t, R, 2, MODE, CB, DC, MON>;
    if (tps == 4) return gf_half_sweep_kernel<real_t, R, 4, MODE, CB, DC, MON>;
    return nullptr;
}

#if GF_INST_PART == 0
// cb: Coulomb reading B; dc: fp32 heatbath kernel with the double chain at every site (the relaxation kernels pick
// their chain at run time); mon: relaxation kernel with the fused F / theta monitor (1: stop test only, 2: partials, duty)
static sweep_fn pick(int tps, int mode, bool cb, bool dc, int mon)
{
    if (mode == MODE_HEATBATH) return mon == 0 ? GF_NAME(pick_heatbath)(tps, cb, dc) : nullptr;
    if (mon != 0) return GF_NAME(pick_monitor)(tps, mode, cb, mon);
    if (mode == MODE_OVERRELAX) return cb ? pick_tps<MODE_OVERRELAX, true, false, 0>(tps) : pick_tps<MODE_OVERRELAX, false, false, 0>(tps);
    if (mode == MODE_VARIANT) return cb ? pick_tps<MODE_VARIANT, true, false, 0>(tps) : pick_tps<MODE_VARIANT, false, false, 0>(tps);
    return nullptr;
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
#endif // part 0

#if GF_INST_PART == 1
template <int MODE, bool CB>
static sweep_fn pick_mon(int tps, int mon)
{
    if (mon == 2) return pick_tps<MODE, CB, false, 2>(tps);
    if (mon == 1) return pick_tps<MODE, CB, false, 1>(tps);
    return nullptr;
}

sweep_fn GF_NAME(pick_monitor)(int tps, int mode, bool cb, int mon)
{
    if (mode == MODE_OVERRELAX) return cb ? pick_mon<MODE_OVERRELAX, true>(tps, mon) : pick_mon<MODE_OVERRELAX, false>(tps, mon);
    if (mode == MODE_VARIANT) return cb ? pick_mon<MODE_VARIANT, true>(tps, mon) : pick_mon<MODE_VARIANT, false>(tps, mon);
    return nullptr;
}
#endif // part 1

#if GF_INST_PART == 2
sweep_fn GF_NAME(pick_heatbath)(int tps, bool cb, bool dc)
{
#if !GF_INST_FP64
    if (dc) return cb ? pick_tps<MODE_HEATBATH, true, true, 0>(tps) : pick_tps<MODE_HEATBATH, false, true, 0>(tps);
#endif
    (void)dc;
    return cb ? pick_tps<MODE_HEATBATH, true, false, 0>(tps) : pick_tps<MODE_HEATBATH, false, false, 0>(tps);
}
#endif // part 2

} // namespace gf
