// gf_api.cu -- the C ABI of libgf.so (include/gf.h): argument checking, context, launch sequencing.
// No arithmetic of the method lives here; every step runs in the kernels of gf_sweep.cuh / gf_aux.cu.
#include <cstdarg>
#include <cstdio>
#include <climits>
#include <cstring>
#include <new>

#include "../../include/gf.h"
#include "gf_internal.h"
#include "gf_sweep.cuh"

using namespace gf;

struct gf_ctx {
    int Nx, Ny, Nz, Nt;               // Nt: timeslices this context owns (a t-slab: t_begin .. t_begin + Nt - 1 of Nt_global)
    int slab, t_begin, Nt_global;     // slab != 0: L.Nt = Nt + 1, the extra (last) slice is the ghost of slice t_begin - 1
    unsigned Hs, H_own;               // half-sites per timeslice; half-sites owned (= Nt * Hs; L.H counts the ghost too)
    int precision, gauge, R;
    Lattice L;
    int tps, block;
    int reunit_every;
    int l2_reversal;
    int ld_policy, st_policy;         // L2 eviction policy of the sweep's link loads / stores
    int pdl;                          // programmatic dependent launch of consecutive half-sweeps
    int prefetch;                     // L2 prefetch distance of the sweep kernels, in sites (0 = off)
    int coulomb_b;                    // Coulomb reading B: temporal links transformed once per call (C12)
    void* d_gfield;                   // its accumulated g(x): V links of 18 reals
    int chain;                        // fp32: precision of the site chain (CHAIN_*)
    float watch_threshold;            // hybrid chain: conditioning number below which a half-sweep counts as rough
    float fix_threshold;              // heatbath: |k| below which a site update is redone in double
    int* d_rough;                     // hybrid chain: ring of ROUGH_RING flags + 4 words for two diagnostic counters
    unsigned long long call_sweeps;   // sweeps since the start of the current API call (cadence of the reunitarisation)
    int force_rough;                  // hybrid chain: run the double chain regardless of the flags (relaxation sweeps inside an annealing)
    unsigned long long half_sweeps;   // half-sweeps of any kind since creation (alternates the traversal direction)
    unsigned long long launches;
    unsigned* d_trials;
    cudaStream_t last_stream;
    double* d_partials;               // reduction partials
    double* d_out;                    // reduction results: [0] total, [1] max slice, [2..2+Nt) slices
    double* h_out;                    // pinned mirror of d_out
    int bx;
    // fused F / theta monitor of gf_fix / gf_fix_slices (lazily allocated; sized for one launch shape)
    int monitor;                      // 0: the paper's separate check kernel, 1: fused where it applies and pays (default), 2: fused where it applies
    int fix_lag, fix_fused;           // form of the last gf_fix / gf_fix_slices on this context (-1: none yet); gf_fix_last_form
    char* d_mon;                      // MonitorState, theta_t[2 Nt], frozen_from[Nt] | group | partials
    char* h_mon;                      // pinned: two copies of the prefix up to `frozen`
    size_t mon_prefix, mon_bytes;
    int mon_blocks, mon_groups;       // partials per plane, duty blocks per timeslice the buffer was sized for
    cudaEvent_t mon_event[2];
    // host-buffer path staging (lazily allocated)
    double* d_canon;
    void* d_native;
    // pipelined host path (gf_overrelax_host_batch): three staging slots, three streams
    struct BatchSlot { void* canon; void* native; double* res; cudaEvent_t in, comp, out; } slot[3];
    cudaStream_t batch_stream[3];     // H2D, compute, D2H
    size_t batch_canon_bytes;         // staging size the slots were allocated for (0: not allocated)
    double* h_batch; size_t h_batch_doubles; // pinned results
    char err[512];
};

static char g_create_err[512] = "";
static int update_to_mode(int update, int* mode, int* variant);
static int reduce_to_host(gf_ctx* c, const void* U, bool theta, const char* who);

static int fail(gf_ctx* ctx, int code, const char* fmt, ...)
{
    char* dst = ctx ? ctx->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

static int cuda_fail(gf_ctx* ctx, cudaError_t e, const char* what)
{
    return fail(ctx, e == cudaErrorMemoryAllocation ? GF_ENOMEM : GF_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

static size_t real_size(const gf_ctx* c) { return c->precision == GF_FP64 ? 8 : 4; }

extern "C" const char* gf_last_error(const gf_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

static int create_impl(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int precision, int gauge, int slab, int t_begin,
                       int Nt_global)
{
    if (out == nullptr) return fail(nullptr, GF_EINVAL, "gf_create: out is NULL");
    *out = nullptr;
    const int N[4] = {Nx, Ny, Nz, Nt};
    for (int d = 0; d < 4; ++d)
        if (N[d] < 2 || (N[d] & 1))
            return fail(nullptr, GF_EINVAL, "gf_create: extent %d is %d; every extent must be even and >= 2 (C5)", d, N[d]);
    const unsigned long long V = (unsigned long long)Nx * Ny * Nz * (Nt + (slab ? 1 : 0)); // the allocation: ghost slice included
    if (V >= (1ull << 31)) return fail(nullptr, GF_EINVAL, "gf_create: volume %llu >= 2^31", V);
    if (precision != GF_FP32 && precision != GF_FP64) return fail(nullptr, GF_EINVAL, "gf_create: unknown precision %d", precision);
    if (gauge != GF_LANDAU && gauge != GF_COULOMB) return fail(nullptr, GF_EINVAL, "gf_create: unknown gauge %d", gauge);

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, GF_ECUDA, "gf_create: no CUDA device (%s); this library has no CPU path",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");

    gf_ctx* c = new (std::nothrow) gf_ctx();
    if (c == nullptr) return fail(nullptr, GF_ENOMEM, "gf_create: host allocation failed");
    c->Nx = Nx; c->Ny = Ny; c->Nz = Nz; c->Nt = Nt;
    c->precision = precision; c->gauge = gauge; c->R = 18;
    c->slab = slab; c->t_begin = t_begin; c->Nt_global = Nt_global;
    c->L.Nxh = Nx / 2; c->L.Ny = Ny; c->L.Nz = Nz; c->L.Nt = Nt + (slab ? 1 : 0); c->L.H = (unsigned)(V / 2);
    c->L.Hp = (c->L.H + 31u) & ~31u;
    c->Hs = (unsigned)(Nx / 2) * (unsigned)Ny * (unsigned)Nz;
    c->H_own = c->Hs * (unsigned)Nt;
    c->tps = 0;   // 0 = automatic: resolved per (precision, storage, mode) by auto_tps()
    c->block = 0; // 0 = automatic
    c->reunit_every = -1; // automatic: reunit_due()
    c->l2_reversal = 1;
    c->ld_policy = POLICY_NORMAL; c->st_policy = POLICY_EVICT_LAST; // measured best: profiles/r1_variants.md
    c->pdl = 1;
    c->prefetch = -1; // automatic
    c->chain = CHAIN_HYBRID; c->watch_threshold = 1.0f; c->fix_threshold = 0.15f; c->d_rough = nullptr;
    c->coulomb_b = -1; c->d_gfield = nullptr; // automatic: reading B in fp32, A in fp64 (uses_reading_b)
    c->call_sweeps = 0; c->half_sweeps = 0; c->launches = 0; c->force_rough = 0;
    c->d_trials = nullptr; c->last_stream = nullptr;
    c->d_canon = nullptr; c->d_native = nullptr;
    memset(c->slot, 0, sizeof c->slot);
    c->batch_stream[0] = c->batch_stream[1] = c->batch_stream[2] = nullptr;
    c->batch_canon_bytes = 0; c->h_batch = nullptr; c->h_batch_doubles = 0;
    c->err[0] = 0;
    c->bx = reduce_blocks_per_slice(c->L);
    c->fix_lag = c->fix_fused = -1;
    c->monitor = 1; c->d_mon = nullptr; c->h_mon = nullptr; c->mon_prefix = c->mon_bytes = 0; c->mon_blocks = c->mon_groups = 0;
    c->mon_event[0] = c->mon_event[1] = nullptr;
    const size_t npart = (size_t)c->bx * 2 * Nt;
    c->d_partials = nullptr; c->d_out = nullptr; c->h_out = nullptr;
    if ((e = cudaMalloc(&c->d_partials, npart * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc(&c->d_out, (size_t)(Nt + 2) * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc(&c->d_rough, (ROUGH_RING + 4) * sizeof(int))) != cudaSuccess ||
        (e = cudaMemset(c->d_rough, 0, (ROUGH_RING + 4) * sizeof(int))) != cudaSuccess ||
        (e = cudaMallocHost(&c->h_out, (size_t)(Nt + 2) * sizeof(double))) != cudaSuccess) {
        int rc = cuda_fail(nullptr, e, "gf_create: scratch allocation");
        gf_destroy(c);
        return rc;
    }
    *out = c;
    return GF_OK;
}

extern "C" int gf_create(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int precision, int gauge)
{
    return create_impl(out, Nx, Ny, Nz, Nt, precision, gauge, 0, 0, Nt);
}

extern "C" int gf_create_slab(gf_ctx** out, int Nx, int Ny, int Nz, int Nt_global, int t_begin, int t_end, int precision,
                              int gauge)
{
    if (out != nullptr) *out = nullptr;
    if (Nt_global < 2 || (Nt_global & 1) || t_begin < 0 || t_end > Nt_global || t_end - t_begin < 2 || (t_begin & 1) ||
        ((t_end - t_begin) & 1))
        return fail(nullptr, GF_EINVAL, "gf_create_slab: slab [%d, %d) of %d timeslices; bounds must be even, the slab at least 2 slices "
                                        "(the local checkerboard must be the global one)", t_begin, t_end, Nt_global);
    return create_impl(out, Nx, Ny, Nz, t_end - t_begin, precision, gauge, 1, t_begin, Nt_global);
}

extern "C" void gf_destroy(gf_ctx* c)
{
    if (c == nullptr) return;
    if (c->d_partials) cudaFree(c->d_partials);
    if (c->d_out) cudaFree(c->d_out);
    if (c->d_rough) cudaFree(c->d_rough);
    if (c->d_mon) cudaFree(c->d_mon);
    if (c->h_mon) cudaFreeHost(c->h_mon);
    for (int i = 0; i < 2; ++i) if (c->mon_event[i]) cudaEventDestroy(c->mon_event[i]);
    if (c->h_out) cudaFreeHost(c->h_out);
    for (int i = 0; i < 3; ++i) {
        if (c->slot[i].canon) cudaFree(c->slot[i].canon);
        if (c->slot[i].native) cudaFree(c->slot[i].native);
        if (c->slot[i].res) cudaFree(c->slot[i].res);
        if (c->slot[i].in) cudaEventDestroy(c->slot[i].in);
        if (c->slot[i].comp) cudaEventDestroy(c->slot[i].comp);
        if (c->slot[i].out) cudaEventDestroy(c->slot[i].out);
        if (c->batch_stream[i]) cudaStreamDestroy(c->batch_stream[i]);
    }
    if (c->h_batch) cudaFreeHost(c->h_batch);
    if (c->d_canon) cudaFree(c->d_canon);
    if (c->d_native) cudaFree(c->d_native);
    if (c->d_gfield) cudaFree(c->d_gfield);
    delete c;
}

extern "C" int gf_set_storage(gf_ctx* c, int R)
{
    if (c == nullptr) return GF_EINVAL;
    if (R != 12 && R != 18) return fail(c, GF_EINVAL, "gf_set_storage: reals_per_link must be 12 or 18, got %d", R);
    if (c->d_native != nullptr && R != c->R) { cudaFree(c->d_native); c->d_native = nullptr; }
    if (R != c->R)
        for (int i = 0; i < 3; ++i)
            if (c->slot[i].native) { cudaFree(c->slot[i].native); c->slot[i].native = nullptr; c->batch_canon_bytes = 0; }
    c->R = R;
    return GF_OK;
}

extern "C" size_t gf_field_bytes(const gf_ctx* c)
{
    if (c == nullptr) return 0;
    return (size_t)8 * c->L.Hp * (size_t)c->R * real_size(c); // whole tiles of 32 sites per link block
}

extern "C" int gf_set_tuning(gf_ctx* c, int tps, int block)
{
    if (c == nullptr) return GF_EINVAL;
    if (tps != 0 && tps != 1 && tps != 2 && tps != 4) return fail(c, GF_EINVAL, "gf_set_tuning: threads_per_site must be 1, 2 or 4");
    if (block != 0 && (block < 32 || block > MAX_BLOCK || block % 32)) return fail(c, GF_EINVAL, "gf_set_tuning: block must be a multiple of 32 in [32, %d]", MAX_BLOCK);
    c->tps = tps;     // 0 returns to the automatic choice
    c->block = block;
    return GF_OK;
}

extern "C" int gf_set_reunit(gf_ctx* c, int every)
{
    if (c == nullptr) return GF_EINVAL;
    if (every < -1) return fail(c, GF_EINVAL, "gf_set_reunit: every must be >= 0, or -1 for automatic");
    c->reunit_every = every;
    return GF_OK;
}

extern "C" int gf_set_l2_reversal(gf_ctx* c, int on)
{
    if (c == nullptr) return GF_EINVAL;
    c->l2_reversal = on ? 1 : 0;
    return GF_OK;
}

extern "C" int gf_set_l2_policy(gf_ctx* c, int load_policy, int store_policy)
{
    if (c == nullptr) return GF_EINVAL;
    if (load_policy < 0 || load_policy > 2 || store_policy < 0 || store_policy > 2)
        return fail(c, GF_EINVAL, "gf_set_l2_policy: policies must be 0 (normal), 1 (evict first) or 2 (evict last)");
    c->ld_policy = load_policy;
    c->st_policy = store_policy;
    return GF_OK;
}

extern "C" int gf_set_pdl(gf_ctx* c, int on)
{
    if (c == nullptr) return GF_EINVAL;
    c->pdl = on ? 1 : 0;
    return GF_OK;
}

extern "C" int gf_set_prefetch(gf_ctx* c, int sites)
{
    if (c == nullptr) return GF_EINVAL;
    if (sites < -1) return fail(c, GF_EINVAL, "gf_set_prefetch: distance must be >= 0, or -1 for automatic");
    c->prefetch = sites;
    return GF_OK;
}

extern "C" int gf_set_trial_buffer(gf_ctx* c, unsigned* d_trials)
{
    if (c == nullptr) return GF_EINVAL;
    c->d_trials = d_trials;
    return GF_OK;
}

extern "C" int gf_set_monitor(gf_ctx* c, int fused)
{
    if (c == nullptr) return GF_EINVAL;
    if (fused < 0 || fused > 2) return fail(c, GF_EINVAL, "gf_set_monitor: mode must be 0 (separate check), 1 (automatic) or 2 (fused wherever it applies)");
    c->monitor = fused;
    return GF_OK;
}

extern "C" int gf_monitor_last(gf_ctx* c, int* check_sweep, double* theta_host, double* F_host, double* theta_host_Nt)
{
    if (c == nullptr) return GF_EINVAL;
    if (c->d_mon == nullptr) return fail(c, GF_EINVAL, "gf_monitor_last: no fused fixing loop has run on this context");
    cudaError_t e = cudaStreamSynchronize(c->last_stream);
    if (e == cudaSuccess) e = cudaMemcpy(c->h_mon, c->d_mon, c->mon_prefix, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e, "gf_monitor_last");
    const MonitorState* hs = reinterpret_cast<const MonitorState*>(c->h_mon);
    if (check_sweep) *check_sweep = hs->checks > 0 ? hs->check_sweep : 0;
    if (theta_host) *theta_host = hs->theta;
    if (F_host) *F_host = hs->F;
    if (theta_host_Nt) memcpy(theta_host_Nt, c->h_mon + sizeof(MonitorState), sizeof(double) * (size_t)c->Nt);
    return GF_OK;
}

extern "C" int gf_set_chain(gf_ctx* c, int chain, double watch_threshold, double fix_threshold)
{
    if (c == nullptr) return GF_EINVAL;
    if (chain < 0 || chain > 2) return fail(c, GF_EINVAL, "gf_set_chain: chain must be 0 (fp32), 1 (double) or 2 (hybrid)");
    if (!(watch_threshold >= 0.0 && watch_threshold <= 1e3)) return fail(c, GF_EINVAL, "gf_set_chain: watch_threshold = %g outside [0, 1e3]", watch_threshold);
    if (!(fix_threshold >= 0.0 && fix_threshold <= 1e3)) return fail(c, GF_EINVAL, "gf_set_chain: fix_threshold = %g outside [0, 1e3]", fix_threshold);
    c->chain = chain;
    if (watch_threshold > 0.0) c->watch_threshold = (float)watch_threshold;
    if (fix_threshold > 0.0) c->fix_threshold = (float)fix_threshold;
    return GF_OK;
}

extern "C" int gf_chain_count(gf_ctx* c, unsigned long long* double_launches_host, unsigned long long* double_sites_host)
{
    if (c == nullptr) return GF_EINVAL;
    unsigned long long both[2] = {0ull, 0ull};
    cudaError_t e = cudaStreamSynchronize(c->last_stream);
    if (e == cudaSuccess) e = cudaMemcpy(both, c->d_rough + ROUGH_RING, sizeof both, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e, "gf_chain_count");
    if (double_launches_host) *double_launches_host = both[0];
    if (double_sites_host) *double_sites_host = both[1];
    return GF_OK;
}

extern "C" unsigned long long gf_launch_count(const gf_ctx* c) { return c ? c->launches : 0ull; }

// Launch shape chosen from the measurements in profiles/ (DESIGN.md "Kernels"): the kernel is latency/bandwidth
// bound and wants as many bytes in flight per SM as the register file allows -- few, fat threads in one-warp
// blocks.  fp32 R18: one thread per site (8 links = 144 reals in registers); fp32 R12 and fp64: two threads per
// site (forward+backward links of two directions each), K combined with one warp shuffle.
// Coulomb reading B pays where one thread holds all links of a site (fp32: +14 % at R = 18, +4 % at R = 12); with two
// threads per site the thread that drops the temporal links idles (fp64: -2 %), so automatic = fp32 only.
static bool uses_reading_b(const gf_ctx* c, int mode)
{
    (void)mode;
    if (c->gauge != GF_COULOMB || c->slab) return false; // a slab would have to exchange its g(x) face for the final pass
    return c->coulomb_b < 0 ? c->precision == GF_FP32 : c->coulomb_b != 0;
}

static int auto_tps(const gf_ctx* c, int mode)
{
    if (c->tps) return c->tps;
    if (c->precision == GF_FP32 && uses_reading_b(c, mode)) return 1;
    if (c->precision == GF_FP64) return 2;
    if (mode == MODE_HEATBATH) return 1; // the draw is done once per thread: one thread per site (R12: 0.83 vs 0.65)
    return c->R == 18 ? 1 : 2;
}
// L2 prefetch distance (sites), from the sweep in profiles/r1_variants.md: a quarter of a wave ahead helps the
// variants with more arithmetic per byte (R = 12: +2..3 %, heatbath: +1.5 %); the R = 18 overrelaxation kernels
// already saturate the memory system with their own outstanding loads (fp32: -1 % with prefetch, fp64: neutral).
static int auto_prefetch(const gf_ctx* c, int mode)
{
    if (c->prefetch >= 0) return c->prefetch;
    if (mode == MODE_HEATBATH) return c->precision == GF_FP32 ? (c->R == 18 ? 7104 : 9472) : 0; // fp32 R12: 86.8 -> 82.8 us at 32^4 (r2_variants.md H)
    return c->R == 12 ? 4736 : 0;
}
static int auto_block(const gf_ctx* c) { return c->block ? c->block : 32; }

static cudaError_t launch_sweep(gf_ctx* c, int mode, const SweepParams& p_in, cudaStream_t st)
{
    const int tps = auto_tps(c, mode), block = auto_block(c);
    SweepParams p = p_in;
    p.prefetch = (unsigned)auto_prefetch(c, mode);
    if (mode == MODE_HEATBATH) p.watch_thr2 = c->chain == CHAIN_FP32 ? -1.0f : c->fix_threshold * c->fix_threshold;
    if (c->precision == GF_FP32) return c->R == 18 ? launch_sweep_f32_r18(tps, mode, block, p, st) : launch_sweep_f32_r12(tps, mode, block, p, st);
    return c->R == 18 ? launch_sweep_f64_r18(tps, mode, block, p, st) : launch_sweep_f64_r12(tps, mode, block, p, st);
}

extern "C" int gf_kernel_info(gf_ctx* c, int mode, int* regs, int* local_bytes)
{
    if (c == nullptr) return GF_EINVAL;
    if (mode < 0 || mode > 2) return fail(c, GF_EINVAL, "gf_kernel_info: mode must be 0 (overrelaxation), 1 (heatbath) or 2 (variants)");
    cudaFuncAttributes a;
    cudaError_t e;
    const int tps = auto_tps(c, mode);
    const bool rb = uses_reading_b(c, mode);
    const bool dc = c->precision == GF_FP32 && c->chain == CHAIN_DOUBLE;
    if (c->precision == GF_FP32) e = c->R == 18 ? sweep_attributes_f32_r18(tps, mode, rb, dc, &a) : sweep_attributes_f32_r12(tps, mode, rb, dc, &a);
    else e = c->R == 18 ? sweep_attributes_f64_r18(tps, mode, rb, dc, &a) : sweep_attributes_f64_r12(tps, mode, rb, dc, &a);
    if (e != cudaSuccess) return cuda_fail(c, e, "gf_kernel_info");
    if (regs) *regs = a.numRegs;
    if (local_bytes) *local_bytes = (int)a.localSizeBytes;
    return GF_OK;
}

static SweepParams base_params(gf_ctx* c, void* U)
{
    SweepParams p;
    memset(&p, 0, sizeof p);
    p.U = U;
    p.L = c->L;
    p.nd = c->gauge == GF_COULOMB ? 3 : 4;
    p.omega = 1.0;
    p.ph.T = 1.0;
    p.h_begin = 0;
    p.h_count = c->H_own;
    p.site_offset = c->slab ? (uint32_t)c->t_begin * 2u * c->Hs : 0u;
    p.ld_policy = c->ld_policy;
    p.st_policy = c->st_policy;
    p.pdl = c->pdl;
    p.chain = c->chain;
    p.watch_thr2 = c->watch_threshold * c->watch_threshold;
    p.rough = c->d_rough;
    p.dc_count = reinterpret_cast<unsigned long long*>(c->d_rough + ROUGH_RING);
    return p;
}

extern "C" int gf_pack(gf_ctx* c, const double* canon, void* native, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    if (canon == nullptr || native == nullptr) return fail(c, GF_EINVAL, "gf_pack: NULL pointer");
    c->last_stream = (cudaStream_t)stream;
    cudaError_t e = launch_pack(c->precision, c->R, c->L, c->H_own, canon, native, c->last_stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "gf_pack");
    c->launches += 1;
    return GF_OK;
}

extern "C" int gf_unpack(gf_ctx* c, const void* native, double* canon, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    if (canon == nullptr || native == nullptr) return fail(c, GF_EINVAL, "gf_unpack: NULL pointer");
    c->last_stream = (cudaStream_t)stream;
    cudaError_t e = launch_unpack(c->precision, c->R, c->L, c->H_own, native, canon, c->last_stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "gf_unpack");
    c->launches += 1;
    return GF_OK;
}

// Unitarity policy (C15).  Automatic cadence of the re-orthonormalisation on load (RED half-sweep, every link once):
//   18-real storage: rounding makes the links drift linearly -- fp32 every 16th sweep, fp64 never;
//   12-real storage: the rebuilt third row feeds the norm errors of rows 0,1 back into them, which grows
//   EXPONENTIALLY under large rotations (measured x1.5-1.7 per heatbath sweep at T = 1, both precisions: fp32 loses
//   unitarity after ~50 sweeps, fp64 after ~150) -- every 4th sweep for the hot updates (heatbath, stochastic /
//   microcanonical), every 16th for overrelaxation, in fp32 and fp64.
// The cadence counts the sweeps (of any kind) since the start of the current API call, so that a call's result
// depends on its arguments and the field only, not on the context's history.
static int reunit_every(const gf_ctx* c, bool hot)
{
    int every = c->reunit_every;
    if (every < 0) every = c->R == 12 ? (hot ? 4 : 16) : (c->precision == GF_FP32 ? 16 : 0);
    return every;
}

static bool reunit_due(const gf_ctx* c, bool hot)
{
    const int every = reunit_every(c, hot);
    return every > 0 && ((c->call_sweeps + 1) % (unsigned long long)every) == 0;
}

extern "C" int gf_set_coulomb_reading(gf_ctx* c, int reading_b)
{
    if (c == nullptr) return GF_EINVAL;
    if (c->gauge != GF_COULOMB) return fail(c, GF_EINVAL, "gf_set_coulomb_reading: the context is not in Coulomb gauge");
    c->coulomb_b = reading_b < 0 ? -1 : (reading_b ? 1 : 0);
    return GF_OK;
}

// the per-half-sweep part of the launch parameters
static void set_phase(gf_ctx* c, SweepParams& p, int parity, bool reunit)
{
    p.ph.parity = parity;
    p.ph.reunit = (reunit && parity == 0) ? 1 : 0; // every link is loaded once per half-sweep (C6)
    p.ph.reverse = c->l2_reversal ? (int)(c->half_sweeps & 1ull) : 0;
    // hybrid chain (fp32): the ring position counts the half-sweeps of the call; its first sweep runs the double chain
    p.ph.rough_slot = (int)((2ull * c->call_sweeps + (unsigned)parity) % ROUGH_RING);
    p.ph.rough_force = (c->call_sweeps == 0 || c->force_rough) ? 1 : 0;
}

// start of an API call that sweeps: the sweep counter of the call and, for the hybrid chain, a clean flag ring
static int begin_call(gf_ctx* c, cudaStream_t st)
{
    c->call_sweeps = 0;
    c->last_stream = st;
    if (c->precision == GF_FP32 && c->chain == CHAIN_HYBRID) {
        cudaError_t e = cudaMemsetAsync(c->d_rough, 0, ROUGH_RING * sizeof(int), st);
        if (e != cudaSuccess) return cuda_fail(c, e, "roughness flags");
    }
    return GF_OK;
}

// nsweeps sweeps (RED then BLACK) of one member of the relaxation family on `st`
// sweep0: index of the first of them within the API call that runs them (the counter of the stochastic decisions,
//   C18: it restarts at 0 with every gf_relax call and runs on through the chunks of gf_fix / gf_fix_slices)
// active (may be NULL = all): Nt flags; only the sites of the flagged timeslices are updated, one launch per
// maximal run of consecutive flagged slices (their half-site indices are contiguous) -- C20
static int run_sweeps_core(gf_ctx* c, void* U, int mode, int variant, double param, int nsweeps, int sweep0,
                           unsigned long long seed, cudaStream_t st, const char* who, const unsigned char* active,
                           void* gfield, int* launched = nullptr)
{
    c->last_stream = st;
    SweepParams p = base_params(c, U);
    p.G = gfield;
    p.omega = param;
    p.variant = variant;
    p.key0 = (uint32_t)seed;
    p.key1 = (uint32_t)(seed >> 32);
    for (int sweep = 0; sweep < nsweeps; ++sweep) {
        const bool reunit = reunit_due(c, mode == MODE_VARIANT && variant == VARIANT_STOCHASTIC);
        p.ph.step = (uint32_t)(sweep0 + sweep);
        for (int parity = 0; parity < 2; ++parity) { // RED, BLACK
            set_phase(c, p, parity, reunit);
            if (active == nullptr) {
                cudaError_t e = launch_sweep(c, mode, p, st);
                if (e != cudaSuccess) return cuda_fail(c, e, who);
                c->launches += 1;
                if (launched) *launched += 1;
            } else {
                const unsigned Hs = c->Hs; // half-sites per timeslice
                for (int t = 0; t < c->Nt;) {
                    if (!active[t]) { ++t; continue; }
                    int t1 = t;
                    while (t1 < c->Nt && active[t1]) ++t1;
                    p.h_begin = (unsigned)t * Hs;
                    p.h_count = (unsigned)(t1 - t) * Hs;
                    cudaError_t e = launch_sweep(c, mode, p, st);
                    if (e != cudaSuccess) return cuda_fail(c, e, who);
                    c->launches += 1;
                    if (launched) *launched += 1;
                    t = t1;
                }
            }
            c->half_sweeps += 1;
        }
        c->call_sweeps += 1;
    }
    return GF_OK;
}

extern "C" int gf_convert(gf_ctx* src, const void* U_src, gf_ctx* dst, void* U_dst, void* stream)
{
    if (src == nullptr || dst == nullptr) return GF_EINVAL;
    if (U_src == nullptr || U_dst == nullptr) return fail(dst, GF_EINVAL, "gf_convert: NULL field");
    if (src->Nx != dst->Nx || src->Ny != dst->Ny || src->Nz != dst->Nz || src->Nt != dst->Nt || src->slab != dst->slab)
        return fail(dst, GF_EINVAL, "gf_convert: the two contexts describe different lattices");
    if (U_src == U_dst) return fail(dst, GF_EINVAL, "gf_convert: source and destination must be different buffers");
    dst->last_stream = (cudaStream_t)stream;
    cudaError_t e = launch_convert(src->precision, src->R, dst->precision, dst->R, dst->L, U_src, U_dst, dst->last_stream);
    if (e != cudaSuccess) return cuda_fail(dst, e, "gf_convert");
    dst->launches += 1;
    return GF_OK;
}

// Coulomb reading B (gf_set_coulomb_reading): G = 1, the sweeps leave the temporal links alone and accumulate g(x) in
// G, then one pass transforms the temporal links.  Reading A otherwise.
// reading_b_begin: *gfield = the context's g(x) field set to 1, or NULL when this call runs reading A
static int reading_b_begin(gf_ctx* c, int mode, cudaStream_t st, void** gfield, const char* who)
{
    *gfield = nullptr;
    if (!uses_reading_b(c, mode)) return GF_OK;
    cudaError_t e;
    if (c->d_gfield == nullptr && (e = cudaMalloc(&c->d_gfield, (size_t)c->L.Hp * 2 * 18 * real_size(c))) != cudaSuccess) {
        c->d_gfield = nullptr;
        (void)cudaGetLastError();
        if (c->coulomb_b < 0) { // automatic choice and no room for the g(x) field: reading A needs none
            c->coulomb_b = 0;
            return GF_OK;
        }
        return cuda_fail(c, e, "Coulomb reading B: allocation of the g(x) field");
    }
    if ((e = launch_coulomb_init(c->precision, c->L, c->d_gfield, st)) != cudaSuccess) return cuda_fail(c, e, who);
    c->launches += 1;
    *gfield = c->d_gfield;
    return GF_OK;
}

static int reading_b_end(gf_ctx* c, void* U, void* gfield, cudaStream_t st, const char* who)
{
    if (gfield == nullptr) return GF_OK;
    cudaError_t e = launch_coulomb_finish(c->precision, c->R, c->L, U, gfield, st);
    if (e != cudaSuccess) return cuda_fail(c, e, who);
    c->launches += 1;
    return GF_OK;
}

// One chunk of sweeps with the Coulomb reading-B bracket around it.  If a launch fails after sweeps have been
// enqueued, the temporal links are still transformed with the g(x) accumulated so far (reading_b_end), so that the
// field stays a gauge transform of the input; the first error is the one reported.
static int run_sweeps(gf_ctx* c, void* U, int mode, int variant, double param, int nsweeps, int sweep0,
                      unsigned long long seed, cudaStream_t st, const char* who, const unsigned char* active = nullptr)
{
    if (nsweeps == 0) return GF_OK;
    void* gfield;
    int rc = reading_b_begin(c, mode, st, &gfield, who);
    if (rc != GF_OK) return rc;
    int launched = 0;
    rc = run_sweeps_core(c, U, mode, variant, param, nsweeps, sweep0, seed, st, who, active, gfield, &launched);
    if (rc == GF_OK || launched > 0) {
        char first[512];
        if (rc != GF_OK) memcpy(first, c->err, sizeof first);
        const int rc2 = reading_b_end(c, U, gfield, st, who);
        if (rc != GF_OK) memcpy(c->err, first, sizeof first);
        else rc = rc2;
    }
    return rc;
}

// argument check and dispatch of one member of the relaxation family (gf_relax, and the chunks of gf_fix)
static int relax_chunk(gf_ctx* c, void* U, int update, double param, int nsweeps, int sweep0, unsigned long long seed,
                       cudaStream_t st, const char* who, const unsigned char* active = nullptr)
{
    if (U == nullptr) return fail(c, GF_EINVAL, "%s: U is NULL", who);
    if (nsweeps < 0) return fail(c, GF_EINVAL, "%s: nsweeps = %d < 0", who, nsweeps);
    switch (update) {
    case GF_UPDATE_OVERRELAX2:
        if (!(param >= 1.0 && param < 2.0)) return fail(c, GF_EINVAL, "%s: omega = %g outside [1,2) (PAPER.md:63)", who, param);
        return run_sweeps(c, U, MODE_OVERRELAX, 0, param, nsweeps, sweep0, 0ull, st, who, active);
    case GF_UPDATE_OVERRELAX1:
        if (!(param >= 1.0 && param < 2.0)) return fail(c, GF_EINVAL, "%s: omega = %g outside [1,2) (PAPER.md:63)", who, param);
        return run_sweeps(c, U, MODE_VARIANT, VARIANT_OVERRELAX1, param, nsweeps, sweep0, seed, st, who, active);
    case GF_UPDATE_STOCHASTIC:
        if (!(param >= 0.0 && param <= 1.0)) return fail(c, GF_EINVAL, "%s: probability p = %g outside [0,1]", who, param);
        return run_sweeps(c, U, MODE_VARIANT, VARIANT_STOCHASTIC, param, nsweeps, sweep0, seed, st, who, active);
    default:
        return fail(c, GF_EINVAL, "%s: unknown update %d", who, update);
    }
}

extern "C" int gf_overrelax(gf_ctx* c, void* U, double omega, int nsweeps, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    int rc = begin_call(c, (cudaStream_t)stream);
    if (rc != GF_OK) return rc;
    return relax_chunk(c, U, GF_UPDATE_OVERRELAX2, omega, nsweeps, 0, 0ull, (cudaStream_t)stream, "gf_overrelax");
}

extern "C" int gf_relax(gf_ctx* c, void* U, int update, double param, int nsweeps, unsigned long long seed, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    int rc = begin_call(c, (cudaStream_t)stream);
    if (rc != GF_OK) return rc;
    return relax_chunk(c, U, update, param, nsweeps, 0, seed, (cudaStream_t)stream, "gf_relax");
}

extern "C" int gf_anneal_micro(gf_ctx* c, void* U, double T_start, double T_end, int nsteps, int n_micro,
                               unsigned long long seed, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    if (U == nullptr) return fail(c, GF_EINVAL, "gf_anneal: U is NULL");
    if (!(T_start > 0.0) || !(T_end > 0.0)) return fail(c, GF_EINVAL, "gf_anneal: temperatures must be > 0 (got %g, %g)", T_start, T_end);
    if (nsteps < 0) return fail(c, GF_EINVAL, "gf_anneal: nsteps = %d < 0", nsteps);
    if (n_micro < 0) return fail(c, GF_EINVAL, "gf_anneal_micro: n_micro = %d < 0", n_micro);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = begin_call(c, st);
    if (rc != GF_OK) return rc;
    SweepParams p = base_params(c, U);
    p.key0 = (uint32_t)seed;
    p.key1 = (uint32_t)(seed >> 32);
    if (nsteps == 0) return GF_OK;
    void* gfield; // Coulomb reading B: one g(x) field over the whole call, heatbath and microcanonical sweeps alike
    rc = reading_b_begin(c, MODE_HEATBATH, st, &gfield, "gf_anneal");
    if (rc != GF_OK) return rc;
    p.G = gfield;
    int launched = 0;
    for (int step = 0; step < nsteps && rc == GF_OK; ++step) {
        // T_i = T_start + (T_end - T_start) i / (nsteps - 1)   (C13)
        p.ph.T = nsteps > 1 ? T_start + (T_end - T_start) * (double)step / (double)(nsteps - 1) : T_start;
        p.ph.step = (uint32_t)step;
        p.trials = (step == nsteps - 1) ? c->d_trials : nullptr;
        const bool reunit = reunit_due(c, true);
        for (int parity = 0; parity < 2 && rc == GF_OK; ++parity) {
            set_phase(c, p, parity, reunit);
            cudaError_t e = launch_sweep(c, MODE_HEATBATH, p, st);
            if (e != cudaSuccess) { rc = cuda_fail(c, e, "gf_anneal: kernel launch"); break; }
            c->half_sweeps += 1;
            c->launches += 1;
            launched += 1;
        }
        if (rc != GF_OK) break;
        c->call_sweeps += 1;
        // microcanonical sweeps g -> g^2 (C19): stochastic relaxation with p = 2 > u, i.e. always
        if (n_micro > 0) {
            // the field between heatbath sweeps is rough by construction and the heatbath kernel keeps no roughness flags:
            // fp32 contexts run the site chain of these sweeps in double (hybrid chain forced)
            c->force_rough = 1;
            rc = run_sweeps_core(c, U, MODE_VARIANT, VARIANT_STOCHASTIC, 2.0, n_micro, 0, seed, st,
                                 "gf_anneal_micro: kernel launch", nullptr, gfield, &launched);
            c->force_rough = 0;
        }
    }
    // after a failed launch the temporal links are still transformed with the g(x) accumulated so far (reading B)
    if (rc == GF_OK || launched > 0) {
        char first[512];
        if (rc != GF_OK) memcpy(first, c->err, sizeof first);
        const int rc2 = reading_b_end(c, U, gfield, st, "gf_anneal");
        if (rc != GF_OK) memcpy(c->err, first, sizeof first);
        else rc = rc2;
    }
    return rc;
}

extern "C" int gf_anneal(gf_ctx* c, void* U, double T_start, double T_end, int nsteps, unsigned long long seed, void* stream)
{
    return gf_anneal_micro(c, U, T_start, T_end, nsteps, 0, seed, stream);
}

// ---------------------------------------------------------------------------------------------------------
// single half-sweeps and t-slab faces: what a driver needs to run one configuration sharded in t over several
// contexts (paper_1209_4008_b200/slab.py).  A slab context owns the timeslices
// [t_begin, t_end) and keeps, as one more slice behind them, a ghost copy of the temporal links of slice t_begin - 1:
// the only links a site of the slab shares with another slab (U_t(x - t) of its first slice).  Per half-sweep of
// parity p the ghost is refreshed from the neighbour's last slice (parity block 1 - p: the links whose upper end is
// active), the half-sweep updates it in place, and it is written back.
// ---------------------------------------------------------------------------------------------------------
extern "C" size_t gf_slab_face_bytes(const gf_ctx* c)
{
    if (c == nullptr) return 0;
    return (size_t)c->Hs * (size_t)c->R * real_size(c);
}

static int face_impl(gf_ctx* c, void* U, int which, int block_parity, void* buf, bool pack, cudaStream_t st, const char* who)
{
    if (c == nullptr) return GF_EINVAL;
    if (!c->slab) return fail(c, GF_EINVAL, "%s: not a slab context (gf_create_slab)", who);
    if (U == nullptr || buf == nullptr) return fail(c, GF_EINVAL, "%s: NULL pointer", who);
    if ((which != 0 && which != 1) || (block_parity != 0 && block_parity != 1)) return fail(c, GF_EINVAL, "%s: which and block_parity must be 0 or 1", who);
    c->last_stream = st;
    const int t = which == 0 ? c->Nt - 1 : c->Nt; // last owned slice / ghost slice
    cudaError_t e = launch_face(c->precision, c->R, c->L, c->Hs, t, block_parity, pack, U, buf, st);
    if (e != cudaSuccess) return cuda_fail(c, e, who);
    c->launches += 1;
    return GF_OK;
}

extern "C" int gf_slab_pack_face(gf_ctx* c, const void* U, int which, int block_parity, void* buf_dev, void* stream)
{
    return face_impl(c, const_cast<void*>(U), which, block_parity, buf_dev, true, (cudaStream_t)stream, "gf_slab_pack_face");
}

extern "C" int gf_slab_unpack_face(gf_ctx* c, void* U, int which, int block_parity, const void* buf_dev, void* stream)
{
    return face_impl(c, U, which, block_parity, const_cast<void*>(buf_dev), false, (cudaStream_t)stream, "gf_slab_unpack_face");
}

// one half-sweep on the owned timeslices [t_first, t_first + t_count)
static int half_impl(gf_ctx* c, void* U, int mode, int variant, double param, double T, int parity, int sweep,
                     unsigned long long seed, int t_first, int t_count, cudaStream_t st, const char* who)
{
    if (U == nullptr) return fail(c, GF_EINVAL, "%s: U is NULL", who);
    if (parity != 0 && parity != 1) return fail(c, GF_EINVAL, "%s: parity must be 0 (RED) or 1 (BLACK)", who);
    if (sweep < 0) return fail(c, GF_EINVAL, "%s: sweep = %d < 0", who, sweep);
    if (t_first < 0 || t_count < 0 || t_first + t_count > c->Nt) return fail(c, GF_EINVAL, "%s: timeslices [%d, %d) outside [0, %d)", who, t_first, t_first + t_count, c->Nt);
    if (uses_reading_b(c, mode)) return fail(c, GF_EINVAL, "%s: single half-sweeps run Coulomb reading A (gf_set_coulomb_reading(ctx, 0))", who);
    c->last_stream = st;
    if (t_count == 0) return GF_OK;
    SweepParams p = base_params(c, U);
    p.omega = param;
    p.variant = variant;
    p.key0 = (uint32_t)seed;
    p.key1 = (uint32_t)(seed >> 32);
    c->call_sweeps = (unsigned long long)sweep;
    const bool hot = mode == MODE_HEATBATH || (mode == MODE_VARIANT && variant == VARIANT_STOCHASTIC);
    set_phase(c, p, parity, reunit_due(c, hot));
    p.ph.step = (uint32_t)sweep;
    p.ph.T = T;
    p.trials = c->d_trials;
    p.h_begin = (unsigned)t_first * c->Hs;
    p.h_count = (unsigned)t_count * c->Hs;
    cudaError_t e = launch_sweep(c, mode, p, st);
    if (e != cudaSuccess) return cuda_fail(c, e, who);
    c->launches += 1;
    c->half_sweeps += 1;
    return GF_OK;
}

extern "C" int gf_begin_sweeps(gf_ctx* c, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    return begin_call(c, (cudaStream_t)stream);
}

extern "C" int gf_relax_half(gf_ctx* c, void* U, int update, double param, int parity, int sweep, unsigned long long seed,
                             int t_first, int t_count, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    int mode, variant;
    if (update_to_mode(update, &mode, &variant) != GF_OK) return fail(c, GF_EINVAL, "gf_relax_half: unknown update %d", update);
    if (update == GF_UPDATE_STOCHASTIC ? !(param >= 0.0 && param <= 1.0) : !(param >= 1.0 && param < 2.0))
        return fail(c, GF_EINVAL, "gf_relax_half: parameter %g out of range for update %d", param, update);
    return half_impl(c, U, mode, variant, param, 1.0, parity, sweep, seed, t_first, t_count, (cudaStream_t)stream, "gf_relax_half");
}

extern "C" int gf_anneal_half(gf_ctx* c, void* U, double T, int parity, int step, unsigned long long seed, int t_first,
                              int t_count, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    if (!(T > 0.0)) return fail(c, GF_EINVAL, "gf_anneal_half: temperature must be > 0 (got %g)", T);
    return half_impl(c, U, MODE_HEATBATH, 0, 1.0, T, parity, step, seed, t_first, t_count, (cudaStream_t)stream, "gf_anneal_half");
}

// runs one reduction on last_stream and brings the Nt+2 results to h_out
static int reduce_to_host(gf_ctx* c, const void* U, bool theta, const char* who)
{
    if (U == nullptr) return fail(c, GF_EINVAL, "%s: U is NULL", who);
    const int nd = c->gauge == GF_COULOMB ? 3 : 4;
    cudaStream_t st = c->last_stream;
    cudaError_t e = theta ? launch_theta(c->precision, c->R, c->L, c->Nt, nd, U, c->d_partials, c->d_out, st)
                          : launch_functional(c->precision, c->R, c->L, c->Nt, nd, U, c->d_partials, c->d_out, st);
    if (e != cudaSuccess) return cuda_fail(c, e, who);
    c->launches += 2;
    e = cudaMemcpyAsync(c->h_out, c->d_out, (size_t)(c->Nt + 2) * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(c, e, who);
    return GF_OK;
}

extern "C" int gf_functional(gf_ctx* c, const void* U, double* F_host)
{
    if (c == nullptr) return GF_EINVAL;
    if (F_host == nullptr) return fail(c, GF_EINVAL, "gf_functional: F_host is NULL");
    int rc = reduce_to_host(c, U, false, "gf_functional");
    if (rc != GF_OK) return rc;
    *F_host = c->h_out[0];
    return GF_OK;
}

extern "C" int gf_theta(gf_ctx* c, const void* U, double* theta_host)
{
    if (c == nullptr) return GF_EINVAL;
    if (theta_host == nullptr) return fail(c, GF_EINVAL, "gf_theta: theta_host is NULL");
    int rc = reduce_to_host(c, U, true, "gf_theta");
    if (rc != GF_OK) return rc;
    *theta_host = c->gauge == GF_COULOMB ? c->h_out[1] : c->h_out[0];
    return GF_OK;
}

extern "C" int gf_raw_sums(gf_ctx* c, const void* U, double* F_raw_host, double* theta_raw_host)
{
    if (c == nullptr) return GF_EINVAL;
    const double V = 2.0 * (double)c->H_own, nd = c->gauge == GF_COULOMB ? 3.0 : 4.0;
    int rc;
    if (F_raw_host) {
        if ((rc = reduce_to_host(c, U, false, "gf_raw_sums")) != GF_OK) return rc;
        *F_raw_host = c->h_out[0] * (3.0 * nd * V);
    }
    if (theta_raw_host) {
        if ((rc = reduce_to_host(c, U, true, "gf_raw_sums")) != GF_OK) return rc;
        *theta_raw_host = c->h_out[0] * (3.0 * V);
    }
    return GF_OK;
}

extern "C" int gf_theta_slices(gf_ctx* c, const void* U, double* theta_host_Nt)
{
    if (c == nullptr) return GF_EINVAL;
    if (theta_host_Nt == nullptr) return fail(c, GF_EINVAL, "gf_theta_slices: output is NULL");
    int rc = reduce_to_host(c, U, true, "gf_theta_slices");
    if (rc != GF_OK) return rc;
    memcpy(theta_host_Nt, c->h_out + 2, (size_t)c->Nt * sizeof(double));
    return GF_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Alg. 1 with its stop rule, monitored from inside the sweeps (SweepMonitor, gf_sweep.cuh): theta(S_n) and F(S_n) of
// the state after sweep n are complete when the BLACK half-sweep of sweep n+1 has run, so the loop stops one sweep
// after the sweep that met the tolerance (oracle: orc_fix / orc_fix_slices with lag = 1), and no launch waits for the
// host: sweeps are enqueued in batches, the device state is copied out behind each batch, and the host reads the copy
// of the batch before the one just enqueued.  Launches past the stop return at once.
// ---------------------------------------------------------------------------------------------------------
static int update_to_mode(int update, int* mode, int* variant)
{
    *variant = 0;
    switch (update) {
    case GF_UPDATE_OVERRELAX2: *mode = MODE_OVERRELAX; return GF_OK;
    case GF_UPDATE_OVERRELAX1: *mode = MODE_VARIANT; *variant = VARIANT_OVERRELAX1; return GF_OK;
    case GF_UPDATE_STOCHASTIC: *mode = MODE_VARIANT; *variant = VARIANT_STOCHASTIC; return GF_OK;
    default: return GF_EINVAL;
    }
}

// can this context run the fused monitor with the current launch shape?  every block must lie inside one timeslice;
// fp32 contexts form theta from the fp32 K of the sweep, which resolves it down to ~1e-12 only
// and it pays while checks are frequent: a monitored sweep costs ~4 % more than a plain one and a checked one ~20 %
// (32^4 fp32: 185 / 214 against 178 us), the separate check ~110 us per check -- break-even near one check per 10 sweeps
static bool monitor_applies(const gf_ctx* c, int mode, double tol, int check_every)
{
    if (!c->monitor || c->slab) return false; // slabs: the driver owns the loop (exchange + all-reduce per check)
    if (c->monitor == 1 && check_every > 10) return false;
    const unsigned Hs = c->Hs;
    const unsigned tps = (unsigned)auto_tps(c, mode), block = (unsigned)auto_block(c);
    if ((Hs * tps) % block != 0) return false;
    if (c->precision == GF_FP32 && tol < 1e-10) return false;
    return true;
}

static int monitor_alloc(gf_ctx* c, int blocks, int groups)
{
    const size_t Nt = (size_t)c->Nt;
    const size_t prefix = ((sizeof(MonitorState) + 2 * Nt * sizeof(double) + Nt * sizeof(int) + 63) / 64) * 64;
    const size_t bytes = prefix + 3 * Nt * (size_t)groups * sizeof(double) + 5 * (size_t)blocks * sizeof(double);
    cudaError_t e;
    if (c->d_mon != nullptr && (bytes > c->mon_bytes || blocks != c->mon_blocks || groups != c->mon_groups)) {
        cudaFree(c->d_mon);
        c->d_mon = nullptr;
    }
    if (c->d_mon == nullptr) {
        if ((e = cudaMalloc(&c->d_mon, bytes)) != cudaSuccess) { c->d_mon = nullptr; return cuda_fail(c, e, "monitor: allocation"); }
        c->mon_bytes = bytes; c->mon_blocks = blocks; c->mon_groups = groups; c->mon_prefix = prefix;
    }
    if (c->h_mon == nullptr) {
        if ((e = cudaMallocHost(&c->h_mon, 2 * prefix)) != cudaSuccess) { c->h_mon = nullptr; return cuda_fail(c, e, "monitor: pinned allocation"); }
        for (int i = 0; i < 2; ++i)
            if ((e = cudaEventCreateWithFlags(&c->mon_event[i], cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(c, e, "monitor: event");
    }
    return GF_OK;
}

static int fix_fused(gf_ctx* c, void* U, int update, double param, double tol, int check_every, int max_sweeps,
                     unsigned long long seed, cudaStream_t st, bool slices, int* sweeps_done, int* per_slice,
                     double* theta_host, double* F_host, const char* who)
{
    int mode, variant;
    if (update_to_mode(update, &mode, &variant) != GF_OK) return fail(c, GF_EINVAL, "%s: unknown update %d", who, update);
    const int Nt = c->Nt;
    const unsigned Hs = c->Hs;
    const int tps = auto_tps(c, mode), block = auto_block(c);
    const int bps = (int)(Hs * (unsigned)tps / (unsigned)block), blocks = bps * Nt;
    const int groups = bps < 8 ? bps : 8;
    int rc = monitor_alloc(c, blocks, groups);
    if (rc != GF_OK) return rc;
    // the check before the first sweep: the separate reduction (the BLACK sites of S_0 have no sweep behind them)
    if ((rc = reduce_to_host(c, U, true, who)) != GF_OK) return rc;
    const bool coulomb = c->gauge == GF_COULOMB;
    char* h0 = c->h_mon;
    memset(h0, 0, c->mon_prefix);
    MonitorState* hs = reinterpret_cast<MonitorState*>(h0);
    double* h_theta_t = reinterpret_cast<double*>(h0 + sizeof(MonitorState));
    int* h_from = reinterpret_cast<int*>(h0 + sizeof(MonitorState) + 2 * (size_t)Nt * sizeof(double));
    int active = 0;
    for (int t = 0; t < Nt; ++t) {
        h_theta_t[t] = c->h_out[2 + t];
        const bool fr = slices && c->h_out[2 + t] < tol;
        h_from[t] = fr ? 1 : INT_MAX;
        active += fr ? 0 : 1;
    }
    hs->theta = coulomb ? c->h_out[1] : c->h_out[0];
    hs->any_active = active;
    hs->stop_sweep = -1;
    hs->stop_from = INT_MAX;
    if (slices && active > 0 && active < Nt) {
        // slices frozen before the first sweep: no sweep will ever deliver their share of F (the duty keeps a frozen
        // slice's last values), so it is seeded here from the separate reduction
        if ((rc = reduce_to_host(c, U, false, who)) != GF_OK) return rc;
        const double raw = 3.0 * (coulomb ? 3.0 : 4.0) * 2.0 * (double)c->Hs; // undoes the per-slice normalisation
        for (int t = 0; t < Nt; ++t)
            if (h_from[t] != INT_MAX) h_theta_t[Nt + t] = c->h_out[2 + t] * raw;
    }
    const bool fixed_already = slices ? active == 0 : hs->theta < tol;
    int done = 0;
    if (!fixed_already && max_sweeps > 0) {
        cudaError_t e = cudaMemcpyAsync(c->d_mon, h0, c->mon_prefix, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(c, e, who);
        void* gfield;
        if ((rc = reading_b_begin(c, mode, st, &gfield, who)) != GF_OK) return rc;
        SweepParams p = base_params(c, U);
        p.G = gfield;
        p.omega = param;
        p.variant = variant;
        p.key0 = (uint32_t)seed;
        p.key1 = (uint32_t)(seed >> 32);
        char* d = c->d_mon;
        SweepMonitor m;
        memset(&m, 0, sizeof m);
        m.state = reinterpret_cast<MonitorState*>(d);
        m.theta_t = reinterpret_cast<double*>(d + sizeof(MonitorState));
        m.frozen_from = reinterpret_cast<int*>(d + sizeof(MonitorState) + 2 * (size_t)Nt * sizeof(double));
        m.group = reinterpret_cast<double*>(d + c->mon_prefix);
        double* part = m.group + 3 * (size_t)Nt * groups; // planes: F[0], F[1], post[0], post[1], pre
        m.groups = groups;
        m.blocks_per_slice = bps;
        m.slices = slices ? 1 : 0;
        m.coulomb = coulomb ? 1 : 0;
        m.tol = tol;
        const double V = 2.0 * (double)c->H_own, nd = coulomb ? 3.0 : 4.0;
        m.scale_theta_t = 1.0 / (3.0 * V / Nt);
        m.scale_theta = 1.0 / (3.0 * V);
        m.scale_F = 1.0 / (3.0 * nd * V);
        const int batch_sweeps = 32;
        int enq = 0, batch = 0, launched = 0;
        bool stopped = false;
        while (rc == GF_OK && enq < max_sweeps && !stopped) {
            const int nb = batch_sweeps < max_sweeps - enq ? batch_sweeps : max_sweeps - enq;
            for (int i = enq + 1; i <= enq + nb && rc == GF_OK; ++i) { // sweep i (1-based)
                const bool prev_check = i - 1 >= 1 && (i - 1) % check_every == 0; // theta(S_{i-1}) is being completed
                const bool this_check = i % check_every == 0 && i < max_sweeps;   // theta(S_i) needs RED_{i+1}
                const bool reunit = reunit_due(c, mode == MODE_VARIANT && variant == VARIANT_STOCHASTIC);
                p.ph.step = (uint32_t)(i - 1);
                for (int parity = 0; parity < 2 && rc == GF_OK; ++parity) { // RED, BLACK
                    set_phase(c, p, parity, reunit);
                    p.mon = m;
                    p.mon.sweep = i;
                    if (parity == 0) {
                        p.mon.pre_part = prev_check ? part + 4 * (size_t)blocks : nullptr;
                    } else {
                        if (this_check) {
                            p.mon.F_part = part + (size_t)(i & 1) * blocks;
                            p.mon.post_part = part + (size_t)(2 + (i & 1)) * blocks;
                        }
                        if (prev_check) {
                            p.mon.red_F = part + (size_t)((i - 1) & 1) * blocks;
                            p.mon.red_post = part + (size_t)(2 + ((i - 1) & 1)) * blocks;
                            p.mon.red_pre = part + 4 * (size_t)blocks;
                            p.mon.check_sweep = i - 1;
                        }
                    }
                    e = launch_sweep(c, mode, p, st);
                    if (e != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
                    c->launches += 1;
                    c->half_sweeps += 1;
                    launched += 1;
                }
                c->call_sweeps += 1;
            }
            if (rc != GF_OK) break;
            enq += nb;
            // the device state behind this batch, into the pinned copy of this batch; read the copy of the batch before
            char* hb = c->h_mon + (size_t)(batch & 1) * c->mon_prefix;
            if ((e = cudaMemcpyAsync(hb, c->d_mon, c->mon_prefix, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
                (e = cudaEventRecord(c->mon_event[batch & 1], st)) != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
            if (batch >= 1) {
                if ((e = cudaEventSynchronize(c->mon_event[(batch - 1) & 1])) != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
                stopped = reinterpret_cast<const MonitorState*>(c->h_mon + (size_t)((batch - 1) & 1) * c->mon_prefix)->stop_from != INT_MAX;
            }
            ++batch;
        }
        // after a failed launch the temporal links are still transformed with the g(x) accumulated so far (reading B)
        if (rc == GF_OK || launched > 0) {
            char first[512];
            if (rc != GF_OK) memcpy(first, c->err, sizeof first);
            const int rc2 = reading_b_end(c, U, gfield, st, who);
            if (rc != GF_OK) memcpy(c->err, first, sizeof first);
            else rc = rc2;
        }
        if (rc != GF_OK) return rc;
        if ((e = cudaMemcpyAsync(h0, c->d_mon, c->mon_prefix, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(c, e, who);
        done = hs->stop_from != INT_MAX && hs->stop_from - 1 < enq ? hs->stop_from - 1 : enq;
    }
    if (sweeps_done) *sweeps_done = done;
    if (per_slice)
        for (int t = 0; t < Nt; ++t) per_slice[t] = h_from[t] - 1 < done ? h_from[t] - 1 : done;
    // theta and F of the field as it is returned: the separate reductions, once
    if (theta_host) {
        if ((rc = reduce_to_host(c, U, true, who)) != GF_OK) return rc;
        *theta_host = coulomb ? c->h_out[1] : c->h_out[0];
    }
    if (F_host) return gf_functional(c, U, F_host);
    return GF_OK;
}

// The stop rule of gf_fix / gf_fix_slices is a setting of the context and of nothing else: gf_set_monitor(ctx, 0) is the
// paper's loop (lag 0), any other setting (the default included) the loop of C21 (lag 1), whichever kernels run it.
static int fix_lag(const gf_ctx* c) { return c->monitor ? 1 : 0; }

extern "C" int gf_fix_last_form(const gf_ctx* c, int* lag, int* fused)
{
    if (c == nullptr) return GF_EINVAL;
    if (lag) *lag = c->fix_lag;
    if (fused) *fused = c->fix_fused;
    return GF_OK;
}

// gf_fix_slices with the stop rule of the fused monitor (orc_fix_slices_lag, lag = 1) run with the separate check: a
// slice found below the tolerance at the check after sweep n gets one more sweep and is frozen from sweep n + 2; no
// check at max_sweeps.
static int fix_slices_lag1(gf_ctx* c, void* U, int mode, int variant, double param, double tol, int check_every,
                           int max_sweeps, unsigned long long seed, cudaStream_t st, int* sweeps_done, int* per_slice,
                           double* theta_host, double* F_host)
{
    const char* who = "gf_fix_slices";
    const int Nt = c->Nt;
    unsigned char* mask = new (std::nothrow) unsigned char[Nt];
    int* count = new (std::nothrow) int[Nt];
    int* last = new (std::nothrow) int[Nt]; // last sweep (1-based) that updates the slice; -1: still open
    if (mask == nullptr || count == nullptr || last == nullptr) {
        delete[] mask; delete[] count; delete[] last;
        return fail(c, GF_ENOMEM, "%s: host allocation", who);
    }
    int done = 0, any = 0;
    int rc = reduce_to_host(c, U, true, who);
    for (int t = 0; t < Nt && rc == GF_OK; ++t) { count[t] = 0; last[t] = c->h_out[2 + t] >= tol ? -1 : 0; any |= last[t] < 0; }
    while (rc == GF_OK && any && done < max_sweeps) {
        bool pending = false; // a slice in its one sweep after the check that froze it
        for (int t = 0; t < Nt; ++t) pending = pending || last[t] > done;
        const int next_check = (done / check_every + 1) * check_every;
        const int target = pending ? done + 1 : (next_check < max_sweeps ? next_check : max_sweeps);
        for (int t = 0; t < Nt; ++t) {
            mask[t] = last[t] < 0 || last[t] > done;
            if (mask[t]) count[t] += target - done;
        }
        rc = run_sweeps(c, U, mode, variant, param, target - done, done, seed, st, "gf_fix_slices: kernel launch", mask);
        done = target;
        if (rc == GF_OK && done % check_every == 0 && done < max_sweeps) {
            rc = reduce_to_host(c, U, true, who);
            for (int t = 0; t < Nt && rc == GF_OK; ++t)
                if (last[t] < 0 && c->h_out[2 + t] < tol) last[t] = done + 1;
        }
        any = 0;
        for (int t = 0; t < Nt; ++t) any |= last[t] < 0 || last[t] > done;
    }
    if (rc == GF_OK) rc = reduce_to_host(c, U, true, who); // theta of the field as returned
    if (rc == GF_OK) {
        if (sweeps_done) *sweeps_done = done;
        if (per_slice) memcpy(per_slice, count, sizeof(int) * (size_t)Nt);
        if (theta_host) *theta_host = c->h_out[1];
        if (F_host) rc = gf_functional(c, U, F_host);
    }
    delete[] mask; delete[] count; delete[] last;
    return rc;
}

extern "C" int gf_fix(gf_ctx* c, void* U, int update, double param, double theta_tol, int check_every, int max_sweeps,
                      unsigned long long seed, int* sweeps_done, double* theta_host, double* F_host, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    if (U == nullptr) return fail(c, GF_EINVAL, "gf_fix: U is NULL");
    if (check_every < 1) return fail(c, GF_EINVAL, "gf_fix: check_every = %d < 1", check_every);
    if (max_sweeps < 0) return fail(c, GF_EINVAL, "gf_fix: max_sweeps = %d < 0", max_sweeps);
    if (!(theta_tol >= 0.0)) return fail(c, GF_EINVAL, "gf_fix: theta_tol = %g < 0", theta_tol);
    int done = 0;
    double th = 0.0;
    int rc = begin_call(c, (cudaStream_t)stream);
    if (rc == GF_OK) rc = relax_chunk(c, U, update, param, 0, 0, seed, (cudaStream_t)stream, "gf_fix"); // argument check
    if (rc != GF_OK) return rc;
    {
        int mode, variant;
        update_to_mode(update, &mode, &variant);
        if (monitor_applies(c, mode, theta_tol, check_every)) {
            c->fix_fused = 1;
            c->fix_lag = 1;
            return fix_fused(c, U, update, param, theta_tol, check_every, max_sweeps, seed, (cudaStream_t)stream, false,
                             sweeps_done, nullptr, theta_host, F_host, "gf_fix");
        }
    }
    c->fix_fused = 0;
    c->fix_lag = fix_lag(c);
    rc = gf_theta(c, U, &th);
    if (c->fix_lag == 1) {
        // the stop rule of the fused monitor (C21, orc_fix_lag with lag = 1) run with the separate check, where the fused
        // kernels cannot or would not pay: one more sweep after the check that met the tolerance, no check at max_sweeps.
        // The rule is the context's setting; the launch shape, the precision and the tolerance only pick the kernels.
        int stop_at = -1;
        bool current = true; // th belongs to the field as it is now
        while (rc == GF_OK && th >= theta_tol && done < max_sweeps && done != stop_at) {
            const int next_check = (done / check_every + 1) * check_every;
            const int target = next_check < max_sweeps ? next_check : max_sweeps;
            rc = relax_chunk(c, U, update, param, target - done, done, seed, (cudaStream_t)stream, "gf_fix");
            done = target;
            current = false;
            if (rc == GF_OK && done % check_every == 0 && done < max_sweeps) {
                double th_check = 0.0;
                rc = gf_theta(c, U, &th_check);
                if (rc == GF_OK && th_check < theta_tol) {
                    rc = relax_chunk(c, U, update, param, 1, done, seed, (cudaStream_t)stream, "gf_fix");
                    stop_at = ++done;
                } else if (rc == GF_OK) {
                    th = th_check;
                    current = true;
                }
            }
        }
        if (rc == GF_OK && !current) rc = gf_theta(c, U, &th);
        if (rc != GF_OK) return rc;
        if (sweeps_done) *sweeps_done = done;
        if (theta_host) *theta_host = th;
        if (F_host) return gf_functional(c, U, F_host);
        return GF_OK;
    }
    // Alg. 1: "while precision theta not reached", checked every check_every-th sweep
    while (rc == GF_OK && th >= theta_tol && done < max_sweeps) {
        const int n = check_every < max_sweeps - done ? check_every : max_sweeps - done;
        rc = relax_chunk(c, U, update, param, n, done, seed, (cudaStream_t)stream, "gf_fix");
        done += n;
        if (rc == GF_OK) rc = gf_theta(c, U, &th);
    }
    if (rc != GF_OK) return rc;
    if (sweeps_done) *sweeps_done = done;
    if (theta_host) *theta_host = th;
    if (F_host) return gf_functional(c, U, F_host);
    return GF_OK;
}

extern "C" int gf_fix_slices(gf_ctx* c, void* U, int update, double param, double theta_tol, int check_every,
                             int max_sweeps, unsigned long long seed, int* sweeps_done, int* sweeps_per_slice,
                             double* theta_host, double* F_host, void* stream)
{
    if (c == nullptr) return GF_EINVAL;
    if (c->gauge != GF_COULOMB) return fail(c, GF_EINVAL, "gf_fix_slices: timeslices decouple in Coulomb gauge only (C12)");
    if (U == nullptr) return fail(c, GF_EINVAL, "gf_fix_slices: U is NULL");
    if (check_every < 1) return fail(c, GF_EINVAL, "gf_fix_slices: check_every = %d < 1", check_every);
    if (max_sweeps < 0) return fail(c, GF_EINVAL, "gf_fix_slices: max_sweeps = %d < 0", max_sweeps);
    if (!(theta_tol >= 0.0)) return fail(c, GF_EINVAL, "gf_fix_slices: theta_tol = %g < 0", theta_tol);
    int mode, variant = 0;
    switch (update) {
    case GF_UPDATE_OVERRELAX2: mode = MODE_OVERRELAX; break;
    case GF_UPDATE_OVERRELAX1: mode = MODE_VARIANT; variant = VARIANT_OVERRELAX1; break;
    case GF_UPDATE_STOCHASTIC: mode = MODE_VARIANT; variant = VARIANT_STOCHASTIC; break;
    default: return fail(c, GF_EINVAL, "gf_fix_slices: unknown update %d", update);
    }
    if (update == GF_UPDATE_STOCHASTIC ? !(param >= 0.0 && param <= 1.0) : !(param >= 1.0 && param < 2.0))
        return fail(c, GF_EINVAL, "gf_fix_slices: parameter %g out of range for update %d", param, update);
    cudaStream_t st = (cudaStream_t)stream;
    if (begin_call(c, st) != GF_OK) return GF_ECUDA;
    if (monitor_applies(c, mode, theta_tol, check_every)) {
        c->fix_fused = 1;
        c->fix_lag = 1;
        return fix_fused(c, U, update, param, theta_tol, check_every, max_sweeps, seed, st, true, sweeps_done,
                         sweeps_per_slice, theta_host, F_host, "gf_fix_slices");
    }
    c->fix_fused = 0;
    c->fix_lag = fix_lag(c);
    if (c->fix_lag == 1)
        return fix_slices_lag1(c, U, mode, variant, param, theta_tol, check_every, max_sweeps, seed, st, sweeps_done,
                               sweeps_per_slice, theta_host, F_host);
    const int Nt = c->Nt;
    unsigned char* active = new (std::nothrow) unsigned char[Nt];
    int* count = new (std::nothrow) int[Nt];
    if (active == nullptr || count == nullptr) { delete[] active; delete[] count; return fail(c, GF_ENOMEM, "gf_fix_slices: host allocation"); }
    int done = 0, any = 0;
    int rc = reduce_to_host(c, U, true, "gf_fix_slices");
    for (int t = 0; t < Nt && rc == GF_OK; ++t) { count[t] = 0; active[t] = c->h_out[2 + t] >= theta_tol; any |= active[t]; }
    // Alg. 1 with the stop rule per timeslice: a slice below the tolerance at a check is frozen for good
    while (rc == GF_OK && any && done < max_sweeps) {
        const int n = check_every < max_sweeps - done ? check_every : max_sweeps - done;
        rc = run_sweeps(c, U, mode, variant, param, n, done, seed, st, "gf_fix_slices: kernel launch", active);
        done += n;
        if (rc == GF_OK) rc = reduce_to_host(c, U, true, "gf_fix_slices");
        any = 0;
        for (int t = 0; t < Nt && rc == GF_OK; ++t) {
            if (active[t]) count[t] += n;
            active[t] = active[t] && c->h_out[2 + t] >= theta_tol;
            any |= active[t];
        }
    }
    if (rc == GF_OK) {
        if (sweeps_done) *sweeps_done = done;
        if (sweeps_per_slice) memcpy(sweeps_per_slice, count, sizeof(int) * (size_t)Nt);
        if (theta_host) *theta_host = c->h_out[1];
        if (F_host) rc = gf_functional(c, U, F_host);
    }
    delete[] active;
    delete[] count;
    return rc;
}

// host-buffer path, canonical field in host memory as double (elem = 8) or float (elem = 4)
static int overrelax_host_impl(gf_ctx* c, void* U_host, size_t elem, double omega, int nsweeps, double* F_host,
                               double* theta_host, const char* who)
{
    if (c == nullptr) return GF_EINVAL;
    if (c->slab) return fail(c, GF_EINVAL, "%s: not available on a slab context", who);
    if (U_host == nullptr) return fail(c, GF_EINVAL, "%s: U_canon_host is NULL", who);
    const size_t canon_bytes = (size_t)c->H_own * 2 * 72 * sizeof(double); // staging sized for the larger element
    const size_t copy_bytes = (size_t)c->H_own * 2 * 72 * elem;
    cudaError_t e;
    if (c->d_canon == nullptr && (e = cudaMalloc(&c->d_canon, canon_bytes)) != cudaSuccess) { c->d_canon = nullptr; return cuda_fail(c, e, "host path: staging allocation"); }
    if (c->d_native == nullptr && (e = cudaMalloc(&c->d_native, gf_field_bytes(c))) != cudaSuccess) { c->d_native = nullptr; return cuda_fail(c, e, "host path: staging allocation"); }
    cudaStream_t st = c->last_stream;
    if ((e = cudaMemcpyAsync(c->d_canon, U_host, copy_bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(c, e, "host path: H2D copy");
    int rc;
    if (elem == 8) rc = gf_pack(c, c->d_canon, c->d_native, st);
    else {
        e = launch_pack_f32(c->precision, c->R, c->L, c->H_own, (const float*)c->d_canon, c->d_native, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "host path: pack");
        c->launches += 1;
        rc = GF_OK;
    }
    if (rc == GF_OK) rc = gf_overrelax(c, c->d_native, omega, nsweeps, st);
    if (rc != GF_OK) return rc;
    if (elem == 8) rc = gf_unpack(c, c->d_native, c->d_canon, st);
    else {
        e = launch_unpack_f32(c->precision, c->R, c->L, c->H_own, c->d_native, (float*)c->d_canon, st);
        if (e != cudaSuccess) return cuda_fail(c, e, "host path: unpack");
        c->launches += 1;
    }
    if (rc != GF_OK) return rc;
    if ((e = cudaMemcpyAsync(U_host, c->d_canon, copy_bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(c, e, "host path: D2H copy");
    if (F_host != nullptr && (rc = gf_functional(c, c->d_native, F_host)) != GF_OK) return rc;
    if (theta_host != nullptr && (rc = gf_theta(c, c->d_native, theta_host)) != GF_OK) return rc;
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(c, e, "host path: synchronise");
    return GF_OK;
}

extern "C" int gf_overrelax_host(gf_ctx* c, double* U_host, double omega, int nsweeps, double* F_host, double* theta_host)
{
    return overrelax_host_impl(c, U_host, sizeof(double), omega, nsweeps, F_host, theta_host, "gf_overrelax_host");
}

extern "C" int gf_overrelax_host_f32(gf_ctx* c, float* U_host, double omega, int nsweeps, double* F_host, double* theta_host)
{
    return overrelax_host_impl(c, U_host, sizeof(float), omega, nsweeps, F_host, theta_host, "gf_overrelax_host_f32");
}


// ---------------------------------------------------------------------------------------------------------
// Ensembles from host memory (production gauge fixing: many independent configurations).  The single-configuration
// call above is serial -- H2D, pack, sweeps, unpack, D2H on one stream: at 32^4 fp32 11 ms of PCIe beside 18 ms of
// sweeps.  Here configuration i+1 is uploaded and configuration i-1 downloaded while configuration i is swept: three
// staging slots (canonical + native field each), one stream for each direction of the PCIe link (full duplex) and one
// for the kernels, events between them.  One plain cudaMemcpyAsync per copy.
// ---------------------------------------------------------------------------------------------------------
extern "C" int gf_overrelax_host_batch(gf_ctx* c, void* const* U_canon_host, int n, int element_bytes, double omega, int nsweeps,
                                       double* F_host_n, double* theta_host_n)
{
    if (c == nullptr) return GF_EINVAL;
    const char* who = "gf_overrelax_host_batch";
    if (c->slab) return fail(c, GF_EINVAL, "%s: not available on a slab context", who);
    if (n < 0 || (n > 0 && U_canon_host == nullptr)) return fail(c, GF_EINVAL, "%s: n = %d, U_canon_host = %p", who, n, (const void*)U_canon_host);
    if (element_bytes != 4 && element_bytes != 8) return fail(c, GF_EINVAL, "%s: element_bytes must be 4 (float) or 8 (double)", who);
    if (!(omega >= 1.0 && omega < 2.0)) return fail(c, GF_EINVAL, "%s: omega = %g outside [1,2) (PAPER.md:63)", who, omega);
    if (nsweeps < 0) return fail(c, GF_EINVAL, "%s: nsweeps = %d < 0", who, nsweeps);
    for (int i = 0; i < n; ++i)
        if (U_canon_host[i] == nullptr) return fail(c, GF_EINVAL, "%s: configuration %d is NULL", who, i);
    if (n == 0) return GF_OK;
    const size_t copy_bytes = (size_t)c->H_own * 2 * 72 * (size_t)element_bytes;
    const size_t nres = (size_t)(c->Nt + 2);
    cudaError_t e = cudaSuccess;
    // slots, streams, events, pinned results: allocated once, reused by later calls
    for (int i = 0; i < 3 && e == cudaSuccess; ++i) {
        if (c->batch_stream[i] == nullptr) e = cudaStreamCreateWithFlags(&c->batch_stream[i], cudaStreamNonBlocking);
        gf_ctx::BatchSlot& sl = c->slot[i];
        if (e == cudaSuccess && sl.canon != nullptr && c->batch_canon_bytes < copy_bytes) { cudaFree(sl.canon); sl.canon = nullptr; }
        if (e == cudaSuccess && sl.canon == nullptr) e = cudaMalloc(&sl.canon, copy_bytes);
        if (e == cudaSuccess && sl.native == nullptr) e = cudaMalloc(&sl.native, gf_field_bytes(c));
        if (e == cudaSuccess && sl.res == nullptr) e = cudaMalloc(&sl.res, 2 * nres * sizeof(double));
        if (e == cudaSuccess && sl.in == nullptr) e = cudaEventCreateWithFlags(&sl.in, cudaEventDisableTiming);
        if (e == cudaSuccess && sl.comp == nullptr) e = cudaEventCreateWithFlags(&sl.comp, cudaEventDisableTiming);
        if (e == cudaSuccess && sl.out == nullptr) e = cudaEventCreateWithFlags(&sl.out, cudaEventDisableTiming);
    }
    if (e == cudaSuccess && c->batch_canon_bytes < copy_bytes) c->batch_canon_bytes = copy_bytes;
    if (e == cudaSuccess && c->h_batch_doubles < 2 * nres * (size_t)n) {
        if (c->h_batch) cudaFreeHost(c->h_batch);
        c->h_batch = nullptr;
        e = cudaMallocHost(&c->h_batch, 2 * nres * (size_t)n * sizeof(double));
        c->h_batch_doubles = e == cudaSuccess ? 2 * nres * (size_t)n : 0;
    }
    if (e != cudaSuccess) return cuda_fail(c, e, "gf_overrelax_host_batch: staging allocation");
    cudaStream_t s_in = c->batch_stream[0], s_comp = c->batch_stream[1], s_out = c->batch_stream[2];
    const int nd = c->gauge == GF_COULOMB ? 3 : 4;
    int rc = GF_OK;
    for (int i = 0; i < n && rc == GF_OK; ++i) {
        gf_ctx::BatchSlot& sl = c->slot[i % 3];
        // upload: the slot is free once its previous occupant has been downloaded
        if (i >= 3 && (e = cudaStreamWaitEvent(s_in, sl.out, 0)) != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
        if ((e = cudaMemcpyAsync(sl.canon, U_canon_host[i], copy_bytes, cudaMemcpyHostToDevice, s_in)) != cudaSuccess ||
            (e = cudaEventRecord(sl.in, s_in)) != cudaSuccess || (e = cudaStreamWaitEvent(s_comp, sl.in, 0)) != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
        // pack, sweep, reduce, unpack on the compute stream
        if (element_bytes == 8) rc = gf_pack(c, (const double*)sl.canon, sl.native, s_comp);
        else {
            e = launch_pack_f32(c->precision, c->R, c->L, c->H_own, (const float*)sl.canon, sl.native, s_comp);
            if (e != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
            c->launches += 1;
        }
        if (rc == GF_OK) rc = gf_overrelax(c, sl.native, omega, nsweeps, s_comp);
        if (rc != GF_OK) break;
        if ((e = launch_functional(c->precision, c->R, c->L, c->Nt, nd, sl.native, c->d_partials, sl.res, s_comp)) != cudaSuccess ||
            (e = launch_theta(c->precision, c->R, c->L, c->Nt, nd, sl.native, c->d_partials, sl.res + nres, s_comp)) != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
        c->launches += 4;
        if (element_bytes == 8) rc = gf_unpack(c, sl.native, (double*)sl.canon, s_comp);
        else {
            e = launch_unpack_f32(c->precision, c->R, c->L, c->H_own, sl.native, (float*)sl.canon, s_comp);
            if (e != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
            c->launches += 1;
        }
        if (rc != GF_OK) break;
        // download
        if ((e = cudaEventRecord(sl.comp, s_comp)) != cudaSuccess || (e = cudaStreamWaitEvent(s_out, sl.comp, 0)) != cudaSuccess ||
            (e = cudaMemcpyAsync(U_canon_host[i], sl.canon, copy_bytes, cudaMemcpyDeviceToHost, s_out)) != cudaSuccess ||
            (e = cudaMemcpyAsync(c->h_batch + 2 * nres * (size_t)i, sl.res, 2 * nres * sizeof(double), cudaMemcpyDeviceToHost, s_out)) != cudaSuccess ||
            (e = cudaEventRecord(sl.out, s_out)) != cudaSuccess) { rc = cuda_fail(c, e, who); break; }
    }
    // drain all three streams whatever happened: the host buffers must not be in flight when the call returns
    cudaError_t e1 = cudaStreamSynchronize(s_in), e2 = cudaStreamSynchronize(s_comp), e3 = cudaStreamSynchronize(s_out);
    if (rc != GF_OK) return rc;
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) return cuda_fail(c, e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3), who);
    for (int i = 0; i < n; ++i) {
        const double* r = c->h_batch + 2 * nres * (size_t)i;
        if (F_host_n) F_host_n[i] = r[0];
        if (theta_host_n) theta_host_n[i] = c->gauge == GF_COULOMB ? r[nres + 1] : r[nres];
    }
    return GF_OK;
}
