/*
 * include/gf.h -- C ABI of libgf.so: lattice gauge fixing of 3+1-dimensional SU(3) gauge fields by
 * checkerboard (RED/BLACK) overrelaxation, with the F_g / theta reductions and an SU(2)-heatbath
 * simulated-annealing sweep, on one NVIDIA B200 (sm_100a).
 *
 * Method: Schroeck & Vogt, "Gauge fixing using overrelaxation and simulated annealing on GPUs"
 * (arXiv:1209.4008).  Citations "PAPER.md:<line>" refer to the text of that paper; "Cn" are the readings of
 * DESIGN.md ("Readings of the paper") taken where the paper is silent, ambiguous or garbled.
 *
 * Conventions common to all calls
 *   - Every function returning int returns GF_OK (0) or a negative GF_E* code.  Nothing throws across the
 *     ABI.  gf_last_error(ctx) gives the message of the last failing call on ctx (ctx == NULL: of the last
 *     failing gf_create in this thread's process).
 *   - "device" pointers are CUDA device pointers of the current device, owned by the CALLER (e.g. the
 *     data_ptr() of a torch tensor); the library never frees or reallocates them.  "host" pointers are plain
 *     host memory (pinned memory makes the copies faster, it is not required).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the default stream).  Calls that take a stream only
 *     enqueue work on it and return; they do not synchronise.
 *   - Lattice: extents Nx,Ny,Nz,Nt, all even and >= 2 (checkerboard with periodic boundaries, C5);
 *     V = Nx*Ny*Nz*Nt < 2^31; direction mu = 0,1,2,3 <-> x,y,z,t.
 *   - Canonical exchange layout (fp64, host or device): site s = x + Nx*(y + Ny*(z + Nz*t)); the double at
 *       (((s*4 + mu)*3 + row)*3 + col)*2 + {0: re, 1: im}
 *     is that part of (U_mu(x))_{row,col}.  V*4*18 doubles.
 *   - Native layout (device only; what gf_overrelax / gf_anneal / gf_functional / gf_theta work on):
 *     parity-split, component-major structure of arrays with the site index running fastest
 *     (PAPER.md:124), 12 or 18 reals per link, in 128-bit vectors.  Exact definition:
 *     DESIGN.md "Data layout in HBM".  Produced and consumed only through gf_pack / gf_unpack.
 */
#ifndef GF_H_
#define GF_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gf_ctx gf_ctx; /* opaque; owns reduction scratch, launch configuration, staging buffers */

enum { GF_FP32 = 0, GF_FP64 = 1 };      /* precision of the stored links and of the sweep arithmetic */
enum { GF_LANDAU = 0, GF_COULOMB = 1 }; /* gauge condition */
enum { GF_OK = 0, GF_EINVAL = -1, GF_ECUDA = -2, GF_ENOMEM = -3 };

/* ---- life cycle --------------------------------------------------------------------------------------- */

/* Problem statement of the paper: maximise F_g[U] (eq. 2.1) over gauge transformations by
 * Alg. 1 on an Nx*Ny*Nz*Nt lattice, in Landau gauge (all four mu enter K, F, theta) or
 * Coulomb gauge (mu = x,y,z only, every timeslice fixed independently; the temporal links are still
 * transformed, C12).  Allocates only small device scratch.  *out is NULL on failure.
 * GF_EINVAL: odd or < 2 extent, V >= 2^31, unknown precision / gauge.  GF_ECUDA: no usable device. */
int gf_create(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int precision, int gauge);
void gf_destroy(gf_ctx* ctx);
const char* gf_last_error(const gf_ctx* ctx);

/* Reals stored per link: 18 (default) or 12 (rows 0 and 1 stored, row 2 = conj(row0 x row1) rebuilt on
 * load, C16).  Must be called before the first gf_pack.  GF_EINVAL otherwise. */
int gf_set_storage(gf_ctx* ctx, int reals_per_link);

/* Bytes the caller must allocate (device, 256-byte aligned) for one field in the native layout:
 * 4 * V * reals_per_link * sizeof(real). */
size_t gf_field_bytes(const gf_ctx* ctx);

/* ---- layout conversion (device -> device) --------------------------------------------------------------- */

/* canonical fp64 (device) -> native (device).  fp32: rounds each real to nearest.  R12: drops row 2. */
int gf_pack(gf_ctx* ctx, const double* U_canon_dev, void* U_native_dev, void* stream);
/* native (device) -> canonical fp64 (device).  R12: row 2 is rebuilt from rows 0,1 (C16). */
int gf_unpack(gf_ctx* ctx, const void* U_native_dev, double* U_canon_dev, void* stream);

/* native field of `src` (its precision and storage) -> native field of `dst` (same lattice, any precision / storage):
 * fp32 sweeps followed by an fp64 polish, or 18- <-> 12-real storage (row 2 rebuilt / dropped).  The gauge of the
 * two contexts may differ.  Widening (fp32 -> fp64) re-orthonormalises every link in fp64 (rows 0,1 Gram-Schmidt,
 * row 2 rebuilt), so the result is unitary to fp64 rounding.  GF_EINVAL: different extents, NULL or identical buffers. */
int gf_convert(gf_ctx* src, const void* U_src_native_dev, gf_ctx* dst, void* U_dst_native_dev, void* stream);

/* ---- the sweeps (device, in place, asynchronous on `stream`) --------------------------------------------- */

/* `nsweeps` iterations of Alg. 1: for sublattice = RED (parity 0), BLACK (parity 1): for
 * every site x of the sublattice: K(x) = sum_mu [U_mu(x) + U_mu(x-mu)^dagger] (eq. 2.3, C2); for
 * the SU(2) subgroups (0,1),(0,2),(1,2) in turn (C4): g = maximiser of Re tr[g K] in the subgroup
 * (eq. 2.4, C7), g -> g^omega to second order, reprojected to SU(2) (C9);
 * U_mu(x) <- g U_mu(x), U_mu(x-mu) <- U_mu(x-mu) g^dagger for all four mu.
 * U: native layout, device, updated in place.  omega in [1,2).  nsweeps >= 0.
 * Launches 2*nsweeps kernels on `stream`.  GF_EINVAL: omega outside [1,2), nsweeps < 0, NULL U. */
int gf_overrelax(gf_ctx* ctx, void* U_native_dev, double omega, int nsweeps, void* stream);

/* Simulated annealing "preconditioner" (all details C13/C14): `nsteps` full sweeps
 * (RED then BLACK), step i at temperature T_i = T_start + (T_end - T_start) * i / (nsteps - 1)
 * (nsteps == 1: T_start).  Each site update replaces the overrelaxed maximiser by an SU(2) heatbath draw
 * with weight exp(Re tr[g K] / T) per subgroup (Kennedy-Pendleton sampler), random numbers from
 * Philox4x32-10 keyed by (seed; site, step, parity, subgroup, trial).  The step counter restarts at 0 on
 * every call.  GF_EINVAL: T_start <= 0 or T_end <= 0, nsteps < 0, NULL U. */
int gf_anneal(gf_ctx* ctx, void* U_native_dev, double T_start, double T_end, int nsteps,
              unsigned long long seed, void* stream);

/* The other members of the paper's "family of relaxation algorithms", same sweep, other SU(2) step:
 *   GF_UPDATE_OVERRELAX2: gf_overrelax (param = omega, second-order g^omega);
 *   GF_UPDATE_OVERRELAX1: g^omega "to first order" (C17): h = (1 + omega (g0 - 1), omega gvec) / |.|;
 *   GF_UPDATE_STOCHASTIC: stochastic relaxation (PAPER.md:33 ref. [5]; C18): g -> g^2 with probability param = p in
 *     [0,1], else g; decision u < p from Philox4x32-10 keyed by (seed; site, sweep, parity, subgroup), the sweep
 *     counter restarting at 0 with every gf_relax call (inside gf_fix / gf_fix_slices it runs on through the chunks,
 *     so the decisions of a fixing run do not repeat).  p = 0 is plain relaxation [3], p = 1 a microcanonical sweep.
 * GF_EINVAL: unknown update, omega outside [1,2), p outside [0,1], nsweeps < 0, NULL U. */
enum { GF_UPDATE_OVERRELAX2 = 0, GF_UPDATE_OVERRELAX1 = 1, GF_UPDATE_STOCHASTIC = 2 };
int gf_relax(gf_ctx* ctx, void* U_native_dev, int update, double param, int nsweeps, unsigned long long seed,
             void* stream);

/* gf_anneal with n_micro microcanonical sweeps (g -> g^2 in every subgroup: F unchanged, C19) after every heatbath
 * sweep.  n_micro = 0 is gf_anneal. */
int gf_anneal_micro(gf_ctx* ctx, void* U_native_dev, double T_start, double T_end, int nsteps, int n_micro,
                    unsigned long long seed, void* stream);

/* ---- the reductions (device field -> host scalar; these calls synchronise) ------------------------------- */

/* F = Re sum_{x, mu < Nd} tr U_mu(x) / (N_c * Nd * V)  (eq. 2.1, C1), Nd = 4 (Landau) or 3
 * (Coulomb); F = 1 on the unit field.  Runs on the stream last passed to this ctx and waits for it. */
int gf_functional(gf_ctx* ctx, const void* U_native_dev, double* F_host);
/* theta = (1 / (V N_c)) sum_x tr[Delta(x) Delta(x)^dagger]  (eq. 2.5), Delta(x) the traceless
 * part of (K - K^dagger) / (2i) (C3).  Landau: that number.  Coulomb: max over timeslices of the
 * per-timeslice value (C12). */
int gf_theta(gf_ctx* ctx, const void* U_native_dev, double* theta_host);
/* per-timeslice theta_t = (1 / (V_s N_c)) sum_{x in slice t} tr[Delta Delta^dagger]; theta_host_Nt: Nt doubles */
int gf_theta_slices(gf_ctx* ctx, const void* U_native_dev, double* theta_host_Nt);

/* ---- theta without any allocation ---------------------------------------------------------------------------- */

/* The same theta reduction as gf_theta / gf_theta_slices (same kernels, same summation order), for callers that are
 * not allowed to allocate GPU memory: a host program that claimed the whole GPU for its own memory pool at start-up,
 * or one that runs under a fixed memory budget next to other jobs, cannot let a library call cudaMalloc behind its
 * back (it fails, or eats memory already promised elsewhere), and a measurement loop that checks theta every few
 * sweeps cannot afford the device-wide stall of a cudaMalloc / cudaFree.  Every other reduction here needs a gf_ctx,
 * and gf_create allocates.  This call needs no context and calls no cudaMalloc, cudaFree, cudaMallocHost or any other
 * allocating routine: the field and the output are the caller's, and the only scratch the reduction needs (one partial
 * sum per thread block) is a fixed array compiled into libgf.so.
 *
 *   Nx..Nt, precision, gauge, reals_per_link: as for gf_create / gf_set_storage (no slabs).
 *   U_native_dev: device, the field in the native layout (gf_field_bytes bytes), read only.
 *   out_dev:      device, Nt + 2 doubles owned by the caller, fully overwritten: out[0] = theta of the whole lattice
 *                 (eq. 2.5; what gf_theta returns in Landau gauge), out[1] = max_t theta_t (what gf_theta returns in
 *                 Coulomb gauge), out[2 + t] = theta_t (gf_theta_slices).
 *   stream:       the work is only enqueued; out_dev is valid once the stream has reached this point.
 *   err, err_len: optional host buffer for the message of a failing call (NULL / 0: no message).
 *
 * Limit: the built-in scratch holds gf_theta_static_max_partials() = 131072 doubles (1 MiB).  A lattice needs
 * 2 * Nt * ceil(Nx/2 * Ny * Nz / 256) of them -- 65536 at 64^4, 27648 at 48^3 x 64 -- and a larger one is refused with
 * GF_EINVAL and a message naming both numbers; nothing is launched.  The price of the array: that 1 MiB is held on
 * every GPU a process has loaded libgf.so on, until the process exits, used or not.
 *
 * First call on each device: it looks up where the array lives on that device (once; the device must be current, as
 * for every call here) and remembers it.  That look-up is set-up work, not stream work: make the first call on a device
 * during initialisation, before any stream capture is open.  Later calls only launch the two reduction kernels.
 *
 * Sharing: all calls on one GPU use the same array, and it keeps whatever the last call wrote.  That is harmless --
 * nothing in it has to start at zero, every launch writes each slot before reading it -- but two calls that run on the
 * GPU at the same time (two streams, two host threads) overwrite each other's partial sums and both results are
 * garbage.  Order them: one stream, or an event between them.  gf_theta on a context does not touch this array.
 *
 * GF_EINVAL: extents (odd, < 2, V >= 2^31), unknown precision / gauge / storage, NULL field or output, lattice beyond
 * the limit.  GF_ECUDA: the array's address cannot be resolved, or a launch fails. */
int gf_theta_static(int Nx, int Ny, int Nz, int Nt, int precision, int gauge, int reals_per_link,
                    const void* U_native_dev, double* out_dev, void* stream, char* err, size_t err_len);
size_t gf_theta_static_max_partials(void);

/* ---- Alg. 1 with its stop rule -------------------------------------------------------------------------------- */

/* "while precision theta not reached do" with the check after every `check_every`-th sweep
 * (C11) -- and, with the default setting, ending ONE SWEEP LATER than the paper's loop: sweeps_done =
 * n + 1 for the first checked sweep n with theta < theta_tol, and no check at n = max_sweeps (C21).  Coulomb: theta =
 * max over timeslices (C12).  sweeps_done / theta_host / F_host (each may be NULL) receive the number of sweeps and theta
 * and F of the field as returned.
 * The STOP RULE is a setting of the context and of nothing else (gf_set_monitor): the same arguments give the same
 * sweeps_done whatever the launch shape (gf_set_tuning), the precision, the tolerance or check_every.
 *   gf_set_monitor(ctx, 1 or 2) -- 1 is the default: the rule above (oracle: orc_fix_lag(lag = 1)).
 *   gf_set_monitor(ctx, 0): the paper's loop (oracle: orc_fix_lag(lag = 0)): gf_theta; while theta >= theta_tol and
 *     fewer than max_sweeps sweeps done: min(check_every, max_sweeps - done) sweeps; gf_theta.
 * Which KERNELS run the default rule is a matter of speed only (gf_fix_last_form tells):
 *   fused monitor: theta and F of the state after sweep n are accumulated by the sweep kernels themselves -- the BLACK
 *     half-sweep of sweep n leaves K(x) of its sites in registers, the RED half-sweep of sweep n+1 builds K(x) of the
 *     other half from that state before updating it -- and reduced on the device in a fixed order while sweep n+1 runs
 *     (which is where the one-sweep lag comes from).  No pass over the field per check, no host synchronisation per
 *     check: sweeps are enqueued in batches of 32 and launches past the stop return at once.  theta before the first
 *     sweep and theta / F of the returned field come from the separate reductions.  Taken when every thread block of the
 *     sweep lies inside one timeslice ((Nx Ny Nz / 2) * threads per site divisible by the block size; true for every
 *     lattice of BASELINE.json but 4^4 in fp64), for fp32 contexts when theta_tol >= 1e-10 (theta formed from the fp32 K
 *     of the sweep resolves ~1e-12), and, with setting 1, when check_every <= 10 (where it pays).
 *   separate check (the paper's second kernel) otherwise: the same rule with gf_theta at every check and
 *     one more sweep after the check that met the tolerance; synchronises at every check.  fp64 fields are bit-identical
 *     between the two; fp32 fields agree to the fp32 tolerance (the fused form sees theta through the fp32 K).
 * Errors as gf_relax; GF_EINVAL also for check_every < 1, max_sweeps < 0. */
int gf_fix(gf_ctx* ctx, void* U_native_dev, int update, double param, double theta_tol, int check_every,
           int max_sweeps, unsigned long long seed, int* sweeps_done, double* theta_host, double* F_host,
           void* stream);

/* Coulomb gauge, "each timeslice fixed independently" (C12, C20): as gf_fix, but a timeslice whose theta_t is below
 * theta_tol at a check is frozen for good (its sites are no longer updated; K, F and theta_t of a slice depend on
 * the spatial links of that slice alone), and the loop ends when no slice is active.  sweeps_done = sweeps of the
 * slowest slice; sweeps_per_slice (Nt ints, may be NULL) the sweeps every slice got.  Default stop rule (gf_set_monitor
 * 1 or 2, whichever kernels run it): the freeze of a slice found below the tolerance after sweep n takes effect from
 * sweep n + 2 (it gets n + 1 sweeps; oracle: orc_fix_slices_lag(lag = 1)); with check_every = 1 every slice stops
 * within one sweep of meeting the tolerance.  gf_set_monitor(ctx, 0): frozen from sweep n + 1 (orc_fix_slices).
 * GF_EINVAL for a Landau ctx. */
int gf_fix_slices(gf_ctx* ctx, void* U_native_dev, int update, double param, double theta_tol, int check_every,
                  int max_sweeps, unsigned long long seed, int* sweeps_done, int* sweeps_per_slice,
                  double* theta_host, double* F_host, void* stream);

/* ---- one configuration sharded over several contexts: t-slabs ("future multi-GPU") --- */

/* A context that owns the timeslices [t_begin, t_end) of an Nx*Ny*Nz*Nt_global lattice.  Its native field
 * (gf_field_bytes) holds the owned slices followed by ONE ghost slice: a copy of the temporal links U_t(x, t_begin - 1)
 * of the slab below (periodic: the last slab for the first), the only links a site update of this slab shares with
 * another slab (as U_t(x - t) of its first slice, read for K(x) and multiplied by g(x)^dagger).  gf_pack / gf_unpack
 * exchange the owned slices only (canonical: the (t_end - t_begin) slices, local t); Nt-sized outputs (gf_theta_slices,
 * gf_fix_slices) have t_end - t_begin entries; gf_functional / gf_theta are those of the owned sites (gf_theta needs
 * a current ghost); the Philox counters carry the site of the WHOLE lattice, so a sharded run takes the decisions of
 * the unsharded one.  Not available on a slab: Coulomb reading B, the fused monitor, the host-buffer path.
 * GF_EINVAL: t_begin or t_end odd (the local checkerboard must be the global one), fewer than 2 slices, bounds
 * outside [0, Nt_global]; otherwise as gf_create. */
int gf_create_slab(gf_ctx** out, int Nx, int Ny, int Nz, int Nt_global, int t_begin, int t_end, int precision, int gauge);
/* Bytes of one face message: the temporal links of one parity block of one timeslice, (Nx Ny Nz / 2) * reals_per_link *
 * sizeof(real).  Per half-sweep one such message crosses every slab boundary in each direction. */
size_t gf_slab_face_bytes(const gf_ctx* ctx);
/* Gather / scatter a face between the native field and a contiguous device buffer of gf_slab_face_bytes.
 * which = 0: the last owned slice; which = 1: the ghost slice.  block_parity: parity of the sites the links start at.
 * Protocol of a half-sweep of parity p on slab r (block_parity = 1 - p throughout): pack(r-1, which 0) -> message ->
 * unpack(r, which 1); half-sweep; pack(r, which 1) -> message -> unpack(r-1, which 0).  GF_EINVAL on a plain context. */
int gf_slab_pack_face(gf_ctx* ctx, const void* U_native_dev, int which, int block_parity, void* buf_dev, void* stream);
int gf_slab_unpack_face(gf_ctx* ctx, void* U_native_dev, int which, int block_parity, const void* buf_dev, void* stream);
/* One half-sweep (Alg. 1's inner "for all x of sublattice") of parity 0 (RED) / 1 (BLACK) on the owned
 * timeslices [t_first, t_first + t_count) -- any context; what a driver interleaves with the face exchange (first
 * slice, interior).  `sweep` (>= 0): index of the sweep within the driver's loop: the counter of the stochastic
 * decisions (C18), of the re-orthonormalisation cadence (C15) and of the hybrid chain; gf_begin_sweeps starts such a
 * loop (what the start of gf_relax does: fp32 contexts forget the roughness of whatever ran before, the first sweep
 * runs the double chain).  update / param / seed as gf_relax.  Coulomb contexts run reading
 * A here.  gf_anneal_half: the same for one heatbath half-sweep at temperature T, `step` the annealing step (C13/C14).
 * GF_EINVAL: bad parity, sweep < 0, timeslices outside the owned range, parameter out of range, reading B forced. */
int gf_begin_sweeps(gf_ctx* ctx, void* stream);
int gf_relax_half(gf_ctx* ctx, void* U_native_dev, int update, double param, int parity, int sweep,
                  unsigned long long seed, int t_first, int t_count, void* stream);
int gf_anneal_half(gf_ctx* ctx, void* U_native_dev, double T, int parity, int step, unsigned long long seed,
                   int t_first, int t_count, void* stream);
/* Un-normalised sums over the owned sites, to be added over the slabs: F_raw = sum_{x, mu < Nd} Re tr U_mu(x) (eq. 2.1),
 * theta_raw = sum_x tr[Delta Delta^dagger] (eq. 2.5; needs a current ghost).  Each output may be NULL.  Synchronises. */
int gf_raw_sums(gf_ctx* ctx, const void* U_native_dev, double* F_raw_host, double* theta_raw_host);

/* ---- host-buffer convenience path (what a user with a configuration in host memory calls) ---------------- */

/* U_canon_host (canonical fp64, V*72 doubles) is copied to the device, packed, swept `nsweeps` times at
 * `omega`, F and theta are reduced, the field is unpacked and copied back into U_canon_host; F_host /
 * theta_host (may be NULL) receive the values after the last sweep.  Device staging buffers live in ctx and
 * are reused between calls.  Synchronous.  GF_ENOMEM when the staging buffers cannot be allocated. */
int gf_overrelax_host(gf_ctx* ctx, double* U_canon_host, double omega, int nsweeps, double* F_host,
                      double* theta_host);

/* The same with the canonical field held as float (V*72 floats, same element order): what a user of an fp32
 * context has in memory; halves the bytes over PCIe.  Works for fp64 contexts too (the field is widened on pack). */
int gf_overrelax_host_f32(gf_ctx* ctx, float* U_canon_host, double omega, int nsweeps, double* F_host,
                          double* theta_host);

/* An ensemble of n configurations in host memory (the shape of production gauge fixing), pipelined: configuration
 * i+1 is copied to the device and configuration i-1 copied back while configuration i is swept -- three staging slots in
 * the context, one stream per direction of the PCIe link and one for the kernels.  U_canon_host: n pointers to canonical
 * fields of element_bytes = 8 (double) or 4 (float) per real, each updated in place exactly as gf_overrelax_host /
 * gf_overrelax_host_f32 would (bit-identical); pinned memory lets the copies overlap, pageable memory is correct but
 * serial.  F_host_n / theta_host_n (n doubles each, may be NULL): F and theta after the last sweep.  Synchronous.
 * GF_EINVAL: n < 0, a NULL configuration, element_bytes not 4 or 8, omega outside [1,2), nsweeps < 0, a slab context.
 * GF_ENOMEM: the staging slots (3 x (canonical + native field)) cannot be allocated. */
int gf_overrelax_host_batch(gf_ctx* ctx, void* const* U_canon_host, int n, int element_bytes, double omega, int nsweeps,
                            double* F_host_n, double* theta_host_n);

/* ---- tuning and diagnostics ------------------------------------------------------------------------------ */

/* Launch shape of the sweep kernels: threads_per_site in {1,2,4} (1: one thread holds all 8 links of a site;
 * 2: two threads hold the links of 2 directions each; 4: one direction each; partial K summed by warp
 * shuffles), block = threads per block (multiple of 32, <= 256).  0 = automatic (the default): chosen per
 * (precision, storage) from the measurements in profiles/. */
int gf_set_tuning(gf_ctx* ctx, int threads_per_site, int block);
/* Unitarity policy (C15): every `every`-th sweep the RED half-sweep re-orthonormalises rows 0,1 of each link on load
 * (and rebuilds row 2).  0 = never, -1 = automatic (default): 18-real storage fp32 every 16th sweep, fp64 never;
 * 12-real storage (both precisions) every 16th overrelaxation sweep and every 4th heatbath / stochastic /
 * microcanonical sweep -- with 12 reals the rebuilt row feeds norm errors back and they grow exponentially under
 * large rotations (C15).  The cadence counts the sweeps since the start of the current API call
 * (gf_overrelax, gf_relax, gf_anneal, gf_fix, ...: sweeps 16, 32, ... of each call), so a call's result depends on
 * its arguments and the field only, not on what the context did before. */
int gf_set_reunit(gf_ctx* ctx, int every);
/* Alternate the block traversal direction between consecutive half-sweeps so that the tail of one
 * half-sweep, still in L2, is what the next one reads first (1 = on, default; 0 = off). */
int gf_set_l2_reversal(gf_ctx* ctx, int on);
/* L2 eviction policy of the link accesses of the sweep kernels: 0 = normal, 1 = evict first, 2 = evict last.
 * Default (0, 2): loads keep the normal policy, stores ask L2 to keep
 * the freshly written lines, which the next half-sweep (traversing in the opposite direction) reads first. */
int gf_set_l2_policy(gf_ctx* ctx, int load_policy, int store_policy);
/* Programmatic dependent launch of consecutive half-sweeps (1 = on, default): the next half-sweep's grid becomes
 * resident while the current one drains and waits on the device before it touches the field. */
int gf_set_pdl(gf_ctx* ctx, int on);
/* L2 prefetch distance of the sweep kernels, in sites along the traversal direction: every thread prefetches
 * into L2 the lines that the thread `sites` further on will load.  0 = off, -1 = automatic (default; chosen per
 * precision / storage / sweep kind from the measurements in profiles/). */
int gf_set_prefetch(gf_ctx* ctx, int sites);
/* Coulomb gauge, treatment of the temporal links (C12): 0 = reading A: every half-sweep moves and multiplies all 8
 * links of a site; 1 = reading B; -1 = automatic (default): B in fp32 (+14 % at one thread per site), A in fp64, and
 * A when the site field cannot be allocated.  Reading B: the sweeps (relaxation and annealing alike) leave the
 * temporal links in memory, accumulate g(x) in a site field owned by the context (V * 18 reals) and
 * transform the temporal links once at the end of each call -- 14/16 of the bytes, same result up to rounding.
 * gf_anneal / gf_anneal_micro keep one site field over the whole call.  GF_EINVAL for a Landau context. */
int gf_set_coulomb_reading(gf_ctx* ctx, int reading_b);
/* Stop rule and kernels of the fixing loops gf_fix / gf_fix_slices.  0 = the paper's loop, separate check kernel (lag 0).
 * 1 (default) and 2 = the rule of C21 (lag 1: the loop ends, or a timeslice freezes, one sweep after the check that met
 * the tolerance; no check at max_sweeps) -- the two differ in speed only: 1 takes the fused monitor where it applies and
 * check_every <= 10 (a monitored sweep costs ~4 % more than a plain one, a checked one ~20 %, a separate check about
 * 0.6 sweeps: the fused form wins while checks are frequent), 2 wherever it applies; elsewhere the separate check kernel
 * runs the same rule.  GF_EINVAL otherwise. */
int gf_set_monitor(gf_ctx* ctx, int fused);
/* Form of the last gf_fix / gf_fix_slices on this context (each output may be NULL): *lag = 0 the paper's stop rule,
 * 1 the rule of C21 (one sweep past the check that met the tolerance); *fused = 1 if the sweep kernels monitored theta
 * themselves, 0 if the separate check kernel ran.  Both -1 before the first such call. */
int gf_fix_last_form(const gf_ctx* ctx, int* lag, int* fused);
/* The last check completed by a fused fixing loop on this context: the sweep n it belongs to (0: none yet), theta
 * (Coulomb: max over timeslices) and F of the state after that sweep, the per-timeslice theta_t (Nt doubles).  Each
 * output may be NULL.  Synchronises.  GF_EINVAL if no fused loop has run. */
int gf_monitor_last(gf_ctx* ctx, int* check_sweep, double* theta_host, double* F_host, double* theta_host_Nt);
/* fp32 contexts, precision of the site chain.  The links are fp32 in memory and in the link
 * products; the site chain -- K(x), the three SU(2) steps, K <- G K -- is ill-conditioned where the projected block k
 * of K or the expanded g^omega is small, and a BLACK half-sweep inherits the rounding of the RED one through its K.
 * Relaxation sweeps (gf_overrelax, gf_relax, gf_fix*):
 *   chain = 2 (default, hybrid): a half-sweep runs the chain in double (K accumulated exactly from the fp32 links, G
 *     rounded to fp32 once) while the field is rough -- iff one of the two half-sweeps before it had a step with
 *     conditioning number |k| |h| below watch_threshold (default 1.0; |k|: norm of the projected block, |h|: norm of the
 *     expanded g^omega before its reprojection, 1 for the gf_relax variants), and during the first sweep of every call
 *     -- and in fp32 once it is smooth.  Every link then meets the fp32 tolerance of 5e-5 after one sweep against an
 *     fp64 evaluation; on a nearly fixed field only the first sweep of a call takes the double chain.
 *   chain = 1: always double (about -7 % at 18 reals, -30 % at 12 reals).  chain = 0: always fp32 (a few 1e-5 of the
 *     sites of a random-gauge start miss 5e-5).
 * Annealing sweeps (gf_anneal*): chain = 2 (default): fp32 chain, draw on the special-function unit, in three tiers:
 *   (i) the accepted delta is taken again with 1-ulp fp32 functions where its SFU error would move the links by more
 *   than ~8e-6; (ii) a site is redone in double from the stored fp32 links inside the same kernel (K, the draw, the link
 *   products; one rounding at the store) where the projected block has |k| below fix_threshold (default 0.15) in one of
 *   its three steps, where an accept test fell inside the SFU error band of its threshold, or where (i) is still too
 *   coarse -- 8e-5 of the sites at T = 1.4, none below T ~ 0.1.  Accept decisions: 1e-7 of the draws differ from an fp64
 *   evaluation.  Links, one half-sweep at a time against an fp64 evaluation of the same stored input: all within 5e-5
 *   at every temperature (measured max 3e-5 on 7 M sites at T = 1.4).  Over a whole step the BLACK half-sweep reads RED
 *   links that carry their fp32 storage rounding and a site with a small block amplifies it by 1/|k|: against an fp64
 *   run of the whole step about 7e-6 of the sites of a 7 M-site lattice end beyond 5e-5 at T = 1.4 (max 1.3e-4), none
 *   below T ~ 0.5.  chain = 1: the double chain at every site (about -17 %): the same per-half-sweep bound; it cannot
 *   remove the whole-step tail, which sits in the stored input (measured 4e-6 of the sites, max 7.6e-5) -- only an fp64
 *   context does.  chain = 0: plain fp32, no tiers.
 * A threshold of 0 keeps the current value.  Ignored by fp64 contexts.  GF_EINVAL: chain outside 0..2, a threshold < 0
 * or > 1e3.
 * gf_chain_count (each output may be NULL; synchronises the stream): half-sweep launches that ran the double chain and
 * site updates redone in double, since gf_create. */
int gf_set_chain(gf_ctx* ctx, int chain, double watch_threshold, double fix_threshold);
int gf_chain_count(gf_ctx* ctx, unsigned long long* double_launches_host, unsigned long long* double_sites_host);
/* Optional debug output of gf_anneal: d_trials (device, V*3 unsigned, index 3*s + subgroup) receives the
 * number of Kennedy-Pendleton trials of every (site, subgroup) of the LAST step; NULL switches it off. */
int gf_set_trial_buffer(gf_ctx* ctx, unsigned* d_trials);
/* Number of kernels this ctx has launched so far. */
unsigned long long gf_launch_count(const gf_ctx* ctx);
/* Diagnostic: the double-precision functions of the fp64 annealing draw (C14) evaluated on n given Philox words x_i
 * (device): neglog_dev[i] = -ln u_i, sin_dev[i] = sin(2 pi u_i), cos_dev[i] = cos(2 pi u_i), u_i = (2 (x_i >> 9) + 1) 2^-24.
 * The kernels use their own branch-free versions of these functions (24-bit arguments); this call lets
 * a test check them over the whole domain.  Each output may be NULL.  Asynchronous on `stream`.  GF_EINVAL: NULL words, n < 0. */
int gf_debug_kp_math(const unsigned* words_dev, int n, double* neglog_dev, double* sin_dev, double* cos_dev, void* stream);
/* Registers per thread and local-memory bytes per thread (spills; for the fp32 annealing kernels also the stack frame of
 * their rare double-precision redo path, 200-300 bytes that the hot path never touches) of the sweep kernel that the current
 * (precision, storage, gauge reading, tuning) selects; mode 0 = overrelaxation, 1 = heatbath, 2 = gf_relax variants. */
int gf_kernel_info(gf_ctx* ctx, int mode, int* regs_per_thread, int* local_bytes_per_thread);

#ifdef __cplusplus
}
#endif
#endif /* GF_H_ */
