/* mpmc.h — C ABI of the B200-native checkerboard cell sweep for hard disks.
 *
 * Method: Anderson, Jankowski, Grubb, Engel, Glotzer, "Massively parallel Monte Carlo for many-particle
 * simulations on GPUs" (arxiv 1211.1646).  Citations are lines of /root/reference/PAPER.md.
 *   - one sweep = Algorithm 1 (L60-93): the four checkerboard sets (eq. 1) in a random order, each an
 *     Algorithm-2 sub-sweep (L164-236) over all cells of the set, then a random cell shift, Algorithm 4
 *     (L270-342, L350-354);
 *   - positions live in the cell list in cell-local coordinates (L148-154), n_max = 4 slots per cell (L152);
 *   - pressure from the pair-distance histogram near contact (L366-382, eq. 4-6).
 * The readings taken where the paper is silent or garbled are listed in DESIGN.md "Readings".
 *
 * Conventions for every call
 *   - Return value: 0 (MPMC_OK) or a negative MPMC_ERR_* code; nothing throws across the ABI.
 *   - "device" pointers are CUDA device pointers on the device current at mpmc_create; "host" pointers are
 *     ordinary host memory.  The library NEVER allocates or frees device memory: the caller provides one
 *     workspace (mpmc_workspace_bytes) that must outlive the context, and every in/out buffer.
 *   - All device work is enqueued on the CUDA stream given at creation (a cudaStream_t cast to void*;
 *     NULL = legacy default stream).  Calls that return host values synchronise that stream; the others are
 *     asynchronous.  Conditions detected on the device (cell overflow, bad input) set a sticky error word
 *     that the next synchronising call returns.
 *   - There is no CPU fallback: without a CUDA device every call except mpmc_workspace_bytes*, mpmc_strerror
 *     and mpmc_version fails with MPMC_ERR_CUDA.
 */
#ifndef MPMC_H_
#define MPMC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mpmc_ctx mpmc_ctx; /* opaque host object; owns no device memory */

/* error codes */
#define MPMC_OK 0
#define MPMC_ERR_ARG (-1)           /* bad argument (NULL pointer, N = 0, n_s > 32, both/neither precision flag ...) */
#define MPMC_ERR_BOX (-2)           /* box too small: fewer than 2 cells of width >= sigma along an axis, or too many cells */
#define MPMC_ERR_WORKSPACE (-3)     /* workspace NULL, misaligned (256 B) or smaller than mpmc_workspace_bytes */
#define MPMC_ERR_OVERLAP (-4)       /* loaded positions overlap, or a coordinate is NaN / outside [0, L] */
#define MPMC_ERR_CELL_OVERFLOW (-5) /* more than n_max = 4 disks in one cell (possible only when w >= sqrt(2) sigma) */
#define MPMC_ERR_CUDA (-6)          /* CUDA runtime error (no device, launch failure ...) */
#define MPMC_ERR_STATE (-7)         /* no positions loaded yet */
#define MPMC_ERR_TOO_LARGE (-8)     /* a size beyond the fixed capacity of a no-allocation entry point (see its comment) */

/* flags for mpmc_create: exactly one precision bit */
#define MPMC_FP64 0x1u  /* local coordinates and all move arithmetic in double */
#define MPMC_FP32 0x2u  /* ... in float (the paper's benchmarks, L390); pressure histogram still in double */
#define MPMC_DISC 0x4u   /* trial moves uniform in the DISC of radius d (the paper's rng.inCircle(d), L190) instead of the
                           square [-d, d]^2 of reading A2; runs on the 4-slot fused tile kernel for n_s = 4, otherwise on
                           the general persistent kernel */
/* ablations of PAPER.md section 2.4 / Table 1 (L114-142); both leave the chain valid only in the sense the paper discusses */
#define MPMC_NO_PARTICLE_SHUFFLE 0x8u  /* visit the disks of a cell in slot order (the paper shows a pressure bias) */
#define MPMC_NO_SET_SHUFFLE 0x10u     /* run the checkerboard sets in the fixed order a, b, c, d (harmless per the paper) */
#define MPMC_NO_RESIDENT 0x20u        /* do not use the cluster-resident kernel for small systems (below): every sweep on the
                                      * fused tile kernels or the general kernel, as for large systems.  Same trajectory; for
                                      * tests of those kernels on small inputs and for A/B timing */
#define MPMC_DEBUG 0x100u /* record per-cell accept masks and the accept-sequence digest (tests only; slower) */

/* Bytes of device workspace mpmc_create needs for this system (0 on invalid arguments).  Pure host arithmetic.
 * w_target: requested minimum cell width; <= sigma (e.g. 0) means "smallest width >= sigma that divides the box"
 * (BASELINE.json configs; reading A11), a value in (sigma, sqrt(2) sigma) gives the paper's regime (L152). */
size_t mpmc_workspace_bytes(uint64_t N, const double box[2], double sigma, uint32_t flags);
size_t mpmc_workspace_bytes_ex(uint64_t N, const double box[2], double sigma, double w_target, uint32_t flags);

/* Create a simulation of N hard disks of diameter sigma in the periodic box [0,Lx) x [0,Ly)  (L25, L362).
 *   box      host, {Lx, Ly}
 *   d        maximum displacement: trial moves are uniform in [-d, d]^2 (reading A2), or in the disc of radius d
 *            with MPMC_DISC
 *   n_s      trial moves per non-empty active cell per sub-sweep (the paper's n_M, L95, L358); 0..32
 *   seed     user seed, fixed for the run (L170); keys the Philox4x32-10 streams (reading A9)
 *   workspace  device, 256-byte aligned, >= mpmc_workspace_bytes(...); owned by the caller
 *   cuda_stream  cudaStream_t as void*
 * Derived, not passed: mx, my = largest even cell counts with cell width w = L/m >= max(sigma, w_target)
 * (rounded to the working precision); the simulated box is L_eff = m * w (mpmc_geometry). */
int mpmc_create(mpmc_ctx** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s,
                uint64_t seed, uint32_t flags, void* workspace, size_t workspace_bytes, void* cuda_stream);
int mpmc_create_ex(mpmc_ctx** out, uint64_t N, const double box[2], double sigma, double d, uint32_t n_s,
                   uint64_t seed, uint32_t flags, double w_target, void* workspace, size_t workspace_bytes,
                   void* cuda_stream);
int mpmc_destroy(mpmc_ctx* ctx);

/* Geometry chosen at creation (all host out-pointers, any may be NULL): m = {mx, my}, w = {wx, wy} (the working-
 * precision cell widths as doubles), L_eff = {mx*wx, my*wy}. */
int mpmc_geometry(const mpmc_ctx* ctx, uint32_t m[2], double w[2], double L_eff[2]);

/* Cell-list build (L148-154): xy = device, N x 2 interleaved doubles, global coordinates in [0, L].  Slots of a
 * cell are filled in ascending disk index (reading A13).  Resets the grid origin, the sweep index and the
 * counters.  Synchronises; returns MPMC_ERR_OVERLAP / MPMC_ERR_CELL_OVERFLOW for bad input. */
int mpmc_load_positions(mpmc_ctx* ctx, const double* xy);

/* k full sweeps of Algorithm 1 (four sub-sweeps + shift each).  How they run is chosen at creation
 * (mpmc_debug_config tells): a small system (n_s = 4, up to ~1e4 - 2e4 cells) in ONE launch of the cluster-resident kernel for
 * all k; otherwise one fused tile-kernel launch per sweep (n_s = 4, or n_s = 8 at w ~ sigma with the square proposal),
 * otherwise one persistent cooperative launch for all k.  Every path gives the same trajectory bit for bit.
 * Asynchronous.  All random draws are functions of (seed, sweep index, cell): the per-sweep set order and shift are
 * evaluated on the device, or by the host at launch time and passed as kernel arguments; there is no device->host traffic
 * inside the loop. */
int mpmc_sweep(mpmc_ctx* ctx, uint64_t k);

/* Unpack (L154): xy_out = device, N x 2 doubles, written in the original disk order;
 * X = (origin + cell*w + local) wrapped into [0, L_eff).  Asynchronous. */
int mpmc_get_positions(mpmc_ctx* ctx, double* xy_out);

/* out = host, {attempted, accepted, rejected_boundary, rejected_overlap} since the last load.  attempted counts
 * n_s per non-empty active cell (reading A10; eta = attempted / time, L421).  Synchronises. */
int mpmc_acceptance(mpmc_ctx* ctx, uint64_t out[4]);

/* Contact pressure (L366-382).  hist_out = host, nbins counts of unordered pairs with r in [sigma + i dr,
 * sigma + (i+1) dr), computed on the device in double; g_contact = polynomial fit (unweighted least squares,
 * given degree < nbins) of g(R_i) (eq. 5-6) extrapolated to r = sigma; p_star = eq. 4.  hist_out, g_contact,
 * p_star may each be NULL.  nbins <= 4096.  Synchronises. */
int mpmc_pressure_contact(mpmc_ctx* ctx, double dr, uint32_t nbins, uint32_t degree, uint64_t* hist_out,
                          double* g_contact, double* p_star);

/* Contact pressure averaged over samples — the paper's procedure (L384: a sample every 200 sweeps; eq. 5 averages n[r_i]
 * over configurations before the fit).
 *   mpmc_pressure_accumulate  adds the pair histogram of the CURRENT state (same bins and arithmetic as
 *       mpmc_pressure_contact) to an accumulator in the workspace and counts one sample.  Asynchronous: no host
 *       synchronisation per sample.  The first sample after a reset fixes (dr, nbins); other values are MPMC_ERR_ARG.
 *   mpmc_pressure_accumulated  hist_out = host, nbins summed counts (may be NULL); *samples = number of samples (may be
 *       NULL); g_contact / p_star (each may be NULL) = eq. 5-6 on the sample-averaged histogram, polynomial fit of the
 *       given degree extrapolated to r = sigma, and eq. 4.  Synchronises.  MPMC_ERR_STATE with no sample.
 *   mpmc_pressure_reset  empties the accumulator (mpmc_load_positions does NOT).
 *   mpmc_pressure_from_histogram  the same estimator on a caller's histogram (host, nbins counts summed over `samples`
 *       configurations of THIS system — e.g. blocks of accumulated histograms added up).  Host arithmetic only. */
int mpmc_pressure_accumulate(mpmc_ctx* ctx, double dr, uint32_t nbins);
int mpmc_pressure_accumulated(mpmc_ctx* ctx, uint32_t degree, uint64_t* hist_out, uint64_t* samples, double* g_contact,
                              double* p_star);
int mpmc_pressure_reset(mpmc_ctx* ctx);
int mpmc_pressure_from_histogram(const mpmc_ctx* ctx, const uint64_t* hist, uint64_t samples, double dr, uint32_t nbins,
                                 uint32_t degree, double* g_contact, double* p_star);

/* Contact histogram without any allocation (for callers that cannot call cudaMalloc: code under CUDA graph capture,
 * serving loops, harnesses that forbid it).  The same pair histogram as mpmc_pressure_contact (L366-382; same kernels, same
 * bins, same double-precision arithmetic: the counts are identical), but the kernels' scratch — the device histogram the
 * blocks add their counts to — is NOT the workspace's: it is a file-scope `static __device__` array of
 * MPMC_NOALLOC_MAX_BINS 64-bit counters (8 KB) inside the library, which every GPU that loads the library holds until the
 * process exits.  The call makes no cudaMalloc / cudaFree and no allocating library call, on the device or the host.
 *   hist_out = DEVICE, nbins uint64 counts of unordered pairs with r in [sigma + i dr, sigma + (i+1) dr), owned by the
 *       caller, written on the context's stream.  Asynchronous: no host synchronisation.
 *   nbins > MPMC_NOALLOC_MAX_BINS: MPMC_ERR_TOO_LARGE, nothing is launched (use mpmc_pressure_contact, up to 4096 bins).
 *   The context's device must be the current device (MPMC_ERR_ARG otherwise): the array's device address is resolved
 *       once per device, with that device current, on the first call.
 *   ALL calls on one GPU — of any context, on any stream, from any thread — share the one array, which keeps the last
 *       call's counts: every call clears the bins it uses first, and two calls that OVERLAP on the GPU (different
 *       streams or contexts, no ordering between them) race and both return garbage.  Calls on one stream are ordered.
 *   MPMC_ERR_STATE with no positions loaded; device-detected errors are reported by the next synchronising call. */
#define MPMC_NOALLOC_MAX_BINS 1024u
int mpmc_contact_histogram_noalloc(mpmc_ctx* ctx, double dr, uint32_t nbins, uint64_t* hist_out);

/* Test hooks: single pieces of Algorithm 1 at the current sweep index (do not advance it). */
int mpmc_debug_sub_sweep(mpmc_ctx* ctx, uint32_t checkerboard_set /*0=a(0,0) 1=b(1,0) 2=c(0,1) 3=d(1,1)*/);
/* delta in [0, w) of the chosen axis (Algorithm 1 draws it from [0, w/2), L90; the pull form of Algorithm 4 takes
 * entrants from one neighbour only, so a larger delta is MPMC_ERR_ARG). */
int mpmc_debug_shift(mpmc_ctx* ctx, uint32_t direction /*0:+x 1:-x 2:+y 3:-y*/, double delta);

/* Test hook: the state in a layout-independent canonical form, cell c = y*mx + x.  Device out-pointers (any may
 * be NULL): counts u32[M]; slab real[M][4][2] (real = float or double per the precision flag; unused slots 0);
 * ids u32[M][4] (unused 0xFFFFFFFF); accept_mask u32[M] (bit s = move s of the cell accepted in the last sweep;
 * needs MPMC_DEBUG).  Host out-pointers (any may be NULL): origin[2], sweep index, accept-sequence digest.
 * Synchronises. */
int mpmc_debug_state(mpmc_ctx* ctx, void* counts, void* slab, void* ids, void* accept_mask, double origin[2],
                     uint64_t* sweep, uint64_t* digest);

/* Test hook: out = host, {sweeps done by the fused tile kernel, sweeps done by the general persistent kernel} since
 * the last load (the tile kernel serves cell widths w ~ sigma and hands a sweep to the general
 * kernel only when more cells hold 3 or 4 disks than it can carry).  Synchronises. */
int mpmc_debug_path(mpmc_ctx* ctx, uint64_t out[2]);

/* Test hook (host values only): how mpmc_sweep will run this context.  out = host, {slots per cell of the fused tile
 * kernel: 2 (tile.cuh, w ~ sigma), 4 (tile4.cuh) or 0 (no tile kernel: every sweep on the general persistent kernel);
 * CTAs (= tiles) of the tile kernel; tiles per row of tiles (first group of rows, see mpmc_debug_tiling);
 * tiles along y; threads per tile CTA; dynamic shared memory per tile CTA in bytes; CTAs of the general kernel; threads
 * per CTA of the general kernel; CTAs of the cluster-resident kernel (cluster.cuh; 0 = not used: the system is too large
 * for one cluster's shared memory, n_s != 4, or MPMC_NO_RESIDENT) — when non-zero, mpmc_sweep(k) is ONE launch of that
 * kernel and the tile kernel's entries describe what MPMC_NO_RESIDENT would use; its tiles along x; along y; its dynamic
 * shared memory per CTA in bytes}. */
int mpmc_debug_config(const mpmc_ctx* ctx, uint32_t out[12]);

/* Profiling hook.  A library built with -DMPMC_PHASE_CLOCKS (paper_1211_1646_b200/phase_clocks.py) makes the 2-slot tile
 * kernel record a clock mark at each of its phase boundaries; this call copies the marks of the LAST launch to the host:
 * out = host, room for max_tiles x 32 values; max_tiles x *marks are written, row = tile; value 0 of a row is the global
 * nanosecond timer at the start of the tile's work, values 1-8 are SM cycle counters (clock64) at the ends of: wait for
 * the previous sweep, load, sub-sweeps 1-4, shift, (unused); the rest are marks inside the load phase and before it
 * (paper_1211_1646_b200/phase_clocks.py names them).  *marks = values per row (at most 32), 0 in an ordinary build
 * (nothing is written to out).  A context on the cluster-resident kernel gets one row per CTA of the cluster instead:
 * {sweeps of the last call, SM cycles thread 0 spent in the sub-sweeps, at the cluster barriers, in the shift, in the whole
 * loop}.  MPMC_ERR_STATE unless the context runs the 2-slot tile kernel or the cluster-resident kernel.  Synchronises. */
int mpmc_debug_phase_clocks(mpmc_ctx* ctx, uint64_t* out, uint32_t max_tiles, uint32_t* marks);

/* Test hook (pure host arithmetic, no device needed): the tiling the fused tile kernels would use for a grid of
 * 2 hx x 2 hy cells when a cell takes cell_bytes of shared memory, an SM offers smem_max bytes and the device has sms
 * SMs.  out = {a, rows, plane stride in cells, na, hyA, tiles}: the tiles form `rows` rows; the first na rows hold a tiles
 * each and share the half-rows [0, hyA) evenly, the other rows hold a + 1 tiles each and share the rest (a uniform
 * a x rows grid has na = rows, hyA = hy).  Every tile (rounded up to even sizes) plus a halo of 5 cells on each side fits
 * smem_max and is no wider than the grid; MPMC_ERR_BOX if no such tiling exists (grids under 12 cells across). */
int mpmc_debug_tiling(uint32_t hx, uint32_t hy, size_t cell_bytes, size_t smem_max, uint32_t sms, uint32_t out[6]);

/* Test hook: Philox4x32-10 evaluated ON THE DEVICE by the same routine the kernels use.
 * ctr = device u32[n][4], key = host u32[2], out = device u32[n][4]; enqueued on cuda_stream and synchronised. */
int mpmc_debug_philox(const uint32_t* ctr, const uint32_t key[2], uint32_t* out, uint32_t n, void* cuda_stream);

const char* mpmc_strerror(int code);
const char* mpmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MPMC_H_ */
