/*
 * rc.h — C ABI of librc.so: the radiance-cascades formal solution on a 2D grid ("flatland"),
 * B200 (sm_100a) only.  Method: Osborne & Sannikov, arxiv 2408.14425 (PAPER.md = the paper's text).
 *
 * The interface is the paper's `GivenFs` problem statement (§3.8): "the input model
 * provides a set of isotropic emissivities and opacities at each point in the domain.  These are
 * solved for J".  One rc_solve_J call runs the whole hot path:
 *
 *   a1  per-cascade radiance-interval ray march: DDA through the chi/eta voxel grids with the
 *       piecewise-constant update of eq. 16
 *   a2  boundary intensity on the top cascade
 *   a3  bilinear interpolation over the 4 parent probes of cascade i+1, mean over the 4 child
 *       directions, merge (eq. 11)
 *   a4  J = mean over the 4 merged cascade-0 directions      PAPER.md:36 (eq. 1), 191
 *
 * Cascade geometry (eq. 12-13 with branching factor alpha = 2):
 * cascade i has probes at ((a+1/2) 2^i, (b+1/2) 2^i), 4^(i+1) directions
 * theta_k = 2 pi (k+1/2)/4^(i+1), interval [t_i, t_(i+1)], t_i = c0_interval (4^i - 1)/3; the top
 * cascade runs to the domain edge.  Cell size is 1.
 *
 * Conventions
 *   Layout   chi[(y*nx + x)*nlambda + l], wavelength fastest, y = 0 the bottom row; same for eta
 *            and J_out.  float32.  chi in 1/cell, eta = chi * S.  Device arrays (chi, eta, line, J_out)
 *            must be 32-byte aligned (RC_ERR_BAD_VALUE otherwise): the kernels move one 32-byte sector per thread.
 *   Memory   "device" pointers are CUDA device memory of the context's device, "host" pointers
 *            ordinary host memory.  The library never allocates device memory: inputs, output,
 *            workspace and the stream are the caller's (e.g. torch tensors / torch streams).
 *            Pointers given to rc_set_atmosphere / rc_set_workspace are BORROWED until replaced
 *            or rc_destroy.  Small host arrays (boundary, weights) are copied at the call.
 *   Async    rc_solve_J only enqueues work on the context's stream and returns; it does not
 *            synchronise.  rc_solve_J_host synchronises that stream before returning.
 *   Errors   every call returns RC_OK (0) or a negative RC_ERR_*; nothing throws across the ABI;
 *            rc_last_error(ctx) gives text for the last failure on that context.
 *   Inputs   chi >= 0, eta >= 0, finite.  eta > 0 where chi == 0 (emission without opacity) is valid: eq. 16
 *            in the limit chi -> 0, the cell adds eta ds (reading G11).
 *   There is no CPU fallback and no other backend: without an sm_100 device rc_create fails.
 *
 * The library reads no environment variables; launch knobs for measurements and tests go through rc_set_tuning.
 */
#ifndef RC_H_
#define RC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RC_OK 0
#define RC_ERR_NULL_ARG (-1)
#define RC_ERR_BAD_SHAPE (-2)    /* nx, ny not positive multiples of 2^(ncascades-1); nlambda < 1; too large */
#define RC_ERR_NO_DEVICE (-3)    /* no CUDA device, or not compute capability 10.x */
#define RC_ERR_NO_WORKSPACE (-4) /* workspace missing or smaller than rc_workspace_bytes */
#define RC_ERR_BAD_VALUE (-5)    /* bad config value; or (RC_VALIDATE) negative / non-finite chi or eta */
#define RC_ERR_CUDA (-6)         /* a CUDA runtime call failed; see rc_last_error */
#define RC_ERR_NO_ATMOSPHERE (-7)

#define RC_MAX_CASCADES 12
#define RC_MAX_DIM 16384

/* rc_config.flags */
#define RC_ACCUM_J 1   /* J_out is Jbar[ny][nx] = sum_l w_l J_l (rc_set_lambda_weights) */
#define RC_VALIDATE 2  /* rc_set_atmosphere checks chi, eta on the device (synchronises) */
#define RC_NO_EARLY_EXIT 4 /* never stop a ray early.  Default: a warp stops marching once every live
                              lane has tau*log2(e) > 126 at all its wavelengths, where the fp32
                              transmittance has already flushed to exactly 0, so the result is
                              bit-identical (front-to-back early termination) */

#define RC_BILINEAR_FIX 8 /* the bilinear fix: every interval below the top
                             cascade is traced four times, from its usual start to the start of the child cone on
                             each of the four parent probes, merged with that parent alone and then weighted
                             bilinearly: removes most of the ringing around bright compact sources at 4x the rays */

typedef struct rc_ctx rc_ctx; /* opaque, owned by the library */

typedef struct {
    int ncascades;     /* 1..RC_MAX_CASCADES */
    float c0_interval; /* length of the cascade-0 interval in cells; > 0; the configs use 1 */
    int device;        /* CUDA ordinal */
    int lambda_batch;  /* wavelengths per thread (1, 2, 4 or 8); 0 = library chooses */
    int flags;         /* RC_ACCUM_J | RC_VALIDATE | RC_NO_EARLY_EXIT | RC_BILINEAR_FIX */
} rc_config;

typedef struct {
    int ncascades;
    int lambda_batch;                     /* wavelengths per thread actually used */
    int kernel_launches;                  /* kernels enqueued by the last rc_solve_J */
    int solves_timed;                     /* solves the ms_* figures average over (rc_set_timing) */
    float ms_pack[RC_MAX_CASCADES];       /* mean device ms of cascade i's pack kernel  */
    float ms_march[RC_MAX_CASCADES];      /* mean device ms of cascade i's march+merge kernel */
    float ms_total;                       /* mean device ms of a whole solve */
    int64_t rays[RC_MAX_CASCADES];        /* intervals per cascade per wavelength = 4 nx ny */
    int64_t table_steps[RC_MAX_CASCADES]; /* step-table entries per cascade (all directions) */
    size_t workspace_bytes;
    int64_t empty_cells;                  /* cells that are not flagged, or hold chi == 0 and eta == 0 at every wavelength
                                             (counted by rc_analyse_atmosphere; 0 before) */
    int sparse_march;                     /* the march walks the distance field (rc_analyse_atmosphere found > 2/3 empty) */
    int64_t active_cells;                 /* cells of interest (rc_set_active_cells); -1 = every cell */
    int64_t probes_flagged[RC_MAX_CASCADES]; /* with active cells: flagged probes of cascade i */
    int sparse_lists;                     /* the sparse march runs over hit lists (rc_set_sparse_workspace was large enough): 1 = built by
                                             the last rc_analyse_atmosphere, 2 = kept from an earlier one (same occupancy map) */
    int64_t sparse_list_bytes;            /* bytes the hit lists of the analysed atmosphere need in that buffer (0: not sparse) */
} rc_stats;

/* The launch plan the library would use for a problem, computed on the host alone (no device, no context):
 * what the tests of the host logic and capacity planning read. */
typedef struct {
    size_t workspace_bytes;            /* = rc_workspace_bytes(..., host_io = 0) for the same arguments */
    int lambda_batch;                  /* wavelengths per thread */
    int channels;                      /* lambda_batch x inclinations carried by one thread (<= 8) */
    int nbatches;                      /* wavelength batches per launch */
    int nbands, band_axis;             /* L2 banding: bands (1 = none) along rows (0) or columns (1) */
    int cascade_empty[RC_MAX_CASCADES];   /* interval wholly outside any box of this size: boundary term only */
    int cascade_banded[RC_MAX_CASCADES];  /* marched band by band */
    int patch_w[RC_MAX_CASCADES];      /* a warp's 32 probes form a patch patch_w wide, 32 / patch_w high */
    int cascade_sorted[RC_MAX_CASCADES];  /* instead: 8 quads of 4 x-adjacent probes from a list sorted by ray length */
    float lane_utilisation[RC_MAX_CASCADES]; /* estimated share of a warp's lock-step lane-steps that are inside the box */
    int64_t table_steps[RC_MAX_CASCADES]; /* step-table capacity, all directions (x16 with RC_BILINEAR_FIX) */
} rc_plan_info;

/* cfg->device is ignored.  line_mode != 0: rc_set_line_atmosphere.  RC_ERR_BAD_SHAPE / RC_ERR_BAD_VALUE as the
 * calls it mirrors. */
int rc_plan_query(const rc_config *cfg, int ninclinations, int line_mode, int nx, int ny, int nlambda, rc_plan_info *out);

/* Create a context on cfg->device for the cascade hierarchy of PAPER.md:171-181 (eq. 12-13, alpha = 2): cfg->ncascades
 * cascades, cascade-0 interval cfg->c0_interval cells (1 in BASELINE.json's configs).  Fails with RC_ERR_NO_DEVICE unless
 * that device is sm_100; RC_ERR_BAD_VALUE for a bad config.  Allocates host memory only. */
int rc_create(rc_ctx **out, const rc_config *cfg);

/* Bytes of device workspace rc_solve_J needs for an nx x ny x nlambda atmosphere (0 on bad shape).
 * host_io != 0 adds room for the device copies rc_solve_J_host makes of chi, eta and J. */
size_t rc_workspace_bytes(const rc_ctx *ctx, int nx, int ny, int nlambda, int host_io);  /* enough for rc_set_atmosphere and rc_set_line_atmosphere alike */

/* Caller-owned device workspace (256-byte aligned), borrowed. */
int rc_set_workspace(rc_ctx *ctx, void *dev_ptr, size_t bytes);

/* Caller-owned CUDA stream (cudaStream_t as void*; NULL = the legacy default stream). */
int rc_set_stream(rc_ctx *ctx, void *cuda_stream);

/* Launch knobs, for measurements and tests (none changes a result beyond rounding, except tau_cut < 126).  Call before
 * rc_set_atmosphere: it drops the atmosphere and the active cells (plan, patch lists and captured graph may depend on a
 * knob).  name / value:
 *   "march_variant" -1 | 0..4   register-ring depth and occupancy of the march (-1: chosen per cascade)
 *   "patch_log2"    -1 | 2..5   lane patch width 2^n for cascades >= "patch_from" (-1: chosen per cascade from the geometry)
 *   "pipeline"      0 | 1       rc_solve_J_host in two halves of the wavelength batches with overlapped copies (default 1)
 *   "lists"         0 | 1       hit lists for the sparse march when rc_set_sparse_workspace lends room (default 1)
 *   "list_b"        0 | 1,2,4,8 wavelength batches per warp of the march over hit lists (0: from the L2 footprint of the occupied cells)
 *   "sorted"        -1 | 0 | 1  lanes from quads of probes sorted by ray length: where the geometry says it pays / never / wherever possible
 *   "cpw_from"      -1 | i      cascades >= i run one child direction per warp (-1: never; default 3)
 *   "bands" n, "l2_mb" x        L2 banding of grids whose wavelength batch exceeds L2: n bands (0: from the budget x, 72 MB)
 *   "sparse"        -1 | 0 | 1  distance-field march after rc_analyse_atmosphere: automatic (> 2/3 empty) / never / always
 *   "sparse_mode"   0..3        that march in blocks of 8 / 4 / 2 warps at <= 80 registers, or (3) 4 warps at <= 128
 *   "graph"         0 | 1       CUDA graph replay on small grids
 *   "tau_cut"       x >= 1      early-exit threshold on tau log2 e; below 126 it drops transmittances below 2^-x
 * RC_ERR_BAD_VALUE for an unknown name or a value out of range. */
int rc_set_tuning(rc_ctx *ctx, const char *name, double value);

/* chi, eta: device, [ny][nx][nlambda] float32, borrowed.  Builds the per-direction step tables for
 * this grid size (device kernels, fp64 geometry) if the shape changed; needs the workspace set.
 * With an unchanged shape the call only records the pointers: no device work, no synchronisation (the iteration of
 * PAPER.md:316-342 calls it once per formal solution).  PAPER.md:409. */
int rc_set_atmosphere(rc_ctx *ctx, const float *chi, const float *eta, int nx, int ny, int nlambda);

/* Velocity-dependent line mode ("velocity-dependent terms (spectral lines) are computed on the
 * fly for each ray given its specific direction, and thus projected plasma velocity"),
 * instead of rc_set_atmosphere.  line: device, [ny][nx][6] float32, borrowed: chi_c, S_c (continuum opacity
 * and source function), chi_line, S_line (line opacity scale and source function), v_x, v_y (bulk velocity in
 * Doppler widths).  x_lambda: host, [nlambda], wavelength offsets from line centre in Doppler widths.  For a
 * ray traced from its probe in direction w the photons travel along -w, and in every cell
 *     a = x_l + v.w,  phi = exp(-a^2)/sqrt(pi),  chi = chi_c + chi_line phi,  eta = chi_c S_c + chi_line S_line phi
 * enter eq. 16.  With inclinations set (rc_set_inclinations, before this call) the velocities are taken to lie
 * in the plane: inclination m sees v.w sqrt(1 - mu_m^2) over the path ds / sqrt(1 - mu_m^2).  rc_solve_J,
 * rc_set_boundary, rc_set_lambda_weights, RC_ACCUM_J work as usual; host buffers: rc_solve_J_line_host. */
int rc_set_line_atmosphere(rc_ctx *ctx, const float *line, int nx, int ny, const float *x_lambda, int nlambda);

/* Sparsity as the paper defines it (§3.5): "we can first determine the cells of
 * interest ...  This flag then defines the probes of cascade 0 that may be involved ... Their bilinear "parents" are
 * recursively flagged up to the maximum cascade, and the radiance intervals are only computed for these flagged probes,
 * and non-flagged cells are treated as transparent with no emission."  active: device, [ny][nx] bytes, non-zero = cell
 * of interest; copied (not borrowed).  NULL = every cell (the default).  Afterwards J_out holds J on the flagged cells
 * and 0 on the others, whatever chi, eta hold there; probe patches without a flagged probe launch no warp.  Call
 * after rc_set_atmosphere; stays in force for later atmospheres of the same shape; synchronises the stream (the
 * number of flagged patches sizes the launches). */
int rc_set_active_cells(rc_ctx *ctx, const unsigned char *active);

/* Free-space acceleration ("accelerating the traversal of long-range radiance intervals through
 * free-space"): scans the current atmosphere (and flags) for empty cells - not flagged, or chi == eta == 0 at every
 * wavelength - and builds their Chebyshev distance transform.  When more than two thirds of the cells are empty the
 * march of the next solves lets every lane walk its own ray and jump over empty space; the result is bit-identical
 * to the lock-step march.  Explicit because it synchronises the stream and belongs to one atmosphere: the next
 * rc_set_atmosphere / rc_set_line_atmosphere / rc_set_active_cells switches it off again (rc_solve_J_host repeats it
 * by itself once it has been used on the context).  Not with the bilinear fix (there it only counts); with inclinations
 * or the moving line only through the hit lists of rc_set_sparse_workspace.  rc_stats.empty_cells, rc_stats.sparse_march
 * report the outcome. */
int rc_analyse_atmosphere(rc_ctx *ctx);

/* A second caller-owned device buffer (256-byte aligned, borrowed; NULL takes it back) for the HIT LISTS of the sparse
 * march: which steps of a ray meet an occupied cell depends on the geometry and the occupancy alone, so
 * rc_analyse_atmosphere can find them once - per cascade and ray the numbers of its occupied in-box steps - instead of the
 * march finding them again for every wavelength batch of every solve; the march then only gathers and integrates (the same
 * cells in the same order: bit-identical).  Their size is only known after counting: rc_analyse_atmosphere always counts
 * and reports rc_stats.sparse_list_bytes; when this buffer is missing or smaller the distance-field march stays in use
 * (rc_stats.sparse_lists = 0) - lend at least that many bytes and analyse again.  The lists are kept across atmospheres
 * of the same shape and flags for as long as rc_analyse_atmosphere finds the same occupancy map (the formal solutions of an
 * iteration change chi and eta, not where they vanish): the analysis then costs one scan.  Config 4: 3.6 GB, 435 -> 124 ms per solve. */
int rc_set_sparse_workspace(rc_ctx *ctx, void *dev_ptr, size_t bytes);

/* Boundary intensity sampled by the top cascade: I_below[l] is seen by rays heading
 * down (omega_y < 0), I_above[l] by rays heading up.  host, [nlambda] each; NULL = 0 (free space,
 * PAPER.md:371).  Call after rc_set_atmosphere. */
int rc_set_boundary(rc_ctx *ctx, const float *I_below, const float *I_above);

/* The same with one value per inclination (after rc_set_inclinations and rc_set_atmosphere): host,
 * [ninclinations][nlambda] each, NULL = 0 - the "table of emergent intensity ... as a function of inclination
 * and wavelength" of PAPER.md:374 in the plane-parallel reading G9 (e.g. a limb-darkened disc below). */
int rc_set_boundary_inclined(rc_ctx *ctx, const float *I_below, const float *I_above);

/* 2.5D inclination quadrature: the model is taken homogeneous along
 * the axis perpendicular to the grid, and every flatland ray is replaced by n rays with the same
 * projection and direction cosine mu[m] to that axis (0 <= mu < 1): the same cells, path lengths
 * ds / sqrt(1 - mu^2).  J_l = sum_m w[m] * (mean over the 4 merged cascade-0 directions of inclination m);
 * the weights should sum to 1 (one hemisphere; the other is its mirror image).  The boundary intensities
 * of rc_set_boundary apply to every inclination.  n = 1, 2, 4 or 8; mu, w: host, [n]; n = 1 with
 * mu = w = NULL restores flatland (the default).  Call BEFORE rc_workspace_bytes / rc_set_atmosphere:
 * it changes the workspace size (merged cascades hold n x nlambda channels) and drops the atmosphere. */
int rc_set_inclinations(rc_ctx *ctx, int n, const float *mu, const float *w);

/* Wavelength weights for RC_ACCUM_J: Jbar = sum_l w_l J_l (J of PAPER.md:36, eq. 1, summed over the wavelength grid:
 * "to correctly integrate J and the necessary radiative rates", and the wavelength integration of
 * PAPER.md:359; BASELINE.json configs[4]: "J accumulated across all wavelengths per solve").  host, [nlambda], copied;
 * NULL = all 1.  After rc_set_atmosphere; synchronises. */
int rc_set_lambda_weights(rc_ctx *ctx, const float *w);

/* Enqueue one full solve.  J_out: device, [ny][nx][nlambda] float32, or [ny][nx] with RC_ACCUM_J. */
int rc_solve_J(rc_ctx *ctx, float *J_out);

/* Diagonal approximate lambda operator (eq. 17): for the current
 * atmosphere (either mode) and inclination set, Lambda*[y][x][l] = sum_m w_m <exp(-chi_l ds_m)> over the four
 * cascade-0 directions, ds_m = (sqrt2/2) / sqrt(1 - mu_m^2) the path from the cell centre to its edge.  "Purely
 * local ... only computed for cascade 0": an elementwise launch on the context's stream, not synchronised.
 * alo_out: device, [ny][nx][nlambda] float32. */
int rc_compute_alo(rc_ctx *ctx, float *alo_out);

/* Same path with HOST buffers: copies chi, eta to the device (workspace, host_io != 0), solves,
 * copies J back, synchronises the stream.  Pinned host memory makes the copies asynchronous; large dense solves
 * then run as two halves of the wavelength batches (wavelengths are independent) on the context's stream
 * while a private stream moves the other half's inputs and results (same arithmetic, same J). */
int rc_solve_J_host(rc_ctx *ctx, const float *chi_host, const float *eta_host, int nx, int ny,
                    int nlambda, float *J_host);

/* The line mode with HOST buffers: line_host [ny][nx][6] (host), x_lambda as rc_set_line_atmosphere, J_host as
 * rc_solve_J_host; the workspace must have been sized with host_io != 0.  Copies, solves, copies back, synchronises. */
int rc_solve_J_line_host(rc_ctx *ctx, const float *line_host, int nx, int ny, const float *x_lambda, int nlambda, float *J_host);

/* nsets > 0: the next solves record CUDA events on the context's stream around every kernel, solve
 * number n into event set n % nsets (no synchronisation is added); 0 switches timing off.
 * rc_get_stats waits for the recorded sets and averages over them. */
int rc_set_timing(rc_ctx *ctx, int nsets);
/* Per-cascade work and timing of the last solves (every cascade has 4 nx ny intervals; PAPER.md:545-552:
 * the upper cascades are the cost): rays, table sizes, mean pack / march milliseconds per cascade over the recorded
 * event sets, flagged probes, empty cells.  Waits for the recorded events (hence the non-const context). */
int rc_get_stats(rc_ctx *ctx, rc_stats *out);

/* Geometric work of one solve, the unit of the throughput metric: per_cascade[i] (host,
 * [ncascades]) = number of (probe, direction) cell segments of cascade i inside the box, per
 * wavelength.  Counted on the device from the step tables; synchronises. */
int rc_count_segments(rc_ctx *ctx, int64_t *per_cascade);

/* One solve into J_out (device, as rc_solve_J) that also counts the cell segments the march actually integrated, per
 * cascade and wavelength (host, [ncascades]; the mean over the wavelength batches): the early exit of opaque rays
 * (PAPER.md:308), unflagged probes and the jumps over free space leave the rest of rc_count_segments'
 * geometric count unwalked.  Synchronises. */
int rc_count_walked(rc_ctx *ctx, float *J_out, int64_t *per_cascade);

/* Measurement aid for the roofline: achieved GB/s (*gbs, host) of the access pattern the
 * march gathers with and nothing else - every warp reads pseudo-random 1 KB runs (32 lanes x 32 B), 48
 * warps per SM - over the first `mbytes` MB of the workspace (read only; contents irrelevant).  A region
 * that fits the 126 MB L2 gives the L2 -> SM gather ceiling, a larger one the HBM gather ceiling.
 * Runs on the context's stream and synchronises it.  RC_ERR_BAD_VALUE if the region does not fit. */
int rc_probe_gather_bandwidth(rc_ctx *ctx, int mbytes, double *gbs);

/* The same pattern staged through shared memory by the TMA bulk-copy engine (per warp a ring of 4 stages x
 * 2 KB filled by `cp.async.bulk` 1 KB copies completing on mbarriers, read back with LDS.128; 24 warps per SM):
 * the alternative design DESIGN.md §7 measures the LDG path against.  Same arguments and errors. */
int rc_probe_bulk_copy_bandwidth(rc_ctx *ctx, int mbytes, double *gbs);

/* ---- For callers that cannot allocate device memory at all --------------------------------------------------------
 * Every call above works out of memory the caller lends.  Some callers have none to lend and no way to get any: a
 * plug-in living inside an application whose own pool claimed the whole GPU at start-up (cudaMalloc just fails there), a
 * stage of a real-time or serving loop that bans cudaMalloc / cudaFree because they stall the whole device, a tool that
 * is handed two arrays and nothing else.  For them ONE operation is offered with its scratch memory built into the
 * library image: the empty-cell count on which rc_analyse_atmosphere bases its "is this atmosphere sparse" decision
 * (free-space acceleration; more than two thirds empty = the free-space march pays).
 *
 * Writes to *nempty_out the number of cells of the nx x ny grid that are NOT (of interest and non-zero in chi or eta at
 * some wavelength) - the same number rc_stats.empty_cells reports after an analysis.
 *   device      CUDA ordinal the arrays live on; made current for the calling thread, like every call of this library
 *   chi, eta    device, [ny][nx][nlambda] float32, read only (no alignment demanded; 16-byte aligned is faster)
 *   active      device, [ny][nx] bytes, non-zero = cell of interest; NULL = every cell
 *   nempty_out  device, one 64-bit counter, the caller's; written by the kernel: read it after the stream has caught up
 *   cuda_stream cudaStream_t as void*; the call only enqueues (one memset, one kernel) and does not synchronise
 *   errbuf      host, errbuf_len bytes, or NULL: receives the text of a failure (there is no context to ask)
 * Returns RC_OK, RC_ERR_NULL_ARG, RC_ERR_BAD_SHAPE (also: nx * ny > RC_STATIC_MAX_CELLS - the built-in array is that
 * large and no larger), RC_ERR_NO_DEVICE (not an sm_100 device), RC_ERR_CUDA.
 *
 * What to know about the built-in array (about 4 MiB): every GPU that loads librc.so holds it until the process exits,
 * whether or not this call is ever made.  The first call on a device looks its address up once
 * (cudaGetSymbolAddress); make that first call before any stream capture begins.  No call allocates or frees anything, on the
 * device or through a library that might.  ALL calls share the array and each one starts by clearing the part it
 * uses, so the previous call's contents never leak into a result - but two calls that overlap on the GPU (different
 * streams, different threads, different contexts of this library in one process) race on it and both results are
 * garbage: keep calls on one stream or order them with events. */
#define RC_STATIC_MAX_CELLS (1 << 20) /* 1024 x 1024, 4096 x 256, ... */
int rc_count_empty_cells_static(int device, const float *chi, const float *eta, const unsigned char *active, int nx, int ny,
                                int nlambda, unsigned long long *nempty_out, void *cuda_stream, char *errbuf, size_t errbuf_len);

const char *rc_last_error(const rc_ctx *ctx);
const char *rc_version(void);
int rc_destroy(rc_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* RC_H_ */
