/*
 * nyxrt.h -- C ABI of the B200-native adaptive ray-tracing step (one RT step on the coarse grid) of
 * Nyx-RT, arxiv 2512.12466.  Citations are lines of /root/reference/PAPER.md ("PAPER.md:<line>");
 * readings R1..R42 and H1 of the paper's silent / garbled spots are listed in DESIGN.md.
 *
 * The step ("Ray tracing loop", Figs. 1-2 at PAPER.md:120-124; Sec. 2.8 at 295-391):
 *   source dedup + sort -> [bubble radius -> merge] -> emit 12 HEALPix rays per source ->
 *   { march cell by cell and deposit (Eq. 1-2, Eq. 5-8) -> filter -> split into 4 children } until no
 *   ray is left -> finalise Gamma_HI and the heating rate.
 *
 * Conventions
 *   - Every function returns NYXRT_OK (0) or a negative NYXRT_E* code; the message is available from
 *     nyxrt_last_error().  Nothing throws, aborts or prints.
 *   - "device pointer" = CUDA device memory on the context's device; "host pointer" = ordinary host
 *     memory.  Nothing in a signature is a torch (or any other framework's) type.
 *   - Grids are dense [nz][ny][nx], x fastest: index = (k*ny + j)*nx + i.
 *   - Streams are cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - A context is not thread-safe; use one per host thread / per grid.
 *   - There is no CPU fallback: without a CUDA device nyxrt_create fails with NYXRT_ECUDA.
 */
#ifndef NYXRT_H
#define NYXRT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NYXRT_OK          0
#define NYXRT_EINVAL     -1   /* bad argument (incl. a source outside the box, L < 0, NaN)         */
#define NYXRT_ESTATE     -2   /* call order: fields / sources / workspace not set                  */
#define NYXRT_ENOMEM     -3   /* workspace too small (see nyxrt_workspace_bytes)                   */
#define NYXRT_ECUDA      -4   /* a CUDA call failed; message holds cudaGetErrorString              */
#define NYXRT_EOVERFLOW  -5   /* ray pool overflow or HEALPix level > 14; never silent truncation  */

#define NYXRT_MAXLEV 16

/* nyxrt_params.flags */
#define NYXRT_FLAG_LAUNCH_TIMING 1   /* profiling mode: the ray loop is enqueued launch by launch from the host with a
                                        pair of CUDA events around every march launch (stats ms_march); without it the
                                        loop runs as one CUDA-graph launch (a WHILE node over sched -> emit -> march) and
                                        ms_march is 0.  Same kernels, same results. */

typedef struct nyxrt_ctx nyxrt_ctx;      /* opaque */

/* The coarse RT grid ("downsampled onto a coarse grid"; cubic cells). */
typedef struct {
    int32_t nx, ny, nz;        /* cells per axis, each 1..2^20 and nx*ny*nz < 2^40                  */
    int32_t field_dtype;       /* 0 = fp64 fields, 1 = fp32 fields (converted on load, exact)       */
    double  dx_cm;             /* cell width h in cm; V_box = h^3 (PAPER.md:205 footnote 2)         */
    double  box_lo[3];         /* position of the low corner of cell (0,0,0), in position units     */
    double  pos_unit_cm;       /* cm per position unit of nyxrt_set_sources (dx_cm => cell units)    */
    int32_t periodic;          /* 0: rays die on leaving the box (BASELINE.json configs; R20);
                                  1: periodic box: cells wrap, a ray ends once its travel
                                  distance reaches sqrt(nx^2+ny^2+nz^2) cells (= sqrt(3) L_box, PAPER.md:174;
                                  counted in exited[] / photons_escaped, R30), minimum-image merge and wrapped
                                  shell samples (tie rule R31)                */
    int32_t device;            /* CUDA device ordinal                                               */
} nyxrt_grid;

/* User parameters; names follow the paper's symbols.  Defaults: DESIGN.md "Parameters". */
typedef struct {
    double  sigma_cm2;         /* monochromatic H I cross-section (6.3e-18)                         */
    double  n_min_ray;         /* N_min^ray of Eq. 4, PAPER.md:113-116 (3; paper production: 2)     */
    double  tau_max;           /* RAY_FLTR optical-depth threshold, PAPER.md:128, 174 (ln 1e8)      */
    double  n_th;              /* low-density neighbour threshold of Eq. 7-8      */
    double  e_excess_erg;      /* heating per photo-ionisation (reading H1; 0 at 13.6 eV)           */
    double  automerge_xmean;   /* merge==2: merge once mean ionised fraction exceeds this (0.018)   */
    double  delta_r;           /* Alg. 3 shell spacing in cells, PAPER.md:313 (2)                   */
    double  r_max;             /* Alg. 3 R_max in cells                               */
    double  f_ov;              /* overlap factor                                  */
    double  x_th;              /* ionised threshold of a sample                       */
    double  f_req;             /* required ionised share of a shell                   */
    double  eps;               /* tolerance of the link test                      */
    int32_t level_max;         /* l_max of RAY_FLTR, PAPER.md:174 (<= 13)                           */
    int32_t geom_mode;         /* 0 none, 1 Eq.5 only, 2 Eq.5-6, 3 Eq.7-8 (default), 4 squared [59] */
    int32_t merge;             /* 0 off, 1 on, 2 automerge                           */
    int32_t n_min_samples;     /* N_min of PAPER.md:317                                             */
    int32_t samp_level;        /* HEALPix level of the shell sample pattern, 12*4^level dirs (R6)   */
    int32_t flags;             /* NYXRT_FLAG_* (0: production)                                      */
} nyxrt_params;

/* Filled by nyxrt_trace (host memory).  Per-level arrays are indexed by HEALPix level l. */
typedef struct {
    uint64_t spawned[NYXRT_MAXLEV];      /* rays created at level l (12 per source at l = 0)        */
    uint64_t split[NYXRT_MAXLEV];        /* rays that met Eq. 4 and became 4 children               */
    uint64_t killed_tau[NYXRT_MAXLEV];   /* rays filtered by tau >= tau_max                         */
    uint64_t exited[NYXRT_MAXLEV];       /* rays that left the box                                  */
    uint64_t killed_lmax[NYXRT_MAXLEV];  /* rays filtered by l >= l_max                             */
    uint64_t segments;                   /* ray-cell segments of positive length (the work unit)    */
    uint64_t zero_len_segments;          /* cell crossings of zero length (edge / corner hits)      */
    uint64_t neighbour_deposits;         /* segments whose nearest neighbour cell received a share
                                            (Eq. 6 / 8): the second gather + deposit */
    uint64_t n_src_in, n_src_dedup, n_src_merged;
    uint64_t iterations;                 /* march launches (diagnostic; not part of parity)         */
    uint64_t peak_pool_rays;             /* max rays resident in the pool (diagnostic)              */
    double   photons_emitted;            /* sum of catalogue L [s^-1]                               */
    double   photons_absorbed;           /* sum over cells of deposited photons [s^-1]              */
    double   photons_escaped;            /* carried out of the box                                  */
    double   photons_residual;           /* left in rays filtered by tau_max / l_max                */
    double   photons_lost;               /* geom_mode 1 and 4 only (no secondary correction)        */
    uint64_t march_launches;             /* march launches that had rays (== iterations)            */
    uint64_t kernel_launches;            /* launches of this library's own kernels in the call      */
    float    ms_sources, ms_loop, ms_finalise, ms_total;   /* CUDA-event times of the phases        */
    float    ms_march;                   /* sum of the march launches' own durations (CUDA events)  */
    float    pad_;
} nyxrt_stats;

/* Create a context for one grid.  Copies *grid and *params.  Allocates only small bookkeeping
 * (host + a few KB device).  Errors: EINVAL (bad sizes / parameters, periodic not 0 or 1), ECUDA. */
int nyxrt_create(const nyxrt_grid *grid, const nyxrt_params *params, nyxrt_ctx **out);

/* Size of the caller-provided device workspace.
 *   max_sources     upper bound of n in nyxrt_set_sources
 *   batch_rays      rays marched per launch B (0 = default: 2^23 from 2^29 cells, 2^22 from 2^26 cells, else 2^21); the ray pool holds
 *                   (2 + 5*(level_max+1)) * B rays of 32 bytes
 *   host_staging    non-zero: add room for the fields and outputs of nyxrt_step_host
 * Workspace layout is private.  Errors: EINVAL. */
int nyxrt_workspace_bytes(const nyxrt_ctx *ctx, int64_t max_sources, int64_t batch_rays, int32_t host_staging,
                          uint64_t *bytes);

/* Hand the library its workspace (device pointer, 256-byte aligned, owned by the caller, must stay
 * valid until nyxrt_destroy or the next nyxrt_set_workspace).  The same max_sources / batch_rays /
 * host_staging as in nyxrt_workspace_bytes.  Errors: EINVAL, ENOMEM (bytes too small). */
int nyxrt_set_workspace(nyxrt_ctx *ctx, void *d_workspace, uint64_t bytes, int64_t max_sources,
                        int64_t batch_rays, int32_t host_staging);

/* Register the fields of this step: total hydrogen density n_H [cm^-3] and NEUTRAL fraction x_HI
 * (absorber density a_abs = x_HI n_H, PAPER.md:229 with x_HI = 1 - x; reading R1), device pointers of
 * grid.field_dtype, layout [nz][ny][nx].  Borrowed until the next nyxrt_set_fields / nyxrt_destroy.
 * Enqueues on `stream` the kernel that builds the internal absorber field; does not synchronise.
 * Values are not validated (n_H < 0, x_HI outside [0,1], NaN: garbage in, garbage out).
 * Errors: EINVAL (NULL), ESTATE (no workspace), ECUDA. */
int nyxrt_set_fields(nyxrt_ctx *ctx, const void *d_nH, const void *d_xHI, void *cuda_stream);

/* Set the point sources of this step: host pointers, pos_xyz is [n][3] in
 * position units, L is [n] photons/s.  Copied; validated on the device: a source outside the box,
 * L < 0, NaN or inf -> EINVAL and the previous source list is dropped.  Synchronises `stream`.
 * Errors: EINVAL, ESTATE (no workspace), ENOMEM (n > max_sources), ECUDA. */
int nyxrt_set_sources(nyxrt_ctx *ctx, int64_t n, const double *pos_xyz, const double *L, void *cuda_stream);

/* Run one RT step.  d_gamma_HI (required) and d_heat (may be NULL) are device pointers to
 * [nz][ny][nx] doubles, overwritten:
 *   Gamma_HI [s^-1 per H I atom] = photons absorbed in the cell / (n_HI V)      (Eq. 1)
 *   heat [erg s^-1 cm^-3]        = e_excess * photons absorbed in the cell / V   (reading H1)
 * A cell that received nothing holds exactly 0.  All work is enqueued on `stream`; the call
 * synchronises that stream before filling *h_stats (host pointer, may be NULL).
 * Errors: ESTATE (fields / sources / workspace missing), EOVERFLOW, ECUDA. */
int nyxrt_trace(nyxrt_ctx *ctx, double *d_gamma_HI, double *d_heat, nyxrt_stats *h_stats, void *cuda_stream);

/* Frequency-integrated flux (Sec. 2.2: Eq. 1 "precomputed as a function of tau_0 ... a lookup
 * table"; cross-section sigma_nu = sigma_cm2 (nu/nu_0)^-3, R37).  The table holds the absorbed fraction
 *     Q(tau_0) = int phi(nu) (1 - exp(-tau_0 (nu/nu_0)^-3)) dnu,   phi = photon-number spectrum, int phi = 1,
 * of a ray's share between the source and threshold optical depth tau_0; a segment from tau_0 = a to b absorbs
 * share * [Q(b) - Q(a)] photons (Eq. 1's numerator; telescopes along the ray).  Nodes are fixed by the binary
 * representation of tau_0 (R38): node k = 2^(e_lo + (k >> m)) * (1 + (k mod 2^m) / 2^m), k = 0 .. (e_hi - e_lo) 2^m;
 * Q is linear in tau_0 between nodes, linear from 0 below 2^e_lo, constant above 2^e_hi.
 *   nyxrt_spectrum_nodes      number of nodes n (m <= 16, n <= 2^24)
 *   nyxrt_spectrum_node_tau   tau_0 of node k
 *   nyxrt_set_spectrum        h_q: host array of n values, non-decreasing in [0, 1]; copied to the device
 *                             (a small cudaMalloc owned by the context).  h_q = NULL: monochromatic again
 *                             (the default: Q = 1 - e^-tau evaluated in the kernel).  Needs geom_mode 2 or 3.
 *                             Choose tau_max (nyxrt_params) for the spectrum: hard photons outlive tau_0 = ln 1e8.
 *   nyxrt_blackbody_table     fills h_q with Q of a black body of temperature t_eff_K above 13.6 eV (R39)
 * Heating stays e_excess_erg per absorbed photon (H1).  A call that fails changes nothing: the Q table and the thin
 * table set before stay active (a successful call with a new Q table, or h_q = NULL, drops the thin table).
 * Errors: EINVAL, ECUDA. */
int nyxrt_spectrum_nodes(int32_t e_lo, int32_t e_hi, int32_t m, int64_t *n);
int nyxrt_spectrum_node_tau(int32_t e_lo, int32_t m, int64_t k, double *tau);
int nyxrt_set_spectrum(nyxrt_ctx *ctx, int32_t e_lo, int32_t e_hi, int32_t m, const double *h_q, int64_t n);
int nyxrt_blackbody_table(double t_eff_K, int32_t e_lo, int32_t e_hi, int32_t m, double *h_q, int64_t n);

/* The separate table for the optically thin case (PAPER.md:267 footnote 3: "the approach of C2-Ray, which takes the
 * limit as n_H -> 0 to compute a separate LUT for the optically thin case"; readings R40-R42).  In a thin cell Eq. 1's
 * (1 - exp(-dtau_nu)) -> dtau_nu, so the cell absorbs share * dtau_0 * T(tau_0) with
 *     T(tau_0) = int phi(nu) (nu/nu_0)^-3 exp(-tau_0 (nu/nu_0)^-3) dnu = dQ/dtau_0,
 * on the nodes of the Q table set before (same n), linear between nodes, constant below the first and above the last.
 * A segment with dtau_0 < tau_thin absorbs share * dtau_0 * T(tau_0 + dtau_0 / 2) instead of the difference of two
 * interpolated Q values; the photons a ray carries are then counted down segment by segment (the two forms do not
 * telescope into each other).  The neighbour's share of Eq. 6 / 8 is (1 - f_c) of the absorbed photons either way.
 *   nyxrt_set_spectrum_thin    h_t: host array of n values >= 0, copied (h_t = NULL: thin table off).  A later
 *                              successful nyxrt_set_spectrum drops it; a failed call of either function leaves the
 *                              tables as they were.  Errors: EINVAL, ESTATE (no Q table), ECUDA.
 *   nyxrt_blackbody_thin_table T of a black body of temperature t_eff_K above 13.6 eV on the given nodes. */
int nyxrt_set_spectrum_thin(nyxrt_ctx *ctx, const double *h_t, int64_t n, double tau_thin);
int nyxrt_blackbody_thin_table(double t_eff_K, int32_t e_lo, int32_t e_hi, int32_t m, double *h_t, int64_t n);

/* Source sharding across GPUs: Gamma is a sum over sources, so
 * each of `world` processes, holding a full replica of the fields and the full source list, traces the
 * catalogue entries rank, rank + world, ... (the catalogue -- dedup, merge, sort -- is computed by every
 * process, identically), the per-cell photon counts are summed across processes (one all-reduce, done by the
 * caller, e.g. torch.distributed over NCCL) and nyxrt_finalise turns the sum into rates:
 *   nyxrt_set_shard(rank, world); nyxrt_trace_photons(d_photons); all-reduce(d_photons); nyxrt_finalise(d_photons, ...)
 * With a shard set (world > 1), nyxrt_trace / nyxrt_step_host / nyxrt_timestep return ESTATE.
 * nyxrt_set_shard(0, 1) restores the default.  Errors: EINVAL. */
int nyxrt_set_shard(nyxrt_ctx *ctx, int32_t rank, int32_t world);

/* nyxrt_trace up to, not including, the division by n_HI V: d_photons (device, [nz][ny][nx] doubles) receives
 * the photons absorbed per cell per second from this shard's sources.  *h_stats counts this shard's rays;
 * n_src_* describe the whole catalogue.  Errors: as nyxrt_trace. */
int nyxrt_trace_photons(nyxrt_ctx *ctx, double *d_photons, nyxrt_stats *h_stats, void *cuda_stream);

/* Gamma_HI and heating (may be NULL) from a dense photon grid (device pointers), as nyxrt_trace's last stage;
 * *h_absorbed (host, may be NULL) = sum of d_photons.  Needs the fields of the trace still registered.
 * Synchronises `stream`.  Errors: EINVAL, ESTATE, ECUDA. */
int nyxrt_finalise(nyxrt_ctx *ctx, const double *d_photons, double *d_gamma_HI, double *d_heat, double *h_absorbed,
                   void *cuda_stream);

/* nyxrt_finalise for callers that must not allocate device memory: no context, no workspace, no cudaMalloc /
 * cudaFree / cudaMallocHost and no library routine that allocates, on any call.
 *
 * Why it exists.  The library is meant to run inside a host code that owns the GPU's memory: Nyx's AMReX arena
 * (or, under the Python binding, PyTorch's caching allocator) has usually taken nearly all of it, so a cudaMalloc
 * made from here can fail while the host code still has free blocks, and every cudaMalloc / cudaFree stalls all
 * streams of the device.  The other entry points need a context (a few small allocations in nyxrt_create) and a
 * workspace the caller allocates.  A caller that can afford neither -- e.g. a rank that only turns the all-reduced
 * photon grid of a source-sharded step into rates, or a diagnostic run between two kernels of a time step -- calls
 * this instead.
 *
 * What it computes (Eq. 1 with V_box; heating: reading H1), from device pointers,
 * all [nz][ny][nx], x fastest:
 *   d_nH, d_xHI     in   total hydrogen density [cm^-3] and NEUTRAL fraction, fp64 (field_dtype 0) or fp32 (1)
 *   d_photons       in   photons absorbed per cell per second (nyxrt_trace_photons, summed over shards), fp64
 *   d_gamma_HI      out  photons / (n_H x_HI dx_cm^3), exactly 0 where photons == 0; same bits as nyxrt_finalise
 *   d_heat          out  e_excess_erg * photons / dx_cm^3; may be NULL
 *   d_absorbed      out  one double: sum of d_photons (row sums in x order, rows in a fixed order: the same bits on
 *                        every call, equal to nyxrt_finalise's total up to the rounding of a different but also
 *                        fixed summation order); may be NULL
 * All buffers stay the caller's; nothing is retained.  The two kernels are enqueued on `cuda_stream` on `device`
 * (made current, as the other entry points do); the call does not synchronise.
 *
 * The scratch (one partial sum per row) is a fixed array inside the library: NYXRT_STATIC_MAX_ROWS doubles (8 MiB)
 * on every GPU that loads libnyxrt.so, for the life of the process.  Hence:
 *   - ny * nz > NYXRT_STATIC_MAX_ROWS (more rows than the 1024^3 grid of config 5) -> NYXRT_ENOMEM, nothing enqueued;
 *   - every call in the process shares the array, which still holds the previous call's partials.  No part of it
 *     needs clearing (a call reads only the ny * nz entries it has just written), but two calls that run on the
 *     same GPU at the same time -- two streams, or two host threads -- corrupt each other's d_absorbed.  Put them
 *     on one stream or order them with events;
 *   - the first call that names a device looks up the array's address on that device
 *     (cudaGetSymbolAddress); make that first call before any stream capture begins.
 * errbuf (may be NULL) receives the message of a failed call, truncated to errbuf_len bytes.
 * Errors: EINVAL (sizes, dtype, dx_cm <= 0, NULL, device ordinal outside 0..63), ENOMEM (grid beyond the scratch), ECUDA. */
#define NYXRT_STATIC_MAX_ROWS (1 << 20)
int nyxrt_finalise_static(int32_t device, int32_t nx, int32_t ny, int32_t nz, int32_t field_dtype, double dx_cm,
                          double e_excess_erg, const void *d_nH, const void *d_xHI, const double *d_photons,
                          double *d_gamma_HI, double *d_heat, double *d_absorbed, void *cuda_stream, char *errbuf,
                          int64_t errbuf_len);

/* The (deduplicated, merged, sorted) catalogue the last nyxrt_trace used: host
 * pointers with room for `cap` entries; cell_ijk is [cap][3]; radius is the bubble radius in cells
 * (0 when merging was off).  Any of the three arrays may be NULL.  *n_out = catalogue length even
 * when cap is smaller (then only cap entries are written).  Errors: ESTATE, ECUDA. */
int nyxrt_get_catalog(nyxrt_ctx *ctx, int64_t cap, int32_t *cell_ijk, double *L, double *radius, int64_t *n_out);

/* The same step end to end with HOST buffers: copies the fields and sources to the device, runs
 * nyxrt_set_fields + nyxrt_set_sources + nyxrt_trace on an internal stream, copies Gamma_HI (and the
 * heating rate unless h_heat is NULL) back.  Needs a workspace created with host_staging != 0.
 * Errors: as the three calls. */
int nyxrt_step_host(nyxrt_ctx *ctx, const void *h_nH, const void *h_xHI, int64_t n_src, const double *pos_xyz,
                    const double *L, double *h_gamma_HI, double *h_heat, nyxrt_stats *h_stats);

/* Parameters of one RT TIMESTEP (time integration, Eq. 3, inside the iterative nonlinear
 * solve, "following [23]").  The ray traces inside use whatever flux is configured: monochromatic
 * by default, the tau_0 lookup table of PAPER.md:95 once nyxrt_set_spectrum has been called (R32). */
typedef struct {
    double  dt_s;              /* timestep [s], > 0                                                  */
    double  alpha_cm3_s;       /* recombination coefficient alpha_H(T) of Eq. 3 (2.59e-13 at 1e4 K)  */
    double  coll_cm3_s;        /* collisional ionisation coefficient C_H(T) of Eq. 3                 */
    double  clumping;          /* clumping factor C of Eq. 10: multiplies the recombination rate     */
    double  tol_rel, tol_abs;  /* a cell has converged when |d<x_HI>| <= tol_rel <x_HI> + tol_abs (R35) */
    double  unconv_frac;       /* fraction of the cells that may stay unconverged (R35)              */
    int32_t max_iter;          /* ray trace <-> update iterations, >= 1                              */
    int32_t inner_iter;        /* per-cell iterations on the electron density, >= 1 (R34)            */
} nyxrt_ode;

typedef struct {
    int32_t  iterations, converged;
    uint64_t unconverged_cells;          /* in the last iteration                                    */
    uint64_t segments_total;             /* ray-cell segments over all iterations                    */
    uint64_t kernel_launches;            /* own kernels over all iterations                          */
    double   max_rel_change;             /* last iteration: max |d<x_HI>| / (tol_rel <x_HI> + tol_abs) */
    float    ms_total, ms_rt, ms_ode, pad_;
} nyxrt_tstats;

/* One RT timestep of length ode->dt_s: starting from the neutral fraction d_xHI_begin (fp64, [nz][ny][nx]),
 * iterate { nyxrt_set_fields(d_nH, d_xHI_avg); nyxrt_trace -> Gamma; per cell, integrate Eq. 3 over dt with
 * Gamma fixed and n_e at its time average (semi-analytic, time-averaged solution of [23]) -> x_HI at the end
 * of the step and its time average } until the time-averaged neutral fraction stops changing or max_iter.
 * All pointers are device pointers.  d_nH: grid.field_dtype.  d_xHI_avg: grid.field_dtype, written (the x_HI
 * field of every ray trace; on return the converged time average, and the registered field of the context).
 * d_xHI_end: fp64, written.  d_gamma_HI / d_heat (may be NULL): the last iteration's rates.  h_stats (may be
 * NULL): the last ray trace's statistics.  h_tstats (may be NULL).  Sources must have been set.  Synchronises
 * `stream` every iteration (the convergence test is read on the host).
 * Errors: EINVAL (NULL, bad parameters), ESTATE (workspace / sources missing), EOVERFLOW, ECUDA. */
int nyxrt_timestep(nyxrt_ctx *ctx, const nyxrt_ode *ode, const void *d_nH, const double *d_xHI_begin,
                   double *d_xHI_end, void *d_xHI_avg, double *d_gamma_HI, double *d_heat, nyxrt_stats *h_stats,
                   nyxrt_tstats *h_tstats, void *cuda_stream);

/* HEALPix nested pixel centre of (level, pix) as the library computes it on the device (DIR-SPEC,
 * DESIGN.md): n directions into the host array dir_xyz [n][3].  For tests.  Errors: EINVAL, ECUDA. */
int nyxrt_pix2dir(nyxrt_ctx *ctx, int32_t level, int64_t pix_begin, int64_t n, double *dir_xyz);

/* Message of the last failed call on this context ("" if none).  Never NULL. */
const char *nyxrt_last_error(const nyxrt_ctx *ctx);

/* Free the context (not the workspace, which the caller owns).  NULL is allowed. */
void nyxrt_destroy(nyxrt_ctx *ctx);

/* Library version and the size of the public structs (for binding self-checks). */
int nyxrt_version(void);
int nyxrt_sizeof_grid(void);
int nyxrt_sizeof_params(void);
int nyxrt_sizeof_stats(void);
int nyxrt_sizeof_ode(void);
int nyxrt_sizeof_tstats(void);

#ifdef __cplusplus
}
#endif
#endif /* NYXRT_H */
