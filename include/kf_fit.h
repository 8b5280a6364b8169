/*
 * kf_fit.h -- C ABI of libkf_fit.so: batched per-track Kalman-filter track fit on one B200.
 *
 * What it computes (arxiv 2105.01796, "A GPU-based Kalman Filter for Track Fitting"):
 *   for every track independently the Kalman step loop of PAPER.md:55-60 --
 *   propagate the bound parameters (loc0, loc1, phi, theta, q/p, t) and their 6x6
 *   covariance to the next measurement surface with a 4th-order Runge-Kutta-Nystrom stepper,
 *   transporting the 8x8 free Jacobian alongside and applying the local<->global Jacobians at both
 *   ends; combine the prediction with the surface's 2-D measurement in the
 *   gain-matrix formalism; add the material effects of the surface;
 *   then, optionally, the Rauch-Tung-Striebel smoother "with the stored Jacobians between states"
 *   (PAPER.md:62, 75).  The four track-specific data sets of PAPER.md:174-180 (measurements,
 *   starting parameters, fit configuration, results) are the four argument groups below; the
 *   "global data shared by different tracks" (geometry, field) are kf_geometry / kf_field.
 *   The exact arithmetic (the paper prints none) is stated in DESIGN.md "The algorithm".
 *
 * All of it runs in hand-written sm_100a CUDA kernels, in IEEE double precision by default (kf_options.precision
 * MIXED: float operands with the smoother's 6x6 solve in double, the paper's own operating point).  There is no CPU
 * fallback: without a CUDA device every compute entry point returns KF_ERR_CUDA.
 *
 * Conventions
 *   units      mm, GeV, e.  q/p in 1/GeV.  t is c*t in mm (1 ns = 299.792458 mm).  Field in tesla.
 *   bound      x = (loc0, loc1, phi, theta, q/p, t) on a plane with centre c and orthonormal
 *              u, v, n = u x v:  r = c + loc0 u + loc1 v,  T = (cos phi sin theta, sin phi sin theta, cos theta);
 *              on a cylinder or a disc (loc0, loc1) are the chart of that kind (KF_SURFACE_* below).
 *   SoA        per-track arrays are component-major: element (component k, track i) of a
 *              double[K][N] array lives at [k * N + i].
 *   cov        6x6 symmetric, packed upper triangle row-major, 21 values:
 *              (00 01 02 03 04 05 11 12 13 14 15 22 23 24 25 33 34 35 44 45 55).
 *   pointers   every array pointer is a DEVICE pointer (8-byte aligned) unless the field says HOST;
 *              the descriptor structs themselves are small HOST structs read during the call.
 *
 * Ownership and ordering
 *   The caller owns every buffer including the workspace (kf_fit_batch_static alone uses a fixed array inside
 *   the library image instead; see there).  The library allocates no device or
 *   pinned memory, never frees and never synchronises: kf_fit_batch validates the descriptors on
 *   the host, enqueues its kernels on `cuda_stream` (a cudaStream_t; NULL = the legacy default
 *   stream) and returns.  Inputs are read-only.  Buffers must stay valid until the stream has run
 *   past the call.  No state of a fit survives the call; what the library does keep is bookkeeping
 *   only: per calling thread, the text of the last CUDA error, the launch count of the last call
 *   (kf_last_launch_count) and the stage-event hook (kf_set_stage_events); per process, the list of
 *   kernels whose dynamic shared-memory limit has been raised (a one-time cudaFuncSetAttribute).
 *
 * Errors
 *   0 = everything enqueued.  KF_ERR_ARG / KF_ERR_UNSUPPORTED / KF_ERR_WORKSPACE are decided on the
 *   host before anything is enqueued: outputs are untouched.  KF_ERR_CUDA means a CUDA call failed
 *   while enqueuing: kernels and copies enqueued before the failure still run (outputs may be
 *   partly written); in kf_fit_batch_host_pipelined the worker streams are joined back onto
 *   `cuda_stream` before the call returns, so the caller's stream remains an ordering point for
 *   reusing the buffers.  Per-track problems never fail a call: they set KF_ST_* bits.
 */
#ifndef KF_FIT_H
#define KF_FIT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KF_VERSION 109          /* major * 100 + minor */
#define KF_GEOM_STRIDE 20       /* doubles per surface record */
#define KF_MAX_SUBSTEPS 1024    /* cap on primary RKN sub-steps per leg (max_step_mm) */

/* return codes */
enum {
  KF_OK = 0,
  KF_ERR_ARG = -1,        /* null / ill-formed descriptor */
  KF_ERR_UNSUPPORTED = -2,/* unsupported option combination */
  KF_ERR_WORKSPACE = -3,  /* workspace too small (see kf_workspace_bytes) */
  KF_ERR_CUDA = -4,       /* CUDA error at launch (text: kf_last_cuda_error) */
  KF_ERR_STATIC_LIMIT = -5 /* kf_fit_batch_static only: the batch needs more scratch than KF_STATIC_WORKSPACE_BYTES */
};

/* per-track status bits (never fail the call) */
enum {
  KF_ST_PROPAGATION = 1,   /* n.T <= 1e-6 or a non-finite state: next surface not reachable. Track stops. */
  KF_ST_NOT_POSITIVE = 2,  /* S = H C H^T + V not positive definite (track stops), or a non-positive
                              Cholesky pivot in the smoother (smoothed output falls back to filtered) */
  KF_ST_ENERGY = 4,        /* E' <= m after the energy loss in a layer. Track stops after that layer. */
  KF_ST_NDF = 8,           /* ndf = 2 n_used - 5 <= 0 */
  KF_ST_THETA = 16,        /* sin(theta) <= 1e-12 on arrival: (phi, theta) chart singular. Track stops. */
  KF_ST_FIELD_CLAMPED = 32,/* a field lookup fell outside the grid; the clamped value was used */
  KF_ST_BAD_HITS = 64,     /* hit list not strictly ascending in surf_idx or outside (start, n_surfaces), or CSR
                              offsets of the track outside 0 <= offsets[i] <= offsets[i+1] <= n_meas: track not
                              fitted, outputs hold the start state, its per-hit outputs are left untouched */
  KF_ST_PERIGEE = 128,     /* the extrapolation of first_* to the perigee surface stopped (moving along the axis,
                              non-finite state, theta chart singular): perigee_* hold NaN */
  KF_ST_CANCELLATION = 256 /* Bryson-Frazier backward pass only: first_cov = C- - C- Lam C- cancelled more than 1e6 (an
                              uninformative prior): first_* are valid but may miss the 1e-8 covariance bar; the RTS
                              form (the default) does not have this */
};

/* per-hit flags */
enum { KF_HIT_UNPROCESSED = 0, KF_HIT_USED = 1, KF_HIT_OUTLIER = 2 };

/* field kinds */
enum { KF_FIELD_CONST = 0, KF_FIELD_GRID3 = 1 };

/* kernel variants (kf_options.variant); results agree to round-off.
 *   THREAD_PER_TRACK  one CUDA thread fits one track ("track-level parallelisation")
 *   LANES_PER_TRACK   8 adjacent lanes of a warp fit one track, the 6x6 products split by row and exchanged
 *                     with warp shuffles ("intra-track parallelisation")
 *   AUTO              the measured choice: LANES for batches (or pipeline chunks) of at most
 *                     KF_AUTO_LANES_MAX_TRACKS tracks, THREAD above */
enum { KF_VARIANT_AUTO = 0, KF_VARIANT_THREAD_PER_TRACK = 1, KF_VARIANT_LANES_PER_TRACK = 2 };
#define KF_AUTO_LANES_MAX_TRACKS 2048

/* kf_options.length_sort: ragged batches (tracks whose last hit lies on different surfaces) are fitted in
 * order of decreasing leg count, so that the threads of a warp and the tracks of a record tile finish
 * together; results do not depend on it.  AUTO: considered for a batch (or pipeline chunk) of at least
 * KF_AUTO_SORT_MIN_TRACKS tracks whose hit lists are not dense (n_meas != n_tracks * legs) when the
 * workspace holds the sort's arrays (it does when sized by kf_workspace_bytes); the device then keeps the
 * batch's own order if the mean leg count is within 15 % of the longest track's (nothing to win).
 * ON: always sorted. */
enum { KF_SORT_AUTO = 0, KF_SORT_OFF = 1, KF_SORT_ON = 2 };
#define KF_AUTO_SORT_MIN_TRACKS 8192

/* kf_options.smoother: how the backward pass reaches the smoothed state.
 *   RTS  (default) the Rauch-Tung-Striebel recursion of PAPER.md:62, 75 with the stored Jacobians: one 6x6 SPD solve
 *        per state; every per-leg smoothed state available (KF_STATES_SMOOTH).
 *   BRYSON_FRAZIER  the same smoothed state at the first surface (first_*) from the adjoint recursion of the modified
 *        Bryson-Frazier smoother: no 6x6 solve, 42-double records instead of 55, thread-per-track kernels only.
 *        Agrees with RTS to round-off while kappa = C-_ii / C^s_ii stays moderate (1.6e3 on the configs); loses
 *        kappa * 1e-16 relative to it (an inflated prior), so it is an option, not the default.  Not with
 *        KF_STATES_SMOOTH, not with KF_VARIANT_LANES_PER_TRACK (KF_ERR_UNSUPPORTED). */
enum { KF_SMOOTHER_RTS = 0, KF_SMOOTHER_BRYSON_FRAZIER = 1 };

/* kf_options.precision: the arithmetic the fit runs in.
 *   FP64   (default; the BASELINE.json metric) every operand IEEE double.
 *   MIXED  the paper's operating point ("All the tests use single precision ... with the
 *          exception of the matrix inversion"): inputs are rounded to float on load, the state, the Jacobians, the
 *          covariances and the RTS records (half the workspace, half its HBM traffic) are float, the smoother's 6x6
 *          solve runs in double, results are widened to the double arrays of kf_outputs.  The boundary does not
 *          change.  The fitted parameters move by at most a few per cent of their own standard deviation against the
 *          FP64 fit (resolution-loss table); a hit whose chi2 lies within ~0.05 of the
 *          outlier cut may be classified differently.  Thread-per-track kernels, RTS smoother, at most 1024 surfaces
 *          (KF_ERR_UNSUPPORTED with KF_VARIANT_LANES_PER_TRACK or KF_SMOOTHER_BRYSON_FRAZIER); the perigee
 *          extrapolation of the result (kf_outputs.perigee_*) stays in double. */
enum { KF_PRECISION_FP64 = 0, KF_PRECISION_MIXED = 1 };

/* kf_options.output_states bitmask: which per-leg states to write to kf_outputs.state_* */
enum { KF_STATES_PRED = 1, KF_STATES_FILT = 2, KF_STATES_SMOOTH = 4 };

/* (2) starting parameters -- PAPER.md:177 */
typedef struct kf_tracks_in {
  int64_t n_tracks;       /* N >= 0 */
  const double* params;   /* double[6][N]  start parameters on the start surface */
  const double* cov;      /* double[21][N] start covariance, packed upper triangle */
  int32_t start_surface;  /* index into the geometry; one value for the batch */
} kf_tracks_in;

/* (1) input measurements -- PAPER.md:176; the geometry identifier that links a hit to its
 * surface is surf_idx.  CSR over tracks. */
typedef struct kf_measurements {
  int64_t n_meas;          /* M = offsets[N] */
  const int32_t* offsets;  /* int32[N+1], offsets[0] = 0, non-decreasing */
  const int32_t* surf_idx; /* int32[M], strictly ascending within a track, in (start_surface, n_surfaces) */
  const double* loc;       /* double[2][M] measured local position (loc0 row, then loc1 row) */
  const double* var;       /* double[2][M] per-hit variances, or NULL: use the surface's meas_var */
  const double* cov01;     /* double[M] per-hit covariance (needs var), or NULL: 0 */
} kf_measurements;

/* surface kinds (geometry record entry [18]; "surfaces of different concrete types for different
 * tracking detectors"; reading U33).  The bound vector is (loc0, loc1, phi, theta, q/p, t) on every kind.
 *   PLANE     r = c + loc0 u + loc1 v                                              (PAPER.md:182 boundless planes)
 *   CYLINDER  axis v through c, radius R = entry [12]; azimuth alpha = loc0 / R measured from n towards u:
 *             r = c + R (cos alpha n + sin alpha u) + loc1 v      (loc0 = arc length R alpha, loc1 = along the axis)
 *             reached along the track's direction of motion from inside (navigation outwards)
 *   DISC      the plane through c with normal n in polar coordinates: r = c + loc0 (cos loc1 u + sin loc1 v),
 *             loc0 = rho > 0, loc1 = alpha in (-pi, pi]
 * The angular coordinates are periodic (R alpha: 2 pi R; alpha: 2 pi): a hit is taken on the branch nearest the
 * prediction before the update. */
enum { KF_SURFACE_PLANE = 0, KF_SURFACE_CYLINDER = 1, KF_SURFACE_DISC = 2 };

/* global data: detector geometry -- PAPER.md:168, 174, 182 (boundless planes), 136-138 (other kinds).
 * Surface record, KF_GEOM_STRIDE doubles:
 *   [0..2] centre  [3..5] u  [6..8] v  [9..11] n = u x v (orthonormal)  [12..13] half lengths (informational; the
 *   radius in [12] for a cylinder)  [14] x/X0 along the normal  [15] thickness in mm
 *   [16..17] measurement variances (loc0, loc1)  [18] kind (KF_SURFACE_*, 0 = plane)  [19] unused
 * Navigation order = ascending surface index: a track visits start_surface+1, +2, ... up to the
 * surface of its last hit. */
typedef struct kf_geometry {
  int32_t n_surfaces;
  const double* surfaces;  /* double[n_surfaces][KF_GEOM_STRIDE] */
  double mat_Z, mat_A;     /* one material for the batch: atomic number, mass (g/mol) */
  double mat_rho;          /* density g/cm^3 */
  double mat_I_eV;         /* mean excitation energy */
  int32_t surface_kinds;   /* bit k set = the table holds surfaces of kind k (the table itself is DEVICE memory, which
                              the host-side dispatch does not read).  0 or 1 = planes only: the plane-only kernels run
                              and entry [18] is then ignored by the fit AND by the perigee extrapolation (one exception:
                              kf_options.field_gradient with a GRID3 field runs the general kernels, which read entry
                              [18] of every record -- keep it 0 for planes there).  Any other value selects the
                              general-surface kernels:
                              one thread per track, RTS smoother, at most 1024 surfaces, FP64 or MIXED precision
                              (KF_ERR_UNSUPPORTED with KF_VARIANT_LANES_PER_TRACK or Bryson-Frazier) */
} kf_geometry;

/* global data: magnetic field -- PAPER.md:170 (constant 3x1 vector; inhomogeneous fields need
 * "position-specific field information ... stored and retrieved") */
typedef struct kf_field {
  int32_t kind;        /* KF_FIELD_CONST | KF_FIELD_GRID3 */
  double b[3];         /* CONST: tesla (HOST values) */
  int32_t n[3];        /* GRID3: nodes along x, y, z (each >= 2) */
  double origin[3];    /* GRID3: position of node (0,0,0), mm */
  double spacing[3];   /* GRID3: mm, > 0 */
  const double* grid;  /* GRID3: double[nz][ny][nx][3] tesla, x fastest, component innermost.
                          Trilinear interpolation; outside the grid the clamped value is used. */
  /* GRID3, optional hint (all zero = none): the box of nodes [stage_lo[a], stage_lo[a] + stage_n[a]) per axis that
   * covers where the tracks of the batch go (the detector acceptance).  When it is well-formed (inside the grid,
   * stage_n[a] >= 2) and fits (KF_FIELD_STAGE_MAX_BYTES), the thread-per-track forward kernel keeps that part of
   * the table in shared memory ("position-specific field information ... stored and retrieved", PAPER.md:170;
   * shared memory for the objects of a fit); a lookup outside the box reads the table in global
   * memory.  Results do not depend on the hint (same values, same arithmetic).  kf_field_stage_box fills it. */
  int32_t stage_lo[3];
  int32_t stage_n[3];
} kf_field;
#define KF_FIELD_STAGE_MAX_BYTES (200 * 1024)

/* Fill field->stage_lo / stage_n from a HOST copy of the geometry table: the smallest node box that contains every
 * surface's rectangle (centre +- half lengths along u and v, record entries [12..13]) plus one cell of margin,
 * clipped to the grid; the hint is cleared when the field is not GRID3, the table holds no half lengths, or the box
 * would not fit in KF_FIELD_STAGE_MAX_BYTES of doubles.  Host-only arithmetic, no CUDA call.  Returns KF_OK / KF_ERR_ARG. */
int kf_field_stage_box(const double* surfaces_host, int32_t n_surfaces, kf_field* field);

/* (3) fit configuration -- PAPER.md:179 */
typedef struct kf_options {
  int32_t smooth;         /* 1: run the RTS backward pass */
  int32_t material;       /* 1: Highland scattering noise + Bethe mean energy loss at surfaces with x/X0 > 0 */
  double outlier_chi2;    /* <= 0: off.  Else a hit whose predicted chi2 (2 dof) is > this is flagged, not used */
  int32_t n_corr_steps;   /* RKN correction steps after the primary ones, 0..8 (default 2) */
  double max_step_mm;     /* cap on a primary step; +inf (or <= 0): one primary step per leg */
  double mass_gev;        /* particle mass (> 0) */
  double cov_inflation;   /* multiplies the start covariance (default 1) */
  int32_t output_states;  /* KF_STATES_* bitmask */
  int32_t variant;        /* KF_VARIANT_* */
  int32_t length_sort;    /* KF_SORT_* */
  int32_t smoother;       /* KF_SMOOTHER_* (used when smooth) */
  double step_tolerance_mm; /* > 0: adaptive number of primary RKN steps per leg ("adaptive"): the
                             embedded error estimate eps0 = h^2 |k1-k2-k3+k4|_1 of one trial step over the whole leg
                             gives n = ceil((eps0 / tolerance)^(1/4)) primary steps (at least what max_step_mm asks
                             for, at most KF_MAX_SUBSTEPS), decided once per leg, no accept/reject loop.
                             <= 0 or inf (default 0): off */
  /* perigee surface (used only when kf_outputs.perigee_params is given): the straight line
   * through perigee_center with UNIT direction perigee_axis (the beam axis; default origin, +z) */
  double perigee_center[3];
  double perigee_axis[3];
  int32_t precision;      /* KF_PRECISION_* */
  int32_t field_gradient; /* 1: the transported Jacobian carries the dB/dr terms of a GRID3 field (
                             DESIGN.md reading U32): every stage derivative of the RKN4 step gains lam T_i x (G_i dr_i),
                             G = gradient of the trilinear interpolant.  The states do not change, the covariances do
                             (CFG4: up to a few per cent of a standard deviation on the fitted parameters).  0 (default):
                             neglected (reading U4).  No effect in a constant field.  Runs in the general kernels (FP64,
                             thread per track, RTS; KF_ERR_UNSUPPORTED with MIXED precision, the lanes variant or
                             Bryson-Frazier); the perigee extrapolation neglects the terms either way */
} kf_options;

/* (4) results -- PAPER.md:180: status, track states, fitted parameters */
typedef struct kf_outputs {
  double* first_params;   /* double[6][N]  smoothed (or filtered if !smooth) state at the first visited surface */
  double* first_cov;      /* double[21][N] */
  double* last_params;    /* double[6][N]  filtered state at the last visited surface */
  double* last_cov;       /* double[21][N] */
  double* chi2;           /* double[N]     sum of predicted-residual chi2 over used hits */
  int32_t* ndf;           /* int32[N]      2 n_used - 5 */
  uint32_t* status;       /* uint32[N]     KF_ST_* bits */
  int32_t* n_used;        /* int32[N] */
  int32_t* n_outliers;    /* int32[N] */
  int32_t* n_holes;       /* int32[N]      visited surfaces without a hit */
  /* optional (NULL = skip).  Per-leg arrays are dense over (leg, track) with
   * Lmax = n_surfaces - 1 - start_surface legs: element (leg l, component k, track i) at
   * [(l * K + k) * N + i].  Legs a track did not visit are left untouched. */
  double* state_params[3];/* double[Lmax][6][N]  for PRED, FILT, SMOOTH (index = log2 of the bit) */
  double* state_cov[3];   /* double[Lmax][21][N] */
  double* hit_chi2;       /* double[M]  predicted chi2 of every processed hit (0 if unprocessed) */
  uint8_t* hit_flags;     /* uint8[M]   KF_HIT_* */
  double* rk_err_max;     /* double[N]  largest embedded RKN error estimate h^2 |k1-k2-k3+k4|_1, mm */
  /* optional, both or neither: the fitted parameters on the perigee surface:
   * first_* extrapolated (backwards, no material) to the point of closest approach to the line of
   * kf_options.perigee_*, as (d0, z0, phi, theta, q/p, t) with d0 = D.(a x T)/|a x T|, z0 = D.a, D = r - centre,
   * and their covariance J first_cov J^T.  One more kernel after the fit.  DESIGN.md U27-U30. */
  double* perigee_params; /* double[6][N] */
  double* perigee_cov;    /* double[21][N] */
} kf_outputs;

/* Fill `opt` with the defaults: smooth 1, material 0, outlier off, n_corr_steps 2, max_step inf,
 * no step tolerance, muon mass, inflation 1, no per-leg states, variant AUTO, length sort AUTO, perigee line = the z axis
 * through the origin, precision FP64, field gradient neglected. */
void kf_default_options(kf_options* opt);

/* Bytes of device workspace kf_fit_batch needs for n_tracks tracks and n_legs_max =
 * n_surfaces - 1 - start_surface legs per track: the RTS records (55 values of the precision's type + a flag byte per
 * leg and track) and leg counts (only when smooth), then the
 * length sort's permutation and counters (4.5 B per track).  A workspace that holds only the first part is
 * accepted: the batch is then fitted unsorted (KF_SORT_ON: KF_ERR_WORKSPACE). */
size_t kf_workspace_bytes(int64_t n_tracks, int32_t n_legs_max, const kf_options* opt);

/* Enqueue the fit of one batch on `cuda_stream`.  Returns KF_OK or a negative KF_ERR_*. */
int kf_fit_batch(const kf_tracks_in* tracks, const kf_measurements* meas, const kf_geometry* geom,
                 const kf_field* field, const kf_options* opt, const kf_outputs* out,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* The same fit for a caller that has no device memory to give as workspace and may not allocate any.
 *
 * Who that is: kf_fit_batch leaves the RTS records, leg counts and length-sort arrays to a caller-owned workspace,
 * which assumes the caller can get one.  Some cannot.  A reconstruction module plugged into an experiment's event
 * framework gets its input and output buffers from the framework's device-memory pool and is forbidden to call the
 * CUDA allocator itself (the pool is the memory budget).  An online-trigger or other latency-bound thread may not
 * call cudaMalloc / cudaFree once the run has started, because those calls take driver-wide locks and cudaFree
 * waits for the whole device: one late allocation stalls every stream.  A process on a GPU whose memory is already
 * handed out to its neighbours cannot count on a late cudaMalloc succeeding at all.
 *
 * What it does: the workspace lives in a KF_STATIC_WORKSPACE_BYTES array that is part of the library image
 * (a file-scope `static __device__ __align__(256)` array in kf_fit.cu).  The call allocates nothing, frees nothing and
 * calls no allocating library routine; apart from the workspace it is kf_fit_batch argument for argument (same
 * validation, same kernels, same results bit for bit), with `tracks`, `meas`, `geom`, `field`, `out` still the
 * caller's DEVICE buffers.
 *
 * Limit: the batch must satisfy kf_workspace_bytes(n_tracks, n_legs_max, opt) <= KF_STATIC_WORKSPACE_BYTES (64 MiB:
 * about 5,000 tracks x 30 legs in FP64 with smoothing, 10,000 in MIXED precision; any number without smoothing up
 * to the sort arrays' 4.5 B per track).  A larger batch is refused with KF_ERR_STATIC_LIMIT before anything is
 * enqueued, outputs untouched: split it, or use kf_fit_batch with a workspace.  The price of the array: every GPU
 * on which this process uses the library gives up those 64 MiB from the moment the library's code is loaded onto it
 * until the process exits, whether or not this entry point is ever called.
 *
 * First call on a device: the first call made while a given device is current looks up the array's device address
 * on that device (cudaGetSymbolAddress, which may also load the library's module there) and remembers it; later
 * calls on that device reuse it.  Make that first call with the device current, outside any stream capture, e.g.
 * once at start-up with n_tracks = 0 (which does the look-up and enqueues nothing).  A failed look-up returns
 * KF_ERR_CUDA and is retried by the next call.
 *
 * One array, shared: every call on a device, from whatever thread or stream, uses the same bytes, and the array
 * keeps what the previous call left in it.  Nothing in it has to be cleared by the caller: the only part that must
 * start at zero, the length sort's counters, is cleared on `cuda_stream` by the call itself (as in kf_fit_batch),
 * and every record and leg count is written by the forward kernel before the backward pass reads it.  But two calls
 * whose kernels can run at the same time on one GPU (different streams without an ordering between them, or two
 * host threads) overwrite each other's records and give wrong results without any error: order them on one
 * stream, or with events.  Calls on different GPUs do not interfere (each GPU has its own copy of the array). */
#define KF_STATIC_WORKSPACE_BYTES (64u * 1024u * 1024u)
int kf_fit_batch_static(const kf_tracks_in* tracks, const kf_measurements* meas, const kf_geometry* geom,
                        const kf_field* field, const kf_options* opt, const kf_outputs* out, void* cuda_stream);

/* End-to-end variant for HOST buffers (the paper's offload runtime):
 * every array pointer in tracks/meas/geom/field/out is a HOST pointer (pinned memory for
 * asynchronous copies).  The call copies the inputs into `device_arena` (caller-owned device
 * memory of at least kf_host_arena_bytes), runs kf_fit_batch there and copies the requested
 * outputs back, all enqueued on `cuda_stream`; it does not synchronise. */
size_t kf_host_arena_bytes(int64_t n_tracks, int64_t n_meas, int32_t n_surfaces, int32_t start_surface,
                           const kf_field* field, const kf_options* opt, int has_var, int has_cov01);
int kf_fit_batch_host(const kf_tracks_in* tracks, const kf_measurements* meas, const kf_geometry* geom,
                      const kf_field* field, const kf_options* opt, const kf_outputs* out,
                      void* device_arena, size_t arena_bytes, void* cuda_stream);

/* The same with the copies and the fit of different track ranges overlapped (the paper's multi-stream
 * offload): the tracks are cut into chunks of `chunk_tracks` (rounded up to a multiple of
 * 128 tracks; 0 = max(16384, N / (4 n_streams))); chunk c runs its H2D copies, its forward and RTS
 * kernels and its D2H copies in order on streams[c % n_streams].  The whole call is ordered after the work
 * already enqueued on `cuda_stream`, and `cuda_stream` continues only after every chunk has finished
 * (fork/join through the caller-owned events, which need no timing).  All handles are caller-owned;
 * meas->offsets is read on the host during the call.  Returns like kf_fit_batch_host. */
#define KF_MAX_STREAMS 8
typedef struct kf_pipeline {
  int32_t n_streams;                 /* 1..KF_MAX_STREAMS */
  void* streams[KF_MAX_STREAMS];     /* cudaStream_t handles */
  void* events[KF_MAX_STREAMS + 1];  /* cudaEvent_t handles, n_streams + 1 of them */
  int64_t chunk_tracks;              /* >= 0 */
} kf_pipeline;
int kf_fit_batch_host_pipelined(const kf_tracks_in* tracks, const kf_measurements* meas, const kf_geometry* geom,
                                const kf_field* field, const kf_options* opt, const kf_outputs* out,
                                void* device_arena, size_t arena_bytes, void* cuda_stream,
                                const kf_pipeline* pipe);

/* Number of kernels the last kf_fit_batch* call of this thread enqueued (for launch accounting). */
int kf_last_launch_count(void);

/* Optional per-kernel timing for the roofline report.  After this call every kf_fit_batch of the
 * calling thread records the three caller-owned CUDA events (cudaEvent_t handles created with
 * timing enabled) on its stream: events3[0] before the forward-filter kernel, events3[1] after it
 * (= before the RTS kernel), events3[2] after the RTS kernel (or after the forward kernel when
 * !smooth).  events3 == NULL switches the recording off again.  The events are only recorded,
 * never waited on. */
void kf_set_stage_events(void* const* events3);

/* Sustained FP64 FMA throughput probe (roofline denominator): runs a dependent-chain DFMA kernel
 * `iters` long on every SM, on `cuda_stream`, synchronises, and returns TFLOP/s (2 flop per FMA),
 * or a negative KF_ERR_*.  Not part of the fit. */
double kf_probe_fp64_tflops(int iters, void* cuda_stream);

const char* kf_status_string(int rc);
const char* kf_last_cuda_error(void);
int kf_version(void);

#ifdef __cplusplus
}
#endif
#endif
