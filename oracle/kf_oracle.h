/*
 * kf_oracle.h -- CPU ORACLE for the batched per-track Kalman-filter track fit.
 *
 * TEST INFRASTRUCTURE ONLY.  This is a plain, slow, double-precision restatement of the method,
 * written from the paper (arxiv 2105.01796, /root/reference/PAPER.md: the Kalman step list at
 * lines 55-60, the RTS smoother with stored Jacobians at line 62, the Runge-Kutta-Nystrom
 * transport with local<->global Jacobians at line 128) and, where the paper prints no formula,
 * from the readings collected in SURVEY.md section 8(c) / DESIGN.md "Readings".  It shares no
 * code, header, constant table or helper with the CUDA path (paper_2105_01796_b200/csrc, include/).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  The product path never does.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): analytic helix, 4th-order convergence,
 * zero-field straight line, finite-difference Jacobian, noiseless recovery, weighted least
 * squares at zero field, KF+RTS == global linear least squares, covariance invariants,
 * chi2/pull statistics, the worked material table, trilinear exactness, option limits; for the cylinder and disc
 * surface kinds and the field-gradient terms of the step Jacobian (tests/test_oracle_surfaces.py): closed-form
 * helix <-> cylinder, straight line <-> cylinder / disc, finite-difference Jacobians between every pair of kinds,
 * chain rule through mixed kinds, disc = plane in polar coordinates, tangent-plane material, whole-fit pulls;
 * gradient of the interpolant exact on a linear field, finite differences of the step and of the propagation in
 * non-uniform tables.  No function below is "parity unpinned".
 *
 * Conventions:
 *   bound vector  x = (loc0, loc1, phi, theta, q/p, t)
 *   free  vector  f = (rx, ry, rz, t, Tx, Ty, Tz, q/p)          8 components
 *   units: mm, GeV, e; q/p in 1/GeV; t is c*t in mm; field in tesla at the interface
 *   geometry: packed table, 20 doubles per surface:
 *       center[3] u[3] v[3] n[3] half_len[2] x_over_X0 thickness_mm meas_var[2] kind pad
 *       kind 0 = plane (loc = u, v coordinates), 1 = cylinder (axis v through the centre, radius = half_len[0],
 *       loc0 = R alpha with alpha from n towards u, loc1 along the axis), 2 = disc (the plane in polar coordinates,
 *       loc0 = rho, loc1 = alpha from u towards v)      -- PAPER.md:136-138, reading U33
 *   all matrices are dense row-major; all pointers are HOST pointers.
 */
#ifndef KF_ORACLE_H
#define KF_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KFO_GEOM_STRIDE 20

enum { KFO_FIELD_CONST = 0, KFO_FIELD_GRID3 = 1 };

/* per-track status bits */
enum {
  KFO_ST_PROPAGATION = 1,   /* n.T <= 1e-6 or non-finite state: surface not reachable         */
  KFO_ST_NOT_POSITIVE = 2,  /* S not positive definite in the update, or non-positive pivot in the RTS inverse */
  KFO_ST_ENERGY = 4,        /* E' <= m in the material step                                    */
  KFO_ST_NDF = 8,           /* ndf <= 0                                                        */
  KFO_ST_THETA = 16,        /* sin(theta) <= 1e-12: (phi, theta) chart singular                */
  KFO_ST_FIELD_CLAMPED = 32,/* a field lookup fell outside the grid (clamped value used)       */
  KFO_ST_BAD_HITS = 64,     /* hit list not strictly ascending / outside (start, n_surfaces)   */
  KFO_ST_PERIGEE = 128      /* the extrapolation to the perigee (line) surface stopped          */
};

/* hit flags */
enum { KFO_HIT_UNPROCESSED = 0, KFO_HIT_USED = 1, KFO_HIT_OUTLIER = 2 };

typedef struct {
  int32_t kind;        /* KFO_FIELD_CONST | KFO_FIELD_GRID3 */
  double b[3];         /* CONST: field in tesla */
  int32_t n[3];        /* GRID3: nodes along x, y, z */
  double origin[3];    /* mm */
  double spacing[3];   /* mm */
  const double* grid;  /* [nz][ny][nx][3] tesla, x fastest, component innermost */
} kfo_field;

typedef struct {
  int32_t smooth;        /* run the RTS backward pass */
  int32_t material;      /* apply Highland noise + Bethe mean loss at surfaces with x/X0 > 0 */
  double outlier_chi2;   /* <= 0: off; else hits with predicted chi2 > cut are flagged, not used */
  int32_t n_corr_steps;  /* correction steps after the primary sub-steps (default 2) */
  double max_step_mm;    /* primary step cap (inf: one primary step per leg) */
  double mass_gev;
  double cov_inflation;  /* multiplies the whole start covariance */
  double mat_Z, mat_A, mat_rho, mat_I_eV; /* one material for the batch (silicon in the configs) */
  double step_tolerance_mm; /* > 0: adaptive step count per leg (U31); <= 0 or inf: off */
  int32_t field_gradient;   /* 1: the step Jacobian carries the dB/dr terms of a grid field (U32); 0: neglected (U4) */
} kfo_options;

/* --- step-level entry points (pinned one by one in tests/test_oracle_steps.py) ------------- */

/* B(r) in tesla; *clamped is OR-ed with 1 when r is outside the grid. */
void kfo_field_at(const kfo_field* fld, const double r[3], double b_tesla[3], int32_t* clamped);

/* dB_c/dr_a of the trilinear interpolant at r in tesla/mm, G[c * 3 + a]; zero along an axis on which the lookup is
 * clamped, zero for a constant field. */
void kfo_field_gradient_at(const kfo_field* fld, const double r[3], double G_tesla_per_mm[9]);

/* One RKN4 step of length h on the free vector; Dstep is the 8x8 step Jacobian (field gradient
 * neglected, or with the dB/dr terms of the trilinear interpolant when field_gradient != 0),
 * *eps the embedded error estimate h^2 |k1-k2-k3+k4|_1. */
void kfo_rkn4_step(const kfo_field* fld, double mass_gev, const double f[8], double h,
                   double f_out[8], double Dstep[64], double* eps, int32_t* clamped, int32_t field_gradient);

/* bound state on surface `from` -> bound state on surface `to` (any kinds) with the 6x6 Jacobian.
 * Returns 0 or the status bit that stopped the propagation. */
int32_t kfo_propagate(const kfo_field* fld, const kfo_options* opt, const double x[6],
                      const double* surf_from, const double* surf_to, double x_out[6],
                      double J[36], double free_out[8], double* rk_err, int32_t* clamped);

/* bound state (x, C) on plane `surf_from` -> bound state (d0, z0, phi, theta, q/p, t) with covariance on
 * the line surface through line_c with unit direction line_a: the perigee surface of PAPER.md:70, 85
 * (closest approach to the axis); J is the 6x6 Jacobian.  Returns 0 or the stopping status bit. */
int32_t kfo_to_line(const kfo_field* fld, const kfo_options* opt, const double x[6], const double C[36],
                    const double* surf_from, const double line_c[3], const double line_a[3],
                    double x_out[6], double C_out[36], double J[36], int32_t* clamped);

/* gain-matrix update with a 2-D hit: returns 0, or KFO_ST_NOT_POSITIVE. */
int32_t kfo_update(const double xp[6], const double Cp[36], const double m[2], const double V[4],
                   double xf[6], double Cf[36], double* chi2);

/* material at a surface from the filtered state: x -> x (q/p changed), C -> G C G^T + Q, g = dlam'/dlam.
 * Returns 0 or KFO_ST_ENERGY. theta0 / dE (GeV) are diagnostics for the material pin. */
int32_t kfo_material(const kfo_options* opt, const double* surf, const double xf[6],
                     const double Cf[36], double x_out[6], double C_out[36], double* g,
                     double* theta0, double* dE_gev);

/* one RTS step: smoothed (k+1) + records -> smoothed (k). Returns 0 or KFO_ST_NOT_POSITIVE. */
int32_t kfo_rts_step(const double xf_k[6], const double Cf_k[36], const double F_k1[36],
                     const double xp_k1[6], const double Cp_k1[36], const double xs_k1[6],
                     const double Cs_k1[36], double xs_k[6], double Cs_k[36]);

/* --- the batch fit -------------------------------------------------------------------------
 * Inputs (host, AoS): params0 [N][6], cov0 [N][6][6], CSR hits (offsets [N+1], surf_idx [M],
 * loc [M][2], optional var [M][2] and cov01 [M], NULL -> surface meas_var), geometry table.
 * Outputs (host; any pointer may be NULL to skip): first/last params [N][6] and cov [N][6][6],
 * chi2 [N], ndf/status/counters [N], per-leg states [N][Lmax][6] / [N][Lmax][6][6] with
 * Lmax = n_surfaces - 1 - start_surface (legs not visited are filled with NaN), per-hit
 * chi2 [M] and flags [M], rk_err_max [N].
 * Tracks are fitted independently under an OpenMP parallel-for over tracks
 * (the paper's CPU parallelisation); n_threads <= 0 keeps the OpenMP default.
 * Returns the number of threads used (> 0), or < 0 on a malformed call. */
int32_t kfo_fit_batch(int64_t n_tracks, const double* params0, const double* cov0,
                      int32_t start_surface, const int32_t* offsets, const int32_t* surf_idx,
                      const double* loc, const double* var, const double* cov01,
                      int32_t n_surfaces, const double* geometry, const kfo_field* fld,
                      const kfo_options* opt, double* first_params, double* first_cov,
                      double* last_params, double* last_cov, double* chi2, int32_t* ndf,
                      uint32_t* status, int32_t* n_used, int32_t* n_outliers, int32_t* n_holes,
                      double* st_pred_params, double* st_pred_cov, double* st_filt_params,
                      double* st_filt_cov, double* st_smooth_params, double* st_smooth_cov,
                      double* hit_chi2, uint8_t* hit_flags, double* rk_err_max,
                      int32_t n_threads);

/* perigee parameters (d0, z0, phi, theta, q/p, t) and covariance of N fitted tracks: kfo_to_line applied to
 * first_params [N][6] / first_cov [N][6][6], which live on geometry surface on_surface[i].  out_* as the
 * inputs; a stopped extrapolation sets KFO_ST_PERIGEE in status[i] and NaN outputs.  Returns 0, or < 0. */
int32_t kfo_perigee_batch(int64_t n_tracks, const double* first_params, const double* first_cov,
                          const int32_t* on_surface, const double* geometry, const kfo_field* fld,
                          const kfo_options* opt, const double line_c[3], const double line_a[3],
                          double* out_params, double* out_cov, uint32_t* status);

/* Which arithmetic this build of the oracle runs in (kf_oracle.c "the arithmetic type"): sizeof the type of
 * every operand (8 = double: the oracle; 16 = x87 long double: the arbiter; 4 = float: the paper's operating
 * point) and of the smoother's 6x6 solve (8, 16, 8).  The interface is double in every build. */
int32_t kfo_real_bytes(void);
int32_t kfo_solve_real_bytes(void);

#ifdef __cplusplus
}
#endif
#endif
