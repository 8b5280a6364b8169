/*
 * kf_oracle.c -- CPU ORACLE (test infrastructure, see kf_oracle.h).
 *
 * Step-by-step restatement of the per-track Kalman fit, in the order and notation of
 * SURVEY.md section 8(c) C.2 (the paper names the steps at PAPER.md:55-62 and 128 but prints no
 * formula; the formulas below are derived from the definitions those passages name).
 * Dense row-major matrices, plain loops, IEEE double, no blocking, no structure exploitation,
 * no fused or reordered arithmetic.  Build: gcc -O2 -ffp-contract=off -fopenmp.
 */
#include "kf_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <tgmath.h> /* sin, cos, sqrt, fabs, ... follow the type of their argument */

/* ---- the arithmetic type -------------------------------------------------------------------
 * Every quantity of the fit is a `real`; the interface (kf_oracle.h) stays in double and converts
 * at the door.  Three builds of this one file (oracle/__init__.py):
 *   real = double       the oracle proper (BASELINE.json metric: FP64)
 *   real = long double  the ARBITER: the same algorithm in x87 80-bit arithmetic (64-bit mantissa), used by the
 *                       tests to tell which of two double-precision results is nearer the exact one where the
 *                       conditioning of the inputs exceeds the parity bars
 *   real = float        the paper's operating point ("All the tests use single precision ...
 *                       with the exception of the matrix inversion"): every operand float, the 6x6 solve of the
 *                       smoother in double (`sreal`).  Built with -fsingle-precision-constant so that literals
 *                       do not promote an expression to double.
 * Constants are written once as double literals: the long-double build uses the same (double-rounded) values,
 * so that it differs from the double build by arithmetic round-off only. */
#ifndef KFO_REAL
#define KFO_REAL double
#endif
#ifndef KFO_SOLVE_REAL
#define KFO_SOLVE_REAL double
#endif
typedef KFO_REAL real;
typedef KFO_SOLVE_REAL sreal; /* type of the smoother's 6x6 solve */
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- constants (the CUDA path carries its own copy) ------------- */
static const real TESLA_TO_GEV_PER_MM = 2.99792458e-4; /* 1 T = 2.99792458e-4 GeV/(e mm) */
static const real ME_GEV = 0.51099895e-3;              /* electron mass */
static const real K_BETHE = 0.307075;                  /* MeV mol^-1 cm^2 */
static const real NT_MIN = 1e-6;                       /* surface reachable if n.T > NT_MIN */
static const real SIN_THETA_MIN = 1e-12;
static const int MAX_SUBSTEPS = 1024;
static const real PI = 3.14159265358979323846;

/* ---- the descriptors of kf_oracle.h with their numbers as `real` (converted once per call) ---- */
typedef struct {
  int32_t kind;
  real b[3];
  int32_t n[3];
  real origin[3], spacing[3];
  const double* grid; /* the table itself stays as given; every node value read is converted to real */
} field_r;
typedef struct {
  int32_t smooth, material, n_corr_steps;
  real outlier_chi2, max_step_mm, mass_gev, cov_inflation, mat_Z, mat_A, mat_rho, mat_I_eV, step_tolerance_mm;
  int32_t field_gradient; /* 1: the step Jacobian carries the dB/dr terms of a grid field (reading U32) */
} options_r;

/* ---- tiny dense helpers ------------------------------------------------------------------- */
static void cross3(const real a[3], const real b[3], real c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
static real dot3(const real a[3], const real b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}
/* C (n x m) = A (n x k) * B (k x m) */
static void matmul(int n, int k, int m, const real* A, const real* B, real* C) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < m; ++j) {
      real s = 0.0;
      for (int l = 0; l < k; ++l) s += A[i * k + l] * B[l * m + j];
      C[i * m + j] = s;
    }
}
/* C (n x m) = A (n x k) * B^T, B is (m x k) */
static void matmul_bt(int n, int k, int m, const real* A, const real* B, real* C) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < m; ++j) {
      real s = 0.0;
      for (int l = 0; l < k; ++l) s += A[i * k + l] * B[j * k + l];
      C[i * m + j] = s;
    }
}
static void symmetrise6(real C[36]) {
  for (int i = 0; i < 6; ++i)
    for (int j = i + 1; j < 6; ++j) {
      real a = 0.5 * (C[i * 6 + j] + C[j * 6 + i]);
      C[i * 6 + j] = a;
      C[j * 6 + i] = a;
    }
}
static int all_finite(const real* a, int n) {
  for (int i = 0; i < n; ++i)
    if (!isfinite(a[i])) return 0;
  return 1;
}
static real wrap_pi(real a) { /* into (-pi, pi]: a - 2 pi ceil((a - pi) / (2 pi)); NaN for a non-finite a */
  if (a > PI || a <= -PI) a = a - (2.0 * PI) * ceil((a - PI) / (2.0 * PI));
  return a;
}

/* ---- field (C.2.2 "Field") ----------------------------------------------------------------- */
static void field_at_r(const field_r* fld, const real r[3], real b[3], int32_t* clamped) {
  if (fld->kind == KFO_FIELD_CONST) {
    b[0] = fld->b[0]; b[1] = fld->b[1]; b[2] = fld->b[2];
    return;
  }
  /* trilinear: per axis f = (r_a - origin_a)/spacing_a, i = clamp(floor f, 0, n_a-2),
     w = clamp(f - i, 0, 1); outside the grid the clamped value is used */
  int idx[3];
  real w[3];
  for (int a = 0; a < 3; ++a) {
    real f = (r[a] - fld->origin[a]) / fld->spacing[a];
    real fl = floor(f);
    if (fl < 0.0) fl = 0.0;
    if (fl > (real)(fld->n[a] - 2)) fl = (real)(fld->n[a] - 2);
    real ww = f - fl;
    if (ww < 0.0) { ww = 0.0; if (clamped) *clamped |= 1; }
    if (ww > 1.0) { ww = 1.0; if (clamped) *clamped |= 1; }
    idx[a] = (int)fl;
    w[a] = ww;
  }
  const int nx = fld->n[0], ny = fld->n[1];
  b[0] = b[1] = b[2] = 0.0;
  for (int dz = 0; dz < 2; ++dz)
    for (int dy = 0; dy < 2; ++dy)
      for (int dx = 0; dx < 2; ++dx) {
        real wt = (dx ? w[0] : 1.0 - w[0]) * (dy ? w[1] : 1.0 - w[1]) * (dz ? w[2] : 1.0 - w[2]);
        const double* node =
            fld->grid + 3 * ((size_t)(idx[2] + dz) * ny * nx + (size_t)(idx[1] + dy) * nx + (idx[0] + dx));
        b[0] += wt * (real)node[0];
        b[1] += wt * (real)node[1];
        b[2] += wt * (real)node[2];
      }
}

static void field_internal(const field_r* fld, const real r[3], real B[3], int32_t* clamped) {
  real bt[3];
  field_at_r(fld, r, bt, clamped);
  for (int a = 0; a < 3; ++a) B[a] = bt[a] * TESLA_TO_GEV_PER_MM; /* dT/ds = lam T x B */
}

/* dB_c/dr_a of the trilinear interpolant at r, in GeV/(e mm) per mm: G[c * 3 + a].  Along an axis on which the
 * lookup is clamped (r outside the grid) the interpolant is constant: zero derivative.  CONST field: zero. */
static void field_gradient_internal(const field_r* fld, const real r[3], real G[9]) {
  for (int i = 0; i < 9; ++i) G[i] = 0.0;
  if (fld->kind == KFO_FIELD_CONST) return;
  int idx[3], inside[3];
  real w[3];
  for (int a = 0; a < 3; ++a) {
    real f = (r[a] - fld->origin[a]) / fld->spacing[a];
    real fl = floor(f);
    if (fl < 0.0) fl = 0.0;
    if (fl > (real)(fld->n[a] - 2)) fl = (real)(fld->n[a] - 2);
    real ww = f - fl;
    inside[a] = 1;
    if (ww < 0.0) { ww = 0.0; inside[a] = 0; }
    if (ww > 1.0) { ww = 1.0; inside[a] = 0; }
    idx[a] = (int)fl;
    w[a] = ww;
  }
  const int nx = fld->n[0], ny = fld->n[1];
  for (int a = 0; a < 3; ++a) {
    if (!inside[a]) continue;
    /* d/dr_a of sum_corners prod_b w_b(d_b) node: the factor of axis a becomes (+1 or -1) / spacing_a */
    for (int dz = 0; dz < 2; ++dz)
      for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx) {
          const int d[3] = {dx, dy, dz};
          real wt = 1.0;
          for (int b = 0; b < 3; ++b) {
            if (b == a) wt *= (d[b] ? 1.0 : -1.0) / fld->spacing[a];
            else wt *= (d[b] ? w[b] : 1.0 - w[b]);
          }
          const double* node =
              fld->grid + 3 * ((size_t)(idx[2] + dz) * ny * nx + (size_t)(idx[1] + dy) * nx + (idx[0] + dx));
          for (int c = 0; c < 3; ++c) G[c * 3 + a] += wt * (real)node[c] * TESLA_TO_GEV_PER_MM;
        }
  }
}

/* M(B) a := a x B */
static void cross_matrix(const real B[3], real M[9]) {
  M[0] = 0.0;   M[1] = B[2];  M[2] = -B[1];
  M[3] = -B[2]; M[4] = 0.0;   M[5] = B[0];
  M[6] = B[1];  M[7] = -B[0]; M[8] = 0.0;
}

/* ---- C.2.2: one RKN4 step with its step Jacobian -------------------------------------------- */
static void rkn4_step_r(const field_r* fld, real mass, const real f[8], real h, real fo[8],
                   real Ds[64], real* eps, int32_t* clamped, int grad) {
  const real* r = f;
  const real t = f[3];
  const real* T = f + 4;
  const real lam = f[7];
  real B1[3], B2[3], B3[3], k1[3], k2[3], k3[3], k4[3], tmp[3], rm[3], re[3];
  real T2[3], T3[3], T4[3];

  /* stages; the field is sampled at 3 points, stages 2 and 3 share the midpoint */
  field_internal(fld, r, B1, clamped);
  cross3(T, B1, tmp);
  for (int a = 0; a < 3; ++a) k1[a] = lam * tmp[a];
  for (int a = 0; a < 3; ++a) rm[a] = r[a] + 0.5 * h * T[a] + 0.125 * h * h * k1[a];
  field_internal(fld, rm, B2, clamped);
  for (int a = 0; a < 3; ++a) T2[a] = T[a] + 0.5 * h * k1[a];
  cross3(T2, B2, tmp);
  for (int a = 0; a < 3; ++a) k2[a] = lam * tmp[a];
  for (int a = 0; a < 3; ++a) T3[a] = T[a] + 0.5 * h * k2[a];
  cross3(T3, B2, tmp);
  for (int a = 0; a < 3; ++a) k3[a] = lam * tmp[a];
  for (int a = 0; a < 3; ++a) re[a] = r[a] + h * T[a] + 0.5 * h * h * k3[a];
  field_internal(fld, re, B3, clamped);
  for (int a = 0; a < 3; ++a) T4[a] = T[a] + h * k3[a];
  cross3(T4, B3, tmp);
  for (int a = 0; a < 3; ++a) k4[a] = lam * tmp[a];

  /* state */
  real Tn[3], norm = 0.0;
  for (int a = 0; a < 3; ++a) {
    fo[a] = r[a] + h * T[a] + h * h / 6.0 * (k1[a] + k2[a] + k3[a]);
    Tn[a] = T[a] + h / 6.0 * (k1[a] + 2.0 * k2[a] + 2.0 * k3[a] + k4[a]);
    norm += Tn[a] * Tn[a];
  }
  norm = sqrt(norm);
  for (int a = 0; a < 3; ++a) fo[4 + a] = Tn[a] / norm;
  const real dtds = sqrt(1.0 + mass * mass * lam * lam); /* dt/ds = 1/beta, |q| = 1 */
  fo[3] = t + h * dtds;
  fo[7] = lam;

  /* embedded error estimate (diagnostic only) */
  real e = 0.0;
  for (int a = 0; a < 3; ++a) e += fabs(k1[a] - k2[a] - k3[a] + k4[a]);
  if (eps) *eps = h * h * e;

  if (!Ds) return;
  if (grad) {
    /* Step Jacobian WITH the field-gradient terms (reading U32): the derivative of the stage arithmetic above,
     * column by column.  For the variation (dr, dT, dlam) of the step's input, with G_i = dB/dr at stage point i:
     *   dk1 = dlam (T x B1) + lam (dT x B1 + T x (G1 dr))
     *   dr2 = dr + (h/2) dT + (h^2/8) dk1,  dT2 = dT + (h/2) dk1,  dk2 = dlam (T2 x B2) + lam (dT2 x B2 + T2 x (G2 dr2))
     *   dT3 = dT + (h/2) dk2 (same point),                         dk3 = dlam (T3 x B2) + lam (dT3 x B2 + T3 x (G2 dr2))
     *   dr4 = dr + h dT + (h^2/2) dk3,      dT4 = dT + h dk3,      dk4 = dlam (T4 x B3) + lam (dT4 x B3 + T4 x (G3 dr4))
     *   dr' = dr + h dT + (h^2/6)(dk1 + dk2 + dk3),   dT' = dT + (h/6)(dk1 + 2 dk2 + 2 dk3 + dk4)
     * (h fixed: the dependence of the step length on the state is the path-length correction's business; the
     * normalisation of T' is left out as in the gradient-free Jacobian below). */
    real G1[9], G2[9], G3[9];
    field_gradient_internal(fld, r, G1);
    field_gradient_internal(fld, rm, G2);
    field_gradient_internal(fld, re, G3);
    memset(Ds, 0, 64 * sizeof(real));
    for (int col = 0; col < 8; ++col) {
      real dr[3] = {0.0, 0.0, 0.0}, dT[3] = {0.0, 0.0, 0.0}, dlam = 0.0, dt = 0.0;
      if (col < 3) dr[col] = 1.0;
      else if (col == 3) dt = 1.0;
      else if (col < 7) dT[col - 4] = 1.0;
      else dlam = 1.0;
      real dk1[3], dk2[3], dk3[3], dk4[3], dB[3], a1[3], a2[3], a3[3], drs[3], dTs[3];
      /* stage 1 */
      matmul(3, 3, 1, G1, dr, dB);
      cross3(T, B1, a1); cross3(dT, B1, a2); cross3(T, dB, a3);
      for (int a = 0; a < 3; ++a) dk1[a] = dlam * a1[a] + lam * (a2[a] + a3[a]);
      /* stage 2 */
      for (int a = 0; a < 3; ++a) { drs[a] = dr[a] + 0.5 * h * dT[a] + 0.125 * h * h * dk1[a]; dTs[a] = dT[a] + 0.5 * h * dk1[a]; }
      matmul(3, 3, 1, G2, drs, dB);
      cross3(T2, B2, a1); cross3(dTs, B2, a2); cross3(T2, dB, a3);
      for (int a = 0; a < 3; ++a) dk2[a] = dlam * a1[a] + lam * (a2[a] + a3[a]);
      /* stage 3: same point, direction T3 */
      for (int a = 0; a < 3; ++a) dTs[a] = dT[a] + 0.5 * h * dk2[a];
      cross3(T3, B2, a1); cross3(dTs, B2, a2); cross3(T3, dB, a3);
      for (int a = 0; a < 3; ++a) dk3[a] = dlam * a1[a] + lam * (a2[a] + a3[a]);
      /* stage 4 */
      for (int a = 0; a < 3; ++a) { drs[a] = dr[a] + h * dT[a] + 0.5 * h * h * dk3[a]; dTs[a] = dT[a] + h * dk3[a]; }
      matmul(3, 3, 1, G3, drs, dB);
      cross3(T4, B3, a1); cross3(dTs, B3, a2); cross3(T4, dB, a3);
      for (int a = 0; a < 3; ++a) dk4[a] = dlam * a1[a] + lam * (a2[a] + a3[a]);
      for (int a = 0; a < 3; ++a) {
        Ds[a * 8 + col] = dr[a] + h * dT[a] + h * h / 6.0 * (dk1[a] + dk2[a] + dk3[a]);
        Ds[(4 + a) * 8 + col] = dT[a] + h / 6.0 * (dk1[a] + 2.0 * dk2[a] + 2.0 * dk3[a] + dk4[a]);
      }
      Ds[3 * 8 + col] = dt + h * mass * mass * lam / dtds * dlam;
      Ds[7 * 8 + col] = dlam;
    }
    return;
  }
  /* step Jacobian, field gradient neglected (reading U4) */
  real M1[9], M2[9], M3[9], d1[9], d2[9], d3[9], d4[9], P[9];
  cross_matrix(B1, M1);
  cross_matrix(B2, M2);
  cross_matrix(B3, M3);
  for (int i = 0; i < 9; ++i) d1[i] = lam * M1[i];
  for (int i = 0; i < 9; ++i) P[i] = 0.5 * h * d1[i];
  P[0] += 1.0; P[4] += 1.0; P[8] += 1.0;
  matmul(3, 3, 3, M2, P, d2);
  for (int i = 0; i < 9; ++i) d2[i] *= lam;
  for (int i = 0; i < 9; ++i) P[i] = 0.5 * h * d2[i];
  P[0] += 1.0; P[4] += 1.0; P[8] += 1.0;
  matmul(3, 3, 3, M2, P, d3);
  for (int i = 0; i < 9; ++i) d3[i] *= lam;
  for (int i = 0; i < 9; ++i) P[i] = h * d3[i];
  P[0] += 1.0; P[4] += 1.0; P[8] += 1.0;
  matmul(3, 3, 3, M3, P, d4);
  for (int i = 0; i < 9; ++i) d4[i] *= lam;

  real l1[3], l2[3], l3[3], l4[3], q[3], c1[3], c2[3];
  cross3(T, B1, l1);
  cross3(T2, B2, c1);
  for (int a = 0; a < 3; ++a) q[a] = 0.5 * h * l1[a];
  cross3(q, B2, c2);
  for (int a = 0; a < 3; ++a) l2[a] = c1[a] + lam * c2[a];
  cross3(T3, B2, c1);
  for (int a = 0; a < 3; ++a) q[a] = 0.5 * h * l2[a];
  cross3(q, B2, c2);
  for (int a = 0; a < 3; ++a) l3[a] = c1[a] + lam * c2[a];
  cross3(T4, B3, c1);
  for (int a = 0; a < 3; ++a) q[a] = h * l3[a];
  cross3(q, B3, c2);
  for (int a = 0; a < 3; ++a) l4[a] = c1[a] + lam * c2[a];

  memset(Ds, 0, 64 * sizeof(real));
  for (int i = 0; i < 8; ++i) Ds[i * 8 + i] = 1.0;
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) {
      /* dr'/dT = h I + h^2/6 (d1+d2+d3);  dT'/dT = I + h/6 (d1+2d2+2d3+d4) */
      Ds[i * 8 + (4 + j)] = (i == j ? h : 0.0) + h * h / 6.0 * (d1[i * 3 + j] + d2[i * 3 + j] + d3[i * 3 + j]);
      Ds[(4 + i) * 8 + (4 + j)] =
          (i == j ? 1.0 : 0.0) + h / 6.0 * (d1[i * 3 + j] + 2.0 * d2[i * 3 + j] + 2.0 * d3[i * 3 + j] + d4[i * 3 + j]);
    }
    Ds[i * 8 + 7] = h * h / 6.0 * (l1[i] + l2[i] + l3[i]);                        /* dr'/dlam */
    Ds[(4 + i) * 8 + 7] = h / 6.0 * (l1[i] + 2.0 * l2[i] + 2.0 * l3[i] + l4[i]);  /* dT'/dlam */
  }
  Ds[3 * 8 + 7] = h * mass * mass * lam / dtds; /* dt'/dlam */
}

/* ---- surfaces ("surfaces of different concrete types for different tracking detectors";
 * DESIGN.md reading U33).  Record entry [18] = kind:
 *   0 PLANE     centre c, orthonormal u, v, n = u x v;  r = c + loc0 u + loc1 v
 *   1 CYLINDER  axis v through c, radius R = entry [12], azimuth alpha = loc0 / R measured from n towards u:
 *               r = c + R (cos alpha n + sin alpha u) + loc1 v     (loc0 = R alpha: the arc length, loc1: along the axis)
 *   2 DISC      the plane through c with normal n in polar coordinates: r = c + rho (cos alpha u + sin alpha v),
 *               loc0 = rho > 0, loc1 = alpha in (-pi, pi]
 * Each kind provides: local -> global with the tangent vectors dr/dloc; global -> local with the rows dloc/dr;
 * the unit normal at a point; the straight-line path length from (r, T) to the surface. */
enum { SURF_PLANE = 0, SURF_CYLINDER = 1, SURF_DISC = 2 };
static int surf_kind(const real* s) { return (int)s[18]; }

static void local_to_global(const real* s, real l0, real l1, real r[3], real e0[3], real e1[3]) {
  const real *c = s, *u = s + 3, *v = s + 6, *n = s + 9;
  const int kind = surf_kind(s);
  if (kind == SURF_CYLINDER) {
    const real R = s[12], al = l0 / R, ca = cos(al), sa = sin(al);
    for (int a = 0; a < 3; ++a) {
      r[a] = c[a] + R * (ca * n[a] + sa * u[a]) + l1 * v[a];
      e0[a] = -sa * n[a] + ca * u[a]; /* dr/dloc0 = (1/R) dr/dalpha */
      e1[a] = v[a];
    }
  } else if (kind == SURF_DISC) {
    const real ca = cos(l1), sa = sin(l1);
    for (int a = 0; a < 3; ++a) {
      r[a] = c[a] + l0 * (ca * u[a] + sa * v[a]);
      e0[a] = ca * u[a] + sa * v[a];          /* dr/drho */
      e1[a] = l0 * (-sa * u[a] + ca * v[a]);  /* dr/dalpha */
    }
  } else {
    for (int a = 0; a < 3; ++a) {
      r[a] = c[a] + l0 * u[a] + l1 * v[a];
      e0[a] = u[a];
      e1[a] = v[a];
    }
  }
}

/* unit normal of the surface at the point r (which lies on it) */
static void surface_normal(const real* s, const real r[3], real nrm[3]) {
  const real *c = s, *v = s + 6, *n = s + 9;
  if (surf_kind(s) == SURF_CYLINDER) {
    real d[3] = {r[0] - c[0], r[1] - c[1], r[2] - c[2]};
    const real z = dot3(d, v);
    real dp[3] = {d[0] - z * v[0], d[1] - z * v[1], d[2] - z * v[2]};
    const real rho = sqrt(dot3(dp, dp));
    for (int a = 0; a < 3; ++a) nrm[a] = dp[a] / rho;
  } else {
    for (int a = 0; a < 3; ++a) nrm[a] = n[a];
  }
}

/* local coordinates of the point r on the surface and the rows g0 = dloc0/dr, g1 = dloc1/dr */
static void global_to_local(const real* s, const real r[3], real* l0, real* l1, real g0[3], real g1[3]) {
  const real *c = s, *u = s + 3, *v = s + 6, *n = s + 9;
  const real d[3] = {r[0] - c[0], r[1] - c[1], r[2] - c[2]};
  const int kind = surf_kind(s);
  if (kind == SURF_CYLINDER) {
    const real R = s[12];
    const real dn = dot3(d, n), du = dot3(d, u);
    const real al = atan2(du, dn), rho2 = dn * dn + du * du;
    *l0 = R * al;
    *l1 = dot3(d, v);
    for (int a = 0; a < 3; ++a) {
      g0[a] = R * (dn * u[a] - du * n[a]) / rho2; /* R dalpha/dr */
      g1[a] = v[a];
    }
  } else if (kind == SURF_DISC) {
    const real du = dot3(d, u), dv = dot3(d, v);
    const real rho = sqrt(du * du + dv * dv);
    *l0 = rho;
    *l1 = atan2(dv, du);
    for (int a = 0; a < 3; ++a) {
      g0[a] = (du * u[a] + dv * v[a]) / rho;
      g1[a] = (du * v[a] - dv * u[a]) / (rho * rho);
    }
  } else {
    *l0 = dot3(u, d);
    *l1 = dot3(v, d);
    for (int a = 0; a < 3; ++a) {
      g0[a] = u[a];
      g1[a] = v[a];
    }
  }
}

/* Straight-line path length h from (r, T) to the surface.  Planes and discs: h = n.(c - r)/(n.T), n.T > NT_MIN.
 * Cylinder: with d, T projected on the plane normal to the axis, |d_p + h T_p|^2 = R^2, i.e. a h^2 + 2 b h + c0 = 0,
 * a = |T_p|^2, b = d_p.T_p, c0 = |d_p|^2 - R^2; the root taken is the larger of the two textbook roots
 * (-b -+ sqrt(b^2 - a c0)) / a: the crossing ahead for a track inside the cylinder (c0 < 0), and the root next to the
 * point once the track is within round-off of the surface and moving outwards.  Returns 0 when the surface cannot
 * be reached. */
static int path_to_surface(const real* s, const real r[3], const real T[3], real* h) {
  const real *c = s, *v = s + 6, *n = s + 9;
  if (surf_kind(s) == SURF_CYLINDER) {
    const real R = s[12];
    real d[3] = {r[0] - c[0], r[1] - c[1], r[2] - c[2]};
    const real dz = dot3(d, v), tz = dot3(T, v);
    real dp[3], tp[3];
    for (int a = 0; a < 3; ++a) { dp[a] = d[a] - dz * v[a]; tp[a] = T[a] - tz * v[a]; }
    const real a2 = dot3(tp, tp), b = dot3(dp, tp), c0 = dot3(dp, dp) - R * R;
    const real disc = b * b - a2 * c0;
    if (!(disc > 0.0)) return 0;            /* the line misses the cylinder, or runs along its axis (a = 0) */
    const real sq = sqrt(disc);
    if (!(b + sq > NT_MIN * R)) return 0;   /* reading U33: grazing, or moving inwards from on / outside the surface */
    /* the textbook roots (-b -+ sqrt(b^2 - a c0)) / a, both formed; sq > 0 and a > 0, so root_hi > root_lo.  Inside the
     * cylinder (c0 < 0) they straddle zero and root_hi is the crossing ahead; on the surface to round-off and moving
     * outwards root_hi is the one next to the point (the correction), root_lo the crossing far behind.  Either way
     * the larger root.  (Its cancellation next to the surface is an absolute error of eps b / a ~ 1e-14 mm in h: no
     * stable rearrangement is needed at the 1e-10 bars, and none is used -- the kernel's form is not copied here.) */
    const real root_lo = (-b - sq) / a2, root_hi = (-b + sq) / a2;
    *h = root_hi > root_lo ? root_hi : root_lo;
    return 1;
  }
  const real nT = dot3(n, T);
  if (!(nT > NT_MIN)) return 0;
  real dr[3] = {c[0] - r[0], c[1] - r[1], c[2] - r[2]};
  *h = dot3(n, dr) / nT;
  return 1;
}

/* ---- C.2.1 - C.2.3: bound -> bound propagation with the 6x6 Jacobian ------------------------ */
static int32_t propagate_r(const field_r* fld, const options_r* opt, const real x[6],
                      const real* sf, const real* st, real xo[6], real J[36],
                      real free_out[8], real* rk_err, int32_t* clamped) {
  const real mass = opt->mass_gev;

  /* C.2.1 bound -> free on the start surface */
  const real sphi = sin(x[2]), cphi = cos(x[2]), sth = sin(x[3]), cth = cos(x[3]);
  real f[8], e0[3], e1[3];
  local_to_global(sf, x[0], x[1], f, e0, e1);
  f[3] = x[5];
  f[4] = cphi * sth; f[5] = sphi * sth; f[6] = cth;
  f[7] = x[4];
  real Jb2f[48];
  memset(Jb2f, 0, sizeof(Jb2f));
  for (int a = 0; a < 3; ++a) {
    Jb2f[a * 6 + 0] = e0[a];
    Jb2f[a * 6 + 1] = e1[a];
  }
  Jb2f[3 * 6 + 5] = 1.0;
  Jb2f[4 * 6 + 2] = -sphi * sth; Jb2f[4 * 6 + 3] = cphi * cth;
  Jb2f[5 * 6 + 2] = cphi * sth;  Jb2f[5 * 6 + 3] = sphi * cth;
  Jb2f[6 * 6 + 2] = 0.0;         Jb2f[6 * 6 + 3] = -sth;
  Jb2f[7 * 6 + 4] = 1.0;

  /* C.2.2 stepping: exactly n_sub + n_corr RKN4 steps, no tolerance test, no early exit */
  real D[64], Ds[64], Dn[64];
  memset(D, 0, sizeof(D));
  for (int i = 0; i < 8; ++i) D[i * 8 + i] = 1.0;
  real errmax = 0.0;
  int n_sub = 1;
  {
    real s0;
    if (!path_to_surface(st, f, f + 4, &s0)) return KFO_ST_PROPAGATION;
    /* A cylinder is reached from inside (kf_fit.h KF_SURFACE_CYLINDER; reading U33): the first aim of a leg
     * must lie ahead.  A start point outside the cylinder and moving away from it has its chosen root behind it
     * (s0 <= 0) -- that is "cannot be reached", not a step backwards.  (Moving inwards from outside, the chosen root's
     * denominator is negative and path_to_surface has already refused.)  Later aims of the same leg may be slightly
     * negative: they are corrections around the surface. */
    if (surf_kind(st) == SURF_CYLINDER && !(s0 > 0.0)) return KFO_ST_PROPAGATION;
    if (isfinite(opt->max_step_mm) && opt->max_step_mm > 0.0) {
      real q = ceil(fabs(s0) / opt->max_step_mm * (1.0 - 1e-12));
      if (!(q >= 1.0)) q = 1.0;
      if (q > (real)MAX_SUBSTEPS) q = (real)MAX_SUBSTEPS;
      n_sub = (int)q;
    }
    /* Adaptive step count ("adaptive Runge-Kutta-Nystrom"; reading U31): the embedded
     * error estimate eps0 of ONE trial step over the whole leg (the step itself is discarded) fixes the number of
     * primary steps.  eps = h^2 |k1-k2-k3+k4|_1 falls with the fourth power of the step, so
     * n = ceil((eps0 / tol)^(1/4)) steps bring the estimate of each to about tol.  A rule on a number, decided once
     * per leg before any step is taken: no accept/reject loop. */
    if (isfinite(opt->step_tolerance_mm) && opt->step_tolerance_mm > 0.0) {
      real ft[8], Dt_[64], e0 = 0.0;
      rkn4_step_r(fld, mass, f, s0, ft, Dt_, &e0, clamped, 0);
      real q = ceil(sqrt(sqrt(e0 / opt->step_tolerance_mm)) * (1.0 - 1e-12));
      if (!(q >= 1.0)) q = 1.0;
      if (q > (real)MAX_SUBSTEPS) q = (real)MAX_SUBSTEPS;
      if ((int)q > n_sub) n_sub = (int)q;
    }
  }
  const int n_steps = n_sub + opt->n_corr_steps;
  for (int is = 0; is < n_steps; ++is) {
    real h;
    if (!path_to_surface(st, f, f + 4, &h)) return KFO_ST_PROPAGATION;
    if (is < n_sub) h = h / (real)(n_sub - is); /* the last primary step aims at the surface */
    real fn[8], e = 0.0;
    rkn4_step_r(fld, mass, f, h, fn, Ds, &e, clamped, opt->field_gradient);
    if (e > errmax) errmax = e;
    matmul(8, 8, 8, Ds, D, Dn);
    memcpy(D, Dn, sizeof(D));
    memcpy(f, fn, sizeof(f));
    if (!all_finite(f, 8)) return KFO_ST_PROPAGATION;
  }
  if (rk_err) *rk_err = errmax;

  /* C.2.3 free -> bound with the path-length correction */
  const real* r = f;
  const real* T = f + 4;
  const real lam = f[7];
  real nt[3];
  surface_normal(st, r, nt); /* planes, discs: the record's n; cylinder: the radial direction at r */
  const real nT = dot3(nt, T);
  if (!(nT > NT_MIN)) return KFO_ST_PROPAGATION;
  real B[3], TxB[3];
  field_internal(fld, r, B, clamped);
  cross3(T, B, TxB);
  real fp[8] = {T[0], T[1], T[2], sqrt(1.0 + mass * mass * lam * lam),
                  lam * TxB[0], lam * TxB[1], lam * TxB[2], 0.0};
  real w[8] = {nt[0] / nT, nt[1] / nT, nt[2] / nT, 0.0, 0.0, 0.0, 0.0, 0.0};
  real Pm[64];
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 8; ++j) Pm[i * 8 + j] = (i == j ? 1.0 : 0.0) - fp[i] * w[j];
  real Dt[64];
  matmul(8, 8, 8, Pm, D, Dt);

  const real thn = acos(T[2] > 1.0 ? 1.0 : (T[2] < -1.0 ? -1.0 : T[2]));
  const real phn = atan2(T[1], T[0]);
  const real s2 = sin(thn), c2 = cos(thn), sp = sin(phn), cp = cos(phn);
  if (!(s2 > SIN_THETA_MIN)) return KFO_ST_THETA;
  real g0[3], g1[3];
  global_to_local(st, r, &xo[0], &xo[1], g0, g1);
  xo[2] = phn;
  xo[3] = thn;
  xo[4] = lam;
  xo[5] = f[3];
  real Jf2b[48];
  memset(Jf2b, 0, sizeof(Jf2b));
  for (int a = 0; a < 3; ++a) {
    Jf2b[0 * 8 + a] = g0[a];
    Jf2b[1 * 8 + a] = g1[a];
  }
  Jf2b[2 * 8 + 4] = -sp / s2; Jf2b[2 * 8 + 5] = cp / s2; Jf2b[2 * 8 + 6] = 0.0;
  Jf2b[3 * 8 + 4] = cp * c2;  Jf2b[3 * 8 + 5] = sp * c2; Jf2b[3 * 8 + 6] = -s2;
  Jf2b[4 * 8 + 7] = 1.0;
  Jf2b[5 * 8 + 3] = 1.0;
  real A68[48];
  matmul(6, 8, 8, Jf2b, Dt, A68);
  matmul(6, 8, 6, A68, Jb2f, J);
  if (free_out) memcpy(free_out, f, sizeof(f));
  if (!all_finite(xo, 6) || !all_finite(J, 36)) return KFO_ST_PROPAGATION;
  return 0;
}

/* ---- perigee: bound state on a plane -> bound state on a LINE surface --------
 * The perigee surface of the paper is "defined at the point of closest approach to a reference
 * point"; there loc0, loc1 "become the transverse and longitudinal impact parameters d0 and z0".
 * Here (readings U27-U30) the surface is a straight line through c with unit direction
 * a (the beam axis).  With D = r - c and D_perp = D - (D.a) a, the state is ON the surface when
 *     g(r, T) = D_perp . T = 0            (closest approach of the tangent to the axis),
 * and its local coordinates are  d0 = D . e_d,  e_d = (a x T)/|a x T|,   z0 = D . a.
 * Stepping: the same fixed policy as for planes (n_sub + n_corr RKN4 steps, no accept/reject), each
 * step aimed with the Newton root of g along the track:  h = -g / (dg/ds),
 * dg/ds = 1 - (a.T)^2 + lam D_perp . (T x B)  (the curvature term keeps the convergence quadratic when the
 * track passes the axis at a distance); h may be negative (the perigee lies behind the first plane).
 * Jacobian: J = J_f2b (I - f' w^T) D J_b2f with w = grad g / (dg/ds),
 *   grad_r g = T - (a.T) a,  grad_T g = D_perp,  dg/ds = 1 - (a.T)^2 + lam D_perp . (T x B);
 *   J_f2b rows: d0: e_d on r (its T-derivative vanishes on the surface, where D_perp || e_d),
 *   z0: a on r, angles / q/p / t as for planes.
 * C_out = J C J^T.  No material is crossed.  Returns 0 or the status bit that stopped it. */
static int32_t to_line_r(const field_r* fld, const options_r* opt, const real x[6], const real C[36],
                    const real* sf, const real lc[3], const real la[3], real xo[6], real Co[36],
                    real J[36], int32_t* clamped) {
  const real mass = opt->mass_gev;
  const real sphi = sin(x[2]), cphi = cos(x[2]), sth = sin(x[3]), cth = cos(x[3]);
  real f[8], e0[3], e1[3];
  local_to_global(sf, x[0], x[1], f, e0, e1);
  f[3] = x[5];
  f[4] = cphi * sth; f[5] = sphi * sth; f[6] = cth;
  f[7] = x[4];
  real Jb2f[48];
  memset(Jb2f, 0, sizeof(Jb2f));
  for (int a = 0; a < 3; ++a) {
    Jb2f[a * 6 + 0] = e0[a];
    Jb2f[a * 6 + 1] = e1[a];
  }
  Jb2f[3 * 6 + 5] = 1.0;
  Jb2f[4 * 6 + 2] = -sphi * sth; Jb2f[4 * 6 + 3] = cphi * cth;
  Jb2f[5 * 6 + 2] = cphi * sth;  Jb2f[5 * 6 + 3] = sphi * cth;
  Jb2f[6 * 6 + 2] = 0.0;         Jb2f[6 * 6 + 3] = -sth;
  Jb2f[7 * 6 + 4] = 1.0;

  real D[64], Ds[64], Dn[64];
  memset(D, 0, sizeof(D));
  for (int i = 0; i < 8; ++i) D[i * 8 + i] = 1.0;
  int n_sub = 1;
  for (int is = 0;; ++is) {
    const real* T = f + 4;
    const real aT = dot3(la, T);
    const real den = 1.0 - aT * aT;
    if (!(den > 1e-12)) return KFO_ST_PROPAGATION; /* moving along the axis: no closest approach */
    real dl[3] = {f[0] - lc[0], f[1] - lc[1], f[2] - lc[2]};
    const real da = dot3(dl, la);
    real dperp[3] = {dl[0] - da * la[0], dl[1] - da * la[1], dl[2] - da * la[2]};
    /* Newton step on g along the track: dg/ds = 1 - (a.T)^2 + lam D_perp . (T x B) */
    real Bs[3], TxBs[3];
    field_internal(fld, f, Bs, clamped);
    cross3(T, Bs, TxBs);
    const real slope = den + f[7] * dot3(dperp, TxBs);
    if (!(fabs(slope) > 1e-12)) return KFO_ST_PROPAGATION;
    real h = -dot3(dperp, T) / slope;
    if (is == 0 && isfinite(opt->max_step_mm) && opt->max_step_mm > 0.0) {
      real q = ceil(fabs(h) / opt->max_step_mm * (1.0 - 1e-12));
      if (!(q >= 1.0)) q = 1.0;
      if (q > (real)MAX_SUBSTEPS) q = (real)MAX_SUBSTEPS;
      n_sub = (int)q;
    }
    if (is >= n_sub + opt->n_corr_steps) break;
    if (is < n_sub) h = h / (real)(n_sub - is);
    real fn[8], e = 0.0;
    rkn4_step_r(fld, mass, f, h, fn, Ds, &e, clamped, 0); /* the perigee extrapolation neglects dB/dr (U32) */
    matmul(8, 8, 8, Ds, D, Dn);
    memcpy(D, Dn, sizeof(D));
    memcpy(f, fn, sizeof(f));
    if (!all_finite(f, 8)) return KFO_ST_PROPAGATION;
  }

  const real* r = f;
  const real* T = f + 4;
  const real lam = f[7];
  const real aT = dot3(la, T);
  real dl[3] = {r[0] - lc[0], r[1] - lc[1], r[2] - lc[2]};
  const real da = dot3(dl, la);
  real dperp[3] = {dl[0] - da * la[0], dl[1] - da * la[1], dl[2] - da * la[2]};
  real B[3], TxB[3];
  field_internal(fld, r, B, clamped);
  cross3(T, B, TxB);
  real fp[8] = {T[0], T[1], T[2], sqrt(1.0 + mass * mass * lam * lam),
                  lam * TxB[0], lam * TxB[1], lam * TxB[2], 0.0};
  const real dgds = 1.0 - aT * aT + lam * dot3(dperp, TxB);
  if (!(fabs(dgds) > 1e-12)) return KFO_ST_PROPAGATION;
  real w[8] = {(T[0] - aT * la[0]) / dgds, (T[1] - aT * la[1]) / dgds, (T[2] - aT * la[2]) / dgds, 0.0,
                 dperp[0] / dgds, dperp[1] / dgds, dperp[2] / dgds, 0.0};
  real Pm[64], Dt[64];
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 8; ++j) Pm[i * 8 + j] = (i == j ? 1.0 : 0.0) - fp[i] * w[j];
  matmul(8, 8, 8, Pm, D, Dt);

  const real thn = acos(T[2] > 1.0 ? 1.0 : (T[2] < -1.0 ? -1.0 : T[2]));
  const real phn = atan2(T[1], T[0]);
  const real s2 = sin(thn), c2 = cos(thn), sp = sin(phn), cp = cos(phn);
  if (!(s2 > SIN_THETA_MIN)) return KFO_ST_THETA;
  real ed[3];
  cross3(la, T, ed);
  const real edn = sqrt(dot3(ed, ed));
  for (int a = 0; a < 3; ++a) ed[a] /= edn;
  xo[0] = dot3(dl, ed);
  xo[1] = da;
  xo[2] = phn;
  xo[3] = thn;
  xo[4] = lam;
  xo[5] = f[3];
  real Jf2b[48];
  memset(Jf2b, 0, sizeof(Jf2b));
  for (int a = 0; a < 3; ++a) {
    Jf2b[0 * 8 + a] = ed[a];
    Jf2b[1 * 8 + a] = la[a];
  }
  Jf2b[2 * 8 + 4] = -sp / s2; Jf2b[2 * 8 + 5] = cp / s2; Jf2b[2 * 8 + 6] = 0.0;
  Jf2b[3 * 8 + 4] = cp * c2;  Jf2b[3 * 8 + 5] = sp * c2; Jf2b[3 * 8 + 6] = -s2;
  Jf2b[4 * 8 + 7] = 1.0;
  Jf2b[5 * 8 + 3] = 1.0;
  real A68[48], JC[36];
  matmul(6, 8, 8, Jf2b, Dt, A68);
  matmul(6, 8, 6, A68, Jb2f, J);
  matmul(6, 6, 6, J, C, JC);
  matmul_bt(6, 6, 6, JC, J, Co);
  symmetrise6(Co);
  if (!all_finite(xo, 6) || !all_finite(J, 36) || !all_finite(Co, 36)) return KFO_ST_PROPAGATION;
  return 0;
}

/* ---- C.2.4: gain-matrix update ------------------------------------------------ */
static int32_t update_r(const real xp[6], const real Cp[36], const real m[2], const real V[4],
                   real xf[6], real Cf[36], real* chi2) {
  /* H = first two rows of I6 */
  const real r0 = m[0] - xp[0], r1 = m[1] - xp[1];
  const real S00 = Cp[0] + V[0], S01 = Cp[1] + V[1], S10 = Cp[6] + V[2], S11 = Cp[7] + V[3];
  const real det = S00 * S11 - S01 * S10;
  if (!(S00 > 0.0 && det > 0.0)) return KFO_ST_NOT_POSITIVE; /* S must be positive definite */
  const real Si00 = S11 / det, Si01 = -S01 / det, Si10 = -S10 / det, Si11 = S00 / det;
  *chi2 = r0 * (Si00 * r0 + Si01 * r1) + r1 * (Si10 * r0 + Si11 * r1);
  real K[12]; /* 6x2 = C H^T S^-1 */
  for (int i = 0; i < 6; ++i) {
    K[i * 2 + 0] = Cp[i * 6 + 0] * Si00 + Cp[i * 6 + 1] * Si10;
    K[i * 2 + 1] = Cp[i * 6 + 0] * Si01 + Cp[i * 6 + 1] * Si11;
  }
  for (int i = 0; i < 6; ++i) xf[i] = xp[i] + K[i * 2 + 0] * r0 + K[i * 2 + 1] * r1;
  /* C+ = (I - K H) C- */
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j)
      Cf[i * 6 + j] = Cp[i * 6 + j] - (K[i * 2 + 0] * Cp[0 * 6 + j] + K[i * 2 + 1] * Cp[1 * 6 + j]);
  symmetrise6(Cf);
  return 0;
}

/* ---- C.2.5: material after the update -------------------------------------------------------- */
static int32_t material_r(const options_r* opt, const real* surf, const real xf[6],
                     const real Cf[36], real xo[6], real Co[36], real* g_out,
                     real* theta0_out, real* dE_out) {
  real n[3], rpos[3], e0_[3], e1_[3];
  local_to_global(surf, xf[0], xf[1], rpos, e0_, e1_);
  surface_normal(surf, rpos, n); /* planes, discs: the record's n; cylinder: the radial direction at the state */
  const real xX0 = surf[14], thick = surf[15];
  const real m = opt->mass_gev;
  const real lam = xf[4];
  const real sth = sin(xf[3]), cth = cos(xf[3]), sph = sin(xf[2]), cph = cos(xf[2]);
  const real T[3] = {cph * sth, sph * sth, cth};
  const real p = 1.0 / fabs(lam);
  const real E = sqrt(p * p + m * m);
  const real beta = p / E, gamma = E / m;
  const real cfac = 1.0 / fabs(dot3(n, T)); /* path factor */

  /* multiple scattering, Highland (PDG form) */
  const real X = xX0 * cfac;
  const real theta0 = 0.0136 / (beta * p) * sqrt(X) * (1.0 + 0.038 * log(X / (beta * beta)));

  /* mean energy loss, Bethe with the asymptotic density correction */
  const real bg = p / m;
  const real I_exc = opt->mat_I_eV * 1e-9; /* GeV */
  const real ZA = opt->mat_Z / opt->mat_A;
  const real Wmax = 2.0 * ME_GEV * bg * bg / (1.0 + 2.0 * gamma * ME_GEV / m + (ME_GEV / m) * (ME_GEV / m));
  const real hwp = 28.816e-9 * sqrt(opt->mat_rho * ZA); /* GeV */
  real dhalf = log(hwp / I_exc) + log(bg) - 0.5;
  if (dhalf < 0.0) dhalf = 0.0;
  const real dedx_mass =
      K_BETHE * ZA / (beta * beta) * (0.5 * log(2.0 * ME_GEV * bg * bg * Wmax / (I_exc * I_exc)) - beta * beta - dhalf);
  /* MeV cm^2/g * g/cm^3 = MeV/cm -> GeV/mm: 1e-3 * 0.1 */
  const real dE = dedx_mass * opt->mat_rho * 1e-3 * 0.1 * thick * cfac;
  if (theta0_out) *theta0_out = theta0;
  if (dE_out) *dE_out = dE;
  const real E2 = E - dE;
  if (!(E2 > m)) return KFO_ST_ENERGY;
  const real p2 = sqrt(E2 * E2 - m * m);
  const real lam2 = (lam < 0.0 ? -1.0 : 1.0) / p2;
  const real g = (p * p * p * E2) / (p2 * p2 * p2 * E); /* dlam'/dlam, dE held constant */
  if (g_out) *g_out = g;

  for (int i = 0; i < 6; ++i) xo[i] = xf[i];
  xo[4] = lam2;
  real G[36], GC[36];
  memset(G, 0, sizeof(G));
  for (int i = 0; i < 6; ++i) G[i * 6 + i] = 1.0;
  G[4 * 6 + 4] = g;
  matmul(6, 6, 6, G, Cf, GC);
  matmul_bt(6, 6, 6, GC, G, Co);
  Co[2 * 6 + 2] += theta0 * theta0 / (sth * sth); /* Q_phiphi */
  Co[3 * 6 + 3] += theta0 * theta0;               /* Q_thetatheta */
  symmetrise6(Co);
  return 0;
}

/* ---- X = C^-1 B for an SPD 6x6 C (reading U19): Gaussian elimination with partial pivoting on the
 * correlation-scaled matrix R = D^-1 C D^-1, D = diag(sqrt(C_ii)), followed by back substitution.
 * A solve, not an explicit inverse: forming C^-1 and multiplying costs a factor cond(R) in accuracy,
 * which the cancellation in C^s = C+ + A (C^s' - C-') A^T then amplifies by |C+| / |C^s| (up to 1e6
 * for an inflated prior; pinned against the long-double build in tests/test_oracle_precision.py).
 * Independent of the CUDA path, which uses an un-pivoted Cholesky.
 * The whole routine runs in `sreal`: the paper keeps its matrix inversion in double whatever the
 * operand type, so the float build converts in and out here. -------- */

/* determinant of the leading k x k block of the 6x6 matrix R, by pivoted elimination */
static sreal leading_minor6(const sreal R[36], int k) {
  sreal T[36], det = 1.0;
  for (int i = 0; i < k; ++i)
    for (int j = 0; j < k; ++j) T[i * k + j] = R[i * 6 + j];
  for (int c = 0; c < k; ++c) {
    int piv = c;
    for (int i = c + 1; i < k; ++i)
      if (fabs(T[i * k + c]) > fabs(T[piv * k + c])) piv = i;
    if (T[piv * k + c] == 0.0) return 0.0;
    if (piv != c) {
      for (int j = 0; j < k; ++j) { sreal t = T[c * k + j]; T[c * k + j] = T[piv * k + j]; T[piv * k + j] = t; }
      det = -det;
    }
    det *= T[c * k + c];
    for (int i = c + 1; i < k; ++i) {
      const sreal f = T[i * k + c] / T[c * k + c];
      for (int j = c; j < k; ++j) T[i * k + j] -= f * T[c * k + j];
    }
  }
  return det;
}

static int32_t solve_spd6(const real Cin[36], const real Bin[36], real Xout[36]) {
  sreal C[36], B[36], X[36];
  for (int i = 0; i < 36; ++i) { C[i] = (sreal)Cin[i]; B[i] = (sreal)Bin[i]; }
  sreal s[6], R[36], Y[36];
  for (int i = 0; i < 6; ++i) {
    if (!(C[i * 6 + i] > 0.0)) return KFO_ST_NOT_POSITIVE;
    s[i] = sqrt(C[i * 6 + i]);
  }
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) {
      R[i * 6 + j] = C[i * 6 + j] / (s[i] * s[j]);
      Y[i * 6 + j] = B[i * 6 + j] / s[i]; /* R (D X) = D^-1 B */
    }
  /* the status decision is the definition: a symmetric matrix is positive definite iff its six leading
     principal minors are positive (Sylvester's criterion) */
  for (int k = 1; k <= 6; ++k)
    if (!(leading_minor6(R, k) > 0.0)) return KFO_ST_NOT_POSITIVE;
  for (int k = 0; k < 6; ++k) {
    int piv = k;
    for (int i = k + 1; i < 6; ++i)
      if (fabs(R[i * 6 + k]) > fabs(R[piv * 6 + k])) piv = i;
    if (piv != k)
      for (int j = 0; j < 6; ++j) {
        sreal t = R[k * 6 + j]; R[k * 6 + j] = R[piv * 6 + j]; R[piv * 6 + j] = t;
        t = Y[k * 6 + j]; Y[k * 6 + j] = Y[piv * 6 + j]; Y[piv * 6 + j] = t;
      }
    if (R[k * 6 + k] == 0.0) return KFO_ST_NOT_POSITIVE;
    for (int i = k + 1; i < 6; ++i) {
      const sreal f = R[i * 6 + k] / R[k * 6 + k];
      for (int j = k; j < 6; ++j) R[i * 6 + j] -= f * R[k * 6 + j];
      for (int j = 0; j < 6; ++j) Y[i * 6 + j] -= f * Y[k * 6 + j];
    }
  }
  for (int c = 0; c < 6; ++c)
    for (int i = 5; i >= 0; --i) {
      sreal v = Y[i * 6 + c];
      for (int j = i + 1; j < 6; ++j) v -= R[i * 6 + j] * X[j * 6 + c];
      X[i * 6 + c] = v / R[i * 6 + i];
    }
  for (int i = 0; i < 6; ++i) /* undo the scaling: X <- D^-1 (D X) */
    for (int c = 0; c < 6; ++c) Xout[i * 6 + c] = (real)(X[i * 6 + c] / s[i]);
  return 0;
}

/* ---- C.2.6: one RTS step ("stored Jacobians between states") ------------------- */
static int32_t rts_step_r(const real xf[6], const real Cf[36], const real F[36],
                     const real xp1[6], const real Cp1[36], const real xs1[6],
                     const real Cs1[36], real xs[6], real Cs[36]) {
  real FC[36], At[36], A[36];
  matmul(6, 6, 6, F, Cf, FC);          /* F C+_k  (C+ symmetric: = (C+ F^T)^T) */
  int32_t rc = solve_spd6(Cp1, FC, At); /* A_k^T = (C-_{k+1})^-1 F C+_k */
  if (rc) return rc;
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) A[i * 6 + j] = At[j * 6 + i]; /* A_k = C+_k F^T (C-_{k+1})^-1 */
  real dx[6];
  for (int i = 0; i < 6; ++i) dx[i] = xs1[i] - xp1[i];
  dx[2] = wrap_pi(dx[2]);
  for (int i = 0; i < 6; ++i) {
    real s = 0.0;
    for (int j = 0; j < 6; ++j) s += A[i * 6 + j] * dx[j];
    xs[i] = xf[i] + s;
  }
  real dC[36], AdC[36], AdCAt[36];
  for (int i = 0; i < 36; ++i) dC[i] = Cs1[i] - Cp1[i];
  matmul(6, 6, 6, A, dC, AdC);
  matmul_bt(6, 6, 6, AdC, A, AdCAt);
  for (int i = 0; i < 36; ++i) Cs[i] = Cf[i] + AdCAt[i];
  symmetrise6(Cs);
  if (!all_finite(xs, 6) || !all_finite(Cs, 36)) return KFO_ST_NOT_POSITIVE;
  return 0;
}

/* ---- double <-> real at the interface ------------------------------------------------------------------- */
static void get(real* dst, const double* src, int n) {
  for (int i = 0; i < n; ++i) dst[i] = (real)src[i];
}
static void put(double* dst, const real* src, int n) {
  for (int i = 0; i < n; ++i) dst[i] = (double)src[i];
}
static field_r field_to_real(const kfo_field* f) {
  field_r o;
  o.kind = f->kind;
  for (int a = 0; a < 3; ++a) {
    o.b[a] = (real)f->b[a];
    o.n[a] = f->n[a];
    o.origin[a] = (real)f->origin[a];
    o.spacing[a] = (real)f->spacing[a];
  }
  o.grid = f->grid;
  return o;
}
static options_r options_to_real(const kfo_options* p) {
  options_r o;
  o.smooth = p->smooth; o.material = p->material; o.n_corr_steps = p->n_corr_steps;
  o.outlier_chi2 = (real)p->outlier_chi2; o.max_step_mm = (real)p->max_step_mm; o.mass_gev = (real)p->mass_gev;
  o.cov_inflation = (real)p->cov_inflation; o.mat_Z = (real)p->mat_Z; o.mat_A = (real)p->mat_A;
  o.mat_rho = (real)p->mat_rho; o.mat_I_eV = (real)p->mat_I_eV; o.step_tolerance_mm = (real)p->step_tolerance_mm;
  o.field_gradient = p->field_gradient;
  return o;
}

/* ---- C.2: the per-track loop ----------------------------------------------------------------- */
typedef struct {
  real xp[6], Cp[36], F[36], xf[6], Cf[36];
} leg_record;

static void fill_nan(double* a, size_t n) {
  for (size_t i = 0; i < n; ++i) a[i] = NAN;
}

int32_t kfo_fit_batch(int64_t N, const double* params0, const double* cov0, int32_t start,
                      const int32_t* offsets, const int32_t* surf_idx, const double* loc,
                      const double* var, const double* cov01, int32_t n_surfaces,
                      const double* geom_in, const kfo_field* fld_in, const kfo_options* opt_in,
                      double* first_params, double* first_cov, double* last_params,
                      double* last_cov, double* chi2_out, int32_t* ndf_out, uint32_t* status_out,
                      int32_t* n_used_out, int32_t* n_out_out, int32_t* n_holes_out,
                      double* sp_par, double* sp_cov, double* sf_par, double* sf_cov,
                      double* ss_par, double* ss_cov, double* hit_chi2, uint8_t* hit_flags,
                      double* rk_err_max, int32_t n_threads) {
  if (N < 0 || !params0 || !cov0 || !offsets || !geom_in || !fld_in || !opt_in) return -1;
  if (start < 0 || start >= n_surfaces) return -1;
  const int Lmax = n_surfaces - 1 - start;
  /* the shared global data (geometry, field, options) as `real`, once */
  const field_r fld_v = field_to_real(fld_in);
  const options_r opt_v = options_to_real(opt_in);
  const field_r* fld = &fld_v;
  const options_r* opt = &opt_v;
  real* geom = (real*)malloc(sizeof(real) * (size_t)n_surfaces * KFO_GEOM_STRIDE);
  if (!geom) return -1;
  for (size_t a = 0; a < (size_t)n_surfaces * KFO_GEOM_STRIDE; ++a) geom[a] = (real)geom_in[a];
  int used_threads = 1;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#pragma omp parallel
  {
#pragma omp single
    used_threads = omp_get_num_threads();
  }
#endif

#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < N; ++i) {
    const int32_t o0 = offsets[i], o1 = offsets[i + 1];
    uint32_t status = 0;
    real x[6], C[36];
    for (int a = 0; a < 6; ++a) x[a] = (real)params0[i * 6 + a];
    for (int a = 0; a < 36; ++a) C[a] = opt->cov_inflation * (real)cov0[i * 36 + a];
    real first_x[6], first_C[36], last_x[6], last_C[36];
    memcpy(first_x, x, sizeof(x)); memcpy(first_C, C, sizeof(C));
    memcpy(last_x, x, sizeof(x));  memcpy(last_C, C, sizeof(C));
    real chi2 = 0.0, errmax = 0.0;
    int n_used = 0, n_outl = 0, n_holes = 0, nleg = 0;

    if (sp_par) fill_nan(sp_par + (size_t)i * Lmax * 6, (size_t)Lmax * 6);
    if (sp_cov) fill_nan(sp_cov + (size_t)i * Lmax * 36, (size_t)Lmax * 36);
    if (sf_par) fill_nan(sf_par + (size_t)i * Lmax * 6, (size_t)Lmax * 6);
    if (sf_cov) fill_nan(sf_cov + (size_t)i * Lmax * 36, (size_t)Lmax * 36);
    if (ss_par) fill_nan(ss_par + (size_t)i * Lmax * 6, (size_t)Lmax * 6);
    if (ss_cov) fill_nan(ss_cov + (size_t)i * Lmax * 36, (size_t)Lmax * 36);
    for (int32_t j = o0; j < o1; ++j) {
      if (hit_chi2) hit_chi2[j] = 0.0;
      if (hit_flags) hit_flags[j] = KFO_HIT_UNPROCESSED;
    }

    /* the hit list must be strictly ascending in surface index, inside (start, n_surfaces) */
    int ok = 1;
    {
      int32_t prev_s = start;
      for (int32_t j = o0; j < o1; ++j) {
        if (!(surf_idx[j] > prev_s && surf_idx[j] < n_surfaces)) { ok = 0; break; }
        prev_s = surf_idx[j];
      }
    }
    leg_record* rec = NULL;
    if (!ok) {
      status |= KFO_ST_BAD_HITS;
    } else if (o1 > o0) {
      const int n_target = surf_idx[o1 - 1] - start; /* reading U7: visit every surface up to the last hit */
      rec = (leg_record*)malloc(sizeof(leg_record) * (size_t)n_target);
      real g_prev = 1.0;
      int32_t hp = o0, prev = start;
      for (int32_t s = start + 1; s <= start + n_target; ++s) {
        const real* sf = geom + (size_t)prev * KFO_GEOM_STRIDE;
        const real* st = geom + (size_t)s * KFO_GEOM_STRIDE;
        leg_record* R = &rec[nleg];
        real J[36], e = 0.0;
        int32_t clamped = 0;
        int32_t rc = propagate_r(fld, opt, x, sf, st, R->xp, J, NULL, &e, &clamped);
        if (clamped) status |= KFO_ST_FIELD_CLAMPED;
        if (rc) { status |= (uint32_t)rc; break; }
        if (e > errmax) errmax = e;
        /* F = J G_prev (G_prev = diag(1,1,1,1,g,1) of the previous surface's energy loss) */
        real G[36], JC[36];
        memset(G, 0, sizeof(G));
        for (int a = 0; a < 6; ++a) G[a * 6 + a] = 1.0;
        G[4 * 6 + 4] = g_prev;
        matmul(6, 6, 6, J, G, R->F);
        /* C- = J C J^T  (C already holds G C+ G^T + Q of the previous surface) */
        matmul(6, 6, 6, J, C, JC);
        matmul_bt(6, 6, 6, JC, J, R->Cp);
        symmetrise6(R->Cp);

        if (hp < o1 && surf_idx[hp] == s) {
          real V[4];
          if (var) {
            V[0] = (real)var[(size_t)hp * 2 + 0];
            V[3] = (real)var[(size_t)hp * 2 + 1];
            V[1] = V[2] = cov01 ? (real)cov01[hp] : 0.0;
          } else {
            V[0] = st[16]; V[3] = st[17]; V[1] = V[2] = 0.0;
          }
          real c2 = 0.0, xf[6], Cf[36];
          real m[2] = {(real)loc[(size_t)hp * 2 + 0], (real)loc[(size_t)hp * 2 + 1]};
          /* angular local coordinates (reading U33): the hit is taken on the branch nearest the prediction -- the arc
             length R alpha of a cylinder has period 2 pi R, the azimuth of a disc 2 pi.  A residual already inside
             (-P/2, P/2] leaves the hit untouched. */
          {
            const int kind = surf_kind(st);
            const int a = kind == SURF_CYLINDER ? 0 : 1;
            const real period = kind == SURF_CYLINDER ? 2.0 * PI * st[12] : (kind == SURF_DISC ? 2.0 * PI : 0.0);
            if (period > 0.0) {
              const real d = m[a] - R->xp[a];
              if (d > 0.5 * period || d <= -0.5 * period) m[a] = m[a] - period * ceil((d - 0.5 * period) / period);
            }
          }
          rc = update_r(R->xp, R->Cp, m, V, xf, Cf, &c2);
          if (rc) { status |= (uint32_t)rc; break; }
          if (opt->outlier_chi2 > 0.0 && c2 > opt->outlier_chi2) { /* reading U9: strictly greater */
            memcpy(R->xf, R->xp, sizeof(xf));
            memcpy(R->Cf, R->Cp, sizeof(Cf));
            n_outl++;
            if (hit_flags) hit_flags[hp] = KFO_HIT_OUTLIER;
          } else {
            memcpy(R->xf, xf, sizeof(xf));
            memcpy(R->Cf, Cf, sizeof(Cf));
            chi2 += c2;
            n_used++;
            if (hit_flags) hit_flags[hp] = KFO_HIT_USED;
          }
          if (hit_chi2) hit_chi2[hp] = (double)c2;
          hp++;
        } else { /* hole */
          memcpy(R->xf, R->xp, sizeof(R->xf));
          memcpy(R->Cf, R->Cp, sizeof(R->Cf));
          n_holes++;
        }
        nleg++;
        memcpy(last_x, R->xf, sizeof(last_x));
        memcpy(last_C, R->Cf, sizeof(last_C));

        if (opt->material && st[14] > 0.0) { /* reading U6: after the update, at every visited surface */
          real g = 1.0;
          rc = material_r(opt, st, R->xf, R->Cf, x, C, &g, NULL, NULL);
          if (rc) { status |= (uint32_t)rc; break; }
          g_prev = g;
        } else {
          memcpy(x, R->xf, sizeof(x));
          memcpy(C, R->Cf, sizeof(C));
          g_prev = 1.0;
        }
        prev = s;
      }

      if (nleg > 0) {
        memcpy(first_x, rec[0].xf, sizeof(first_x));
        memcpy(first_C, rec[0].Cf, sizeof(first_C));
      }
      for (int k = 0; k < nleg; ++k) {
        size_t o = (size_t)i * Lmax + k;
        if (sp_par) put(sp_par + o * 6, rec[k].xp, 6);
        if (sp_cov) put(sp_cov + o * 36, rec[k].Cp, 36);
        if (sf_par) put(sf_par + o * 6, rec[k].xf, 6);
        if (sf_cov) put(sf_cov + o * 36, rec[k].Cf, 36);
      }

      /* C.2.6 RTS backward pass over the visited surfaces */
      if (opt->smooth && nleg > 0) {
        real xs[6], Cs[36];
        memcpy(xs, rec[nleg - 1].xf, sizeof(xs));
        memcpy(Cs, rec[nleg - 1].Cf, sizeof(Cs));
        size_t o = (size_t)i * Lmax + (nleg - 1);
        if (ss_par) put(ss_par + o * 6, xs, 6);
        if (ss_cov) put(ss_cov + o * 36, Cs, 36);
        for (int k = nleg - 2; k >= 0; --k) {
          real xn[6], Cn[36];
          int32_t rc = rts_step_r(rec[k].xf, rec[k].Cf, rec[k + 1].F, rec[k + 1].xp,
                                    rec[k + 1].Cp, xs, Cs, xn, Cn);
          if (rc) { /* fall back to the filtered states for the remaining surfaces */
            status |= (uint32_t)rc;
            for (int kk = k; kk >= 0; --kk) {
              size_t oo = (size_t)i * Lmax + kk;
              if (ss_par) put(ss_par + oo * 6, rec[kk].xf, 6);
              if (ss_cov) put(ss_cov + oo * 36, rec[kk].Cf, 36);
            }
            memcpy(xs, rec[0].xf, sizeof(xs));
            memcpy(Cs, rec[0].Cf, sizeof(Cs));
            break;
          }
          memcpy(xs, xn, sizeof(xs));
          memcpy(Cs, Cn, sizeof(Cs));
          o = (size_t)i * Lmax + k;
          if (ss_par) put(ss_par + o * 6, xs, 6);
          if (ss_cov) put(ss_cov + o * 36, Cs, 36);
        }
        memcpy(first_x, xs, sizeof(first_x));
        memcpy(first_C, Cs, sizeof(first_C));
      }
    }
    free(rec);

    const int ndf = 2 * n_used - 5; /* time is never measured: 5, not 6 (reading U10) */
    if (ndf <= 0) status |= KFO_ST_NDF;
    if (first_params) put(first_params + i * 6, first_x, 6);
    if (first_cov) put(first_cov + i * 36, first_C, 36);
    if (last_params) put(last_params + i * 6, last_x, 6);
    if (last_cov) put(last_cov + i * 36, last_C, 36);
    if (chi2_out) chi2_out[i] = (double)chi2;
    if (ndf_out) ndf_out[i] = ndf;
    if (status_out) status_out[i] = status;
    if (n_used_out) n_used_out[i] = n_used;
    if (n_out_out) n_out_out[i] = n_outl;
    if (n_holes_out) n_holes_out[i] = n_holes;
    if (rk_err_max) rk_err_max[i] = (double)errmax;
  }
  free(geom);
  return used_threads;
}

/* ---- perigee of every fitted track: first_* (on the first visited surface, or on the start surface for a
 * track that completed no leg) extrapolated to the line surface.  on_surface[i] = geometry index of the
 * surface first_* of track i lives on.  A track whose extrapolation stops gets KFO_ST_PERIGEE OR-ed into
 * status[i] (plus FIELD_CLAMPED when a lookup was clamped) and NaN outputs. */
int32_t kfo_perigee_batch(int64_t N, const double* first_params, const double* first_cov,
                          const int32_t* on_surface, const double* geometry, const kfo_field* fld_in,
                          const kfo_options* opt_in, const double line_c[3], const double line_a[3],
                          double* out_params, double* out_cov, uint32_t* status) {
  if (N < 0 || !first_params || !first_cov || !on_surface || !geometry || !fld_in || !opt_in || !out_params || !out_cov)
    return -1;
  const field_r fld = field_to_real(fld_in);
  const options_r opt = options_to_real(opt_in);
  const real lc[3] = {(real)line_c[0], (real)line_c[1], (real)line_c[2]};
  const real la[3] = {(real)line_a[0], (real)line_a[1], (real)line_a[2]};
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    real x[6], C[36], sf[KFO_GEOM_STRIDE], xo[6], Co[36], J[36];
    get(x, first_params + i * 6, 6);
    get(C, first_cov + i * 36, 36);
    get(sf, geometry + (size_t)on_surface[i] * KFO_GEOM_STRIDE, KFO_GEOM_STRIDE);
    int32_t clamped = 0;
    const int32_t rc = to_line_r(&fld, &opt, x, C, sf, lc, la, xo, Co, J, &clamped);
    if (rc != 0) {
      fill_nan(out_params + i * 6, 6);
      fill_nan(out_cov + i * 36, 36);
      if (status) status[i] |= KFO_ST_PERIGEE;
    } else {
      put(out_params + i * 6, xo, 6);
      put(out_cov + i * 36, Co, 36);
    }
    if (status && clamped) status[i] |= KFO_ST_FIELD_CLAMPED;
  }
  return 0;
}

/* ---- the step-level entry points of kf_oracle.h: double in, the step in `real`, double out ---------------- */
void kfo_field_at(const kfo_field* fld_in, const double r[3], double b_tesla[3], int32_t* clamped) {
  const field_r fld = field_to_real(fld_in);
  real rr[3], b[3];
  get(rr, r, 3);
  field_at_r(&fld, rr, b, clamped);
  put(b_tesla, b, 3);
}

void kfo_field_gradient_at(const kfo_field* fld_in, const double r[3], double G_tesla_per_mm[9]) {
  const field_r fld = field_to_real(fld_in);
  real rr[3], G[9];
  get(rr, r, 3);
  field_gradient_internal(&fld, rr, G);
  for (int i = 0; i < 9; ++i) G_tesla_per_mm[i] = (double)(G[i] / TESLA_TO_GEV_PER_MM);
}

void kfo_rkn4_step(const kfo_field* fld_in, double mass_gev, const double f[8], double h, double f_out[8],
                   double Dstep[64], double* eps, int32_t* clamped, int32_t field_gradient) {
  const field_r fld = field_to_real(fld_in);
  real fr[8], fo[8], Ds[64], e = 0.0;
  get(fr, f, 8);
  rkn4_step_r(&fld, (real)mass_gev, fr, (real)h, fo, Dstep ? Ds : NULL, &e, clamped, field_gradient);
  put(f_out, fo, 8);
  if (Dstep) put(Dstep, Ds, 64);
  if (eps) *eps = (double)e;
}

int32_t kfo_propagate(const kfo_field* fld_in, const kfo_options* opt_in, const double x[6],
                      const double* surf_from, const double* surf_to, double x_out[6], double J[36],
                      double free_out[8], double* rk_err, int32_t* clamped) {
  const field_r fld = field_to_real(fld_in);
  const options_r opt = options_to_real(opt_in);
  real xr[6], sf[KFO_GEOM_STRIDE], st[KFO_GEOM_STRIDE], xo[6], Jr[36], fo[8], e = 0.0;
  get(xr, x, 6);
  get(sf, surf_from, KFO_GEOM_STRIDE);
  get(st, surf_to, KFO_GEOM_STRIDE);
  const int32_t rc = propagate_r(&fld, &opt, xr, sf, st, xo, Jr, fo, &e, clamped);
  if (rc) return rc;
  put(x_out, xo, 6);
  put(J, Jr, 36);
  if (free_out) put(free_out, fo, 8);
  if (rk_err) *rk_err = (double)e;
  return 0;
}

int32_t kfo_to_line(const kfo_field* fld_in, const kfo_options* opt_in, const double x[6], const double C[36],
                    const double* surf_from, const double line_c[3], const double line_a[3], double x_out[6],
                    double C_out[36], double J[36], int32_t* clamped) {
  const field_r fld = field_to_real(fld_in);
  const options_r opt = options_to_real(opt_in);
  real xr[6], Cr[36], sf[KFO_GEOM_STRIDE], lc[3], la[3], xo[6], Co[36], Jr[36];
  get(xr, x, 6);
  get(Cr, C, 36);
  get(sf, surf_from, KFO_GEOM_STRIDE);
  get(lc, line_c, 3);
  get(la, line_a, 3);
  const int32_t rc = to_line_r(&fld, &opt, xr, Cr, sf, lc, la, xo, Co, Jr, clamped);
  if (rc) return rc;
  put(x_out, xo, 6);
  put(C_out, Co, 36);
  put(J, Jr, 36);
  return 0;
}

int32_t kfo_update(const double xp[6], const double Cp[36], const double m[2], const double V[4], double xf[6],
                   double Cf[36], double* chi2) {
  real xpr[6], Cpr[36], mr[2], Vr[4], xfr[6], Cfr[36], c2 = 0.0;
  get(xpr, xp, 6);
  get(Cpr, Cp, 36);
  get(mr, m, 2);
  get(Vr, V, 4);
  const int32_t rc = update_r(xpr, Cpr, mr, Vr, xfr, Cfr, &c2);
  if (rc) return rc;
  put(xf, xfr, 6);
  put(Cf, Cfr, 36);
  *chi2 = (double)c2;
  return 0;
}

int32_t kfo_material(const kfo_options* opt_in, const double* surf, const double xf[6], const double Cf[36],
                     double x_out[6], double C_out[36], double* g, double* theta0, double* dE_gev) {
  const options_r opt = options_to_real(opt_in);
  real sr[KFO_GEOM_STRIDE], xfr[6], Cfr[36], xo[6], Co[36], gr = 1.0, th = 0.0, dE = 0.0;
  get(sr, surf, KFO_GEOM_STRIDE);
  get(xfr, xf, 6);
  get(Cfr, Cf, 36);
  const int32_t rc = material_r(&opt, sr, xfr, Cfr, xo, Co, &gr, &th, &dE);
  if (theta0) *theta0 = (double)th;
  if (dE_gev) *dE_gev = (double)dE;
  if (rc) return rc;
  put(x_out, xo, 6);
  put(C_out, Co, 36);
  if (g) *g = (double)gr;
  return 0;
}

int32_t kfo_rts_step(const double xf_k[6], const double Cf_k[36], const double F_k1[36], const double xp_k1[6],
                     const double Cp_k1[36], const double xs_k1[6], const double Cs_k1[36], double xs_k[6],
                     double Cs_k[36]) {
  real xf[6], Cf[36], F[36], xp1[6], Cp1[36], xs1[6], Cs1[36], xs[6], Cs[36];
  get(xf, xf_k, 6);
  get(Cf, Cf_k, 36);
  get(F, F_k1, 36);
  get(xp1, xp_k1, 6);
  get(Cp1, Cp_k1, 36);
  get(xs1, xs_k1, 6);
  get(Cs1, Cs_k1, 36);
  const int32_t rc = rts_step_r(xf, Cf, F, xp1, Cp1, xs1, Cs1, xs, Cs);
  if (rc) return rc;
  put(xs_k, xs, 6);
  put(Cs_k, Cs, 36);
  return 0;
}

/* which arithmetic this build runs in: bytes of `real` and of the 6x6 solve's type */
int32_t kfo_real_bytes(void) { return (int32_t)sizeof(real); }
int32_t kfo_solve_real_bytes(void) { return (int32_t)sizeof(sreal); }
