// kf_device.cuh -- device-side arithmetic of the per-track Kalman fit (sm_100a, IEEE double).
//
// One thread owns one track; every matrix below is a fully unrolled register array.  The
// structure the method guarantees is exploited everywhere:
//   * the 8x8 free Jacobian D keeps its r and t columns as unit vectors (the field gradient is
//     neglected, reading U4), so only the blocks  P = dr/dT0 (3x3), p = dr/dlam (3),
//     Q = dT/dT0 (3x3), q = dT/dlam (3) and sigma = dt/dlam are carried: 25 numbers, not 64;
//   * the bound Jacobian J has row q/p = e_qp and column t = e_t: 25 non-trivial entries;
//   * H selects loc0, loc1; covariances are packed upper triangles (21 numbers).
// Citations: PAPER.md:55-62 (Kalman step, RTS with stored Jacobians), PAPER.md:128 (RKN transport,
// local<->global Jacobians), PAPER.md:119 (8x8 global covariance), PAPER.md:168 (material).
// This file shares nothing with oracle/ (its own constants, its own formulas' arrangement).
#pragma once

#include <cstdint>

namespace kf {

// ---- constants (this path's own copy) -----------------------------------------------------------
__device__ constexpr double kTeslaToGeVPerMm = 2.99792458e-4;  // 1 T in GeV/(e mm): dT/ds = lam T x B
__device__ constexpr double kElectronMass = 0.51099895e-3;     // GeV
__device__ constexpr double kBetheK = 0.307075;                // MeV mol^-1 cm^2
__device__ constexpr double kNdotTMin = 1e-6;
__device__ constexpr double kSinThetaMin = 1e-12;
__device__ constexpr double kPi = 3.14159265358979323846;

enum : unsigned {
  ST_PROPAGATION = 1u, ST_NOT_POSITIVE = 2u, ST_ENERGY = 4u, ST_NDF = 8u, ST_THETA = 16u,
  ST_FIELD_CLAMPED = 32u, ST_BAD_HITS = 64u
};

constexpr int FIELD_CONST = 0;
constexpr int FIELD_GRID3 = 1;

// packed upper-triangle index of a symmetric 6x6 (i <= j)
__host__ __device__ constexpr int IX(int i, int j) { return i * 6 - (i * (i - 1)) / 2 + (j - i); }
// symmetric access with any order
__host__ __device__ constexpr int SX(int i, int j) { return i <= j ? IX(i, j) : IX(j, i); }

struct FieldDesc {
  double b[3];        // CONST: field already in GeV/(e mm)
  int n[3];           // GRID3 nodes
  double origin[3];
  double spacing[3];
  const double* grid; // [nz][ny][nx][3] tesla
};

struct MaterialDesc {
  double mass;        // GeV
  double ZA;          // Z / A
  double rho;         // g/cm^3
  double I_gev;       // mean excitation energy, GeV
  double log_hwp_I;   // ln(hbar omega_p / I)
};

// ---- 3-vector helpers ----------------------------------------------------------------------------
__device__ __forceinline__ void cross(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
__device__ __forceinline__ double dot(const double a[3], const double b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

// ---- field --------------------------------------------------------------------------------------
// B(r) in GeV/(e mm).  GRID3: trilinear, clamped outside (status bit 32).
template <int FIELD>
__device__ __forceinline__ void field_at(const FieldDesc& F, const double r[3], double B[3],
                                         unsigned& status) {
  if constexpr (FIELD == FIELD_CONST) {
    B[0] = F.b[0]; B[1] = F.b[1]; B[2] = F.b[2];
  } else {
    int idx[3];
    double w[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double f = (r[a] - F.origin[a]) / F.spacing[a];
      double fl = floor(f);
      fl = fmax(fl, 0.0);
      fl = fmin(fl, (double)(F.n[a] - 2));
      double ww = f - fl;
      if (ww < 0.0) { ww = 0.0; status |= ST_FIELD_CLAMPED; }
      if (ww > 1.0) { ww = 1.0; status |= ST_FIELD_CLAMPED; }
      idx[a] = (int)fl;
      w[a] = ww;
    }
    const int nx = F.n[0];
    const size_t row = (size_t)nx * 3;
    const size_t slab = row * (size_t)F.n[1];
    const double* base = F.grid + (size_t)idx[2] * slab + (size_t)idx[1] * row + (size_t)idx[0] * 3;
    double acc[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int dz = 0; dz < 2; ++dz)
#pragma unroll
      for (int dy = 0; dy < 2; ++dy) {
        const double* nd = base + dz * slab + dy * row;  // two x-adjacent nodes: 6 contiguous doubles
        const double wyz = (dy ? w[1] : 1.0 - w[1]) * (dz ? w[2] : 1.0 - w[2]);
        const double w0 = (1.0 - w[0]) * wyz, w1 = w[0] * wyz;
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[c] += w0 * __ldg(nd + c) + w1 * __ldg(nd + 3 + c);
      }
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = acc[c] * kTeslaToGeVPerMm;
  }
}

// out[:, c] = lam * (X[:, c] x B) for the three columns of the row-major 3x3 X:  out = lam M(B) X
__device__ __forceinline__ void cross_columns(const double X[9], const double B[3], double lam,
                                              double out[9]) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    out[0 + c] = lam * (X[3 + c] * B[2] - X[6 + c] * B[1]);
    out[3 + c] = lam * (X[6 + c] * B[0] - X[0 + c] * B[2]);
    out[6 + c] = lam * (X[0 + c] * B[1] - X[3 + c] * B[0]);
  }
}

// ---- one RKN4 step (DESIGN.md "The algorithm" A.2) -------------------------------------------------
// Advances (r, t, T) by a step of length h and returns the step-Jacobian blocks
//   A = dr'/dT, a = dr'/dlam, Bm = dT'/dT, b = dT'/dlam, tau = dt'/dlam   (dr'/dr = I, dT'/dr = 0).
template <int FIELD>
__device__ __forceinline__ void rkn4_step(const FieldDesc& F, double mass, double r[3], double& t,
                                          double T[3], double lam, double h, double A[9],
                                          double a[3], double Bm[9], double b[3], double& tau,
                                          double& eps, unsigned& status) {
  double B1[3], B2[3], B3[3];
  const double hh = 0.5 * h;
  // stage 1
  field_at<FIELD>(F, r, B1, status);
  double l1[3], k1[3];
  cross(T, B1, l1);  // dk1/dlam
#pragma unroll
  for (int i = 0; i < 3; ++i) k1[i] = lam * l1[i];
  double d[9];  // current dk_i/dT
  d[0] = 0.0;            d[1] = lam * B1[2];   d[2] = -lam * B1[1];
  d[3] = -lam * B1[2];   d[4] = 0.0;           d[5] = lam * B1[0];
  d[6] = lam * B1[1];    d[7] = -lam * B1[0];  d[8] = 0.0;
  double SA[9], SB[9];  // d1+d2+d3 and d1+2d2+2d3+d4
#pragma unroll
  for (int i = 0; i < 9; ++i) { SA[i] = d[i]; SB[i] = d[i]; }
  double sa[3], sb[3];  // l1+l2+l3 and l1+2l2+2l3+l4
#pragma unroll
  for (int i = 0; i < 3; ++i) { sa[i] = l1[i]; sb[i] = l1[i]; }

  // stage 2 (midpoint)
  double rm[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) rm[i] = r[i] + hh * T[i] + 0.125 * h * h * k1[i];
  field_at<FIELD>(F, rm, B2, status);
  double X[9], v[3], k2[3], l2[3];
#pragma unroll
  for (int i = 0; i < 9; ++i) X[i] = hh * d[i];
  X[0] += 1.0; X[4] += 1.0; X[8] += 1.0;
  cross_columns(X, B2, lam, d);  // d2
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = T[i] + hh * k1[i];
  cross(v, B2, k2);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] += lam * hh * l1[i];
  cross(v, B2, l2);
#pragma unroll
  for (int i = 0; i < 3; ++i) k2[i] *= lam;
#pragma unroll
  for (int i = 0; i < 9; ++i) { SA[i] += d[i]; SB[i] += 2.0 * d[i]; }
#pragma unroll
  for (int i = 0; i < 3; ++i) { sa[i] += l2[i]; sb[i] += 2.0 * l2[i]; }

  // stage 3 (same field point)
  double k3[3], l3[3];
#pragma unroll
  for (int i = 0; i < 9; ++i) X[i] = hh * d[i];
  X[0] += 1.0; X[4] += 1.0; X[8] += 1.0;
  cross_columns(X, B2, lam, d);  // d3
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = T[i] + hh * k2[i];
  cross(v, B2, k3);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] += lam * hh * l2[i];
  cross(v, B2, l3);
#pragma unroll
  for (int i = 0; i < 3; ++i) k3[i] *= lam;
#pragma unroll
  for (int i = 0; i < 9; ++i) { SA[i] += d[i]; SB[i] += 2.0 * d[i]; }
#pragma unroll
  for (int i = 0; i < 3; ++i) { sa[i] += l3[i]; sb[i] += 2.0 * l3[i]; }

  // stage 4 (end point)
  double re[3], k4[3], l4[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) re[i] = r[i] + h * T[i] + 0.5 * h * h * k3[i];
  field_at<FIELD>(F, re, B3, status);
#pragma unroll
  for (int i = 0; i < 9; ++i) X[i] = h * d[i];
  X[0] += 1.0; X[4] += 1.0; X[8] += 1.0;
  cross_columns(X, B3, lam, d);  // d4
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = T[i] + h * k3[i];
  cross(v, B3, k4);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] += lam * h * l3[i];
  cross(v, B3, l4);
#pragma unroll
  for (int i = 0; i < 3; ++i) k4[i] *= lam;
#pragma unroll
  for (int i = 0; i < 9; ++i) SB[i] += d[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) sb[i] += l4[i];

  // Jacobian blocks
  const double h6 = h / 6.0, h26 = h * h / 6.0;
#pragma unroll
  for (int i = 0; i < 9; ++i) { A[i] = h26 * SA[i]; Bm[i] = h6 * SB[i]; }
  A[0] += h; A[4] += h; A[8] += h;
  Bm[0] += 1.0; Bm[4] += 1.0; Bm[8] += 1.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) { a[i] = h26 * sa[i]; b[i] = h6 * sb[i]; }
  const double dtds = sqrt(1.0 + mass * mass * lam * lam);
  tau = h * mass * mass * lam / dtds;

  // error estimate (diagnostic)
  eps = h * h * (fabs(k1[0] - k2[0] - k3[0] + k4[0]) + fabs(k1[1] - k2[1] - k3[1] + k4[1]) +
                 fabs(k1[2] - k2[2] - k3[2] + k4[2]));

  // state
  double Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = r[i] + h * T[i] + h26 * (k1[i] + k2[i] + k3[i]);
    Tn[i] = T[i] + h6 * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
  }
  const double nrm = sqrt(Tn[0] * Tn[0] + Tn[1] * Tn[1] + Tn[2] * Tn[2]);
#pragma unroll
  for (int i = 0; i < 3; ++i) T[i] = Tn[i] / nrm;
  t += h * dtds;
}

// 3x3 row-major helpers
__device__ __forceinline__ void mat3_mul(const double A[9], const double B[9], double C[9]) {
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      C[i * 3 + j] = A[i * 3 + 0] * B[0 + j] + A[i * 3 + 1] * B[3 + j] + A[i * 3 + 2] * B[6 + j];
}
__device__ __forceinline__ void mat3_vec(const double A[9], const double x[3], double y[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) y[i] = A[i * 3 + 0] * x[0] + A[i * 3 + 1] * x[1] + A[i * 3 + 2] * x[2];
}

// The bound-to-bound Jacobian, non-trivial part: Ja rows (loc0, loc1, phi, theta) x columns
// (loc0, loc1, phi, theta, qp); Jt = row t over the same columns.  Row qp = e_qp, column t = e_t.
struct BoundJacobian {
  double Ja[4][5];
  double Jt[5];
};

// ---- propagate a bound state from surface sf to surface st (A.1 - A.3) ---------------------------
// trig = (sin phi, cos phi, sin theta, cos theta) of x.  Returns 0 or the stopping status bit.
template <int FIELD>
__device__ __forceinline__ unsigned propagate(const FieldDesc& F, double mass, int n_corr,
                                              double max_step, const double* __restrict__ sf,
                                              const double* __restrict__ st, const double x[6],
                                              const double trig[4], double xo[6], BoundJacobian& J,
                                              double& errmax, unsigned& status) {
  const double sphi = trig[0], cphi = trig[1], sth = trig[2], cth = trig[3];
  // A.1 bound -> free
  double r[3], T[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) r[i] = sf[i] + x[0] * sf[3 + i] + x[1] * sf[6 + i];
  T[0] = cphi * sth; T[1] = sphi * sth; T[2] = cth;
  const double lam = x[4];
  double t = x[5];
  const double Tphi[3] = {-sphi * sth, cphi * sth, 0.0};
  const double Tth[3] = {cphi * cth, sphi * cth, -sth};
  const double nt[3] = {st[9], st[10], st[11]};
  const double ct[3] = {st[0], st[1], st[2]};

  // A.2 stepping: n_sub primary steps + n_corr correction steps, no accept/reject
  double P[9], Q[9], p[3], q[3], sigma = 0.0;
  int n_sub = 1;
  {
    const double nT = dot(nt, T);
    if (!(nT > kNdotTMin)) return ST_PROPAGATION;
    if (max_step > 0.0 && max_step < 1.0e300) {
      const double dr[3] = {ct[0] - r[0], ct[1] - r[1], ct[2] - r[2]};
      const double s0 = dot(nt, dr) / nT;
      double qn = ceil(fabs(s0) / max_step * (1.0 - 1e-12));
      if (!(qn >= 1.0)) qn = 1.0;
      if (qn > 1024.0) qn = 1024.0;
      n_sub = (int)qn;
    }
  }
  const int n_steps = n_sub + n_corr;
  for (int is = 0; is < n_steps; ++is) {
    const double nT = dot(nt, T);
    if (!(nT > kNdotTMin)) return ST_PROPAGATION;
    const double dr[3] = {ct[0] - r[0], ct[1] - r[1], ct[2] - r[2]};
    double h = dot(nt, dr) / nT;
    if (is < n_sub) h = h / (double)(n_sub - is);
    double A[9], a[3], Bm[9], b[3], tau, eps;
    rkn4_step<FIELD>(F, mass, r, t, T, lam, h, A, a, Bm, b, tau, eps, status);
    errmax = fmax(errmax, eps);
    if (is == 0) {
#pragma unroll
      for (int i = 0; i < 9; ++i) { P[i] = A[i]; Q[i] = Bm[i]; }
#pragma unroll
      for (int i = 0; i < 3; ++i) { p[i] = a[i]; q[i] = b[i]; }
      sigma = tau;
    } else {
      // D <- Dstep D:  P += A Q,  p += A q + a,  Q = Bm Q,  q = Bm q + b,  sigma += tau
      double AQ[9], Aq[3], BQ[9], Bq[3];
      mat3_mul(A, Q, AQ);
      mat3_vec(A, q, Aq);
      mat3_mul(Bm, Q, BQ);
      mat3_vec(Bm, q, Bq);
#pragma unroll
      for (int i = 0; i < 9; ++i) { P[i] += AQ[i]; Q[i] = BQ[i]; }
#pragma unroll
      for (int i = 0; i < 3; ++i) { p[i] += Aq[i] + a[i]; q[i] = Bq[i] + b[i]; }
      sigma += tau;
    }
    const double fin = r[0] + r[1] + r[2] + T[0] + T[1] + T[2] + t;
    if (!(fabs(fin) < 1.0e300)) return ST_PROPAGATION;  // catches NaN and Inf
  }

  // A.3 free -> bound with the path-length correction  D~ = (I - f' w^T) D
  const double nT = dot(nt, T);
  if (!(nT > kNdotTMin)) return ST_PROPAGATION;
  double Bend[3], TxB[3];
  field_at<FIELD>(F, r, Bend, status);
  cross(T, Bend, TxB);
  const double dtds = sqrt(1.0 + mass * mass * lam * lam);
  const double kf_[3] = {lam * TxB[0], lam * TxB[1], lam * TxB[2]};  // dT/ds
  const double w[3] = {nt[0] / nT, nt[1] / nT, nt[2] / nT};

  const double sth2 = sqrt(T[0] * T[0] + T[1] * T[1]);
  if (!(sth2 > kSinThetaMin)) return ST_THETA;
  const double cth2 = T[2];
  const double cph2 = T[0] / sth2, sph2 = T[1] / sth2;
  const double gphi[3] = {-sph2 / sth2, cph2 / sth2, 0.0};
  const double gth[3] = {cph2 * cth2, sph2 * cth2, -sth2};
  const double* ut = st + 3;
  const double* vt = st + 6;

  // columns of D J_b2f as (cr, ct_, cT); then c -= f' (w . cr); then rows of J_f2b
  auto project = [&](int c, double cr[3], double ctime, double cT[3]) {
    const double wd = dot(w, cr);
#pragma unroll
    for (int i = 0; i < 3; ++i) { cr[i] -= T[i] * wd; cT[i] -= kf_[i] * wd; }
    ctime -= dtds * wd;
    J.Ja[0][c] = ut[0] * cr[0] + ut[1] * cr[1] + ut[2] * cr[2];
    J.Ja[1][c] = vt[0] * cr[0] + vt[1] * cr[1] + vt[2] * cr[2];
    J.Ja[2][c] = gphi[0] * cT[0] + gphi[1] * cT[1];
    J.Ja[3][c] = gth[0] * cT[0] + gth[1] * cT[1] + gth[2] * cT[2];
    J.Jt[c] = ctime;
  };
  {
    double cr[3] = {sf[3], sf[4], sf[5]}, cT[3] = {0.0, 0.0, 0.0};
    project(0, cr, 0.0, cT);
  }
  {
    double cr[3] = {sf[6], sf[7], sf[8]}, cT[3] = {0.0, 0.0, 0.0};
    project(1, cr, 0.0, cT);
  }
  {
    double cr[3], cT[3];
    mat3_vec(P, Tphi, cr);
    mat3_vec(Q, Tphi, cT);
    project(2, cr, 0.0, cT);
  }
  {
    double cr[3], cT[3];
    mat3_vec(P, Tth, cr);
    mat3_vec(Q, Tth, cT);
    project(3, cr, 0.0, cT);
  }
  {
    double cr[3] = {p[0], p[1], p[2]}, cT[3] = {q[0], q[1], q[2]};
    project(4, cr, sigma, cT);
  }

  const double dr[3] = {r[0] - ct[0], r[1] - ct[1], r[2] - ct[2]};
  xo[0] = dot(ut, dr);
  xo[1] = dot(vt, dr);
  xo[2] = atan2(T[1], T[0]);
  xo[3] = acos(fmin(fmax(T[2], -1.0), 1.0));
  xo[4] = lam;
  xo[5] = t;
  double chk = xo[0] + xo[1] + xo[5];
#pragma unroll
  for (int c = 0; c < 5; ++c) chk += J.Ja[0][c] + J.Ja[1][c] + J.Ja[2][c] + J.Ja[3][c] + J.Jt[c];
  if (!(fabs(chk) < 1.0e300)) return ST_PROPAGATION;
  return 0u;
}

// ---- C- = J C J^T with the structure of J (A.4) -----------------------------------------------------
__device__ __forceinline__ void transport_covariance(const BoundJacobian& J, const double C[21],
                                                     double Cp[21]) {
  // M = J C : rows a = 0..3 and t; row qp of M is row qp of C
  double Ma[4][6], Mt[6];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      double s = J.Ja[i][0] * C[SX(0, k)];
#pragma unroll
      for (int l = 1; l < 5; ++l) s += J.Ja[i][l] * C[SX(l, k)];
      Ma[i][k] = s;
    }
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    double s = C[SX(5, k)];
#pragma unroll
    for (int l = 0; l < 5; ++l) s += J.Jt[l] * C[SX(l, k)];
    Mt[k] = s;
  }
  // C- = M J^T, upper triangle
#pragma unroll
  for (int i = 0; i < 4; ++i) {
#pragma unroll
    for (int j = i; j < 4; ++j) {
      double s = Ma[i][0] * J.Ja[j][0];
#pragma unroll
      for (int l = 1; l < 5; ++l) s += Ma[i][l] * J.Ja[j][l];
      Cp[IX(i, j)] = s;
    }
    Cp[IX(i, 4)] = Ma[i][4];
    double s = Ma[i][5];
#pragma unroll
    for (int l = 0; l < 5; ++l) s += Ma[i][l] * J.Jt[l];
    Cp[IX(i, 5)] = s;
  }
  Cp[IX(4, 4)] = C[IX(4, 4)];
  {
    double s = C[IX(4, 5)];  // M[qp][t]
#pragma unroll
    for (int l = 0; l < 5; ++l) s += C[SX(4, l)] * J.Jt[l];
    Cp[IX(4, 5)] = s;
  }
  {
    double s = Mt[5];
#pragma unroll
    for (int l = 0; l < 5; ++l) s += Mt[l] * J.Jt[l];
    Cp[IX(5, 5)] = s;
  }
}

// ---- gain-matrix update with a 2-D hit (A.5) ----------------------------------------
// Returns false when S is not positive definite.  xf/Cf may alias nothing of xp/Cp.
__device__ __forceinline__ bool gain_update(const double xp[6], const double Cp[21], double m0,
                                            double m1, double v00, double v01, double v11,
                                            double xf[6], double Cf[21], double& chi2) {
  const double r0 = m0 - xp[0], r1 = m1 - xp[1];
  const double S00 = Cp[IX(0, 0)] + v00, S01 = Cp[IX(0, 1)] + v01, S11 = Cp[IX(1, 1)] + v11;
  const double det = S00 * S11 - S01 * S01;
  if (!(S00 > 0.0 && det > 0.0)) return false;
  const double idet = 1.0 / det;
  const double i00 = S11 * idet, i01 = -S01 * idet, i11 = S00 * idet;
  chi2 = r0 * (i00 * r0 + i01 * r1) + r1 * (i01 * r0 + i11 * r1);
  double K0[6], K1[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    const double c0 = Cp[SX(i, 0)], c1 = Cp[SX(i, 1)];
    K0[i] = c0 * i00 + c1 * i01;
    K1[i] = c0 * i01 + c1 * i11;
    xf[i] = xp[i] + K0[i] * r0 + K1[i] * r1;
  }
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = i; j < 6; ++j)
      Cf[IX(i, j)] = Cp[IX(i, j)] - (K0[i] * Cp[SX(0, j)] + K1[i] * Cp[SX(1, j)]);
  return true;
}

// ---- material at a surface, after the update (A.6) -----------------------------------
// trig = sin/cos of the filtered phi, theta.  On success: lam -> lam', C -> G C G^T + Q in place.
__device__ __forceinline__ bool apply_material(const MaterialDesc& Mt, const double* __restrict__ surf,
                                               const double trig[4], double& lam, double C[21],
                                               double& g) {
  const double sphi = trig[0], cphi = trig[1], sth = trig[2], cth = trig[3];
  const double T[3] = {cphi * sth, sphi * sth, cth};
  const double m = Mt.mass;
  const double p = 1.0 / fabs(lam);
  const double E = sqrt(p * p + m * m);
  const double beta = p / E, gamma = E / m, bg = p / m;
  const double cfac = 1.0 / fabs(surf[9] * T[0] + surf[10] * T[1] + surf[11] * T[2]);
  // Highland
  const double X = surf[14] * cfac;
  const double b2 = beta * beta;
  const double theta0 = 0.0136 / (beta * p) * sqrt(X) * (1.0 + 0.038 * log(X / b2));
  // Bethe, asymptotic density correction
  const double me = kElectronMass;
  const double rme = me / m;
  const double Wmax = 2.0 * me * bg * bg / (1.0 + 2.0 * gamma * rme + rme * rme);
  const double dhalf = fmax(0.0, Mt.log_hwp_I + log(bg) - 0.5);
  const double dedx =
      kBetheK * Mt.ZA / b2 * (0.5 * log(2.0 * me * bg * bg * Wmax / (Mt.I_gev * Mt.I_gev)) - b2 - dhalf);
  const double dE = dedx * Mt.rho * 1e-3 * 0.1 * surf[15] * cfac;
  const double E2 = E - dE;
  if (!(E2 > m)) return false;
  const double p2 = sqrt(E2 * E2 - m * m);
  g = (p * p * p * E2) / (p2 * p2 * p2 * E);
  lam = (lam < 0.0 ? -1.0 : 1.0) / p2;
  // C <- G C G^T + Q : row/column qp scaled by g
#pragma unroll
  for (int i = 0; i < 6; ++i)
    if (i != 4) C[SX(i, 4)] *= g;
  C[IX(4, 4)] *= g * g;
  const double t2 = theta0 * theta0;
  C[IX(2, 2)] += t2 / (sth * sth);
  C[IX(3, 3)] += t2;
  return true;
}

// ---- one RTS step (A.7) --------------------------------------------------------------------
// F = J G stored as 26 numbers: Fa[4][5], Ft[5] (column qp already scaled by g) and g.
// In: filtered (xf, Cf) at k, record k+1 (xp1, Cp1, F), smoothed (xs, Cs) at k+1 (updated in place).
__device__ __forceinline__ bool rts_step(const double xf[6], const double Cf[21],
                                         const double Fa[4][5], const double Ft[5], double g,
                                         const double xp1[6], const double Cp1[21], double xs[6],
                                         double Cs[21]) {
  // Cholesky C-_{k+1} = L L^T without pivoting; L[i][j] (i >= j) kept at packed (j, i)
  double L[21], inv[6];
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    double s = Cp1[IX(j, j)];
#pragma unroll
    for (int k = 0; k < j; ++k) s -= L[IX(k, j)] * L[IX(k, j)];
    if (!(s > 0.0)) return false;
    const double d = sqrt(s);
    L[IX(j, j)] = d;
    inv[j] = 1.0 / d;
#pragma unroll
    for (int i = j + 1; i < 6; ++i) {
      double u = Cp1[IX(j, i)];
#pragma unroll
      for (int k = 0; k < j; ++k) u -= L[IX(k, i)] * L[IX(k, j)];
      L[IX(j, i)] = u * inv[j];
    }
  }
  // A = C+ F^T (C-)^-1, one row at a time: w = row of C+ F^T, solve L L^T a = w
  double A[6][6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    double w[6];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      double s = Cf[SX(i, 0)] * Fa[j][0];
#pragma unroll
      for (int k = 1; k < 5; ++k) s += Cf[SX(i, k)] * Fa[j][k];
      w[j] = s;
    }
    w[4] = Cf[SX(i, 4)] * g;
    {
      double s = Cf[SX(i, 5)];
#pragma unroll
      for (int k = 0; k < 5; ++k) s += Cf[SX(i, k)] * Ft[k];
      w[5] = s;
    }
#pragma unroll
    for (int r = 0; r < 6; ++r) {  // L y = w
      double s = w[r];
#pragma unroll
      for (int k = 0; k < r; ++k) s -= L[IX(k, r)] * w[k];
      w[r] = s * inv[r];
    }
#pragma unroll
    for (int r = 5; r >= 0; --r) {  // L^T a = y
      double s = w[r];
#pragma unroll
      for (int k = r + 1; k < 6; ++k) s -= L[IX(r, k)] * w[k];
      w[r] = s * inv[r];
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) A[i][j] = w[j];
  }
  // x^s_k = x+_k + A (x^s_{k+1} - x-_{k+1}),  phi difference wrapped into (-pi, pi]
  double dx[6];
#pragma unroll
  for (int j = 0; j < 6; ++j) dx[j] = xs[j] - xp1[j];
  if (dx[2] > kPi) dx[2] -= 2.0 * kPi;
  else if (dx[2] <= -kPi) dx[2] += 2.0 * kPi;
  // C^s_k = C+_k + A (C^s_{k+1} - C-_{k+1}) A^T
  double dC[21];
#pragma unroll
  for (int k = 0; k < 21; ++k) dC[k] = Cs[k] - Cp1[k];
  double chk = 0.0;
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    double s = xf[i];
#pragma unroll
    for (int j = 0; j < 6; ++j) s += A[i][j] * dx[j];
    xs[i] = s;
    chk += s;
    double AdC[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      double u = A[i][0] * dC[SX(0, j)];
#pragma unroll
      for (int k = 1; k < 6; ++k) u += A[i][k] * dC[SX(k, j)];
      AdC[j] = u;
    }
#pragma unroll
    for (int j = i; j < 6; ++j) {
      double u = Cf[IX(i, j)];
#pragma unroll
      for (int k = 0; k < 6; ++k) u += AdC[k] * A[j][k];
      Cs[IX(i, j)] = u;
      chk += u;
    }
  }
  return fabs(chk) < 1.0e300;
}

}  // namespace kf
