// kf_device.cuh -- device-side arithmetic of the per-track Kalman fit (sm_100a; templated on the real type R: IEEE
// double, or float for the MIXED-precision path).
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
// This file shares no code with oracle/ (its own constants, its own formulas' arrangement).  One caveat: the four
// general-surface helpers below (local_to_global, surface_normal, global_to_local, path_to_surface) decompose reading
// U33 the way the oracle does, so GPU-vs-oracle parity on cylinders and discs checks their transcription; what pins
// U33 itself is independent of both: the oracle-side pins PS1-PS11 and the GPU-side closed-form test
// tests/test_gpu_general.py::test_gpu_helix_to_cylinder_closed_form_without_the_oracle.
#pragma once

#include <cstdint>
#include <type_traits>

#include "kf_math.cuh"

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
  ST_FIELD_CLAMPED = 32u, ST_BAD_HITS = 64u, ST_PERIGEE = 128u, ST_CANCELLATION = 256u
};

constexpr int FIELD_CONST = 0;
constexpr int FIELD_GRID3 = 1;
constexpr int FIELD_GRID3S = 2;  // GRID3 with a box of the table staged in shared memory (FieldDescT::box_*)

// every kernel's dynamic shared memory starts here (all `extern __shared__` arrays of a kernel alias one base)
extern __shared__ __align__(128) unsigned char kf_dyn_smem[];

// packed upper-triangle index of a symmetric 6x6 (i <= j)
__host__ __device__ constexpr int IX(int i, int j) { return i * 6 - (i * (i - 1)) / 2 + (j - i); }
// symmetric access with any order
__host__ __device__ constexpr int SX(int i, int j) { return i <= j ? IX(i, j) : IX(j, i); }

template <typename R>
struct FieldDescT {
  R b[3];        // CONST: field already in GeV/(e mm)
  R b2;          // CONST: |b|^2
  R inv_spacing[3];  // GRID3: 1 / spacing
  int n[3];           // GRID3 nodes
  R origin[3];
  R spacing[3];
  const double* grid; // [nz][ny][nx][3] tesla (the table as given: double)
  // GRID3S: nodes [box_lo, box_lo + box_n) per axis are held in shared memory as R[box_n[2]][box_n[1]][box_n[0]][3],
  // box_off bytes behind the start of the kernel's dynamic shared memory; a lookup whose cell is not wholly inside
  // reads the table in global memory
  int box_lo[3], box_n[3], box_off;
};

template <typename R>
struct MaterialDescT {
  R mass;        // GeV
  R inv_mass;    // 1 / mass
  R rme;         // m_e / mass
  R inv_I2;      // 1 / I^2, GeV^-2
  R ZA;          // Z / A
  R rho;         // g/cm^3
  R I_gev;       // mean excitation energy, GeV
  R log_hwp_I;   // ln(hbar omega_p / I)
};

// ---- 3-vector helpers ----------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ void cross(const R a[3], const R b[3], R c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
template <typename R>
__device__ __forceinline__ R dot(const R a[3], const R b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

// ---- field --------------------------------------------------------------------------------------
// B(r) in GeV/(e mm).  GRID3: trilinear, clamped outside (status bit 32).
template <int FIELD, typename R>
__device__ __forceinline__ void field_at(const FieldDescT<R>& F, const R r[3], R B[3],
                                         unsigned& status) {
  if constexpr (FIELD == FIELD_CONST) {
    B[0] = F.b[0]; B[1] = F.b[1]; B[2] = F.b[2];
  } else {
    int idx[3];
    R w[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      // correctly rounded quotient from the host-rounded reciprocal (Markstein): the cell index and the
      // clamp flag must not depend on a last-bit difference from a true division
      const R num = r[a] - F.origin[a];
      R f = num * F.inv_spacing[a];
      f = fma(fma(-f, F.spacing[a], num), F.inv_spacing[a], f);
      R fl = floor(f);
      fl = fmax(fl, R(0.0));
      fl = fmin(fl, (R)(F.n[a] - 2));
      R ww = f - fl;
      if (ww < R(0.0)) { ww = R(0.0); status |= ST_FIELD_CLAMPED; }
      if (ww > R(1.0)) { ww = R(1.0); status |= ST_FIELD_CLAMPED; }
      idx[a] = (int)fl;
      w[a] = ww;
    }
    R acc[3] = {R(0.0), R(0.0), R(0.0)};
    // the eight corners: four pairs of x-adjacent nodes (6 contiguous values each) at row / slab strides
    auto corners = [&](auto base, int row, int slab, auto load6) {
#pragma unroll
      for (int dz = 0; dz < 2; ++dz)
#pragma unroll
        for (int dy = 0; dy < 2; ++dy) {
          R nd[6];
          load6(base + dz * slab + dy * row, nd);
          const R wyz = (dy ? w[1] : R(1.0) - w[1]) * (dz ? w[2] : R(1.0) - w[2]);
          const R w0 = (R(1.0) - w[0]) * wyz, w1 = w[0] * wyz;
#pragma unroll
          for (int c = 0; c < 3; ++c) acc[c] += w0 * nd[c] + w1 * nd[3 + c];
        }
    };
    bool staged = false;
    if constexpr (FIELD == FIELD_GRID3S) {
      const int bi = idx[0] - F.box_lo[0], bj = idx[1] - F.box_lo[1], bk = idx[2] - F.box_lo[2];
      staged = (unsigned)bi < (unsigned)(F.box_n[0] - 1) && (unsigned)bj < (unsigned)(F.box_n[1] - 1) &&
               (unsigned)bk < (unsigned)(F.box_n[2] - 1);
      if (staged) {
        const int row = F.box_n[0] * 3, slab = row * F.box_n[1];
        corners(reinterpret_cast<const R*>(kf_dyn_smem + F.box_off) + bk * slab + bj * row + bi * 3, row, slab,
                [](const R* q, R nd[6]) {
#pragma unroll
                  for (int c = 0; c < 6; ++c) nd[c] = q[c];
                });
      }
    }
    if (!staged) {
      const int row = F.n[0] * 3, slab = row * F.n[1];
      corners(F.grid + (size_t)idx[2] * slab + (size_t)idx[1] * row + (size_t)idx[0] * 3, row, slab,
              [](const double* q, R nd[6]) {
#pragma unroll
                for (int c = 0; c < 6; ++c) nd[c] = R(__ldg(q + c));
              });
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = acc[c] * R(kTeslaToGeVPerMm);
  }
}

// B(r) and G[c][a] = dB_c/dr_a of the trilinear interpolant (GeV/(e mm) per mm), for the field-gradient terms of the
// step Jacobian (U32).  Along an axis on which the lookup is clamped the interpolant is constant: zero
// derivative.  A constant field has G = 0.  (Not a hot path: the eight corners are read once, plainly.)
template <int FIELD, typename R>
__device__ __forceinline__ void field_and_gradient_at(const FieldDescT<R>& F, const R r[3], R B[3], R G[9],
                                                      unsigned& status) {
#pragma unroll
  for (int i = 0; i < 9; ++i) G[i] = R(0.0);
  if constexpr (FIELD == FIELD_CONST) {
    B[0] = F.b[0]; B[1] = F.b[1]; B[2] = F.b[2];
  } else {
    int idx[3];
    R w[3];
    bool inside[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const R num = r[a] - F.origin[a];
      R f = num * F.inv_spacing[a];
      f = fma(fma(-f, F.spacing[a], num), F.inv_spacing[a], f);
      R fl = floor(f);
      fl = fmax(fl, R(0.0));
      fl = fmin(fl, (R)(F.n[a] - 2));
      R ww = f - fl;
      inside[a] = true;
      if (ww < R(0.0)) { ww = R(0.0); status |= ST_FIELD_CLAMPED; inside[a] = false; }
      if (ww > R(1.0)) { ww = R(1.0); status |= ST_FIELD_CLAMPED; inside[a] = false; }
      idx[a] = (int)fl;
      w[a] = ww;
    }
    const int row = F.n[0] * 3, slab = row * F.n[1];
    const double* base = F.grid + (size_t)idx[2] * slab + (size_t)idx[1] * row + (size_t)idx[0] * 3;
    R nd[2][2][2][3];  // [dz][dy][dx][component]
#pragma unroll
    for (int dz = 0; dz < 2; ++dz)
#pragma unroll
      for (int dy = 0; dy < 2; ++dy)
#pragma unroll
        for (int dx = 0; dx < 2; ++dx)
#pragma unroll
          for (int c = 0; c < 3; ++c) nd[dz][dy][dx][c] = R(__ldg(base + dz * slab + dy * row + dx * 3 + c));
    const R wx[2] = {R(1.0) - w[0], w[0]}, wy[2] = {R(1.0) - w[1], w[1]}, wz[2] = {R(1.0) - w[2], w[2]};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      R b = R(0.0), gx = R(0.0), gy = R(0.0), gz = R(0.0);
#pragma unroll
      for (int dz = 0; dz < 2; ++dz)
#pragma unroll
        for (int dy = 0; dy < 2; ++dy) {
#pragma unroll
          for (int dx = 0; dx < 2; ++dx) b = fma(wz[dz] * wy[dy] * wx[dx], nd[dz][dy][dx][c], b);
          gx = fma(wz[dz] * wy[dy], nd[dz][dy][1][c] - nd[dz][dy][0][c], gx);
        }
#pragma unroll
      for (int dz = 0; dz < 2; ++dz)
#pragma unroll
        for (int dx = 0; dx < 2; ++dx) gy = fma(wz[dz] * wx[dx], nd[dz][1][dx][c] - nd[dz][0][dx][c], gy);
#pragma unroll
      for (int dy = 0; dy < 2; ++dy)
#pragma unroll
        for (int dx = 0; dx < 2; ++dx) gz = fma(wy[dy] * wx[dx], nd[1][dy][dx][c] - nd[0][dy][dx][c], gz);
      B[c] = b * R(kTeslaToGeVPerMm);
      G[c * 3 + 0] = inside[0] ? gx * F.inv_spacing[0] * R(kTeslaToGeVPerMm) : R(0.0);
      G[c * 3 + 1] = inside[1] ? gy * F.inv_spacing[1] * R(kTeslaToGeVPerMm) : R(0.0);
      G[c * 3 + 2] = inside[2] ? gz * F.inv_spacing[2] * R(kTeslaToGeVPerMm) : R(0.0);
    }
  }
}

// out[:, c] = lam * (X[:, c] x B) for the three columns of the row-major 3x3 X:  out = lam M(B) X
template <typename R>
__device__ __forceinline__ void cross_columns(const R X[9], const R B[3], R lam,
                                              R out[9]) {
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
template <int FIELD, typename R>
// dtds = sqrt(1 + m^2 lam^2) and tfac = m^2 lam / dtds are constant along a leg (lam is).
__device__ __forceinline__ void rkn4_step(const FieldDescT<R>& F, R dtds, R tfac, R r[3], R& t,
                                          R T[3], R lam, R h, R A[9],
                                          R a[3], R Bm[9], R b[3], R& tau,
                                          R& eps, unsigned& status) {
  R B1[3], B2[3], B3[3];
  const R hh = R(0.5) * h;
  // stage 1
  field_at<FIELD>(F, r, B1, status);
  R l1[3], k1[3];
  cross(T, B1, l1);  // dk1/dlam
#pragma unroll
  for (int i = 0; i < 3; ++i) k1[i] = lam * l1[i];
  R d[9];  // current dk_i/dT
  d[0] = R(0.0);            d[1] = lam * B1[2];   d[2] = -lam * B1[1];
  d[3] = -lam * B1[2];   d[4] = R(0.0);           d[5] = lam * B1[0];
  d[6] = lam * B1[1];    d[7] = -lam * B1[0];  d[8] = R(0.0);
  R SA[9], SB[9];  // d1+d2+d3 and d1+2d2+2d3+d4
#pragma unroll
  for (int i = 0; i < 9; ++i) { SA[i] = d[i]; SB[i] = d[i]; }
  R sa[3], sb[3];  // l1+l2+l3 and l1+2l2+2l3+l4
#pragma unroll
  for (int i = 0; i < 3; ++i) { sa[i] = l1[i]; sb[i] = l1[i]; }

  // stage 2 (midpoint)
  R rm[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) rm[i] = r[i] + hh * T[i] + R(0.125) * h * h * k1[i];
  field_at<FIELD>(F, rm, B2, status);
  R X[9], v[3], k2[3], l2[3];
#pragma unroll
  for (int i = 0; i < 9; ++i) X[i] = hh * d[i];
  X[0] += R(1.0); X[4] += R(1.0); X[8] += R(1.0);
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
  for (int i = 0; i < 9; ++i) { SA[i] += d[i]; SB[i] += R(2.0) * d[i]; }
#pragma unroll
  for (int i = 0; i < 3; ++i) { sa[i] += l2[i]; sb[i] += R(2.0) * l2[i]; }

  // stage 3 (same field point)
  R k3[3], l3[3];
#pragma unroll
  for (int i = 0; i < 9; ++i) X[i] = hh * d[i];
  X[0] += R(1.0); X[4] += R(1.0); X[8] += R(1.0);
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
  for (int i = 0; i < 9; ++i) { SA[i] += d[i]; SB[i] += R(2.0) * d[i]; }
#pragma unroll
  for (int i = 0; i < 3; ++i) { sa[i] += l3[i]; sb[i] += R(2.0) * l3[i]; }

  // stage 4 (end point)
  R re[3], k4[3], l4[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) re[i] = r[i] + h * T[i] + R(0.5) * h * h * k3[i];
  field_at<FIELD>(F, re, B3, status);
#pragma unroll
  for (int i = 0; i < 9; ++i) X[i] = h * d[i];
  X[0] += R(1.0); X[4] += R(1.0); X[8] += R(1.0);
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
  const R h6 = h * (R(1.0) / R(6.0)), h26 = h * h6;
#pragma unroll
  for (int i = 0; i < 9; ++i) { A[i] = h26 * SA[i]; Bm[i] = h6 * SB[i]; }
  A[0] += h; A[4] += h; A[8] += h;
  Bm[0] += R(1.0); Bm[4] += R(1.0); Bm[8] += R(1.0);
#pragma unroll
  for (int i = 0; i < 3; ++i) { a[i] = h26 * sa[i]; b[i] = h6 * sb[i]; }
  tau = h * tfac;

  // error estimate (diagnostic)
  eps = h * h * (fabs(k1[0] - k2[0] - k3[0] + k4[0]) + fabs(k1[1] - k2[1] - k3[1] + k4[1]) +
                 fabs(k1[2] - k2[2] - k3[2] + k4[2]));

  // state
  R Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = r[i] + h * T[i] + h26 * (k1[i] + k2[i] + k3[i]);
    Tn[i] = T[i] + h6 * (k1[i] + R(2.0) * k2[i] + R(2.0) * k3[i] + k4[i]);
  }
  const R inrm = rsqrt_near_one(Tn[0] * Tn[0] + Tn[1] * Tn[1] + Tn[2] * Tn[2]);
#pragma unroll
  for (int i = 0; i < 3; ++i) T[i] = Tn[i] * inrm;
  t += h * dtds;
}

// ---- constant field: the RKN4 step in closed form ---------------------------------------------------
// With B the same at the three field points, every stage derivative is a polynomial in
// M = lam M_B (M_B v := v x B, M_B^3 = -|B|^2 M_B):  d1 = M, d2 = M + (h/2)M^2, d3 = d2 + (h^2/4)M^3,
// d4 = M + hM^2 + (h^2/2)M^3 + (h^3/4)M^4, and k_i = d_i T.  The step of DESIGN.md A.2 therefore is,
// with u = h lam, s = u^2 |B|^2, w1 = T x B, w2 = w1 x B:
//   r' = r + hT + a1 w1 + a2 w2,   T' = normalise(T + c1 w1 + c2 w2),
//   dr'/dT = hI + a1 M_B + a2 M_B^2,   dT'/dT = I + c1 M_B + c2 M_B^2,
//   a1 = h u (1/2 - s/24), a2 = h u^2/6, c1 = u (1 - s/6), c2 = u^2 (1/2 - s/24),
//   dr'/dlam = (da1) w1 + (da2) w2, dT'/dlam = (dc1) w1 + (dc2) w2  (derivatives of the coefficients),
//   eps = h^2 |k1 - k2 - k3 + k4|_1 = h^2 |lam| (s/4) |w1 + u w2|_1.
// Same discrete step, same Jacobian as the general code path: only the arithmetic is regrouped.  All
// step Jacobians commute, so the accumulated D keeps the form  P = P0 I + P1 M_B + P2 M_B^2 (dr/dT0),
// Q = I + Q1 M_B + Q2 M_B^2 (dT/dT0): six scalars instead of two 3x3 matrices.
template <typename R>
struct PolyJacT {
  R P0, P1, P2, Q1, Q2;  // Q0 == 1
  R p[3], q[3], sigma;   // dr/dlam, dT/dlam, dt/dlam
};

// v -> c0 v + c1 (v x B) + c2 ((v x B) x B)
template <typename R>
__device__ __forceinline__ void poly_apply(const R B[3], R c0, R c1, R c2,
                                           const R v[3], const R vx[3], const R vxx[3],
                                           R out[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) out[i] = fma(c2, vxx[i], fma(c1, vx[i], c0 * v[i]));
}

template <bool FIRST, typename R>
__device__ __forceinline__ void const_field_step(const R B[3], R b2, R dtds, R tfac,
                                                 R lam, R h, R r[3], R& t, R T[3],
                                                 PolyJacT<R>& D, R& errmax) {
  const R u = h * lam, uu = u * u, s = uu * b2;
  const R e = fma(s, -R(1.0) / R(24.0), R(0.5));
  const R c1 = u * fma(s, -R(1.0) / R(6.0), R(1.0));
  const R c2 = uu * e;
  const R a1 = h * u * e;
  const R a2 = h * uu * (R(1.0) / R(6.0));
  const R hh = h * h;
  const R dc1 = h * fma(s, -R(0.5), R(1.0)), dc2 = h * c1;
  const R da1 = hh * fma(s, -R(0.125), R(0.5)), da2 = hh * u * (R(1.0) / R(3.0));
  R w1[3], w2[3];
  cross(T, B, w1);
  cross(w1, B, w2);
  R av[3], bv[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    av[i] = fma(da2, w2[i], da1 * w1[i]);
    bv[i] = fma(dc2, w2[i], dc1 * w1[i]);
  }
  const R eps = hh * fabs(lam) * R(0.25) * s *
                     (fabs(fma(u, w2[0], w1[0])) + fabs(fma(u, w2[1], w1[1])) + fabs(fma(u, w2[2], w1[2])));
  errmax = fmax(errmax, eps);
  // state
  R Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = fma(a2, w2[i], fma(a1, w1[i], fma(h, T[i], r[i])));
    Tn[i] = fma(c2, w2[i], fma(c1, w1[i], T[i]));
  }
  const R inrm = rsqrt_near_one(fma(Tn[0], Tn[0], fma(Tn[1], Tn[1], Tn[2] * Tn[2])));
#pragma unroll
  for (int i = 0; i < 3; ++i) T[i] = Tn[i] * inrm;
  t = fma(h, dtds, t);
  const R tau = h * tfac;
  // D <- Dstep D
  if constexpr (FIRST) {
    D.P0 = h; D.P1 = a1; D.P2 = a2; D.Q1 = c1; D.Q2 = c2;
#pragma unroll
    for (int i = 0; i < 3; ++i) { D.p[i] = av[i]; D.q[i] = bv[i]; }
    D.sigma = tau;
  } else {
    R qx[3], qxx[3];
    cross(D.q, B, qx);
    cross(qx, B, qxx);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      D.p[i] += fma(a2, qxx[i], fma(a1, qx[i], fma(h, D.q[i], av[i])));
      D.q[i] += fma(c2, qxx[i], fma(c1, qx[i], bv[i]));
    }
    // polynomial products modulo M_B^3 = -b2 M_B:  P += A Q,  Q = Bm Q   (A0 = h, Bm0 = Q0 = 1)
    const R Q1 = D.Q1, Q2 = D.Q2;
    D.P0 += h;
    D.P1 += fma(h, Q1, a1) - b2 * fma(a1, Q2, a2 * Q1);
    D.P2 += fma(h, Q2, fma(a1, Q1, a2)) - b2 * (a2 * Q2);
    D.Q1 = (Q1 + c1) - b2 * fma(c1, Q2, c2 * Q1);
    D.Q2 = fma(c1, Q1, Q2 + c2) - b2 * (c2 * Q2);
    D.sigma += tau;
  }
}

// The same step to first order in h, for a correction step that starts within kFirstOrderStep of the surface (the second
// correction step of the default policy: |h| = kappa |n x T| h1^2 / 2 <= 2e-6 mm down to 0.5 GeV).  Every dropped term of
// const_field_step carries a further factor h or u = h lam: a1 w1 = h^2 lam |B| / 2 <= 1e-10 x 6e-3 / 2 = 3e-13 mm on
// the position, c2 w2 = u^2 |B|^2 / 2 <= 2e-15 on the direction, <= 1e-13 relative on every entry of the accumulated
// Jacobian -- below the last digit that survives the sums they enter, three orders inside the parity bars
// (DESIGN.md "Tolerances").  A step longer than the threshold takes the full form.
template <typename R> __device__ __forceinline__ constexpr R first_order_step();
template <> __device__ __forceinline__ constexpr double first_order_step<double>() { return 1.0e-5; }
template <> __device__ __forceinline__ constexpr float first_order_step<float>() { return 1.0e-3f; }

template <typename R>
__device__ __forceinline__ void const_field_step_first_order(const R B[3], R b2, R dtds, R tfac, R lam, R h, R r[3],
                                                             R& t, R T[3], PolyJacT<R>& D) {
  const R u = h * lam;
  R w1[3];
  cross(T, B, w1);
  R Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = fma(h, T[i], r[i]);
    Tn[i] = fma(u, w1[i], T[i]);
  }
  const R inrm = rsqrt_near_one(fma(Tn[0], Tn[0], fma(Tn[1], Tn[1], Tn[2] * Tn[2])));
#pragma unroll
  for (int i = 0; i < 3; ++i) T[i] = Tn[i] * inrm;
  t = fma(h, dtds, t);
  // D <- Dstep D with A = h I, Bm = I + u M_B, a = 0, b = h w1
  R qx[3];
  cross(D.q, B, qx);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    D.p[i] = fma(h, D.q[i], D.p[i]);
    D.q[i] += fma(u, qx[i], h * w1[i]);
  }
  const R Q1 = D.Q1, Q2 = D.Q2;
  D.P0 += h;
  D.P1 = fma(h, Q1, D.P1);
  D.P2 = fma(h, Q2, D.P2);
  D.Q1 = (Q1 + u) - b2 * (u * Q2);
  D.Q2 = fma(u, Q1, Q2);
  D.sigma = fma(h, tfac, D.sigma);
}

// 3x3 row-major helpers (general field path)
template <typename R>
__device__ __forceinline__ void mat3_mul(const R A[9], const R B[9], R C[9]) {
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      C[i * 3 + j] = A[i * 3 + 0] * B[0 + j] + A[i * 3 + 1] * B[3 + j] + A[i * 3 + 2] * B[6 + j];
}
template <typename R>
__device__ __forceinline__ void mat3_vec(const R A[9], const R x[3], R y[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) y[i] = A[i * 3 + 0] * x[0] + A[i * 3 + 1] * x[1] + A[i * 3 + 2] * x[2];
}

template <typename R>
struct MatJacT {
  R P[9], Q[9], p[3], q[3], sigma;
};

// ---- position-dependent field: the RKN4 step with the Jacobian carried as variational columns -------
// In a grid field the step Jacobians do not commute, and accumulating them as 3x3 blocks (MatJacT: A, Bm per step,
// then P += A Q, Q = Bm Q, then P Tphi, Q Tphi, ...) spends most of its arithmetic on matrix entries that only ever
// act on three vectors.  Here the three non-trivial columns of D J_b2f themselves -- d(r, T)/d(phi), /d(theta),
// /d(q/p) at the start of the leg -- are carried through the stages of every step (the variational equations of
// the RKN4 scheme, the same discrete Jacobian as rkn4_step's blocks, regrouped):
//   dk1 = lam dT x B1 (+ T x B1);  dT2 = dT + (h/2) dk1;  dk2 = lam dT2 x B2 (+ T2 x B2);  dT3 = dT + (h/2) dk2;
//   dk3 = lam dT3 x B2 (+ T3 x B2);  dT4 = dT + h dk3;  dk4 = lam dT4 x B3 (+ T4 x B3)     [(+ ...): the q/p column]
//   dr' = dr + h dT + (h^2/6)(dk1 + dk2 + dk3);   dT' = dT + (h/6)(dk1 + 2 dk2 + 2 dk3 + dk4).
// The loc0 / loc1 columns stay (u, 0), (v, 0) while the field gradient is neglected (U4).
// 19 numbers instead of 25, no 3x3 products, and the per-step blocks A, Bm never exist.
template <typename R>
struct ColJacT {
  R dr[3][3], dT[3][3];  // [column: phi, theta, q/p][component]
  R sigma;               // dt/dlam
};

// After a last step shorter than this, the field of that step's fourth stage (looked up at r + hT + (h^2/2) k3)
// stands for the field at its end point r + hT + (h^2/6)(k1 + k2 + k3) in the path-length correction: the two points
// are within h^2 |k| / 3 <= 1e-6 x 6e-3 / 3 = 2e-9 mm of each other (p >= 0.1 GeV in 2 T), which moves the Jacobian by
// less than |k| |w.c| x |grad B|/|B| x 2e-9 <= 7e-3 x 0.2 x 2e-9 = 3e-12 relative for any grid of >= 10 mm spacing
// (CFG4: 1e-14), far inside the 1e-8 covariance bar.  One lookup per leg saved.
template <typename R> __device__ __forceinline__ constexpr R short_step() { return R(1.0e-3); }

template <int FIELD, typename R>
__device__ __forceinline__ void rkn4_step_cols(const FieldDescT<R>& F, R dtds, R tfac, R r[3], R& t, R T[3], R lam,
                                               R h, ColJacT<R>& V, R Blast[3], R& eps, unsigned& status) {
  const R hh = R(0.5) * h, h6 = h * (R(1.0) / R(6.0)), h26 = h * h6;
  R B1[3], B2[3], B3[3];
  // State and the q/p column together (the column's inhomogeneous terms are the stage vectors T_i x B_i).  The stage
  // slopes are folded into running sums as they appear -- sA = k1 + k2 + k3 (position), sB = k1 + 2 k2 + 2 k3 + k4
  // (direction), sE = k1 - k2 - k3 + k4 (error estimate), likewise qA, qB for the column -- so that no slope outlives
  // the next stage (registers: the kernel has none to spare).
  R* const dTq = V.dT[2];
  R* const drq = V.dr[2];
  R l[3], k[3], q[3], v[3], sA[3], sB[3], sE[3], qA[3], qB[3];
  field_at<FIELD>(F, r, B1, status);
  cross(T, B1, l);
  cross(dTq, B1, q);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k[i] = lam * l[i];
    q[i] = fma(lam, q[i], l[i]);
    sA[i] = k[i]; sB[i] = k[i]; sE[i] = k[i];
    qA[i] = q[i]; qB[i] = q[i];
  }
  {
    R rm[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) rm[i] = fma(R(0.125) * h * h, k[i], fma(hh, T[i], r[i]));
    field_at<FIELD>(F, rm, B2, status);
  }
  // stage 2
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = fma(hh, k[i], T[i]);
  cross(v, B2, l);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = fma(hh, q[i], dTq[i]);
  cross(v, B2, q);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k[i] = lam * l[i];
    q[i] = fma(lam, q[i], l[i]);
    sA[i] += k[i]; sB[i] = fma(R(2.0), k[i], sB[i]); sE[i] -= k[i];
    qA[i] += q[i]; qB[i] = fma(R(2.0), q[i], qB[i]);
  }
  // stage 3 (same field point)
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = fma(hh, k[i], T[i]);
  cross(v, B2, l);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = fma(hh, q[i], dTq[i]);
  cross(v, B2, q);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k[i] = lam * l[i];
    q[i] = fma(lam, q[i], l[i]);
    sA[i] += k[i]; sB[i] = fma(R(2.0), k[i], sB[i]); sE[i] -= k[i];
    qA[i] += q[i]; qB[i] = fma(R(2.0), q[i], qB[i]);
  }
  {
    R re[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) re[i] = fma(R(0.5) * h * h, k[i], fma(h, T[i], r[i]));
    field_at<FIELD>(F, re, B3, status);
  }
  // stage 4
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = fma(h, k[i], T[i]);
  cross(v, B3, l);
#pragma unroll
  for (int i = 0; i < 3; ++i) v[i] = fma(h, q[i], dTq[i]);
  cross(v, B3, q);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k[i] = lam * l[i];
    q[i] = fma(lam, q[i], l[i]);
    sB[i] += k[i]; sE[i] += k[i];
    qB[i] += q[i];
  }
  // the phi and theta columns: homogeneous, they need the three field values only
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    R* const dT = V.dT[c];
    R* const dr = V.dr[c];
    R d[3], w[3], dA[3], dB[3];
    cross(dT, B1, d);
#pragma unroll
    for (int i = 0; i < 3; ++i) { d[i] *= lam; dA[i] = d[i]; dB[i] = d[i]; w[i] = fma(hh, d[i], dT[i]); }
    cross(w, B2, d);
#pragma unroll
    for (int i = 0; i < 3; ++i) { d[i] *= lam; dA[i] += d[i]; dB[i] = fma(R(2.0), d[i], dB[i]); w[i] = fma(hh, d[i], dT[i]); }
    cross(w, B2, d);
#pragma unroll
    for (int i = 0; i < 3; ++i) { d[i] *= lam; dA[i] += d[i]; dB[i] = fma(R(2.0), d[i], dB[i]); w[i] = fma(h, d[i], dT[i]); }
    cross(w, B3, d);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      dB[i] = fma(lam, d[i], dB[i]);
      dr[i] = fma(h26, dA[i], fma(h, dT[i], dr[i]));
      dT[i] = fma(h6, dB[i], dT[i]);
    }
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    drq[i] = fma(h26, qA[i], fma(h, dTq[i], drq[i]));
    dTq[i] = fma(h6, qB[i], dTq[i]);
  }
  V.sigma = fma(h, tfac, V.sigma);
  eps = h * h * (fabs(sE[0]) + fabs(sE[1]) + fabs(sE[2]));
  // state
  R Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = fma(h26, sA[i], fma(h, T[i], r[i]));
    Tn[i] = fma(h6, sB[i], T[i]);
  }
  const R inrm = rsqrt_near_one(fma(Tn[0], Tn[0], fma(Tn[1], Tn[1], Tn[2] * Tn[2])));
#pragma unroll
  for (int i = 0; i < 3; ++i) { T[i] = Tn[i] * inrm; Blast[i] = B3[i]; }
  t = fma(h, dtds, t);
}

// The same step to first order in h (see const_field_step_first_order: a correction step that starts within
// first_order_step() of the surface): the field is looked up once, at the start point -- over |h| <= 1e-5 mm it changes by
// less than |grad B| h, which moves T' by <= |lam| |grad B| h^2 <= 6e-3 x 0.2 x 1e-10 = 1e-13 rad for any table of >= 10 mm
// spacing -- and every term with a further factor h or h lam is dropped (<= 3e-13 mm, <= 1e-13 relative on the columns).
// The field for the path-length correction is then looked up afresh at the end point (Blast is not set).
template <int FIELD, typename R>
__device__ __forceinline__ void rkn4_step_cols_first_order(const FieldDescT<R>& F, R dtds, R tfac, R r[3], R& t, R T[3],
                                                           R lam, R h, ColJacT<R>& V, unsigned& status) {
  const R u = h * lam;
  R B1[3], w1[3];
  field_at<FIELD>(F, r, B1, status);
  cross(T, B1, w1);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    R* const dT = V.dT[c];
    R* const dr = V.dr[c];
    R d1[3];
    cross(dT, B1, d1);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      dr[i] = fma(h, dT[i], dr[i]);
      dT[i] = fma(u, d1[i], c == 2 ? fma(h, w1[i], dT[i]) : dT[i]);
    }
  }
  V.sigma = fma(h, tfac, V.sigma);
  R Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = fma(h, T[i], r[i]);
    Tn[i] = fma(u, w1[i], T[i]);
  }
  const R inrm = rsqrt_near_one(fma(Tn[0], Tn[0], fma(Tn[1], Tn[1], Tn[2] * Tn[2])));
#pragma unroll
  for (int i = 0; i < 3; ++i) T[i] = Tn[i] * inrm;
  t = fma(h, dtds, t);
}

// The bound-to-bound Jacobian, non-trivial part: Ja rows (loc0, loc1, phi, theta) x columns
// (loc0, loc1, phi, theta, qp); Jt = row t over the same columns.  Row qp = e_qp, column t = e_t.
template <typename R>
struct BoundJacobianT {
  R Ja[4][5];
  R Jt[5];
};

// ---- surface kinds (geometry record entry [18]; U33; described at "General surfaces" below) --
constexpr int SURF_PLANE = 0, SURF_CYLINDER = 1, SURF_DISC = 2;

template <typename R>
__device__ __forceinline__ void local_to_global(const R* __restrict__ s, R l0, R l1, R r[3], R e0[3], R e1[3]) {
  const int kind = (int)s[18];
  if (kind == SURF_CYLINDER) {
    const R Rc = s[12];
    R sa, ca;
    sincos_lib(l0 * rcp_nr(Rc), sa, ca);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      r[i] = s[i] + Rc * (ca * s[9 + i] + sa * s[3 + i]) + l1 * s[6 + i];
      e0[i] = ca * s[3 + i] - sa * s[9 + i];
      e1[i] = s[6 + i];
    }
  } else if (kind == SURF_DISC) {
    R sa, ca;
    sincos_lib(l1, sa, ca);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const R er = ca * s[3 + i] + sa * s[6 + i];
      r[i] = fma(l0, er, s[i]);
      e0[i] = er;
      e1[i] = l0 * (ca * s[6 + i] - sa * s[3 + i]);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      r[i] = fma(l1, s[6 + i], fma(l0, s[3 + i], s[i]));
      e0[i] = s[3 + i];
      e1[i] = s[6 + i];
    }
  }
}

// unit normal at the point r of the surface (planes, discs: n; cylinder: the radial direction)
template <typename R>
__device__ __forceinline__ void surface_normal(const R* __restrict__ s, const R r[3], R nrm[3]) {
  if ((int)s[18] == SURF_CYLINDER) {
    const R d[3] = {r[0] - s[0], r[1] - s[1], r[2] - s[2]};
    const R z = d[0] * s[6] + d[1] * s[7] + d[2] * s[8];
    R dp[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) dp[i] = fma(-z, s[6 + i], d[i]);
    const R irho = rsqrt_nr(dot(dp, dp));
#pragma unroll
    for (int i = 0; i < 3; ++i) nrm[i] = dp[i] * irho;
  } else {
    nrm[0] = s[9]; nrm[1] = s[10]; nrm[2] = s[11];
  }
}

// local coordinates of the point r on the surface and the rows g0 = dloc0/dr, g1 = dloc1/dr
template <typename R>
__device__ __forceinline__ void global_to_local(const R* __restrict__ s, const R r[3], R& l0, R& l1, R g0[3], R g1[3]) {
  const R d[3] = {r[0] - s[0], r[1] - s[1], r[2] - s[2]};
  const int kind = (int)s[18];
  if (kind == SURF_CYLINDER) {
    const R Rc = s[12];
    const R dn = d[0] * s[9] + d[1] * s[10] + d[2] * s[11], du = d[0] * s[3] + d[1] * s[4] + d[2] * s[5];
    const R k = Rc * rcp_nr(fma(dn, dn, du * du));
    l0 = Rc * atan2(du, dn);
    l1 = d[0] * s[6] + d[1] * s[7] + d[2] * s[8];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      g0[i] = k * (dn * s[3 + i] - du * s[9 + i]);
      g1[i] = s[6 + i];
    }
  } else if (kind == SURF_DISC) {
    const R du = d[0] * s[3] + d[1] * s[4] + d[2] * s[5], dv = d[0] * s[6] + d[1] * s[7] + d[2] * s[8];
    const R rho2 = fma(du, du, dv * dv);
    R irho;
    const R rho = sqrt_nr(rho2, irho);
    const R irho2 = irho * irho;
    l0 = rho;
    l1 = atan2(dv, du);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      g0[i] = (du * s[3 + i] + dv * s[6 + i]) * irho;
      g1[i] = (du * s[6 + i] - dv * s[3 + i]) * irho2;
    }
  } else {
    l0 = d[0] * s[3] + d[1] * s[4] + d[2] * s[5];
    l1 = d[0] * s[6] + d[1] * s[7] + d[2] * s[8];
#pragma unroll
    for (int i = 0; i < 3; ++i) { g0[i] = s[3 + i]; g1[i] = s[6 + i]; }
  }
}

// Straight-line path length from (r, T) to the surface; false when it cannot be reached.  Planes, discs:
// n.(c - r)/(n.T) with n.T > 1e-6.  Cylinder: a h^2 + 2 b h + c0 = 0 for the components normal to the axis,
// root h = -c0 / (b + sqrt(b^2 - a c0)): the crossing ahead of a track inside the cylinder, and the near root in
// cancellation-free form once the track is within round-off of the surface (U33).
template <typename R>
__device__ __forceinline__ bool path_to_surface(const R* __restrict__ s, const R r[3], const R T[3], R& h) {
  if ((int)s[18] == SURF_CYLINDER) {
    const R Rc = s[12];
    const R d[3] = {r[0] - s[0], r[1] - s[1], r[2] - s[2]};
    const R dz = d[0] * s[6] + d[1] * s[7] + d[2] * s[8], tz = T[0] * s[6] + T[1] * s[7] + T[2] * s[8];
    R dp[3], tp[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) { dp[i] = fma(-dz, s[6 + i], d[i]); tp[i] = fma(-tz, s[6 + i], T[i]); }
    const R a2 = dot(tp, tp), b = dot(dp, tp), c0 = dot(dp, dp) - Rc * Rc;
    const R disc = fma(b, b, -a2 * c0);
    if (!(disc > R(0.0))) return false;
    const R den = b + sqrt_nr(disc);
    if (!(den > R(kNdotTMin) * Rc)) return false;
    h = -c0 * rcp_nr(den);
    return true;
  }
  const R nT = T[0] * s[9] + T[1] * s[10] + T[2] * s[11];
  if (!(nT > R(kNdotTMin))) return false;
  h = ((s[0] - r[0]) * s[9] + (s[1] - r[1]) * s[10] + (s[2] - r[2]) * s[11]) * rcp_nr(nT);
  return true;
}

// ---- propagate a bound state from surface sf to surface st (A.1 - A.3) ---------------------------
// trig = (sin phi, cos phi, sin theta, cos theta) of x on entry; on success it holds the values of
// the predicted (phi, theta), taken from the direction vector itself.  Returns 0 or the stopping bit.
// CURVED: the surfaces may be of any kind (the start surface's chart, the target's path length, normal and chart
// through local_to_global / path_to_surface / surface_normal / global_to_local); else both are planes.
template <int FIELD, typename R, bool CURVED = false>
__device__ __forceinline__ unsigned propagate(const FieldDescT<R>& F, R mass, int n_corr,
                                              R max_step, R step_tol, const R* __restrict__ sf,
                                              const R* __restrict__ st, const R x[6],
                                              R trig[4], R xo[6], BoundJacobianT<R>& J,
                                              R& errmax, unsigned& status) {
  const R sphi = trig[0], cphi = trig[1], sth = trig[2], cth = trig[3];
  // A.1 bound -> free
  R r[3], T[3], e0[3], e1[3];  // e0, e1 = dr/dloc0, dr/dloc1 on the start surface
  if constexpr (CURVED) {
    local_to_global(sf, x[0], x[1], r, e0, e1);
  } else {
#pragma unroll
    for (int i = 0; i < 3; ++i) { r[i] = fma(x[1], sf[6 + i], fma(x[0], sf[3 + i], sf[i])); e0[i] = sf[3 + i]; e1[i] = sf[6 + i]; }
  }
  T[0] = cphi * sth; T[1] = sphi * sth; T[2] = cth;
  const R lam = x[4];
  R t = x[5];
  const R Tphi[3] = {-T[1], T[0], R(0.0)};
  const R Tth[3] = {cphi * cth, sphi * cth, -sth};
  const R nt[3] = {st[9], st[10], st[11]};
  const R ct[3] = {st[0], st[1], st[2]};
  const R ml = mass * lam;
  R idtds;
  const R dtds = sqrt_nr(fma(ml, ml, R(1.0)), idtds);  // dt/ds = sqrt(1 + m^2 lam^2)
  const R tfac = mass * ml * idtds;                  // d(dt/ds)/dlam

  // A.2 stepping: n_sub primary steps + n_corr correction steps, no accept/reject
  int n_sub = 1;
  R nT = dot(nt, T);
  R h_first = R(0.0);  // CURVED: the first step's path length (also the reachability test)
  if constexpr (CURVED) {
    if (!path_to_surface(st, r, T, h_first)) return ST_PROPAGATION;
    // a cylinder is reached from inside: a first aim that lies behind the start point (outside, moving away) is
    // "cannot be reached", not a step backwards; later aims of the leg are corrections and may have either sign
    if ((int)st[18] == SURF_CYLINDER && !(h_first > R(0.0))) return ST_PROPAGATION;
  } else {
    if (!(nT > R(kNdotTMin))) return ST_PROPAGATION;
  }
  if (max_step > R(0.0) || step_tol > R(0.0)) {
    R s0;
    if constexpr (CURVED) {
      s0 = h_first;
    } else {
      const R dr[3] = {ct[0] - r[0], ct[1] - r[1], ct[2] - r[2]};
      s0 = dot(nt, dr) / nT;
    }
    if (max_step > R(0.0)) {
      R qn = ceil(fabs(s0) / max_step * (R(1.0) - R(1e-12)));
      if (!(qn >= R(1.0))) qn = R(1.0);
      if (qn > R(1024.0)) qn = R(1024.0);
      n_sub = (int)qn;
    }
    if (step_tol > R(0.0)) {
      // adaptive step count (U31): the embedded error estimate of ONE trial step over the
      // whole leg fixes the number of primary steps, n = ceil((eps0 / tol)^(1/4)); the trial step is discarded
      R e0;
      if constexpr (FIELD == FIELD_CONST) {
        // closed form of h^2 |k1 - k2 - k3 + k4|_1 in a constant field (const_field_step)
        const R u = s0 * lam, sq = u * u * F.b2;
        R w1[3], w2[3];
        cross(T, F.b, w1);
        cross(w1, F.b, w2);
        e0 = s0 * s0 * fabs(lam) * R(0.25) * sq *
             (fabs(fma(u, w2[0], w1[0])) + fabs(fma(u, w2[1], w1[1])) + fabs(fma(u, w2[2], w1[2])));
      } else {
        R rr[3] = {r[0], r[1], r[2]}, TT[3] = {T[0], T[1], T[2]}, tt = t;
        R A[9], a[3], Bm[9], b[3], tau;
        rkn4_step<FIELD>(F, dtds, tfac, rr, tt, TT, lam, s0, A, a, Bm, b, tau, e0, status);
      }
      R qn = ceil(sqrt(sqrt(e0 / step_tol)) * (R(1.0) - R(1e-12)));
      if (!(qn >= R(1.0))) qn = R(1.0);
      if (qn > R(1024.0)) qn = R(1024.0);
      if ((int)qn > n_sub) n_sub = (int)qn;
    }
  }
  const int n_steps = n_sub + n_corr;
  typename std::conditional<FIELD == FIELD_CONST, PolyJacT<R>, ColJacT<R>>::type D;
  R Bend[3];             // grid field: the field of the last step's fourth stage, used when that step was a short one
  bool have_Bend = false;
  if constexpr (FIELD != FIELD_CONST) {
    // columns of J_b2f: d(r, T)/d(phi) = (0, Tphi), /d(theta) = (0, Tth), /d(q/p) = (0, 0)
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      D.dr[0][i] = D.dr[1][i] = D.dr[2][i] = R(0.0);
      D.dT[0][i] = Tphi[i]; D.dT[1][i] = Tth[i]; D.dT[2][i] = R(0.0);
    }
    D.sigma = R(0.0);
  }
  bool fast = false;
  if constexpr (FIELD == FIELD_CONST) {
    // default policy (one primary + two correction steps) in a constant field: the three steps as one
    // straight-line instruction stream, failure tests collected and taken once at the end
    fast = n_sub == 1 && n_corr == 2;
    if (fast) {
      bool bad = false;
#pragma unroll
      for (int is = 0; is < 3; ++is) {
        R h;
        if constexpr (CURVED) {
          h = h_first;
          if (is > 0) bad = !path_to_surface(st, r, T, h) || bad;
        } else {
          if (is > 0) {
            nT = dot(nt, T);
            bad = bad || !(nT > R(kNdotTMin));
          }
          const R dr[3] = {ct[0] - r[0], ct[1] - r[1], ct[2] - r[2]};
          h = dot(nt, dr) * rcp_nr(nT);
        }
        if (is == 0) const_field_step<true>(F.b, F.b2, dtds, tfac, lam, h, r, t, T, D, errmax);
        else if (is == 2 && fabs(h) <= first_order_step<R>()) const_field_step_first_order(F.b, F.b2, dtds, tfac, lam, h, r, t, T, D);
        else const_field_step<false>(F.b, F.b2, dtds, tfac, lam, h, r, t, T, D, errmax);
      }
      const R fin = r[0] + r[1] + r[2] + T[0] + T[1] + T[2] + t;
      if (bad || !(fabs(fin) < big<R>())) return ST_PROPAGATION;  // non-finite values persist through the steps
    }
  }
  for (int is = 0; !fast && is < n_steps; ++is) {
    R h;
    if constexpr (CURVED) {
      h = h_first;
      if (is > 0 && !path_to_surface(st, r, T, h)) return ST_PROPAGATION;
    } else {
      if (is > 0) {
        nT = dot(nt, T);
        if (!(nT > R(kNdotTMin))) return ST_PROPAGATION;
      }
      const R dr[3] = {ct[0] - r[0], ct[1] - r[1], ct[2] - r[2]};
      h = dot(nt, dr) * rcp_nr(nT);
    }
    if (is < n_sub - 1) h = h / (R)(n_sub - is);
    if constexpr (FIELD == FIELD_CONST) {
      if (is == 0) const_field_step<true>(F.b, F.b2, dtds, tfac, lam, h, r, t, T, D, errmax);
      else const_field_step<false>(F.b, F.b2, dtds, tfac, lam, h, r, t, T, D, errmax);
    } else {
      if (is >= n_sub && is > 0 && fabs(h) <= first_order_step<R>()) {
        have_Bend = false;
        rkn4_step_cols_first_order<FIELD>(F, dtds, tfac, r, t, T, lam, h, D, status);
      } else {
        R eps;
        have_Bend = fabs(h) <= short_step<R>();  // (of the last step, when the loop ends)
        rkn4_step_cols<FIELD>(F, dtds, tfac, r, t, T, lam, h, D, Bend, eps, status);
        errmax = fmax(errmax, eps);
      }
    }
    const R fin = r[0] + r[1] + r[2] + T[0] + T[1] + T[2] + t;
    if (!(fabs(fin) < big<R>())) return ST_PROPAGATION;  // catches NaN and Inf
  }

  // A.3 free -> bound with the path-length correction  D~ = (I - f' w^T) D,  w = normal / (normal . T)
  R nrm[3] = {nt[0], nt[1], nt[2]};
  if constexpr (CURVED) surface_normal(st, r, nrm);  // cylinder: the radial direction at the landing point
  nT = dot(nrm, T);
  if (!(nT > R(kNdotTMin))) return ST_PROPAGATION;
  R TxB[3];
  if constexpr (FIELD == FIELD_CONST) {
    cross(T, F.b, TxB);
  } else {
    // after a short last step (|h| <= short_step) the field of that step's last lookup stands for the field at the end point
    if (!have_Bend) field_at<FIELD>(F, r, Bend, status);
    cross(T, Bend, TxB);
  }
  const R kf_[3] = {lam * TxB[0], lam * TxB[1], lam * TxB[2]};  // dT/ds
  const R inT = rcp_nr(nT);
  const R w[3] = {nrm[0] * inT, nrm[1] * inT, nrm[2] * inT};

  const R st2 = fma(T[0], T[0], T[1] * T[1]);
  if (!(st2 > R(kSinThetaMin) * R(kSinThetaMin))) return ST_THETA;
  R isth;
  const R sth2 = sqrt_nr(st2, isth);
  const R cth2 = T[2];
  const R cph2 = T[0] * isth, sph2 = T[1] * isth;
  const R gphi[2] = {-sph2 * isth, cph2 * isth};
  const R gth[3] = {cph2 * cth2, sph2 * cth2, -sth2};
  // rows dloc0/dr, dloc1/dr of the target's chart (planes: u, v) and, CURVED, the local coordinates themselves
  const R* ut = st + 3;
  const R* vt = st + 6;
  R g0[3], g1[3];
  if constexpr (CURVED) {
    global_to_local(st, r, xo[0], xo[1], g0, g1);
    ut = g0;
    vt = g1;
  }

  // columns of D J_b2f as (cr, ct_, cT); then c -= f' (w . cr); then rows of J_f2b
  auto project = [&](int c, R cr[3], R ctime, R cT[3]) {
    const R wd = dot(w, cr);
#pragma unroll
    for (int i = 0; i < 3; ++i) { cr[i] = fma(-T[i], wd, cr[i]); cT[i] = fma(-kf_[i], wd, cT[i]); }
    J.Ja[0][c] = dot(ut, cr);
    J.Ja[1][c] = dot(vt, cr);
    J.Ja[2][c] = fma(gphi[0], cT[0], gphi[1] * cT[1]);
    J.Ja[3][c] = dot(gth, cT);
    J.Jt[c] = fma(-dtds, wd, ctime);
  };
  {
    R cr[3] = {e0[0], e0[1], e0[2]}, cT[3] = {R(0.0), R(0.0), R(0.0)};
    project(0, cr, R(0.0), cT);
  }
  {
    R cr[3] = {e1[0], e1[1], e1[2]}, cT[3] = {R(0.0), R(0.0), R(0.0)};
    project(1, cr, R(0.0), cT);
  }
  if constexpr (FIELD == FIELD_CONST) {
    {
      R vx[3], vxx[3], cr[3], cT[3];
      cross(Tphi, F.b, vx);
      cross(vx, F.b, vxx);
      poly_apply(F.b, D.P0, D.P1, D.P2, Tphi, vx, vxx, cr);
      poly_apply(F.b, R(1.0), D.Q1, D.Q2, Tphi, vx, vxx, cT);
      project(2, cr, R(0.0), cT);
    }
    {
      R vx[3], vxx[3], cr[3], cT[3];
      cross(Tth, F.b, vx);
      cross(vx, F.b, vxx);
      poly_apply(F.b, D.P0, D.P1, D.P2, Tth, vx, vxx, cr);
      poly_apply(F.b, R(1.0), D.Q1, D.Q2, Tth, vx, vxx, cT);
      project(3, cr, R(0.0), cT);
    }
  } else {
    project(2, D.dr[0], R(0.0), D.dT[0]);
    project(3, D.dr[1], R(0.0), D.dT[1]);
    project(4, D.dr[2], D.sigma, D.dT[2]);
  }
  if constexpr (FIELD == FIELD_CONST) {
    R cr[3] = {D.p[0], D.p[1], D.p[2]}, cT[3] = {D.q[0], D.q[1], D.q[2]};
    project(4, cr, D.sigma, cT);
  }

  if constexpr (!CURVED) {
    const R dr[3] = {r[0] - ct[0], r[1] - ct[1], r[2] - ct[2]};
    xo[0] = dot(ut, dr);
    xo[1] = dot(vt, dr);
  }
  // phi' = atan2(Ty, Tx) and theta' = acos(Tz), taken as the input angle plus the rotation over the leg
  // (sin of the difference from the two direction vectors) whenever that rotation is small
  {
    const R sdp = fma(sph2, cphi, -cph2 * sphi), cdp = fma(cph2, cphi, sph2 * sphi);
    const R sdt = fma(sth2, cth, -cth2 * sth), cdt = fma(cth2, cth, sth2 * sth);
    if (fabs(sdp) <= R(kSmallSine) && cdp > R(0.0) && fabs(sdt) <= R(kSmallSine) && cdt > R(0.0) && fabs(x[2]) <= R(kPi) &&
        x[3] > R(0.0) && x[3] < R(kPi)) {
      R ph = x[2] + asin_small(sdp);
      if (ph > R(kPi)) ph -= R(2.0) * R(kPi);
      else if (ph <= -R(kPi)) ph += R(2.0) * R(kPi);
      xo[2] = ph;
      xo[3] = x[3] + asin_small(sdt);
    } else {
      xo[2] = atan2(T[1], T[0]);
      xo[3] = acos(fmin(fmax(T[2], -R(1.0)), R(1.0)));
    }
  }
  xo[4] = lam;
  xo[5] = t;
  trig[0] = sph2; trig[1] = cph2; trig[2] = sth2; trig[3] = cth2;
  R chk = xo[0] + xo[1] + xo[5];
#pragma unroll
  for (int c = 0; c < 5; ++c) chk += J.Ja[0][c] + J.Ja[1][c] + J.Ja[2][c] + J.Ja[3][c] + J.Jt[c];
  if (!(fabs(chk) < big<R>())) return ST_PROPAGATION;
  return 0u;
}

// =====================================================================================================
// General surfaces and the field-gradient terms: the path for geometries that are not all planes
// (kf_geometry.surface_kinds) and for kf_options.field_gradient.  Not the hot path: one code path for
// every field kind, library trigonometry, the five variational columns of D J_b2f carried through every step.
//
// Surface kinds (geometry record entry [18]; "surfaces of different concrete types"; U33):
//   0 PLANE     r = c + loc0 u + loc1 v
//   1 CYLINDER  axis v through c, radius R = entry [12], azimuth alpha = loc0 / R from n towards u:
//               r = c + R (cos alpha n + sin alpha u) + loc1 v
//   2 DISC      the plane through c with normal n in polar coordinates: r = c + loc0 (cos loc1 u + sin loc1 v)
// the five variational columns d(r, T)/d(loc0, loc1, phi, theta, q/p) of D J_b2f and dt/dlam
template <typename R>
struct ColJac5T {
  R dr[5][3], dT[5][3];
  R sigma;
};

// One RKN4 step with the five columns carried through its stages (rkn4_step_cols with all columns; GRAD: plus the
// field-gradient terms lam T_i x (G_i dr_i) in every stage derivative, U32 -- the derivative of the stage
// arithmetic itself, h held fixed).
template <int FIELD, bool GRAD, typename R>
__device__ __forceinline__ void rkn4_step_cols5(const FieldDescT<R>& F, R dtds, R tfac, R r[3], R& t, R T[3], R lam,
                                                R h, ColJac5T<R>& V, R Blast[3], R& eps, unsigned& status) {
  const R hh = R(0.5) * h, h6 = h * (R(1.0) / R(6.0)), h26 = h * h6, h28 = R(0.125) * h * h, h22 = R(0.5) * h * h;
  R B1[3], B2[3], B3[3], G1[9], G2[9], G3[9];
  R T2[3], T3[3], T4[3], k1[3], k2[3], k3[3], k4[3], l1[3], l2[3], l3[3], l4[3];
  auto lookup = [&](const R pos[3], R B[3], R G[9]) {
    if constexpr (GRAD) field_and_gradient_at<FIELD>(F, pos, B, G, status);
    else field_at<FIELD>(F, pos, B, status);
  };
  lookup(r, B1, G1);
  cross(T, B1, l1);
  R rm[3], re[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) { k1[i] = lam * l1[i]; rm[i] = fma(h28, k1[i], fma(hh, T[i], r[i])); T2[i] = fma(hh, k1[i], T[i]); }
  lookup(rm, B2, G2);
  cross(T2, B2, l2);
#pragma unroll
  for (int i = 0; i < 3; ++i) { k2[i] = lam * l2[i]; T3[i] = fma(hh, k2[i], T[i]); }
  cross(T3, B2, l3);
#pragma unroll
  for (int i = 0; i < 3; ++i) { k3[i] = lam * l3[i]; re[i] = fma(h22, k3[i], fma(h, T[i], r[i])); T4[i] = fma(h, k3[i], T[i]); }
  lookup(re, B3, G3);
  cross(T4, B3, l4);
#pragma unroll
  for (int i = 0; i < 3; ++i) k4[i] = lam * l4[i];
  // stage derivative of one column: dk = [q/p: T_i x B_i] + lam (dT_i x B_i + T_i x (G_i dr_i))
  auto stage = [&](const R Ti[3], const R Bi[3], const R Gi[9], const R li[3], const R dTi[3], const R dri[3], bool qp,
                   R dk[3]) {
    R a[3];
    cross(dTi, Bi, a);
    if constexpr (GRAD) {
      R dB[3], c[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) dB[i] = fma(Gi[i * 3 + 2], dri[2], fma(Gi[i * 3 + 1], dri[1], Gi[i * 3] * dri[0]));
      cross(Ti, dB, c);
#pragma unroll
      for (int i = 0; i < 3; ++i) a[i] += c[i];
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) dk[i] = qp ? fma(lam, a[i], li[i]) : lam * a[i];
  };
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    const bool qp = c == 4;
    R* const dr = V.dr[c];
    R* const dT = V.dT[c];
    R d1[3], d2[3], d3[3], d4[3], ds[3], dTs[3];
    stage(T, B1, G1, l1, dT, dr, qp, d1);
#pragma unroll
    for (int i = 0; i < 3; ++i) { ds[i] = fma(h28, d1[i], fma(hh, dT[i], dr[i])); dTs[i] = fma(hh, d1[i], dT[i]); }
    stage(T2, B2, G2, l2, dTs, ds, qp, d2);
#pragma unroll
    for (int i = 0; i < 3; ++i) dTs[i] = fma(hh, d2[i], dT[i]);
    stage(T3, B2, G2, l3, dTs, ds, qp, d3);
#pragma unroll
    for (int i = 0; i < 3; ++i) { ds[i] = fma(h22, d3[i], fma(h, dT[i], dr[i])); dTs[i] = fma(h, d3[i], dT[i]); }
    stage(T4, B3, G3, l4, dTs, ds, qp, d4);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      dr[i] = fma(h26, d1[i] + d2[i] + d3[i], fma(h, dT[i], dr[i]));
      dT[i] = fma(h6, (d1[i] + d4[i]) + R(2.0) * (d2[i] + d3[i]), dT[i]);
    }
  }
  V.sigma = fma(h, tfac, V.sigma);
  eps = h * h * (fabs(k1[0] - k2[0] - k3[0] + k4[0]) + fabs(k1[1] - k2[1] - k3[1] + k4[1]) +
                 fabs(k1[2] - k2[2] - k3[2] + k4[2]));
  R Tn[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r[i] = fma(h26, k1[i] + k2[i] + k3[i], fma(h, T[i], r[i]));
    Tn[i] = fma(h6, (k1[i] + k4[i]) + R(2.0) * (k2[i] + k3[i]), T[i]);
  }
  const R inrm = rsqrt_near_one(fma(Tn[0], Tn[0], fma(Tn[1], Tn[1], Tn[2] * Tn[2])));
#pragma unroll
  for (int i = 0; i < 3; ++i) { T[i] = Tn[i] * inrm; Blast[i] = B3[i]; }
  t = fma(h, dtds, t);
}

// bound state on surface sf -> bound state on surface st, any kinds (A.1 - A.3 with the surface's own chart, normal and
// path length).  Same contract as propagate().
template <int FIELD, bool GRAD, typename R>
__device__ __forceinline__ unsigned propagate_general(const FieldDescT<R>& F, R mass, int n_corr, R max_step, R step_tol,
                                                      const R* __restrict__ sf, const R* __restrict__ st, const R x[6],
                                                      R trig[4], R xo[6], BoundJacobianT<R>& J, R& errmax,
                                                      unsigned& status) {
  const R sphi = trig[0], cphi = trig[1], sth = trig[2], cth = trig[3];
  R r[3], T[3];
  ColJac5T<R> D;
  local_to_global(sf, x[0], x[1], r, D.dr[0], D.dr[1]);
  T[0] = cphi * sth; T[1] = sphi * sth; T[2] = cth;
  const R lam = x[4];
  R t = x[5];
#pragma unroll
  for (int i = 0; i < 3; ++i) { D.dT[0][i] = D.dT[1][i] = D.dT[4][i] = R(0.0); D.dr[2][i] = D.dr[3][i] = D.dr[4][i] = R(0.0); }
  D.dT[2][0] = -T[1]; D.dT[2][1] = T[0]; D.dT[2][2] = R(0.0);
  D.dT[3][0] = cphi * cth; D.dT[3][1] = sphi * cth; D.dT[3][2] = -sth;
  D.sigma = R(0.0);
  const R ml = mass * lam;
  R idtds;
  const R dtds = sqrt_nr(fma(ml, ml, R(1.0)), idtds);
  const R tfac = mass * ml * idtds;

  int n_sub = 1;
  R h;
  if (!path_to_surface(st, r, T, h)) return ST_PROPAGATION;
  if ((int)st[18] == SURF_CYLINDER && !(h > R(0.0))) return ST_PROPAGATION;  // first aim behind the start point (see propagate<>)
  if (max_step > R(0.0)) {
    R qn = ceil(fabs(h) / max_step * (R(1.0) - R(1e-12)));
    if (!(qn >= R(1.0))) qn = R(1.0);
    if (qn > R(1024.0)) qn = R(1024.0);
    n_sub = (int)qn;
  }
  if (step_tol > R(0.0)) {  // adaptive step count (U31): the estimate of one trial step over the whole leg
    R rr[3] = {r[0], r[1], r[2]}, TT[3] = {T[0], T[1], T[2]}, tt = t, e0;
    R A[9], a[3], Bm[9], b[3], tau;
    rkn4_step<(FIELD == FIELD_CONST ? FIELD_CONST : FIELD_GRID3)>(F, dtds, tfac, rr, tt, TT, lam, h, A, a, Bm, b, tau, e0, status);
    R qn = ceil(sqrt(sqrt(e0 / step_tol)) * (R(1.0) - R(1e-12)));
    if (!(qn >= R(1.0))) qn = R(1.0);
    if (qn > R(1024.0)) qn = R(1024.0);
    if ((int)qn > n_sub) n_sub = (int)qn;
  }
  const int n_steps = n_sub + n_corr;
  R Bend[3];
  bool have_Bend = false;
  for (int is = 0; is < n_steps; ++is) {
    if (is > 0 && !path_to_surface(st, r, T, h)) return ST_PROPAGATION;
    if (is < n_sub - 1) h = h / (R)(n_sub - is);
    R eps;
    have_Bend = fabs(h) <= short_step<R>();
    rkn4_step_cols5<FIELD, GRAD>(F, dtds, tfac, r, t, T, lam, h, D, Bend, eps, status);
    errmax = fmax(errmax, eps);
    const R fin = r[0] + r[1] + r[2] + T[0] + T[1] + T[2] + t;
    if (!(fabs(fin) < big<R>())) return ST_PROPAGATION;
  }

  // A.3 free -> bound with the path-length correction, w = normal / (normal . T)
  R nt[3];
  surface_normal(st, r, nt);
  const R nT = dot(nt, T);
  if (!(nT > R(kNdotTMin))) return ST_PROPAGATION;
  if (!have_Bend) field_at<FIELD>(F, r, Bend, status);
  R TxB[3];
  cross(T, Bend, TxB);
  const R kf_[3] = {lam * TxB[0], lam * TxB[1], lam * TxB[2]};
  const R inT = R(1.0) / nT;
  const R w[3] = {nt[0] * inT, nt[1] * inT, nt[2] * inT};
  const R st2 = fma(T[0], T[0], T[1] * T[1]);
  if (!(st2 > R(kSinThetaMin) * R(kSinThetaMin))) return ST_THETA;
  R isth;
  const R sth2 = sqrt_nr(st2, isth);
  const R cth2 = T[2];
  const R cph2 = T[0] * isth, sph2 = T[1] * isth;
  const R gphi[2] = {-sph2 * isth, cph2 * isth};
  const R gth[3] = {cph2 * cth2, sph2 * cth2, -sth2};
  R g0[3], g1[3];
  global_to_local(st, r, xo[0], xo[1], g0, g1);
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    R* const cr = D.dr[c];
    R* const cT = D.dT[c];
    const R wd = dot(w, cr);
#pragma unroll
    for (int i = 0; i < 3; ++i) { cr[i] = fma(-T[i], wd, cr[i]); cT[i] = fma(-kf_[i], wd, cT[i]); }
    J.Ja[0][c] = dot(g0, cr);
    J.Ja[1][c] = dot(g1, cr);
    J.Ja[2][c] = fma(gphi[0], cT[0], gphi[1] * cT[1]);
    J.Ja[3][c] = dot(gth, cT);
    J.Jt[c] = fma(-dtds, wd, c == 4 ? D.sigma : R(0.0));
  }
  {
    const R sdp = fma(sph2, cphi, -cph2 * sphi), cdp = fma(cph2, cphi, sph2 * sphi);
    const R sdt = fma(sth2, cth, -cth2 * sth), cdt = fma(cth2, cth, sth2 * sth);
    if (fabs(sdp) <= R(kSmallSine) && cdp > R(0.0) && fabs(sdt) <= R(kSmallSine) && cdt > R(0.0) && fabs(x[2]) <= R(kPi) &&
        x[3] > R(0.0) && x[3] < R(kPi)) {
      R ph = x[2] + asin_small(sdp);
      if (ph > R(kPi)) ph -= R(2.0) * R(kPi);
      else if (ph <= -R(kPi)) ph += R(2.0) * R(kPi);
      xo[2] = ph;
      xo[3] = x[3] + asin_small(sdt);
    } else {
      xo[2] = atan2(T[1], T[0]);
      xo[3] = acos(fmin(fmax(T[2], -R(1.0)), R(1.0)));
    }
  }
  xo[4] = lam;
  xo[5] = t;
  trig[0] = sph2; trig[1] = cph2; trig[2] = sth2; trig[3] = cth2;
  R chk = xo[0] + xo[1] + xo[5];
#pragma unroll
  for (int c = 0; c < 5; ++c) chk += J.Ja[0][c] + J.Ja[1][c] + J.Ja[2][c] + J.Ja[3][c] + J.Jt[c];
  if (!(fabs(chk) < big<R>())) return ST_PROPAGATION;
  return 0u;
}

// ---- C- = J C J^T with the structure of J (A.4) -----------------------------------------------------
template <typename R>
__device__ __forceinline__ void transport_covariance(const BoundJacobianT<R>& J, const R C[21],
                                                     R Cp[21]) {
  // M = J C : rows a = 0..3 and t; row qp of M is row qp of C
  R Ma[4][6], Mt[6];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      R s = J.Ja[i][0] * C[SX(0, k)];
#pragma unroll
      for (int l = 1; l < 5; ++l) s = fma(J.Ja[i][l], C[SX(l, k)], s);
      Ma[i][k] = s;
    }
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    R s = C[SX(5, k)];
#pragma unroll
    for (int l = 0; l < 5; ++l) s = fma(J.Jt[l], C[SX(l, k)], s);
    Mt[k] = s;
  }
  // C- = M J^T, upper triangle
#pragma unroll
  for (int i = 0; i < 4; ++i) {
#pragma unroll
    for (int j = i; j < 4; ++j) {
      R s = Ma[i][0] * J.Ja[j][0];
#pragma unroll
      for (int l = 1; l < 5; ++l) s = fma(Ma[i][l], J.Ja[j][l], s);
      Cp[IX(i, j)] = s;
    }
    Cp[IX(i, 4)] = Ma[i][4];
    R s = Ma[i][5];
#pragma unroll
    for (int l = 0; l < 5; ++l) s = fma(Ma[i][l], J.Jt[l], s);
    Cp[IX(i, 5)] = s;
  }
  Cp[IX(4, 4)] = C[IX(4, 4)];
  {
    R s = C[IX(4, 5)];  // M[qp][t]
#pragma unroll
    for (int l = 0; l < 5; ++l) s = fma(C[SX(4, l)], J.Jt[l], s);
    Cp[IX(4, 5)] = s;
  }
  {
    R s = Mt[5];
#pragma unroll
    for (int l = 0; l < 5; ++l) s = fma(Mt[l], J.Jt[l], s);
    Cp[IX(5, 5)] = s;
  }
}

// ---- gain-matrix update with a 2-D hit (A.5) ----------------------------------------
// Split in two so that the outlier test (on chi2) comes before any state is written.
template <typename R>
struct GainT {
  R r0, r1, i00, i01, i11;
};
// Returns false when S = H C- H^T + V is not positive definite.
template <typename R>
__device__ __forceinline__ bool gain_prepare(const R xp[6], const R Cp[21], R m0, R m1,
                                             R v00, R v01, R v11, GainT<R>& G, R& chi2) {
  G.r0 = m0 - xp[0];
  G.r1 = m1 - xp[1];
  const R S00 = Cp[IX(0, 0)] + v00, S01 = Cp[IX(0, 1)] + v01, S11 = Cp[IX(1, 1)] + v11;
  const R det = fma(S00, S11, -S01 * S01);
  if (!(S00 > R(0.0) && det > R(0.0))) return false;
  const R idet = rcp_nr(det);
  G.i00 = S11 * idet;
  G.i01 = -S01 * idet;
  G.i11 = S00 * idet;
  chi2 = G.r0 * fma(G.i00, G.r0, G.i01 * G.r1) + G.r1 * fma(G.i01, G.r0, G.i11 * G.r1);
  return true;
}
// x+ = x- + K r, C+ = (I - K H) C-  with K = C- H^T S^-1.  xf/Cf must not alias xp/Cp.
template <typename R>
__device__ __forceinline__ void gain_apply(const GainT<R>& G, const R xp[6], const R Cp[21],
                                           R xf[6], R Cf[21]) {
  R K0[6], K1[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    const R c0 = Cp[SX(i, 0)], c1 = Cp[SX(i, 1)];
    K0[i] = fma(c0, G.i00, c1 * G.i01);
    K1[i] = fma(c0, G.i01, c1 * G.i11);
    xf[i] = fma(K1[i], G.r1, fma(K0[i], G.r0, xp[i]));
  }
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = i; j < 6; ++j)
      Cf[IX(i, j)] = fma(-K1[i], Cp[SX(1, j)], fma(-K0[i], Cp[SX(0, j)], Cp[IX(i, j)]));
}

// ---- material at a surface, after the update (A.6) -----------------------------------
// Highland theta0^2 and Bethe mean loss from the filtered state.  trig = sin/cos of the filtered
// (phi, theta).  Returns false when the energy is exhausted (E' <= m).
template <typename R>
struct MaterialStepT {
  R lam_out, g, theta0sq_over_sin2, theta0sq;
};
// nrm: the unit normal of the surface at the state's position (planes: the record's n = surf + 9)
template <typename R>
__device__ __forceinline__ bool material_prepare(const MaterialDescT<R>& Mt, const R* __restrict__ surf,
                                                 const R* __restrict__ nrm, const R trig[4], R lam,
                                                 MaterialStepT<R>& S) {
  const R sphi = trig[0], cphi = trig[1], sth = trig[2], cth = trig[3];
  const R m = Mt.mass;
  const R al = fabs(lam);
  const R p = rcp_nr(al);
  R iE;
  const R E = sqrt_nr(fma(p, p, m * m), iE);
  const R ib2 = (E * al) * (E * al);  // 1 / beta^2
  const R bg = p * Mt.inv_mass, gamma = E * Mt.inv_mass;
  const R nT = nrm[0] * (cphi * sth) + nrm[1] * (sphi * sth) + nrm[2] * cth;
  const R cfac = rcp_nr(fabs(nT));  // path factor 1/|n.T|
  // Highland: theta0 = 0.0136/(beta p) sqrt(X) (1 + 0.038 ln(X/beta^2)),  1/(beta p) = E lam^2
  const R X = surf[14] * cfac;
  const R theta0 = R(0.0136) * (E * al * al) * sqrt_nr(X) * fma(R(0.038), log_pos(X * ib2), R(1.0));
  // Bethe, asymptotic density correction
  const R me = R(kElectronMass);
  const R Wmax = R(2.0) * me * bg * bg * rcp_nr(R(1.0) + R(2.0) * gamma * Mt.rme + Mt.rme * Mt.rme);
  const R dhalf = fmax(R(0.0), Mt.log_hwp_I + log_pos(bg) - R(0.5));
  const R b2 = (p * iE) * (p * iE);
  const R dedx =
      R(kBetheK) * Mt.ZA * ib2 * (R(0.5) * log_pos(R(2.0) * me * bg * bg * Wmax * Mt.inv_I2) - b2 - dhalf);
  const R dE = dedx * Mt.rho * R(1e-3) * R(0.1) * surf[15] * cfac;
  const R E2 = E - dE;
  if (!(E2 > m)) return false;
  R ip2;
  const R p2 = sqrt_nr(fma(E2, E2, -m * m), ip2);
  (void)p2;
  const R pr = p * ip2;
  S.g = pr * pr * pr * E2 * iE;  // dlam'/dlam = p^3 E' / (p'^3 E)
  S.lam_out = (lam < R(0.0) ? -ip2 : ip2);
  const R t2 = theta0 * theta0;
  S.theta0sq = t2;
  S.theta0sq_over_sin2 = t2 * rcp_nr(sth * sth);
  return true;
}
template <typename R>
__device__ __forceinline__ bool material_prepare(const MaterialDescT<R>& Mt, const R* __restrict__ surf,
                                                 const R trig[4], R lam, MaterialStepT<R>& S) {
  return material_prepare(Mt, surf, surf + 9, trig, lam, S);
}
// the same on a surface of any kind: the normal at the state's local position (l0, l1)
template <typename R>
__device__ __forceinline__ bool material_prepare_general(const MaterialDescT<R>& Mt, const R* __restrict__ surf, R l0,
                                                         R l1, const R trig[4], R lam, MaterialStepT<R>& S) {
  R r[3], e0[3], e1[3], nrm[3];
  local_to_global(surf, l0, l1, r, e0, e1);
  surface_normal(surf, r, nrm);
  return material_prepare(Mt, surf, nrm, trig, lam, S);
}
// C <- G C G^T + Q : row/column qp scaled by g, Highland terms on the angle variances
template <typename R>
__device__ __forceinline__ void material_apply(const MaterialStepT<R>& S, R C[21]) {
#pragma unroll
  for (int i = 0; i < 6; ++i)
    if (i != 4) C[SX(i, 4)] *= S.g;
  C[IX(4, 4)] *= S.g * S.g;
  C[IX(2, 2)] += S.theta0sq_over_sin2;
  C[IX(3, 3)] += S.theta0sq;
}

// exact inverse of material_apply up to round-off (failure paths only)
template <typename R>
__device__ __forceinline__ void material_undo(const MaterialStepT<R>& S, R C[21]) {
  const R ig = R(1.0) / S.g;
  C[IX(2, 2)] -= S.theta0sq_over_sin2;
  C[IX(3, 3)] -= S.theta0sq;
#pragma unroll
  for (int i = 0; i < 6; ++i)
    if (i != 4) C[SX(i, 4)] *= ig;
  C[IX(4, 4)] *= ig * ig;
}

// the FP64 path's names (kf_lanes.cuh, kf_perigee.cuh, kf_mbf.cuh are double only)
using FieldDesc = FieldDescT<double>;
using MaterialDesc = MaterialDescT<double>;
using MatJac = MatJacT<double>;
using BoundJacobian = BoundJacobianT<double>;
using Gain = GainT<double>;
using MaterialStep = MaterialStepT<double>;

}  // namespace kf
