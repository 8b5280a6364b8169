// kf_perigee.cuh -- the fitted parameters on the perigee surface (sm_100a, IEEE double).
//
// at a perigee surface -- "defined at the point of closest approach to a reference point" --
// loc0, loc1 "become the transverse and longitudinal impact parameters d0 and z0"; PAPER.md:179-180 lists the
// fitted parameters on the target surface among the results, and the pulls of Fig. 5 are
// perigee pulls.  DESIGN.md readings U27-U30: the surface is a straight line (centre c, unit axis a); with
// D = r - c, D_perp = D - (D.a) a the state is on it when g = D_perp . T = 0; d0 = D . (a x T)/|a x T|,
// z0 = D . a.  first_* (the smoothed state entering the first visited layer) is taken there with the same
// fixed stepping policy as a leg (n_sub + n_corr RKN4 steps, each aimed with the Newton root of g along the
// track, h = -g / (dg/ds), dg/ds = 1 - (a.T)^2 + lam D_perp . (T x B); h < 0: the perigee lies behind the
// first plane), the free Jacobian alongside, and the path-length correction w = grad g / (dg/ds) with
// grad_r g = T - (a.T) a, grad_T g = D_perp.  No material is crossed.  One thread per track; 27 doubles in,
// 27 out: this kernel is a footnote to the fit's cost (0.1 ms per 1e6 tracks against 6 ms).
#pragma once

#include "kf_common.cuh"

namespace kf {

struct LineSurface {
  double c[3], a[3];
};

// (x on surface sf) -> (xo on the line, J).  Returns 0 or the stopping bit; `status` collects FIELD_CLAMPED.
// any_kind: the call runs in the general-surface kernels (kf_geometry.surface_kinds > 1), so record entry [18] says
// which chart sf has; false: planes only, entry [18] is NOT read (include/kf_fit.h: "entry [18] is then ignored").
template <int FIELD>
__device__ __forceinline__ unsigned propagate_to_line(const FieldDesc& F, double mass, int n_corr, double max_step,
                                                      bool any_kind,
                                                      const double* __restrict__ sf, const LineSurface& Ln,
                                                      const double x[6], double xo[6], BoundJacobian& J,
                                                      unsigned& status) {
  double sphi, cphi, sth, cth;
  sincos(x[2], &sphi, &cphi);
  sincos(x[3], &sth, &cth);
  double r[3], T[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) r[i] = sf[i] + x[0] * sf[3 + i] + x[1] * sf[6 + i];
  double e0[3] = {sf[3], sf[4], sf[5]}, e1[3] = {sf[6], sf[7], sf[8]};
  if (any_kind && (int)sf[18] != SURF_PLANE) local_to_global(sf, x[0], x[1], r, e0, e1);  // first_* on a cylinder or a disc (U33)
  T[0] = cphi * sth; T[1] = sphi * sth; T[2] = cth;
  const double lam = x[4];
  double t = x[5];
  const double Tphi[3] = {-T[1], T[0], 0.0};
  const double Tth[3] = {cphi * cth, sphi * cth, -sth};
  const double ml = mass * lam;
  const double dtds = sqrt(1.0 + ml * ml);
  const double tfac = mass * ml / dtds;

  MatJac D;
  int n_sub = 1;
  double dperp[3], aT, den, TxB[3];
  for (int is = 0;; ++is) {
    aT = dot(Ln.a, T);
    den = 1.0 - aT * aT;
    if (!(den > 1e-12)) return ST_PROPAGATION;  // moving along the axis: no closest approach
    const double dl[3] = {r[0] - Ln.c[0], r[1] - Ln.c[1], r[2] - Ln.c[2]};
    const double da = dot(dl, Ln.a);
#pragma unroll
    for (int i = 0; i < 3; ++i) dperp[i] = dl[i] - da * Ln.a[i];
    double Bs[3];
    field_at<FIELD>(F, r, Bs, status);
    cross(T, Bs, TxB);
    const double slope = den + lam * dot(dperp, TxB);  // dg/ds
    if (!(fabs(slope) > 1e-12)) return ST_PROPAGATION;
    double h = -dot(dperp, T) / slope;
    if (is == 0 && max_step > 0.0) {
      double qn = ceil(fabs(h) / max_step * (1.0 - 1e-12));
      if (!(qn >= 1.0)) qn = 1.0;
      if (qn > 1024.0) qn = 1024.0;
      n_sub = (int)qn;
    }
    if (is >= n_sub + n_corr) break;  // (r, T) is the final state; dperp, aT, den, TxB belong to it
    if (is < n_sub) h = h / (double)(n_sub - is);
    double A[9], a[3], Bm[9], b[3], tau, eps;
    rkn4_step<FIELD>(F, dtds, tfac, r, t, T, lam, h, A, a, Bm, b, tau, eps, status);
    if (is == 0) {
#pragma unroll
      for (int i = 0; i < 9; ++i) { D.P[i] = A[i]; D.Q[i] = Bm[i]; }
#pragma unroll
      for (int i = 0; i < 3; ++i) { D.p[i] = a[i]; D.q[i] = b[i]; }
      D.sigma = tau;
    } else {
      double AQ[9], Aq[3], BQ[9], Bq[3];
      mat3_mul(A, D.Q, AQ);
      mat3_vec(A, D.q, Aq);
      mat3_mul(Bm, D.Q, BQ);
      mat3_vec(Bm, D.q, Bq);
#pragma unroll
      for (int i = 0; i < 9; ++i) { D.P[i] += AQ[i]; D.Q[i] = BQ[i]; }
#pragma unroll
      for (int i = 0; i < 3; ++i) { D.p[i] += Aq[i] + a[i]; D.q[i] = Bq[i] + b[i]; }
      D.sigma += tau;
    }
    const double fin = r[0] + r[1] + r[2] + T[0] + T[1] + T[2] + t;
    if (!(fabs(fin) < 1.0e300)) return ST_PROPAGATION;
  }
  if (n_sub + n_corr == 0) {  // no step at all: D = identity
#pragma unroll
    for (int i = 0; i < 9; ++i) { D.P[i] = 0.0; D.Q[i] = (i % 4 == 0) ? 1.0 : 0.0; }
#pragma unroll
    for (int i = 0; i < 3; ++i) { D.p[i] = 0.0; D.q[i] = 0.0; }
    D.sigma = 0.0;
  }

  // free -> bound on the line with the path-length correction D~ = (I - f' w^T) D
  const double dgds = den + lam * dot(dperp, TxB);
  if (!(fabs(dgds) > 1e-12)) return ST_PROPAGATION;
  const double idg = 1.0 / dgds;
  const double wr[3] = {(T[0] - aT * Ln.a[0]) * idg, (T[1] - aT * Ln.a[1]) * idg, (T[2] - aT * Ln.a[2]) * idg};
  const double wT[3] = {dperp[0] * idg, dperp[1] * idg, dperp[2] * idg};
  const double kf_[3] = {lam * TxB[0], lam * TxB[1], lam * TxB[2]};  // dT/ds

  const double st2 = T[0] * T[0] + T[1] * T[1];
  if (!(st2 > kSinThetaMin * kSinThetaMin)) return ST_THETA;
  const double sth2 = sqrt(st2), isth = 1.0 / sth2, cth2 = T[2];
  const double cph2 = T[0] * isth, sph2 = T[1] * isth;
  const double gphi[2] = {-sph2 * isth, cph2 * isth};
  const double gth[3] = {cph2 * cth2, sph2 * cth2, -sth2};
  double ed[3];
  cross(Ln.a, T, ed);
  const double ied = 1.0 / sqrt(dot(ed, ed));
#pragma unroll
  for (int i = 0; i < 3; ++i) ed[i] *= ied;

  auto project = [&](int c, double cr[3], double ctime, double cT[3]) {
    const double wd = dot(wr, cr) + dot(wT, cT);
#pragma unroll
    for (int i = 0; i < 3; ++i) { cr[i] -= T[i] * wd; cT[i] -= kf_[i] * wd; }
    J.Ja[0][c] = dot(ed, cr);
    J.Ja[1][c] = dot(Ln.a, cr);
    J.Ja[2][c] = gphi[0] * cT[0] + gphi[1] * cT[1];
    J.Ja[3][c] = dot(gth, cT);
    J.Jt[c] = ctime - dtds * wd;
  };
  {
    double cr[3] = {e0[0], e0[1], e0[2]}, cT[3] = {0.0, 0.0, 0.0};
    project(0, cr, 0.0, cT);
  }
  {
    double cr[3] = {e1[0], e1[1], e1[2]}, cT[3] = {0.0, 0.0, 0.0};
    project(1, cr, 0.0, cT);
  }
  {
    double cr[3], cT[3];
    mat3_vec(D.P, Tphi, cr);
    mat3_vec(D.Q, Tphi, cT);
    project(2, cr, 0.0, cT);
  }
  {
    double cr[3], cT[3];
    mat3_vec(D.P, Tth, cr);
    mat3_vec(D.Q, Tth, cT);
    project(3, cr, 0.0, cT);
  }
  {
    double cr[3] = {D.p[0], D.p[1], D.p[2]}, cT[3] = {D.q[0], D.q[1], D.q[2]};
    project(4, cr, D.sigma, cT);
  }

  const double dl[3] = {r[0] - Ln.c[0], r[1] - Ln.c[1], r[2] - Ln.c[2]};
  xo[0] = dot(dl, ed);
  xo[1] = dot(dl, Ln.a);
  xo[2] = atan2(T[1], T[0]);
  xo[3] = acos(fmin(fmax(T[2], -1.0), 1.0));
  xo[4] = lam;
  xo[5] = t;
  double chk = xo[0] + xo[1] + xo[2] + xo[3] + xo[5];
#pragma unroll
  for (int c = 0; c < 5; ++c) chk += J.Ja[0][c] + J.Ja[1][c] + J.Ja[2][c] + J.Ja[3][c] + J.Jt[c];
  if (!(fabs(chk) < 1.0e300)) return ST_PROPAGATION;
  return 0u;
}

struct PerigeeParams {
  LineSurface line;
  double* params;  // [6][ldn]
  double* cov;     // [21][ldn]
  int any_kind;    // 1: the fit ran in the general-surface kernels, geometry entry [18] is the surface kind; 0: planes
};

constexpr int kPerigeeBlock = 128;

template <int FIELD>
__global__ void __launch_bounds__(kPerigeeBlock)
kf_perigee_kernel(const __grid_constant__ FitParams P, const __grid_constant__ PerigeeParams G) {
  const long long i = (long long)blockIdx.x * kPerigeeBlock + threadIdx.x;
  if (i >= P.N) return;
  const long long N = P.ldn;
  // first_* lives on the first visited surface, or on the start surface for a track that completed no leg
  const int nleg = P.n_used[i] + P.n_outliers[i] + P.n_holes[i];
  const double* __restrict__ sf = P.geom + (size_t)(P.start + (nleg > 0 ? 1 : 0)) * 20;
  double x[6], C[21];
#pragma unroll
  for (int k = 0; k < 6; ++k) x[k] = P.first_params[k * N + i];
#pragma unroll
  for (int k = 0; k < 21; ++k) C[k] = P.first_cov[k * N + i];
  unsigned status = 0u;
  double xo[6], Co[21];
  BoundJacobian J;
  const unsigned rc = propagate_to_line<FIELD>(P.field, P.mat.mass, P.n_corr, P.max_step, G.any_kind != 0, sf, G.line, x, xo, J, status);
  bool ok = rc == 0u;
  if (ok) {
    transport_covariance(J, C, Co);
    double chk = 0.0;
#pragma unroll
    for (int k = 0; k < 21; ++k) chk += Co[k];
    ok = fabs(chk) < 1.0e300;
  }
  if (!ok) {
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int k = 0; k < 6; ++k) xo[k] = nan;
#pragma unroll
    for (int k = 0; k < 21; ++k) Co[k] = nan;
    status |= ST_PERIGEE;
  }
  store6(G.params, N, i, xo);
  store21(G.cov, N, i, Co);
  if (status) P.status[i] |= status;
}

}  // namespace kf
