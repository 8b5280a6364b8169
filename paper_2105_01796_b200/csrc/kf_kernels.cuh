// kf_kernels.cuh -- the two global kernels of the thread-per-track variant (sm_100a, IEEE double).
//
//   kf_forward_kernel : one thread = one track.  Kalman step loop of PAPER.md:55-60: propagate
//                       (RKN4 + free-Jacobian transport), C- = J C J^T, gain-matrix
//                       update with the surface's 2-D hit, material.
//                       Writes one RTS record per (leg, track): x-, C-, F ("stored Jacobians",
//                       PAPER.md:62) and a one-byte hit flag.
//   kf_rts_kernel     : one thread = one track.  Rauch-Tung-Striebel backward pass
//                       over the records.  The filtered state (x+, C+) is NOT stored: it is
//                       recomputed from (x-, C-, hit, flag) with the same gain-matrix routine, which
//                       trades ~170 flops per leg for 27 doubles of HBM traffic each way
//                       (DESIGN.md "RTS record").
//
// Workspace layout, Np = N rounded up to 32:
//   rec   double[Lmax][kRecDoubles][Np]   component-major within a leg: a warp's 32 tracks write
//                                         32 consecutive doubles per component (256 B, coalesced)
//   flag  uint8 [Lmax][Np]                0 hole, 1 used, 2 outlier
//   nleg  int32 [Np]                      number of legs the forward pass completed
#pragma once

#include "kf_device.cuh"

namespace kf {

constexpr int kRecDoubles = 53;  // x-(6) C-(21) Fa(20) Ft(5) g(1)
constexpr int kRecXp = 0, kRecCp = 6, kRecFa = 27, kRecFt = 47, kRecG = 52;

#ifndef KF_FWD_BLOCK
#define KF_FWD_BLOCK 128
#endif
#ifndef KF_RTS_BLOCK
#define KF_RTS_BLOCK 128
#endif
#ifndef KF_FWD_MIN_BLOCKS
#define KF_FWD_MIN_BLOCKS 1
#endif
#ifndef KF_RTS_MIN_BLOCKS
#define KF_RTS_MIN_BLOCKS 1
#endif

enum : int { OUT_PRED = 1, OUT_FILT = 2, OUT_SMOOTH = 4 };

struct FitParams {
  // inputs
  long long N, Np, M;
  const double* params;   // [6][N]
  const double* cov;      // [21][N]
  int start;
  const int* offsets;     // [N+1]
  const int* surf_idx;    // [M]
  const double* loc;      // [2][M]
  const double* var;      // [2][M] or null
  const double* cov01;    // [M] or null
  int n_surfaces;
  const double* geom;     // [n_surfaces][20]
  int geom_in_smem;
  FieldDesc field;
  MaterialDesc mat;
  // options
  int smooth, n_corr, output_states;
  double outlier_chi2, max_step, inflation;
  // outputs
  double *first_params, *first_cov, *last_params, *last_cov, *chi2;
  int *ndf, *n_used, *n_outliers, *n_holes;
  unsigned* status;
  double* state_params[3];
  double* state_cov[3];
  double* hit_chi2;
  unsigned char* hit_flags;
  double* rk_err_max;
  // workspace
  double* rec;
  unsigned char* legflag;
  int* nleg;
};

__device__ __forceinline__ void store6(double* base, long long stride, long long i, const double v[6]) {
#pragma unroll
  for (int k = 0; k < 6; ++k) base[k * stride + i] = v[k];
}
__device__ __forceinline__ void store21(double* base, long long stride, long long i, const double v[21]) {
#pragma unroll
  for (int k = 0; k < 21; ++k) base[k * stride + i] = v[k];
}

// stage the geometry table in shared memory once per CTA (5 KB for 31 planes)
__device__ __forceinline__ const double* stage_geometry(const FitParams& P, double* smem) {
  if (!P.geom_in_smem) return P.geom;
  const int n = P.n_surfaces * 20;
  for (int k = threadIdx.x; k < n; k += blockDim.x) smem[k] = P.geom[k];
  __syncthreads();
  return smem;
}


// indices of the 9 numbers the material step changes: q/p, C(i,4) for i = 0..5, C(2,2), C(3,3)
__device__ __forceinline__ void stash_save(double* s, int stride, const double x[6], const double C[21]) {
  s[0] = x[4];
#pragma unroll
  for (int k = 0; k < 6; ++k) s[(1 + k) * stride] = C[SX(k, 4)];
  s[7 * stride] = C[IX(2, 2)];
  s[8 * stride] = C[IX(3, 3)];
}
__device__ __forceinline__ void stash_restore(const double* s, int stride, double x[6], double C[21]) {
  x[4] = s[0];
#pragma unroll
  for (int k = 0; k < 6; ++k) C[SX(k, 4)] = s[(1 + k) * stride];
  C[IX(2, 2)] = s[7 * stride];
  C[IX(3, 3)] = s[8 * stride];
}

// =====================================================================================================
// Forward filter.  Dynamic shared memory: [geometry table if geom_in_smem][9 doubles per thread].
template <int FIELD, bool MATERIAL>
__global__ void __launch_bounds__(KF_FWD_BLOCK, KF_FWD_MIN_BLOCKS)
kf_forward_kernel(const __grid_constant__ FitParams P) {
  extern __shared__ double s_dyn[];
  const double* __restrict__ G = stage_geometry(P, s_dyn);
  double* stash = s_dyn + (P.geom_in_smem ? P.n_surfaces * 20 : 0) + threadIdx.x;
  const int sstride = blockDim.x;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.N) return;
  const long long N = P.N, Np = P.Np;

  const int o0 = P.offsets[i], o1 = P.offsets[i + 1];
  double x[6], C[21];
#pragma unroll
  for (int k = 0; k < 6; ++k) x[k] = P.params[k * N + i];
#pragma unroll
  for (int k = 0; k < 21; ++k) C[k] = P.inflation * P.cov[k * N + i];

  unsigned status = 0u;
  // the hit list must be strictly ascending in surface index, inside (start, n_surfaces)
  int n_target = 0;
  {
    bool ok = true;
    int prev_s = P.start;
    for (int j = o0; j < o1; ++j) {
      const int s = P.surf_idx[j];
      if (!(s > prev_s && s < P.n_surfaces)) { ok = false; break; }
      prev_s = s;
    }
    if (!ok) status |= ST_BAD_HITS;
    else n_target = prev_s - P.start;  // visit every surface up to the one of the last hit (U7)
  }

  double chi2 = 0.0, errmax = 0.0, g_prev = 1.0;
  int n_used = 0, n_outl = 0, n_holes = 0, nleg = 0, hp = o0;
  bool mat_applied = false;
  double trig[4];
  sincos(x[2], &trig[0], &trig[1]);
  sincos(x[3], &trig[2], &trig[3]);

  for (int l = 0; l < n_target; ++l) {
    const int s = P.start + 1 + l;
    const double* __restrict__ sf = G + (s - 1) * 20;
    const double* __restrict__ st = G + s * 20;
    double xp[6];
    BoundJacobian J;
    double e = 0.0;
    const unsigned rc = propagate<FIELD>(P.field, P.mat.mass, P.n_corr, P.max_step, sf, st, x, trig,
                                         xp, J, e, status);
    if (rc) { status |= rc; break; }
    errmax = fmax(errmax, e);
    double Cp[21];
    transport_covariance(J, C, Cp);

    // RTS record: x-, C-, F = J G_prev, g_prev ("stored Jacobians")
    if (P.smooth) {
      double* __restrict__ R = P.rec + (size_t)l * kRecDoubles * Np + i;
#pragma unroll
      for (int k = 0; k < 6; ++k) R[(kRecXp + k) * Np] = xp[k];
#pragma unroll
      for (int k = 0; k < 21; ++k) R[(kRecCp + k) * Np] = Cp[k];
#pragma unroll
      for (int a = 0; a < 4; ++a) {
#pragma unroll
        for (int c = 0; c < 4; ++c) R[(kRecFa + a * 5 + c) * Np] = J.Ja[a][c];
        R[(kRecFa + a * 5 + 4) * Np] = J.Ja[a][4] * g_prev;
      }
#pragma unroll
      for (int c = 0; c < 4; ++c) R[(kRecFt + c) * Np] = J.Jt[c];
      R[(kRecFt + 4) * Np] = J.Jt[4] * g_prev;
      R[kRecG * Np] = g_prev;
    }

    // gain-matrix update with the surface's hit, or hole
    unsigned char flag = 0;
    const bool has_hit = (hp < o1) && (P.surf_idx[hp] == s);
    if (has_hit) {
      const double m0 = P.loc[hp], m1 = P.loc[P.M + hp];
      double v00, v11, v01 = 0.0;
      if (P.var) {
        v00 = P.var[hp];
        v11 = P.var[P.M + hp];
        if (P.cov01) v01 = P.cov01[hp];
      } else {
        v00 = st[16];
        v11 = st[17];
      }
      double c2 = 0.0;
      if (!gain_update(xp, Cp, m0, m1, v00, v01, v11, x, C, c2)) { status |= ST_NOT_POSITIVE; break; }
      if (P.outlier_chi2 > 0.0 && c2 > P.outlier_chi2) {  // strictly greater: flagged, not used (U9)
#pragma unroll
        for (int k = 0; k < 6; ++k) x[k] = xp[k];
#pragma unroll
        for (int k = 0; k < 21; ++k) C[k] = Cp[k];
        n_outl++;
        flag = 2;
      } else {
        chi2 += c2;
        n_used++;
        flag = 1;
      }
      if (P.hit_chi2) P.hit_chi2[hp] = c2;
      if (P.hit_flags) P.hit_flags[hp] = flag;
      hp++;
    } else {
#pragma unroll
      for (int k = 0; k < 6; ++k) x[k] = xp[k];
#pragma unroll
      for (int k = 0; k < 21; ++k) C[k] = Cp[k];
      n_holes++;
    }
    if (P.smooth) P.legflag[(size_t)l * Np + i] = flag;
    if (P.output_states & OUT_PRED) {
      store6(P.state_params[0] + (size_t)l * 6 * N, N, i, xp);
      store21(P.state_cov[0] + (size_t)l * 21 * N, N, i, Cp);
    }
    if (P.output_states & OUT_FILT) {
      store6(P.state_params[1] + (size_t)l * 6 * N, N, i, x);
      store21(P.state_cov[1] + (size_t)l * 21 * N, N, i, C);
    }
    if (l == 0) {
      store6(P.first_params, N, i, x);
      store21(P.first_cov, N, i, C);
    }
    nleg++;

    // material after the update, at every visited surface (U6).  The 9 numbers it changes are
    // stashed in shared memory so that last_* can be the pre-material filtered state.
    sincos(x[2], &trig[0], &trig[1]);
    sincos(x[3], &trig[2], &trig[3]);
    g_prev = 1.0;
    mat_applied = false;
    if (MATERIAL && st[14] > 0.0) {
      stash_save(stash, sstride, x, C);
      double lam = x[4], g = 1.0;
      if (!apply_material(P.mat, st, trig, lam, C, g)) { status |= ST_ENERGY; break; }
      x[4] = lam;
      g_prev = g;
      mat_applied = true;
    }
  }

  // x, C = state after the last completed leg (start state if none); undo its material step
  if (MATERIAL && mat_applied) stash_restore(stash, sstride, x, C);
  store6(P.last_params, N, i, x);
  store21(P.last_cov, N, i, C);
  if (nleg == 0) {
    store6(P.first_params, N, i, x);
    store21(P.first_cov, N, i, C);
  }

  const int ndf = 2 * n_used - 5;
  if (ndf <= 0) status |= ST_NDF;
  P.chi2[i] = chi2;
  P.ndf[i] = ndf;
  P.status[i] = status;
  P.n_used[i] = n_used;
  P.n_outliers[i] = n_outl;
  P.n_holes[i] = n_holes;
  if (P.rk_err_max) P.rk_err_max[i] = errmax;
  if (P.smooth) P.nleg[i] = nleg;
  for (int j = hp; j < o1; ++j) {  // hits never reached
    if (P.hit_chi2) P.hit_chi2[j] = 0.0;
    if (P.hit_flags) P.hit_flags[j] = 0;
  }
}

// =====================================================================================================
// RTS backward pass.  Record k holds x-_k, C-_k, F_k = dx-_k/dx+_{k-1}.
//   A_k = C+_k F_{k+1}^T (C-_{k+1})^-1,  x^s_k = x+_k + A_k (x^s_{k+1} - x-_{k+1}),
//   C^s_k = C+_k + A_k (C^s_{k+1} - C-_{k+1}) A_k^T.
__device__ __forceinline__ void load_record(const FitParams& P, int l, long long i, double xp[6],
                                            double Cp[21], double Fa[4][5], double Ft[5], double& g) {
  const double* __restrict__ R = P.rec + (size_t)l * kRecDoubles * P.Np + i;
  const long long Np = P.Np;
#pragma unroll
  for (int k = 0; k < 6; ++k) xp[k] = R[(kRecXp + k) * Np];
#pragma unroll
  for (int k = 0; k < 21; ++k) Cp[k] = R[(kRecCp + k) * Np];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int c = 0; c < 5; ++c) Fa[a][c] = R[(kRecFa + a * 5 + c) * Np];
#pragma unroll
  for (int c = 0; c < 5; ++c) Ft[c] = R[(kRecFt + c) * Np];
  g = R[kRecG * Np];
}

// filtered state of leg l, recomputed from its record and hit exactly as the forward pass did
__device__ __forceinline__ void refilter(const FitParams& P, const double* __restrict__ G, int l,
                                         long long i, int& hp, const double xp[6], const double Cp[21],
                                         double xf[6], double Cf[21]) {
  const unsigned char flag = P.legflag[(size_t)l * P.Np + i];
  bool copied = true;
  if (flag != 0) {  // the leg consumed hit hp
    if (flag == 1) {
      const double m0 = P.loc[hp], m1 = P.loc[P.M + hp];
      double v00, v11, v01 = 0.0;
      if (P.var) {
        v00 = P.var[hp];
        v11 = P.var[P.M + hp];
        if (P.cov01) v01 = P.cov01[hp];
      } else {
        const double* st = G + (P.start + 1 + l) * 20;
        v00 = st[16];
        v11 = st[17];
      }
      double c2;
      copied = !gain_update(xp, Cp, m0, m1, v00, v01, v11, xf, Cf, c2);
    }
    hp--;
  }
  if (copied) {
#pragma unroll
    for (int k = 0; k < 6; ++k) xf[k] = xp[k];
#pragma unroll
    for (int k = 0; k < 21; ++k) Cf[k] = Cp[k];
  }
}

__global__ void __launch_bounds__(KF_RTS_BLOCK, KF_RTS_MIN_BLOCKS)
kf_rts_kernel(const __grid_constant__ FitParams P) {
  extern __shared__ double s_dyn[];
  const double* __restrict__ G = stage_geometry(P, s_dyn);
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= P.N) return;
  const long long N = P.N;
  const int nleg = P.nleg[i];
  if (nleg <= 0) return;  // first_* already holds the start state

  // last hit consumed by the forward pass (it may have stopped early)
  const int o0 = P.offsets[i];
  int hp = P.offsets[i + 1] - 1;
  while (hp >= o0 && P.surf_idx[hp] > P.start + nleg) hp--;

  double xp1[6], Cp1[21], Fa1[4][5], Ft1[5], g1;
  double xs[6], Cs[21];
  load_record(P, nleg - 1, i, xp1, Cp1, Fa1, Ft1, g1);
  refilter(P, G, nleg - 1, i, hp, xp1, Cp1, xs, Cs);  // x^s_n = x+_n
  if (P.output_states & OUT_SMOOTH) {
    store6(P.state_params[2] + (size_t)(nleg - 1) * 6 * N, N, i, xs);
    store21(P.state_cov[2] + (size_t)(nleg - 1) * 21 * N, N, i, Cs);
  }
  bool failed = false;
  for (int k = nleg - 2; k >= 0; --k) {
    double xpk[6], Cpk[21], Fak[4][5], Ftk[5], gk;
    load_record(P, k, i, xpk, Cpk, Fak, Ftk, gk);
    double xf[6], Cf[21];
    refilter(P, G, k, i, hp, xpk, Cpk, xf, Cf);
    if (!failed) failed = !rts_step(xf, Cf, Fa1, Ft1, g1, xp1, Cp1, xs, Cs);
    if (failed) {  // fall back to the filtered states for the remaining surfaces
#pragma unroll
      for (int c = 0; c < 6; ++c) xs[c] = xf[c];
#pragma unroll
      for (int c = 0; c < 21; ++c) Cs[c] = Cf[c];
    }
    if (P.output_states & OUT_SMOOTH) {
      store6(P.state_params[2] + (size_t)k * 6 * N, N, i, xs);
      store21(P.state_cov[2] + (size_t)k * 21 * N, N, i, Cs);
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) xp1[c] = xpk[c];
#pragma unroll
    for (int c = 0; c < 21; ++c) Cp1[c] = Cpk[c];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int c = 0; c < 5; ++c) Fa1[a][c] = Fak[a][c];
#pragma unroll
    for (int c = 0; c < 5; ++c) Ft1[c] = Ftk[c];
    g1 = gk;
  }
  store6(P.first_params, N, i, xs);
  store21(P.first_cov, N, i, Cs);
  if (failed) P.status[i] |= ST_NOT_POSITIVE;
}

// ---- sustained FP64 FMA throughput probe (roofline denominator; not part of the fit) -----------------
__global__ void __launch_bounds__(256) kf_dfma_probe_kernel(double* out, int iters, double a, double b) {
  double v[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) v[k] = (double)(threadIdx.x + k) * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = fma(v[k], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += v[k];
  if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace kf
