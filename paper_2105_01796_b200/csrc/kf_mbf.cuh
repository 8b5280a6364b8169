// kf_mbf.cuh -- the backward pass in modified Bryson-Frazier form (sm_100a, IEEE double); kf_options.smoother.
//
// The smoothed state the Rauch-Tung-Striebel recursion of PAPER.md:62, 75 defines (DESIGN.md A.7) can be reached
// without the 6x6 solve per state: with the adjoint pair (lam, Lam), zero behind the last leg,
//     lam~_k = -H^T S_k^-1 r_k + (I - K_k H)^T lam^_k          Lam~_k = H^T S_k^-1 H + (I - K_k H)^T Lam^_k (I - K_k H)
//     lam^_{k-1} = F_k^T lam~_k                                Lam^_{k-1} = F_k^T Lam~_k F_k
//     x^s_k = x-_k - C-_k lam~_k                               C^s_k = C-_k - C-_k Lam~_k C-_k
// (Bierman's form of the Bryson-Frazier smoother; algebraically the RTS result, state by state: K r and the
// process noise are already inside x-, C-, K).  Only the smoothed state at the FIRST leg is formed here (first_*),
// so a leg's record is its gain (r, S^-1; zero for a hole or an outlier), the two leading columns of C- (K = C- H^T
// S^-1 is rebuilt from them) and F: 42 doubles against the 55 of the RTS record, ~400 FP64 instructions per leg
// against ~1,000.  The price is conditioning: C- - C- Lam~ C- cancels kappa = C-_ii / C^s_ii leading digits (1.6e3
// on the configs, harmless; 8e6 with a 1e4-inflated prior, where RTS is 100x better) -- which is why this is an
// option measured beside RTS, not the default, and why it offers no per-leg
// smoothed states.  One CTA = one record tile of KF_TILE tracks, records staged by bulk asynchronous copies as
// in kf_rts_kernel.
#pragma once

#include "kf_rts.cuh"

namespace kf {

constexpr double kMbfKappaMax = 1.0e6;  // ~30 eps kappa against the 1e-8 covariance bar
constexpr int kMbfStages = 2;  // 43 KB per CTA: five CTAs (ten warps) per SM
constexpr size_t kMbfSmem = kMbfStages * kMbfLegBytes + kMbfStages * sizeof(unsigned long long);
static_assert(kMbfLegBytes % 16 == 0, "a tile-leg must be a whole number of 16-byte units (bulk copy)");

__global__ void __launch_bounds__(KF_TILE)
kf_mbf_kernel(const __grid_constant__ FitParams P) {
  extern __shared__ __align__(128) double s_rec[];
  constexpr int kStage = (int)(kMbfLegBytes / sizeof(double));
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(s_rec + kMbfStages * kStage);
  __shared__ int s_nmax;
  const int tid = threadIdx.x;
  const long long tslot = (long long)blockIdx.x * KF_TILE + tid;
  const long long N = P.ldn;
  const bool in_range = tslot < P.N;
  const long long i = in_range && P.perm ? (long long)P.perm[tslot] : tslot;
  const int nleg = in_range ? P.nleg[tslot] : 0;
  if (tid == 0) {
    s_nmax = 0;
#pragma unroll
    for (int s = 0; s < kMbfStages; ++s) mbar_init(&bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (nleg > 0) atomicMax(&s_nmax, nleg);
  __syncthreads();
  const int n = s_nmax;
  if (n <= 0) return;

  const char* __restrict__ tile_base = P.rec + (size_t)blockIdx.x * P.tile_stride;
  auto fetch = [&](int k) {  // record k -> stage k % kMbfStages (one thread)
    const int s = k % kMbfStages;
    mbar_expect_tx(&bar[s], (unsigned)kMbfLegBytes);
    bulk_load(s_rec + s * kStage, tile_base + (size_t)k * P.leg_stride, (unsigned)kMbfLegBytes, &bar[s]);
  };
  if (tid == 0) {
#pragma unroll
    for (int d = 0; d < kMbfStages; ++d)
      if (n - 1 - d >= 0) fetch(n - 1 - d);
  }

  double lam[6], Lam[21];
#pragma unroll
  for (int c = 0; c < 6; ++c) lam[c] = 0.0;
#pragma unroll
  for (int c = 0; c < 21; ++c) Lam[c] = 0.0;
  unsigned phase = 0u;
  for (int k = n - 1; k >= 0; --k) {
    const int sc = k % kMbfStages;
    if (tid == 0 && k - kMbfStages - 1 >= 0)
      bulk_prefetch_l2(tile_base + (size_t)(k - kMbfStages - 1) * P.leg_stride, (unsigned)kMbfLegBytes);
    mbar_wait(&bar[sc], (phase >> sc) & 1u);
    phase ^= 1u << sc;
    if (k < nleg) {
      const double* R = s_rec + sc * kStage + tid;
      // (I - K H)^T . (I - K H) and the hit's information
      const double r0 = KF_R(R, kMbfGain + 0), r1 = KF_R(R, kMbfGain + 1);
      const double i00 = KF_R(R, kMbfGain + 2), i01 = KF_R(R, kMbfGain + 3), i11 = KF_R(R, kMbfGain + 4);
      double K0[6], K1[6];
      {
        double c0[6], c1[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) c0[c] = KF_R(R, kMbfCcol + c);
        c1[0] = c0[1];
#pragma unroll
        for (int c = 1; c < 6; ++c) c1[c] = KF_R(R, kMbfCcol + 5 + c);
#pragma unroll
        for (int c = 0; c < 6; ++c) {
          K0[c] = fma(c0[c], i00, c1[c] * i01);
          K1[c] = fma(c0[c], i01, c1[c] * i11);
        }
      }
      double U0[6], U1[6];
#pragma unroll
      for (int a = 0; a < 6; ++a) {
        double u0 = Lam[SX(a, 0)] * K0[0], u1 = Lam[SX(a, 0)] * K1[0];
#pragma unroll
        for (int b = 1; b < 6; ++b) {
          u0 = fma(Lam[SX(a, b)], K0[b], u0);
          u1 = fma(Lam[SX(a, b)], K1[b], u1);
        }
        U0[a] = u0;
        U1[a] = u1;
      }
      double w00 = 0.0, w01 = 0.0, w11 = 0.0, kl0 = 0.0, kl1 = 0.0;
#pragma unroll
      for (int a = 0; a < 6; ++a) {
        w00 = fma(K0[a], U0[a], w00);
        w01 = fma(K0[a], U1[a], w01);
        w11 = fma(K1[a], U1[a], w11);
        kl0 = fma(K0[a], lam[a], kl0);
        kl1 = fma(K1[a], lam[a], kl1);
      }
      lam[0] -= kl0 + fma(i00, r0, i01 * r1);
      lam[1] -= kl1 + fma(i01, r0, i11 * r1);
#pragma unroll
      for (int b = 2; b < 6; ++b) {
        Lam[IX(0, b)] -= U0[b];
        Lam[IX(1, b)] -= U1[b];
      }
      Lam[IX(0, 0)] += (w00 + i00) - 2.0 * U0[0];
      Lam[IX(0, 1)] += (w01 + i01) - (U0[1] + U1[0]);
      Lam[IX(1, 1)] += (w11 + i11) - 2.0 * U1[1];

      if (k > 0) {
        // through the leg: lam^ = F^T lam~, Lam^ = F^T Lam~ F.  F rows loc0..theta = Fa (column t zero), row qp = g e_qp,
        // row t = (Ft, 1)
        double Fa[4][5], Ft[5];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int c = 0; c < 5; ++c) Fa[a][c] = KF_R(R, kMbfFa + a * 5 + c);
#pragma unroll
        for (int c = 0; c < 5; ++c) Ft[c] = KF_R(R, kMbfFt + c);
        const double g = KF_R(R, kMbfG);
        double ln[6];
#pragma unroll
        for (int c = 0; c < 5; ++c) {
          double s = Ft[c] * lam[5];
#pragma unroll
          for (int a = 0; a < 4; ++a) s = fma(Fa[a][c], lam[a], s);
          ln[c] = s;
        }
        ln[4] = fma(g, lam[4], ln[4]);
        ln[5] = lam[5];
        // T = Lam~ F (6x6, column t of F = e_t)
        double T[6][6];
#pragma unroll
        for (int a = 0; a < 6; ++a) {
#pragma unroll
          for (int c = 0; c < 5; ++c) {
            double s = Lam[SX(a, 5)] * Ft[c];
#pragma unroll
            for (int b = 0; b < 4; ++b) s = fma(Lam[SX(a, b)], Fa[b][c], s);
            T[a][c] = s;
          }
          T[a][4] = fma(Lam[SX(a, 4)], g, T[a][4]);
          T[a][5] = Lam[SX(a, 5)];
        }
#pragma unroll
        for (int c = 0; c < 5; ++c)
#pragma unroll
          for (int d = c; d < 6; ++d) {
            double s = Ft[c] * T[5][d];
#pragma unroll
            for (int a = 0; a < 4; ++a) s = fma(Fa[a][c], T[a][d], s);
            if (c == 4) s = fma(g, T[4][d], s);
            Lam[IX(c, d)] = s;
          }
        Lam[IX(5, 5)] = T[5][5];
#pragma unroll
        for (int c = 0; c < 6; ++c) lam[c] = ln[c];
      }
    }
    // every thread is done with this stage: it takes record k - kMbfStages
    __syncthreads();
    if (tid == 0 && k - kMbfStages >= 0) fetch(k - kMbfStages);
  }

  if (nleg > 0) {
    // smoothed state at the first leg: x^s = x- - C- lam~, C^s = C- - C- Lam~ C-
    const double* __restrict__ FB = reinterpret_cast<const double*>(tile_base + P.first_off) + tid;
    double xp[6], Cp[21];
#pragma unroll
    for (int c = 0; c < 6; ++c) xp[c] = __ldcs(FB + c * KF_TILE);
#pragma unroll
    for (int c = 0; c < 21; ++c) Cp[c] = __ldcs(FB + (6 + c) * KF_TILE);
    double xs[6], Cs[21], chk = 0.0;
    double M[6][6];  // C- Lam~
#pragma unroll
    for (int a = 0; a < 6; ++a) {
      double s = xp[a];
#pragma unroll
      for (int b = 0; b < 6; ++b) s = fma(-Cp[SX(a, b)], lam[b], s);
      xs[a] = s;
      chk += s;
#pragma unroll
      for (int d = 0; d < 6; ++d) {
        double u = Cp[SX(a, 0)] * Lam[SX(0, d)];
#pragma unroll
        for (int b = 1; b < 6; ++b) u = fma(Cp[SX(a, b)], Lam[SX(b, d)], u);
        M[a][d] = u;
      }
    }
#pragma unroll
    for (int a = 0; a < 6; ++a)
#pragma unroll
      for (int d = a; d < 6; ++d) {
        double u = Cp[IX(a, d)];
#pragma unroll
        for (int b = 0; b < 6; ++b) u = fma(-M[a][b], Cp[SX(b, d)], u);
        Cs[IX(a, d)] = u;
        chk += u;
      }
    if (fabs(chk) < 1.0e300) {
      store6(P.first_params, N, i, xs);
      store21(P.first_cov, N, i, Cs);
      // the subtraction above loses kappa = C-_ii / C^s_ii leading digits: tell the caller when that is more than the
      // covariance bar of the parity contract can absorb (an uninformative prior; the RTS form does not have this)
      double kappa = 0.0;
#pragma unroll
      for (int a = 0; a < 6; ++a) kappa = fmax(kappa, Cs[IX(a, a)] > 0.0 ? Cp[IX(a, a)] / Cs[IX(a, a)] : 1.0e300);
      if (kappa > kMbfKappaMax) P.status[i] |= ST_CANCELLATION;
    } else {
      P.status[i] |= ST_NOT_POSITIVE;  // first_* keeps the filtered state the forward pass wrote (U25)
    }
  }
}

}  // namespace kf
