// kf_rts.cuh -- the Rauch-Tung-Striebel backward pass kernels (sm_100a).  Record layout and parameter block: kf_common.cuh.
#pragma once

#include "kf_common.cuh"

namespace kf {

// =====================================================================================================
// RTS backward pass.  Record k holds x-_k, C-_k, F_k = dx-_k/dx+_{k-1}, the hit.
//   A_k = C+_k F_{k+1}^T (C-_{k+1})^-1,  x^s_k = x+_k + A_k (x^s_{k+1} - x-_{k+1}),
//   C^s_k = C+_k + A_k (C^s_{k+1} - C-_{k+1}) A_k^T.
//
// One CTA = one tile of KF_TILE tracks.  The tile's records are contiguous per leg (kLegBytes), so
// one bulk async copy (TMA, cp.async.bulk) per leg brings a record into shared memory while the
// threads compute; two stages hold records k and k+1, and the stage of record k+1 is re-armed with
// record k-1 as soon as every thread has consumed it (before the solves and the triple product).
// Threads read their own column (stride KF_TILE doubles: conflict-free), each value exactly once.

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "KF_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra KF_DONE_%=;\n"
      "bra KF_WAIT_%=;\n"
      "KF_DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, unsigned bytes,
                                          unsigned long long* bar) {
#ifndef KF_RTS_PLAIN_LOADS
  // records are read exactly once: evict-first in L2 (RTS 2.73 -> 2.70 ms on CFG2)
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(smem_dst)),
      "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
  return;
#endif
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
          smem_u32(smem_dst)),
      "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}

__device__ __forceinline__ void bulk_prefetch_l2(const void* gmem_src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem_src), "r"(bytes) : "memory");
}

// values of type R per record stage in shared memory (the flag bytes included, rounded up)
template <typename R>
__host__ __device__ constexpr int stage_values() { return (int)(leg_bytes<R>() / sizeof(R)); }
constexpr int kStageDoubles = stage_values<double>();
static_assert(leg_bytes<double>() % 16 == 0 && leg_bytes<float>() % 16 == 0,
              "a tile-leg must be a whole number of 16-byte units (bulk copy)");
// record column of one thread inside a stage: component c at R[c * KF_TILE]
#define KF_R(R, c) (R)[(c) * KF_TILE]

// filtered state of a leg from its record column R exactly as the forward pass computed it:
// the same gain routine on (x-, C-, hit); a hole or flagged outlier has x+ = x-, C+ = C-.
template <bool PLAIN, typename R>
__device__ __forceinline__ void refilter(const FitParams& P, const R* Rc, unsigned char flag, R gv0,
                                         R gv1, int hp, R xf[6], R Cf[21]) {
  const double* const var = PLAIN ? nullptr : P.var;
  R xp[6], Cp[21];
#pragma unroll
  for (int k = 0; k < 6; ++k) xp[k] = KF_R(Rc, kRecXp + k);
#pragma unroll
  for (int k = 0; k < 21; ++k) Cp[k] = KF_R(Rc, kRecCp + k);
  GainT<R> gn;
  gn.r0 = gn.r1 = gn.i00 = gn.i01 = gn.i11 = R(0.0);
  if (flag == 1) {
    const R m0 = KF_R(Rc, kRecM), m1 = KF_R(Rc, kRecM + 1);
    R v00, v11, v01 = R(0.0);
    if (var) {
      v00 = (R)var[hp];
      v11 = (R)var[P.ldm + hp];
      if (P.cov01) v01 = (R)P.cov01[hp];
    } else {
      v00 = gv0;  // the surface's resolution (geometry table), fetched by the caller
      v11 = gv1;
    }
    R c2;
    if (!gain_prepare(xp, Cp, m0, m1, v00, v01, v11, gn, c2)) gn.i00 = gn.i01 = gn.i11 = R(0.0);
  }
  gain_apply(gn, xp, Cp, xf, Cf);
}

// One RTS step (DESIGN.md A.7), in two parts.  In: (xf, Cf) = filtered state at k, (xs, Cs) = smoothed state
// at k+1, R1 = this thread's column of record k+1 in shared memory (x-, C-, F = J G, g).  Out: (xs, Cs) =
// smoothed state at k.  The record column is dead after its single read, so it doubles as scratch: C+
// goes to the F slots and dC = C^s - C- to the C- slots while the 6x6 solve owns the registers.
//
// Part 1 needs record k+1 only, so it runs BEFORE the wait for record k (it covers the bulk copy's latency):
// dx = x^s_{k+1} - x-_{k+1} (phi wrapped into (-pi, pi]), dC -> scratch, Cholesky C-_{k+1} = L L^T without
// pivoting (scale-invariant), L[i][j] (i >= j) kept at packed (j, i), inv = 1 / diag.
// Returns false on a non-positive pivot.
//
// The 6x6 solve (Cholesky factor and the two triangular solves per row of the gain) always runs in double, whatever the
// operand type R: the paper keeps its matrix inversion in double "because of the difference in implementation of the
// floating-point arithmetic between different hardware".
template <typename R>
__device__ __forceinline__ bool rts_step_pre(R* R1, const R xs[6], const R Cs[21], R dx[6],
                                             double L[21], double inv[6]) {
  bool ok = true;
#pragma unroll
  for (int c = 0; c < 21; ++c) {
    const R cp = KF_R(R1, kRecCp + c);
    L[c] = (double)cp;
    KF_R(R1, kRecCp + c) = Cs[c] - cp;
  }
  // (fixed trip counts with compile-time guards: every index is a constant after unrolling)
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    double s = L[IX(j, j)];
#pragma unroll
    for (int k = 0; k < 6; ++k)
      if (k < j) s = fma(-L[SX(k, j)], L[SX(k, j)], s);
    if (!(s > 0.0)) { ok = false; s = 1.0; }
    L[IX(j, j)] = sqrt_nr(s, inv[j]);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      if (i > j) {
        double u = L[SX(j, i)];
#pragma unroll
        for (int k = 0; k < 6; ++k)
          if (k < j) u = fma(-L[SX(k, i)], L[SX(k, j)], u);
        L[SX(j, i)] = u * inv[j];
      }
    }
  }
#pragma unroll
  for (int j = 0; j < 6; ++j) dx[j] = xs[j] - KF_R(R1, kRecXp + j);
  dx[2] = wrap_pi(dx[2]);
  return ok;
}

// Part 2: W = C+ F^T, A = W (L L^T)^-1, x^s_k = x+_k + A dx, C^s_k = C+_k + A dC A^T.
// Returns false on a non-finite result (C+ is then still in the scratch F slots).
template <typename R>
__device__ __forceinline__ bool rts_step_post(R* R1, const R xf[6], const R Cf[21],
                                              const R dx[6], const double L[21], const double inv[6],
                                              R xs[6], R Cs[21]) {
  // W = C+ F^T, streaming F (rows loc0, loc1, phi, theta over columns loc0..qp; row t; row qp = g e_qp)
  R W[6][6];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    R f[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) f[c] = KF_R(R1, kRecFa + j * 5 + c);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      R s = Cf[SX(i, 0)] * f[0];
#pragma unroll
      for (int c = 1; c < 5; ++c) s = fma(Cf[SX(i, c)], f[c], s);
      W[i][j] = s;
    }
  }
  {
    R f[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) f[c] = KF_R(R1, kRecFt + c);
    const R g = KF_R(R1, kRecG);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      W[i][4] = Cf[SX(i, 4)] * g;
      R s = Cf[SX(i, 5)];
#pragma unroll
      for (int c = 0; c < 5; ++c) s = fma(Cf[SX(i, c)], f[c], s);
      W[i][5] = s;
    }
  }
  // C+ -> scratch (the F slots are consumed)
#pragma unroll
  for (int c = 0; c < 21; ++c) KF_R(R1, kRecFa + c) = Cf[c];

  // A = W (L L^T)^-1 row by row (the two triangular solves in double), x^s_k = x+_k + A dx
  R chk = R(0.0);
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    double y[6];
#pragma unroll
    for (int r = 0; r < 6; ++r) {  // L y = w
      double s = (double)W[i][r];
#pragma unroll
      for (int k = 0; k < r; ++k) s = fma(-L[IX(k, r)], y[k], s);
      y[r] = s * inv[r];
    }
#pragma unroll
    for (int r = 5; r >= 0; --r) {  // L^T a = y
      double s = y[r];
#pragma unroll
      for (int k = r + 1; k < 6; ++k) s = fma(-L[IX(r, k)], y[k], s);
      y[r] = s * inv[r];
    }
#pragma unroll
    for (int r = 0; r < 6; ++r) W[i][r] = (R)y[r];
    R s = xf[i];
#pragma unroll
    for (int j = 0; j < 6; ++j) s = fma(W[i][j], dx[j], s);
    xs[i] = s;
    chk += s;
  }
  // C^s_k = C+_k + A dC A^T  (dC and C+ back from scratch)
  R dC[21];
#pragma unroll
  for (int c = 0; c < 21; ++c) dC[c] = KF_R(R1, kRecCp + c);
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    R T[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      R u = W[i][0] * dC[SX(0, j)];
#pragma unroll
      for (int k = 1; k < 6; ++k) u = fma(W[i][k], dC[SX(k, j)], u);
      T[j] = u;
    }
#pragma unroll
    for (int j = i; j < 6; ++j) {
      R u = KF_R(R1, kRecFa + IX(i, j));
#pragma unroll
      for (int k = 0; k < 6; ++k) u = fma(T[k], W[j][k], u);
      Cs[IX(i, j)] = u;
      chk += u;
    }
  }
  return fabs(chk) < big<R>();
}

// PLAIN: per-surface resolutions and no per-leg smoothed states asked for: those paths are compiled out (2.68 -> 2.61 ms
// on CFG2; like the forward kernel this one has no register to spare for run-time options).
// R: the arithmetic type of the records and of every product (double, or float for the MIXED path); the 6x6 solve is
// double in both (rts_step_pre / rts_step_post).
template <bool PLAIN, typename R = double>
__global__ void __launch_bounds__(KF_TILE, KF_RTS_MIN_BLOCKS)
kf_rts_kernel(const __grid_constant__ FitParams P) {
  constexpr unsigned kLeg = (unsigned)leg_bytes<R>();
  constexpr int kStage = stage_values<R>();
  const double* const o_var = PLAIN ? nullptr : P.var;
  const int o_states = PLAIN ? 0 : P.output_states;
  extern __shared__ __align__(128) unsigned char s_rts_raw[];  // two stages of kLeg bytes, then two mbarriers
  R* const s_rec = reinterpret_cast<R*>(s_rts_raw);
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(s_rts_raw + 2 * (size_t)kLeg);
  __shared__ int s_nmax;
  const int tid = threadIdx.x;
  const long long tslot = (long long)blockIdx.x * KF_TILE + tid;
  const long long N = P.ldn;  // SoA stride
  const bool in_range = tslot < P.N;
  const long long i = in_range && P.perm ? (long long)P.perm[tslot] : tslot;  // the track this slot fitted
  const int nleg = in_range ? P.nleg[tslot] : 0;
  if (tid == 0) {
    s_nmax = 0;
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (nleg > 0) atomicMax(&s_nmax, nleg);
  __syncthreads();
  const int n = s_nmax;
  if (n <= 0) return;  // no track of the tile completed a leg: first_* already holds the start state

  const char* __restrict__ tile_base = P.rec + (size_t)blockIdx.x * P.tile_stride;
  if (tid == 0) {
    mbar_expect_tx(&bar[(n - 1) & 1], kLeg);
    bulk_load(s_rec + ((n - 1) & 1) * kStage, tile_base + (size_t)(n - 1) * P.leg_stride, kLeg,
              &bar[(n - 1) & 1]);
    if (n >= 2) {
      mbar_expect_tx(&bar[(n - 2) & 1], kLeg);
      bulk_load(s_rec + ((n - 2) & 1) * kStage, tile_base + (size_t)(n - 2) * P.leg_stride, kLeg,
                &bar[(n - 2) & 1]);
    }
  }

  // per-hit variances (optional input) are looked up by hit index: start from the last consumed hit
  int hp = 0;
  if (o_var && nleg > 0) {
    const int o0 = P.offsets[i];
    hp = P.offsets[i + 1] - 1;
    while (hp >= o0 && P.surf_idx[hp] > P.start + nleg) hp--;
  }

  R xs[6], Cs[21];
  bool failed = false;
  unsigned phase = 0u;
  for (int k = n - 1; k >= 0; --k) {
    const int sc = k & 1, sn = sc ^ 1;
    // record k-2 is fetched at the end of the next iteration: start it towards L2 now
    if (tid == 0 && k >= 2) bulk_prefetch_l2(tile_base + (size_t)(k - 2) * P.leg_stride, kLeg);
    // the surface's measurement variances come from L2: ask for them before waiting on the record
    R gv0 = R(0.0), gv1 = R(0.0);
    if (!o_var) {
      gv0 = (R)__ldg(P.geom + (P.start + 1 + k) * 20 + 16);
      gv1 = (R)__ldg(P.geom + (P.start + 1 + k) * 20 + 17);
    }
    const R* Rc = s_rec + sc * kStage + tid;
    R* Rn = s_rec + sn * kStage + tid;
    // everything that needs record k+1 only comes before the wait for record k
    const bool step = k < nleg - 1 && !failed;
    R dx[6];
    double L[21], inv[6];
    bool ok = true;
    if (step) ok = rts_step_pre(Rn, xs, Cs, dx, L, inv);
    mbar_wait(&bar[sc], (phase >> sc) & 1u);
    phase ^= 1u << sc;
    if (k < nleg) {
      const unsigned char flag =
          reinterpret_cast<const unsigned char*>(s_rec + sc * kStage)[(size_t)kRecDoubles * KF_TILE * sizeof(R) + tid];
      R xf[6], Cf[21];
      refilter<PLAIN>(P, Rc, flag, gv0, gv1, hp, xf, Cf);
      if (flag != 0) hp--;
      bool smoothed = false;
      if (step) {
        if (ok) {
          smoothed = rts_step_post(Rn, xf, Cf, dx, L, inv, xs, Cs);
          if (!smoothed) {
#pragma unroll
            for (int c = 0; c < 21; ++c) Cf[c] = KF_R(Rn, kRecFa + c);
          }
        }
        if (!smoothed) failed = true;  // U25: this and all earlier surfaces fall back to the filtered states
      }
      if (!smoothed) {  // top of the track, or fallback
#pragma unroll
        for (int c = 0; c < 6; ++c) xs[c] = xf[c];
#pragma unroll
        for (int c = 0; c < 21; ++c) Cs[c] = Cf[c];
      }
      if (o_states & OUT_SMOOTH) {
        store6(P.state_params[2] + (size_t)k * 6 * N, N, i, xs);
        store21(P.state_cov[2] + (size_t)k * 21 * N, N, i, Cs);
      }
    }
    if (k < n - 1) {
      // every thread is done with record k+1 and its scratch (generic-proxy writes ordered before the
      // async-proxy write of the next bulk copy): fetch record k-1 into that stage
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();
      if (tid == 0 && k >= 1) {
        mbar_expect_tx(&bar[sn], kLeg);
        bulk_load(s_rec + sn * kStage, tile_base + (size_t)(k - 1) * P.leg_stride, kLeg, &bar[sn]);
      }
    }
  }
  if (nleg > 0) {
    store6(P.first_params, N, i, xs);
    store21(P.first_cov, N, i, Cs);
    if (failed) P.status[i] |= ST_NOT_POSITIVE;
  }
}

// =====================================================================================================
// RTS backward pass, lanes-per-track variant (kf_lanes.cuh): a group of kLanes lanes owns one track.
// The record of a leg (kRecDoubles doubles of the track's column) is brought into the group's own
// shared-memory slot by per-lane asynchronous copies (lane q fetches components q, q+8, ...), three
// slots deep: records k and k+1 in use, record k-1 in flight.  Re-filtering and the Cholesky factor
// run redundantly in every lane; the rows of W = C+ F^T, of the gain A (two triangular solves per row),
// of A dC and of C^s are one per lane, exchanged with shuffles.  Same arithmetic per element as
// kf_rts_kernel, same fallback rule (U25).
constexpr int kLaneSlotDoubles = 56;                       // kRecDoubles rounded up to an even count
constexpr int kRtsLanesBlock = 128;                        // 16 tracks per CTA
constexpr size_t kRtsLanesSmem = (size_t)(kRtsLanesBlock / kLanes) * 3 * kLaneSlotDoubles * sizeof(double);

__global__ void __launch_bounds__(kRtsLanesBlock)
kf_rts_lanes_kernel(const __grid_constant__ FitParams P) {
  extern __shared__ __align__(16) double s_slots[];
  const long long tslot = ((long long)blockIdx.x * kRtsLanesBlock + threadIdx.x) / kLanes;
  if (tslot >= P.N) return;
  const long long i = P.perm ? (long long)P.perm[tslot] : tslot;
  const long long N = P.ldn;
  const int q = threadIdx.x % kLanes, row = q < 6 ? q : 5;
  const int gbase = (threadIdx.x & 31) & ~(kLanes - 1);
  const unsigned gmask = ((1u << kLanes) - 1u) << gbase;
  const bool lead = q == 0;
  const int nleg = P.nleg[tslot];
  if (nleg <= 0) return;  // first_* already holds the start state

  double* const slots = s_slots + (size_t)(threadIdx.x / kLanes) * 3 * kLaneSlotDoubles;
  const char* __restrict__ tile_base = P.rec + (size_t)(tslot / KF_TILE) * P.tile_stride;
  const int col = (int)(tslot % KF_TILE);
  auto fetch = [&](int k) {  // record k -> slot k % 3 (this lane's share), one copy group
    if (k >= 0) {
      const double* src = reinterpret_cast<const double*>(tile_base + (size_t)k * P.leg_stride) + col;
      double* dst = slots + (k % 3) * kLaneSlotDoubles;
      for (int c = q; c < kRecDoubles; c += kLanes) cp_async8(dst + c, src + (size_t)c * KF_TILE);
    }
    cp_async_commit();
  };
  auto load_flag = [&](int k) -> unsigned char {
    if (k < 0) return 0;
    return reinterpret_cast<const unsigned char*>(tile_base + (size_t)k * P.leg_stride)[(size_t)kRecDoubles * KF_TILE * sizeof(double) + col];
  };
  fetch(nleg - 1);
  fetch(nleg - 2);
  unsigned char f_cur = load_flag(nleg - 1), f_n1 = load_flag(nleg - 2);

  int hp = 0;
  if (P.var) {
    const int o0 = P.offsets[i];
    hp = P.offsets[i + 1] - 1;
    while (hp >= o0 && P.surf_idx[hp] > P.start + nleg) hp--;
  }

  double xs[6], Cs[21];
  bool failed = false;
  for (int k = nleg - 1; k >= 0; --k) {
    const unsigned char f_n2 = load_flag(k - 2);
    asm volatile("cp.async.wait_group 1;" ::: "memory");  // everything but the newest group: record k is here
    __syncwarp(gmask);
    const double* Rc = slots + (k % 3) * kLaneSlotDoubles;
    const double* R1 = slots + ((k + 1) % 3) * kLaneSlotDoubles;

    // filtered state of leg k, as the forward pass computed it (same gain routine)
    double xf[6], Cf[21];
    {
      double xp[6], Cp[21];
#pragma unroll
      for (int c = 0; c < 6; ++c) xp[c] = Rc[kRecXp + c];
#pragma unroll
      for (int c = 0; c < 21; ++c) Cp[c] = Rc[kRecCp + c];
      Gain gn;
      gn.r0 = gn.r1 = gn.i00 = gn.i01 = gn.i11 = 0.0;
      if (f_cur == 1) {
        double v00, v11, v01 = 0.0;
        if (P.var) {
          v00 = P.var[hp];
          v11 = P.var[P.ldm + hp];
          if (P.cov01) v01 = P.cov01[hp];
        } else {
          v00 = __ldg(P.geom + (P.start + 1 + k) * 20 + 16);
          v11 = __ldg(P.geom + (P.start + 1 + k) * 20 + 17);
        }
        double c2;
        if (!gain_prepare(xp, Cp, Rc[kRecM], Rc[kRecM + 1], v00, v01, v11, gn, c2)) gn.i00 = gn.i01 = gn.i11 = 0.0;
      }
      gain_apply(gn, xp, Cp, xf, Cf);
      if (f_cur != 0) hp--;
    }

    bool smoothed = false;
    if (k < nleg - 1 && !failed) {
      // Cholesky C-_{k+1} = L L^T (every lane), L[i][j] (i >= j) at packed (j, i)
      double L[21], inv[6], dC[21];
      bool ok = true;
#pragma unroll
      for (int c = 0; c < 21; ++c) {
        L[c] = R1[kRecCp + c];
        dC[c] = Cs[c] - L[c];
      }
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        double s = L[IX(j, j)];
#pragma unroll
        for (int m = 0; m < 6; ++m)
          if (m < j) s = fma(-L[SX(m, j)], L[SX(m, j)], s);
        if (!(s > 0.0)) { ok = false; s = 1.0; }
        L[IX(j, j)] = sqrt_nr(s, inv[j]);
#pragma unroll
        for (int r = 0; r < 6; ++r) {
          if (r > j) {
            double u = L[SX(j, r)];
#pragma unroll
            for (int m = 0; m < 6; ++m)
              if (m < j) u = fma(-L[SX(m, r)], L[SX(m, j)], u);
            L[SX(j, r)] = u * inv[j];
          }
        }
      }
      double dx[6];
#pragma unroll
      for (int j = 0; j < 6; ++j) dx[j] = xs[j] - R1[kRecXp + j];
      dx[2] = wrap_pi(dx[2]);

      // this lane's row of C+ and of W = C+ F^T
      double cr[6], W[6];
#pragma unroll
      for (int c = 0; c < 6; ++c) cr[c] = sym_row(Cf, row, c);
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        double s = cr[0] * R1[kRecFa + j * 5];
#pragma unroll
        for (int c = 1; c < 5; ++c) s = fma(cr[c], R1[kRecFa + j * 5 + c], s);
        W[j] = s;
      }
      W[4] = cr[4] * R1[kRecG];
      {
        double s = cr[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) s = fma(cr[c], R1[kRecFt + c], s);
        W[5] = s;
      }
      // row of A = W (L L^T)^-1
#pragma unroll
      for (int r = 0; r < 6; ++r) {
        double s = W[r];
#pragma unroll
        for (int m = 0; m < r; ++m) s = fma(-L[IX(m, r)], W[m], s);
        W[r] = s * inv[r];
      }
#pragma unroll
      for (int r = 5; r >= 0; --r) {
        double s = W[r];
#pragma unroll
        for (int m = r + 1; m < 6; ++m) s = fma(-L[IX(r, m)], W[m], s);
        W[r] = s * inv[r];
      }
      // x^s component and the row of A dC
      double xq = vec_sel(xf, row);
#pragma unroll
      for (int j = 0; j < 6; ++j) xq = fma(W[j], dx[j], xq);
      double T[6];
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        double u = W[0] * dC[SX(0, j)];
#pragma unroll
        for (int m = 1; m < 6; ++m) u = fma(W[m], dC[SX(m, j)], u);
        T[j] = u;
      }
      // row of C^s = C+ + (A dC) A^T: the other lanes' rows of A arrive by shuffle
      double Rw[6];
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        double u = cr[j];
#pragma unroll
        for (int m = 0; m < 6; ++m) u = fma(T[m], __shfl_sync(gmask, W[m], gbase + j), u);
        Rw[j] = u;
      }
      double xn[6], Cn[21];
#pragma unroll
      for (int j = 0; j < 6; ++j) xn[j] = __shfl_sync(gmask, xq, gbase + j);
      gather_sym(Rw, Cn, gbase, gmask);
      double chk = 0.0;
#pragma unroll
      for (int j = 0; j < 6; ++j) chk += xn[j];
#pragma unroll
      for (int c = 0; c < 21; ++c) chk += Cn[c];
      smoothed = ok && fabs(chk) < 1.0e300;
      if (smoothed) {
#pragma unroll
        for (int j = 0; j < 6; ++j) xs[j] = xn[j];
#pragma unroll
        for (int c = 0; c < 21; ++c) Cs[c] = Cn[c];
      } else {
        failed = true;  // U25
      }
    }
    if (!smoothed) {  // top of the track, or fallback to the filtered state
#pragma unroll
      for (int c = 0; c < 6; ++c) xs[c] = xf[c];
#pragma unroll
      for (int c = 0; c < 21; ++c) Cs[c] = Cf[c];
    }
    if ((P.output_states & OUT_SMOOTH) && lead) {
      store6(P.state_params[2] + (size_t)k * 6 * N, N, i, xs);
      store21(P.state_cov[2] + (size_t)k * 21 * N, N, i, Cs);
    }
    __syncwarp(gmask);  // every lane is done with record k+1: its slot takes record k-2
    fetch(k - 2);
    f_cur = f_n1;
    f_n1 = f_n2;
  }
  if (lead) {
    store6(P.first_params, N, i, xs);
    store21(P.first_cov, N, i, Cs);
    if (failed) P.status[i] |= ST_NOT_POSITIVE;
  }
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
