// kf_forward.cuh -- the forward Kalman filter kernel (sm_100a).  Record layout and parameter block: kf_common.cuh.
#pragma once

#include "kf_common.cuh"

namespace kf {

// =====================================================================================================
// Forward filter.  Dynamic shared memory: [geometry table if GEOM_SMEM][hit staging, kHitStageBytes].
// Material is applied lazily, at the top of the next leg, so that on exit (x, C) is the filtered
// state of the last completed leg before that layer's material (= last_*); the material step of the
// last surface is still evaluated for its status bit (energy exhausted), as in DESIGN.md A.6.
// GEOM_SMEM: the geometry table is read from shared memory (shared-space loads, their own scoreboard)
// or, for tables too large to stage, from global memory.
//
// LPT = lanes per track.  1: one thread owns one track (the default).  kLanes (8): the lanes-per-track
// variant ("intra-track parallelisation", NS "warp-cooperative lanes-per-track"): the 8 lanes
// of a group run the scalar part of the leg redundantly (identical values, identical branches) and share the
// 6x6 covariance transport row by row, exchanging the rows with warp shuffles; lane 0 of the group stores.
// MBF: the record written is the Bryson-Frazier one (kMbf*, kf_mbf.cuh) instead of the RTS one (kRec*); a template
// parameter because a run-time flag cost the RTS path 2.7 % (3.41 -> 3.51 ms on CFG2: five more registers).
// PLAIN: the call uses the default stepping policy (one primary + two correction steps, no step cap, no tolerance),
// per-surface resolutions, and asks for no per-leg predicted/filtered states and no RKN error estimate: those paths are
// compiled out (measured on CFG2: 3.39 -> 3.15 ms; the run-time tests cost registers in a kernel that has none to spare).
// R: the arithmetic type of the path.  double = the FP64 path (BASELINE.json metric).  float = the MIXED path
// (kf_options.precision; "All the tests use single precision ... with the exception of the
// matrix inversion"): inputs are rounded to float on load, every operand and the RTS record are float, outputs are
// widened on store.  Thread-per-track only (LPT = 1), RTS records only, geometry in shared memory only.
// The constant-field float instantiation is held to 128 registers (512 threads per SM resident: twice the FP64 path's
// warps; no spills); the grid-field one needs 244 and is left alone.
#ifndef KF_FWD_F32_THREADS_PER_SM
#define KF_FWD_F32_THREADS_PER_SM 512
#endif
// MODE: 0 = planes only, field gradient neglected in the Jacobian (the hot path: propagate()); 1 = surfaces of any kind
// (kf_geometry.surface_kinds: planes, cylinders, discs); 2 = any kind + the field-gradient terms of the
// step Jacobian (kf_options.field_gradient).  1 takes propagate<.., CURVED> (the hot path's closed-form
// / column steps with the surfaces' own charts), 2 takes propagate_general() (five columns with the gradient terms).
template <int FIELD, bool MATERIAL, bool GEOM_SMEM, int LPT, int BLOCK, bool MBF, bool PLAIN, typename R = double, int MODE = 0>
__global__ void __launch_bounds__(BLOCK, (std::is_same<R, float>::value && FIELD == FIELD_CONST) ? KF_FWD_F32_THREADS_PER_SM / BLOCK
                                                                                                : KF_FWD_MIN_BLOCKS)
kf_forward_kernel(const __grid_constant__ FitParams P) {
  static_assert(std::is_same<R, double>::value || (LPT == 1 && !MBF && GEOM_SMEM), "the MIXED path: thread per track, RTS records");
  static_assert(MODE == 0 || (LPT == 1 && !MBF && GEOM_SMEM), "general surfaces / gradient terms: thread per track, RTS records");
  static_assert(MODE != 2 || std::is_same<R, double>::value, "the field-gradient terms: FP64");
  const int o_n_corr = PLAIN ? 2 : P.n_corr;
  const R o_max_step = PLAIN ? R(0.0) : (R)P.max_step, o_step_tol = PLAIN ? R(0.0) : (R)P.step_tol;
  const double* const o_var = PLAIN ? nullptr : P.var;
  const int o_states = PLAIN ? 0 : P.output_states;
  double* const o_rk_err = PLAIN ? nullptr : P.rk_err_max;
  const R o_outlier = (R)P.outlier_chi2;
  const FieldDescT<R>& Fd = field_of<R>(P);
  const MaterialDescT<R>& Md = material_of<R>(P);
  static_assert(BLOCK % KF_TILE == 0, "a forward CTA covers whole tiles");
  unsigned char* const s_fwd_raw = kf_dyn_smem;
  const R* __restrict__ G;
  if constexpr (GEOM_SMEM) {
    stage_geometry<R>(P, reinterpret_cast<R*>(s_fwd_raw));
    G = reinterpret_cast<const R*>(s_fwd_raw);
  } else {
    G = reinterpret_cast<const R*>(P.geom);  // (double only, see the static_assert)
  }
  double* const s_dyn = reinterpret_cast<double*>(s_fwd_raw + (GEOM_SMEM ? geom_smem_bytes<R>(P.n_surfaces) : 0));  // hit slots
  if constexpr (FIELD == FIELD_GRID3S) {
    // the box of the field table the host chose (kf_field.stage_*) -> shared memory, once per CTA, as values of type R
    R* const s_box = reinterpret_cast<R*>(kf_dyn_smem + Fd.box_off);
    const int bx = Fd.box_n[0] * 3, by = Fd.box_n[1], bz = Fd.box_n[2];
    const int rows = by * bz;
    for (int e = threadIdx.x; e < rows * bx; e += BLOCK) {
      const int rw = e / bx, c = e - rw * bx, k = rw / by, j = rw - k * by;
      s_box[e] = (R)__ldg(Fd.grid + ((size_t)(Fd.box_lo[2] + k) * Fd.n[1] + (size_t)(Fd.box_lo[1] + j)) * ((size_t)Fd.n[0] * 3) +
                          (size_t)Fd.box_lo[0] * 3 + c);
    }
    __syncthreads();
  }
  const long long tslot = ((long long)blockIdx.x * BLOCK + threadIdx.x) / LPT;
  if (tslot >= P.N) return;    // LPT > 1: a group is 8 aligned lanes, so whole groups leave together
  const long long i = P.perm ? (long long)P.perm[tslot] : tslot;  // the track this slot fits
  const long long N = P.ldn;  // SoA stride
  const int q = LPT > 1 ? (int)(threadIdx.x % LPT) : 0;           // lane within the group
  const int gbase = LPT > 1 ? (int)((threadIdx.x & 31) & ~(LPT - 1)) : 0;  // first lane of the group in its warp
  const unsigned gmask = LPT > 1 ? ((1u << LPT) - 1u) << gbase : 0u;
  const bool lead = LPT == 1 || q == 0;  // the lane that writes the track's results

  int o0 = P.offsets[i], o1 = P.offsets[i + 1];
  // the CSR offsets live in device memory, out of the host validation's sight: a range outside [0, M] or running
  // backwards is a malformed hit list (the track is not fitted and none of its per-hit outputs is touched)
  const bool offsets_ok = o0 >= 0 && o0 <= o1 && (long long)o1 <= P.M;
  if (!offsets_ok) o0 = o1 = 0;
  R x[6], C[21];
#pragma unroll
  for (int k = 0; k < 6; ++k) x[k] = (R)P.params[k * N + i];
#pragma unroll
  for (int k = 0; k < 21; ++k) C[k] = (R)P.inflation * (R)P.cov[k * N + i];

  unsigned status = 0u;
  // the hit list must be strictly ascending in surface index, inside (start, n_surfaces)
  int n_target = 0;
  {
    bool ok = true;
    int prev_s = P.start;
#pragma unroll 8
    for (int j = o0; j < o1; ++j) {  // no early exit: the loads of a track's list stay independent
      const int s = __ldg(P.surf_idx + j);
      ok = ok && (s > prev_s) && (s < P.n_surfaces);
      prev_s = s;
    }
    if (!ok || !offsets_ok) status |= ST_BAD_HITS;
    else n_target = prev_s - P.start;  // visit every surface up to the one of the last hit (U7)
  }
  // the next unconsumed hit is fetched one leg ahead of its use into this thread's own shared-memory
  // slot (two alternating slots), asynchronously
  double* const s_hm = s_dyn + threadIdx.x;  // [slot][2][BLOCK] (the hits as given: doubles)
  int* const s_hs = reinterpret_cast<int*>(s_hm - threadIdx.x + 4 * BLOCK) + threadIdx.x;  // [slot][BLOCK]
  int slot = 0;
  auto fetch_hit = [&](int j, int sl) {
    cp_async4(s_hs + sl * BLOCK, P.surf_idx + j);
    cp_async8(s_hm + (sl * 2 + 0) * BLOCK, P.loc + j);
    cp_async8(s_hm + (sl * 2 + 1) * BLOCK, P.loc + P.ldm + j);
    cp_async_commit();
  };
  if (o0 < o1) fetch_hit(o0, 0);

  // Grid field, thread per track: the covariance is dead weight while the propagation runs (255 registers, spills): it is
  // parked in a shared-memory column of the thread between the gain update of one leg and the covariance transport of the
  // next ([21][BLOCK] values behind the hit slots; conflict-free).
  constexpr bool kParkC = FIELD == FIELD_GRID3 && LPT == 1 && MODE != 2 && std::is_same<R, double>::value;
  R* const s_C = reinterpret_cast<R*>(reinterpret_cast<unsigned char*>(s_dyn) + hit_stage_bytes(BLOCK)) + threadIdx.x;
  auto park_C = [&]() {
    if constexpr (kParkC) {
#pragma unroll
      for (int k = 0; k < 21; ++k) s_C[k * BLOCK] = C[k];
    }
  };
  auto fetch_C = [&]() {
    if constexpr (kParkC) {
#pragma unroll
      for (int k = 0; k < 21; ++k) C[k] = s_C[k * BLOCK];
    }
  };
  park_C();
  R chi2 = R(0.0), errmax = R(0.0);
  int n_used = 0, n_outl = 0, n_holes = 0, nleg = 0, hp = o0;
  R trig[4];
  sincos_lib(x[2], trig[0], trig[1]);
  sincos_lib(x[3], trig[2], trig[3]);
  // this tile's records: [leg][kRecDoubles][KF_TILE] doubles + [KF_TILE] flag bytes per leg
  const int lane_in_tile = LPT == 1 ? threadIdx.x % KF_TILE : (int)(tslot % KF_TILE);
  char* __restrict__ tile_base = P.rec + (size_t)(tslot / KF_TILE) * P.tile_stride;
  char* __restrict__ tile_rec = tile_base + (size_t)lane_in_tile * sizeof(R);
  unsigned char* __restrict__ tile_flag =
      reinterpret_cast<unsigned char*>(tile_base) + (size_t)kRecDoubles * KF_TILE * sizeof(R) + lane_in_tile;

  for (int l = 0; l < n_target; ++l) {
    const int s = P.start + 1 + l;
    const R* __restrict__ sf = G + (s - 1) * 20;
    const R* __restrict__ st = G + s * 20;
    // material of the previous surface, from its filtered state (U6, U16).  C is advanced through
    // the layer only after the propagation succeeded, so that a failed leg leaves (x, C) = last_*.
    R g_prev = R(1.0);
    const R lam_filtered = x[4];
    MaterialStepT<R> ms;
    const bool mat_here = MATERIAL && l > 0 && sf[14] > R(0.0);
    if (mat_here) {
      bool ok_m;
      if constexpr (MODE == 0) ok_m = material_prepare(Md, sf, trig, x[4], ms);
      else ok_m = material_prepare_general(Md, sf, x[0], x[1], trig, x[4], ms);
      if (!ok_m) { status |= ST_ENERGY; break; }
      x[4] = ms.lam_out;
      g_prev = ms.g;
    }
    R xp[6];
    BoundJacobianT<R> J;
    unsigned rc;
    if constexpr (MODE == 0) rc = propagate<FIELD>(Fd, Md.mass, o_n_corr, o_max_step, o_step_tol, sf, st, x, trig, xp, J, errmax, status);
    else if constexpr (MODE == 1) rc = propagate<FIELD, R, true>(Fd, Md.mass, o_n_corr, o_max_step, o_step_tol, sf, st, x, trig, xp, J, errmax, status);
    else rc = propagate_general<FIELD, true>(Fd, Md.mass, o_n_corr, o_max_step, o_step_tol, sf, st, x, trig, xp, J, errmax, status);
    if (rc) {
      status |= rc;
      x[4] = lam_filtered;
      break;
    }
    // RTS record ("stored Jacobians"): x-, F = J G_prev, g_prev go out right away so that the
    // stores drain under the covariance transport; C- and the hit follow it
    R* __restrict__ Rk = reinterpret_cast<R*>(tile_rec + (size_t)l * P.leg_stride);
    if (P.smooth && lead) {
      // the F block sits at kRecFa (RTS record) or kMbfFa (Bryson-Frazier record); Ft and g follow it in both
      R* __restrict__ RF = Rk + (size_t)(MBF ? kMbfFa : kRecFa) * KF_TILE;
      if (!MBF) {
#pragma unroll
        for (int k = 0; k < 6; ++k) KF_REC_STORE(&Rk[(kRecXp + k) * KF_TILE], xp[k]);
      } else if (l == 0) {
        R* __restrict__ FB = reinterpret_cast<R*>(tile_rec + P.first_off);
#pragma unroll
        for (int k = 0; k < 6; ++k) KF_REC_STORE(&FB[k * KF_TILE], xp[k]);
      }
#pragma unroll
      for (int a = 0; a < 4; ++a) {
#pragma unroll
        for (int c = 0; c < 4; ++c) KF_REC_STORE(&RF[(a * 5 + c) * KF_TILE], J.Ja[a][c]);
        KF_REC_STORE(&RF[(a * 5 + 4) * KF_TILE], J.Ja[a][4] * g_prev);
      }
#pragma unroll
      for (int c = 0; c < 4; ++c) KF_REC_STORE(&RF[(kRecFt - kRecFa + c) * KF_TILE], J.Jt[c]);
      KF_REC_STORE(&RF[(kRecFt - kRecFa + 4) * KF_TILE], J.Jt[4] * g_prev);
      KF_REC_STORE(&RF[(kRecG - kRecFa) * KF_TILE], g_prev);
    }
    fetch_C();
    if (mat_here) material_apply(ms, C);
    R Cp[21];
    if constexpr (LPT == 1) transport_covariance(J, C, Cp);
    else transport_covariance_lanes(J, C, Cp, q, gbase, gmask);

    // hit of this surface, if any (fetched during the previous leg); start fetching the one after it
    cp_async_wait_all();
    const bool has_hit = hp < o1 && s_hs[slot * BLOCK] == s;
    R m0 = has_hit ? (R)s_hm[(slot * 2 + 0) * BLOCK] : R(0.0);
    R m1 = has_hit ? (R)s_hm[(slot * 2 + 1) * BLOCK] : R(0.0);
    if constexpr (MODE != 0) {
      // angular local coordinates (U33): the hit is taken on the branch nearest the prediction (period 2 pi R for
      // the arc length on a cylinder, 2 pi for the azimuth on a disc); the record keeps the hit as used, so the RTS kernel's
      // re-filtering sees the same residual
      const int kind = (int)st[18];
      if (has_hit && kind != SURF_PLANE) {
        const R period = kind == SURF_CYLINDER ? R(2.0) * R(kPi) * st[12] : R(2.0) * R(kPi);
        R& m = kind == SURF_CYLINDER ? m0 : m1;
        const R d = m - (kind == SURF_CYLINDER ? xp[0] : xp[1]);
        if (d > R(0.5) * period || d <= -R(0.5) * period) m = m - period * ceil((d - R(0.5) * period) / period);
      }
    }
    if (has_hit && hp + 1 < o1) fetch_hit(hp + 1, slot ^ 1);

    if (P.smooth && lead) {
      if (!MBF) {
#pragma unroll
        for (int k = 0; k < 21; ++k) KF_REC_STORE(&Rk[(kRecCp + k) * KF_TILE], Cp[k]);
        KF_REC_STORE(&Rk[kRecM * KF_TILE], m0);
        KF_REC_STORE(&Rk[(kRecM + 1) * KF_TILE], m1);
      } else {
#pragma unroll
        for (int k = 0; k < 11; ++k) KF_REC_STORE(&Rk[(kMbfCcol + k) * KF_TILE], Cp[k]);  // (0,0..5), (1,1..5)
        if (l == 0) {
          R* __restrict__ FB = reinterpret_cast<R*>(tile_rec + P.first_off);
#pragma unroll
          for (int k = 0; k < 21; ++k) KF_REC_STORE(&FB[(6 + k) * KF_TILE], Cp[k]);
        }
      }
    }

    // gain-matrix update with the surface's hit.  A hole or a flagged outlier runs the
    // same arithmetic with a zero gain (x+ = x-, C+ = C- exactly), so the leg has one code path.
    unsigned char flag = 0;
    GainT<R> gn;
    gn.r0 = gn.r1 = gn.i00 = gn.i01 = gn.i11 = R(0.0);
    if (has_hit) {
      R v00, v11, v01 = R(0.0);
      if (o_var) {
        v00 = (R)o_var[hp];
        v11 = (R)o_var[P.ldm + hp];
        if (P.cov01) v01 = (R)P.cov01[hp];
      } else {
        v00 = st[16];
        v11 = st[17];
      }
      R c2 = R(0.0);
      if (!gain_prepare(xp, Cp, m0, m1, v00, v01, v11, gn, c2)) {
        status |= ST_NOT_POSITIVE;
        if (mat_here && !kParkC) material_undo(ms, C);   // (parked: the column still holds C before the layer)
        x[4] = lam_filtered;
        break;
      }
      if (o_outlier > R(0.0) && c2 > o_outlier) {  // strictly greater: flagged, not used (U9)
        n_outl++;
        flag = 2;
        gn.i00 = gn.i01 = gn.i11 = R(0.0);
      } else {
        chi2 += c2;
        n_used++;
        flag = 1;
      }
      if (P.hit_chi2 && lead) P.hit_chi2[hp] = (double)c2;
      if (P.hit_flags && lead) P.hit_flags[hp] = flag;
      hp++;
      slot ^= 1;
    } else {
      n_holes++;
    }
    if (P.smooth && MBF && lead) {  // the gain as applied: zero for a hole or a flagged outlier
      KF_REC_STORE(&Rk[(kMbfGain + 0) * KF_TILE], gn.r0);
      KF_REC_STORE(&Rk[(kMbfGain + 1) * KF_TILE], gn.r1);
      KF_REC_STORE(&Rk[(kMbfGain + 2) * KF_TILE], gn.i00);
      KF_REC_STORE(&Rk[(kMbfGain + 3) * KF_TILE], gn.i01);
      KF_REC_STORE(&Rk[(kMbfGain + 4) * KF_TILE], gn.i11);
    }
    gain_apply(gn, xp, Cp, x, C);
    park_C();
    // trig holds the angles of x-: rotate by the gain's correction (zero for a hole)
    rotate_trig(trig, x[2], x[2] - xp[2], x[3], x[3] - xp[3]);
    if (P.smooth && !MBF && lead) tile_flag[(size_t)l * P.leg_stride] = flag;
    if ((o_states & OUT_PRED) && lead) {
      store6(P.state_params[0] + (size_t)l * 6 * N, N, i, xp);
      store21(P.state_cov[0] + (size_t)l * 21 * N, N, i, Cp);
    }
    if ((o_states & OUT_FILT) && lead) {
      store6(P.state_params[1] + (size_t)l * 6 * N, N, i, x);
      store21(P.state_cov[1] + (size_t)l * 21 * N, N, i, C);
    }
    if (l == 0 && lead) {
      store6(P.first_params, N, i, x);
      store21(P.first_cov, N, i, C);
    }
    nleg++;
  }

  // (x, C) = filtered state of the last completed leg, before that layer's material (start state if none)
  if (MATERIAL && nleg == n_target && nleg > 0) {  // the last surface's material: status bit only
    const R* __restrict__ sl = G + (P.start + nleg) * 20;
    MaterialStepT<R> ms;
    if (sl[14] > R(0.0)) {
      bool ok_m;
      if constexpr (MODE == 0) ok_m = material_prepare(Md, sl, trig, x[4], ms);
      else ok_m = material_prepare_general(Md, sl, x[0], x[1], trig, x[4], ms);
      if (!ok_m) status |= ST_ENERGY;
    }
  }
  if (!lead) return;
  store6(P.last_params, N, i, x);
  fetch_C();
  store21(P.last_cov, N, i, C);
  if (nleg == 0) {
    store6(P.first_params, N, i, x);
    store21(P.first_cov, N, i, C);
  }

  const int ndf = 2 * n_used - 5;
  if (ndf <= 0) status |= ST_NDF;
  P.chi2[i] = (double)chi2;
  P.ndf[i] = ndf;
  P.status[i] = status;
  P.n_used[i] = n_used;
  P.n_outliers[i] = n_outl;
  P.n_holes[i] = n_holes;
  if (o_rk_err) o_rk_err[i] = (double)errmax;
  if (P.smooth) P.nleg[tslot] = nleg;
  for (int j = hp; j < o1; ++j) {  // hits never reached
    if (P.hit_chi2) P.hit_chi2[j] = 0.0;
    if (P.hit_flags) P.hit_flags[j] = 0;
  }
}
}  // namespace kf
