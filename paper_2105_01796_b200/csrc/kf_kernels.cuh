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
// Workspace layout: tile-major, one tile = KF_TILE tracks = one CTA.
//   rec   [tile][leg]{ double[kRecDoubles][KF_TILE]; uint8 flag[KF_TILE] }   (kLegBytes per tile-leg)
//         a warp's 32 tracks write 32 consecutive doubles per component (256 B, coalesced); the component
//         stride is a compile-time constant (immediate offsets); the RTS kernel fetches one tile-leg with
//         one bulk async copy.  flag: 0 hole, 1 used, 2 outlier.
//   nleg  int32 [tiles * KF_TILE]   number of legs the forward pass completed
#pragma once

#include "kf_device.cuh"
#include "kf_lanes.cuh"

namespace kf {

constexpr int kRecDoubles = 55;  // x-(6) C-(21) Fa(20) Ft(5) g(1) hit(2)
constexpr int kRecXp = 0, kRecCp = 6, kRecFa = 27, kRecFt = 47, kRecG = 52, kRecM = 53;
// record of the Bryson-Frazier backward pass (kf_options.smoother, kf_mbf.cuh): gain (r0 r1 S^-1_00 S^-1_01 S^-1_11;
// zero gain = hole or outlier), the two leading columns of C- (00 01 .. 05 11 .. 15), then F = J G and g as above.
// x- and C- of the FIRST leg only go to a per-tile block behind the tile's legs.
constexpr int kMbfDoubles = 42;
constexpr int kMbfGain = 0, kMbfCcol = 5, kMbfFa = 16, kMbfFt = 36, kMbfG = 41;
constexpr int kMbfFirstDoubles = 27;  // x-(6) C-(21) of leg 0

// tracks per tile of the record layout = threads per CTA of the RTS kernel (one bulk copy per tile-leg);
// the forward kernel's CTA covers KF_FWD_BLOCK / KF_TILE whole tiles
#ifndef KF_TILE
#define KF_TILE 64
#endif
// threads per forward CTA: KF_FWD_BLOCK for batches that fill the chip more than once (measured on CFG2: 256
// threads 3.38-3.40 ms, 128 threads 3.46-3.48 ms), KF_FWD_BLOCK_SMALL for smaller ones and for the lanes variant
// (more CTAs, so more SMs take part while a batch is latency-bound)
#ifndef KF_FWD_BLOCK
#define KF_FWD_BLOCK 256
#endif
#ifndef KF_FWD_BLOCK_SMALL
#define KF_FWD_BLOCK_SMALL 128
#endif
static_assert(KF_FWD_BLOCK % KF_TILE == 0 && KF_FWD_BLOCK_SMALL % KF_TILE == 0 && KF_TILE % 32 == 0, "a forward CTA covers whole tiles; a tile covers whole warps");
// bytes of one tile-leg: kRecDoubles values of the path's arithmetic type per track + one flag byte per track
template <typename R>
__host__ __device__ constexpr size_t leg_bytes() { return (size_t)kRecDoubles * KF_TILE * sizeof(R) + KF_TILE; }
constexpr size_t kLegBytes = leg_bytes<double>();  // the FP64 path's record + flags
#ifndef KF_FWD_MIN_BLOCKS
#define KF_FWD_MIN_BLOCKS 1
#endif
#ifndef KF_RTS_MIN_BLOCKS
#define KF_RTS_MIN_BLOCKS 1
#endif

// record stores: written once, read much later by the RTS kernel -> streaming stores (evict-first in L2), so that
// 13 GB of records passing through do not push the field grid and the hit lists out of L2
#ifdef KF_REC_PLAIN_STORES
#define KF_REC_STORE(ptr, v) (*(ptr) = (v))
#else
#define KF_REC_STORE(ptr, v) __stcs((ptr), (v))
#endif
enum : int { OUT_PRED = 1, OUT_FILT = 2, OUT_SMOOTH = 4 };

struct FitParams {
  // inputs
  long long N, M;       // tracks of this launch; hits of the batch
  long long ldn, ldm;   // leading dimensions of the SoA track arrays / hit arrays (>= N, >= M): a launch over a
                        // sub-range of a batch gets base pointers advanced by its first track and ldn = batch size
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
  FieldDescT<float> field_f;   // the same two descriptors rounded to float: what the MIXED-precision kernels read
  MaterialDescT<float> mat_f;
  // options
  int smooth, n_corr, output_states;
  double outlier_chi2, max_step, step_tol, inflation;
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
  char* rec;            // [tile][leg]{ double[kRecDoubles][KF_TILE]; uint8 flag[KF_TILE] }
  size_t leg_stride;    // = kLegBytes
  size_t tile_stride;   // = Lmax * kLegBytes
  int* nleg;            // [slots] legs the forward pass completed, by SLOT
  int mbf;              // 1: Bryson-Frazier records (kMbf*), 0: RTS records (kRec*)
  int mixed;            // 1: float operands and records (kf_options.precision MIXED), 0: double
  size_t first_off;     // mbf: byte offset of a tile's first-leg block [kMbfFirstDoubles][KF_TILE] from its base
  // length sort of ragged batches (kf_sort.cuh): slot -> track.  Records and nleg are indexed by slot (the
  // position in launch order), every caller-visible array by track.  nullptr: slot == track.
  const int* perm;
};

template <typename R>
__device__ __forceinline__ void store6(double* base, long long stride, long long i, const R v[6]) {
#pragma unroll
  for (int k = 0; k < 6; ++k) base[k * stride + i] = (double)v[k];
}
template <typename R>
__device__ __forceinline__ void store21(double* base, long long stride, long long i, const R v[21]) {
#pragma unroll
  for (int k = 0; k < 21; ++k) base[k * stride + i] = (double)v[k];
}
// the descriptors of the kernel's arithmetic type
template <typename R> __device__ __forceinline__ const FieldDescT<R>& field_of(const struct FitParams& P);
template <typename R> __device__ __forceinline__ const MaterialDescT<R>& material_of(const struct FitParams& P);

__device__ __forceinline__ unsigned smem_u32(const void* p) {
  return static_cast<unsigned>(__cvta_generic_to_shared(p));
}
// per-thread asynchronous global -> shared copies (LDGSTS): completion is tracked by copy groups, not by
// the register scoreboards, so a fetch in flight never holds up an unrelated load of the same thread
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// bytes of the forward kernel's hit staging area: two alternating slots of (loc0, loc1, surface) per thread
constexpr size_t hit_stage_bytes(int block) { return (size_t)block * (2 * 2 * sizeof(double) + 2 * sizeof(int)); }

template <> __device__ __forceinline__ const FieldDescT<double>& field_of<double>(const FitParams& P) { return P.field; }
template <> __device__ __forceinline__ const FieldDescT<float>& field_of<float>(const FitParams& P) { return P.field_f; }
template <> __device__ __forceinline__ const MaterialDescT<double>& material_of<double>(const FitParams& P) { return P.mat; }
template <> __device__ __forceinline__ const MaterialDescT<float>& material_of<float>(const FitParams& P) { return P.mat_f; }

// stage the geometry table in shared memory once per CTA (5 KB for 31 planes; half that in float), converted to the
// kernel's arithmetic type
template <typename R>
__device__ __forceinline__ void stage_geometry(const FitParams& P, R* smem) {
  const int n = P.n_surfaces * 20;
  for (int k = threadIdx.x; k < n; k += blockDim.x) smem[k] = (R)P.geom[k];
  __syncthreads();
}
// bytes the staged table takes (a multiple of 16: the hit slots behind it hold doubles)
template <typename R>
__host__ __device__ constexpr size_t geom_smem_bytes(int n_surfaces) {
  return ((size_t)n_surfaces * 20 * sizeof(R) + 15) / 16 * 16;
}


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
template <int FIELD, bool MATERIAL, bool GEOM_SMEM, int LPT, int BLOCK, bool MBF, bool PLAIN, typename R = double>
__global__ void __launch_bounds__(BLOCK, (std::is_same<R, float>::value && FIELD == FIELD_CONST) ? KF_FWD_F32_THREADS_PER_SM / BLOCK
                                                                                                : KF_FWD_MIN_BLOCKS)
kf_forward_kernel(const __grid_constant__ FitParams P) {
  static_assert(std::is_same<R, double>::value || (LPT == 1 && !MBF && GEOM_SMEM), "the MIXED path: thread per track, RTS records");
  const int o_n_corr = PLAIN ? 2 : P.n_corr;
  const R o_max_step = PLAIN ? R(0.0) : (R)P.max_step, o_step_tol = PLAIN ? R(0.0) : (R)P.step_tol;
  const double* const o_var = PLAIN ? nullptr : P.var;
  const int o_states = PLAIN ? 0 : P.output_states;
  double* const o_rk_err = PLAIN ? nullptr : P.rk_err_max;
  const R o_outlier = (R)P.outlier_chi2;
  const FieldDescT<R>& Fd = field_of<R>(P);
  const MaterialDescT<R>& Md = material_of<R>(P);
  static_assert(BLOCK % KF_TILE == 0, "a forward CTA covers whole tiles");
  extern __shared__ __align__(16) unsigned char s_fwd_raw[];
  const R* __restrict__ G;
  if constexpr (GEOM_SMEM) {
    stage_geometry<R>(P, reinterpret_cast<R*>(s_fwd_raw));
    G = reinterpret_cast<const R*>(s_fwd_raw);
  } else {
    G = reinterpret_cast<const R*>(P.geom);  // (double only, see the static_assert)
  }
  double* const s_dyn = reinterpret_cast<double*>(s_fwd_raw + (GEOM_SMEM ? geom_smem_bytes<R>(P.n_surfaces) : 0));  // hit slots
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
      if (!material_prepare(Md, sf, trig, x[4], ms)) { status |= ST_ENERGY; break; }
      x[4] = ms.lam_out;
      g_prev = ms.g;
    }
    R xp[6];
    BoundJacobianT<R> J;
    const unsigned rc = propagate<FIELD>(Fd, Md.mass, o_n_corr, o_max_step, o_step_tol, sf, st, x, trig,
                                         xp, J, errmax, status);
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
    if (mat_here) material_apply(ms, C);
    R Cp[21];
    if constexpr (LPT == 1) transport_covariance(J, C, Cp);
    else transport_covariance_lanes(J, C, Cp, q, gbase, gmask);

    // hit of this surface, if any (fetched during the previous leg); start fetching the one after it
    cp_async_wait_all();
    const bool has_hit = hp < o1 && s_hs[slot * BLOCK] == s;
    const R m0 = has_hit ? (R)s_hm[(slot * 2 + 0) * BLOCK] : R(0.0);
    const R m1 = has_hit ? (R)s_hm[(slot * 2 + 1) * BLOCK] : R(0.0);
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
        if (mat_here) material_undo(ms, C);
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
    if (sl[14] > R(0.0) && !material_prepare(Md, sl, trig, x[4], ms)) status |= ST_ENERGY;
  }
  if (!lead) return;
  store6(P.last_params, N, i, x);
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
