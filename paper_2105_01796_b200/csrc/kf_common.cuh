// kf_common.cuh -- what the two global kernels of the fit share: record layout, parameter block, small device helpers.
// (kf_forward.cuh: kf_forward_kernel; kf_rts.cuh: kf_rts_kernel, kf_rts_lanes_kernel.)
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
constexpr int kSortBins = 64;    // length sort (kf_sort.cuh): lengths are quantised into at most this many bins

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
constexpr size_t kMbfLegBytes = (size_t)kMbfDoubles * KF_TILE * sizeof(double);  // Bryson-Frazier record (no flag byte)
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
__host__ __device__ constexpr size_t hit_stage_bytes(int block) { return (size_t)block * (2 * 2 * sizeof(double) + 2 * sizeof(int)); }

// bytes of the grid-field kernels' parking area for the covariance (kf_forward.cuh): 21 values per thread behind the hit slots
template <typename R>
__host__ __device__ constexpr size_t cov_park_bytes(int block) { return (size_t)block * 21 * sizeof(R); }

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

}  // namespace kf
