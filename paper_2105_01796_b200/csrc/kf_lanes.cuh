// kf_lanes.cuh -- the lanes-per-track variant's cooperative 6x6 algebra (sm_100a, IEEE double).
//
// PAPER.md:126-128 describes an "intra-track parallelisation": the matrix operations of one fit spread
// over the threads of a block with the per-track objects in shared memory; it won below ~1000 tracks and
// lost above.  The north star asks for the B200 form of that idea as a measured
// alternative: a group of kLanes = 8 adjacent lanes of a warp owns one track.  The scalar part of a leg
// (stepping, gain, material) runs redundantly in every lane -- identical inputs, identical instructions,
// hence identical values and branches -- and the 6x6 products are split by ROW: lane q (q < 6) computes
// row q, rows are exchanged with warp shuffles restricted to the group's lanes.  No shared memory, no
// block-level barrier.  Which variant runs when is a measured choice (DESIGN.md "Thread-per-track or
// lanes-per-track").
#pragma once

#include "kf_device.cuh"

namespace kf {

constexpr int kLanes = 8;

// element (row, c) of a packed symmetric 6x6 for a lane-dependent row (c is a compile-time constant
// after unrolling): a chain of selects instead of a dynamically indexed register array
__device__ __forceinline__ double sym_row(const double C[21], int row, int c) {
  double v = C[SX(0, c)];
#pragma unroll
  for (int r = 1; r < 6; ++r) v = (row == r) ? C[SX(r, c)] : v;
  return v;
}

// x[row] for a lane-dependent row
__device__ __forceinline__ double vec_sel(const double x[6], int row) {
  double v = x[0];
#pragma unroll
  for (int r = 1; r < 6; ++r) v = (row == r) ? x[r] : v;
  return v;
}

// every lane of the group receives the packed upper triangle assembled from the lanes' rows:
// out[IX(i, j)] = rowvals[j] of lane i (i <= j)
__device__ __forceinline__ void gather_sym(const double rowvals[6], double out[21], int gbase, unsigned gmask) {
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = i; j < 6; ++j) out[IX(i, j)] = __shfl_sync(gmask, rowvals[j], gbase + i);
}

// C- = J C J^T (DESIGN.md A.4), row `q` of the result per lane, then all rows to all lanes.
// Lanes 6 and 7 repeat row 5 (their values are never read).
__device__ __forceinline__ void transport_covariance_lanes(const BoundJacobian& J, const double C[21],
                                                           double Cp[21], int q, int gbase, unsigned gmask) {
  const int row = q < 6 ? q : 5;
  // row of the full 6x6 J: rows 0..3 = Ja (column t zero), row 4 = e_qp, row 5 = (Jt, 1)
  double Jr[6];
#pragma unroll
  for (int l = 0; l < 5; ++l) {
    double v = J.Ja[0][l];
    v = (row == 1) ? J.Ja[1][l] : v;
    v = (row == 2) ? J.Ja[2][l] : v;
    v = (row == 3) ? J.Ja[3][l] : v;
    v = (row == 4) ? (l == 4 ? 1.0 : 0.0) : v;
    v = (row == 5) ? J.Jt[l] : v;
    Jr[l] = v;
  }
  Jr[5] = (row == 5) ? 1.0 : 0.0;
  // M row = Jr C
  double Mr[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    double s = Jr[0] * C[SX(0, k)];
#pragma unroll
    for (int l = 1; l < 6; ++l) s = fma(Jr[l], C[SX(l, k)], s);
    Mr[k] = s;
  }
  // row of C- = Mr J^T
  double Rw[6];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    double s = Mr[0] * J.Ja[j][0];
#pragma unroll
    for (int l = 1; l < 5; ++l) s = fma(Mr[l], J.Ja[j][l], s);
    Rw[j] = s;
  }
  Rw[4] = Mr[4];
  {
    double s = Mr[5];
#pragma unroll
    for (int l = 0; l < 5; ++l) s = fma(Mr[l], J.Jt[l], s);
    Rw[5] = s;
  }
  gather_sym(Rw, Cp, gbase, gmask);
}

}  // namespace kf
