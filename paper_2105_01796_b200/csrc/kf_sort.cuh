// kf_sort.cuh -- length sort of ragged batches (sm_100a).
//
// Every track visits the surfaces from start+1 up to the surface of its LAST hit (U7), so in a
// ragged batch (BASELINE.json configs[3], configs[4]: tracks that leave the acceptance stop early) the
// tracks of one warp run different numbers of legs: ncu on CFG4 shows 14.2 of 32 threads active per
// executed instruction in both kernels, and the RTS kernel walks every 64-track tile for the longest
// track in it.  The remedy is a counting sort by the number of legs, longest first: slot s of the launch
// fits track perm[s]; RTS records and leg counts are indexed by slot, every caller-visible array by
// track.  Three tiny kernels over the CSR offsets (8 B read per track): histogram, exclusive scan over
// at most kSortBins bins in descending length, scatter.  Inside a bin the tracks of one block keep their
// ascending order, blocks follow each other in the order their atomics land: each track's fit is independent
// (PAPER.md:119), so the results do not depend on the slot a track runs in (tested bit for bit).
#pragma once

#include "kf_common.cuh"

namespace kf {

constexpr int kSortBlock = 256;

struct SortParams {
  long long N, M;      // tracks of the launch; hits of the batch
  const int* offsets;   // [N+1]
  const int* surf_idx;  // [M]
  int start, lmax;      // legs of a track = surface of its last hit - start, clamped to [0, lmax]
  int* bins;            // [kSortBins] histogram, then running cursors (zeroed by the caller before the launch)
  int* perm;            // [N] out
  int force;            // 1: sort whatever the spread of the lengths (KF_SORT_ON)
};

__device__ __forceinline__ int sort_bin_of(const SortParams& S, long long i) {
  const int o0 = S.offsets[i], o1 = S.offsets[i + 1];
  int len = 0;
  if (o1 > o0 && o0 >= 0 && (long long)o1 <= S.M) len = __ldg(S.surf_idx + (o1 - 1)) - S.start;  // else: malformed, not fitted
  len = max(0, min(len, S.lmax));
  // longest first: bin 0 holds the longest tracks
  const int b = S.lmax < kSortBins ? len : (int)(((long long)len * (kSortBins - 1)) / S.lmax);
  return min(S.lmax, kSortBins - 1) - b;
}

__global__ void __launch_bounds__(kSortBlock) kf_sort_hist_kernel(const __grid_constant__ SortParams S) {
  __shared__ int h[kSortBins];
  if (threadIdx.x < kSortBins) h[threadIdx.x] = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * kSortBlock + threadIdx.x;
  if (i < S.N) atomicAdd(&h[sort_bin_of(S, i)], 1);
  __syncthreads();
  if (threadIdx.x < kSortBins && h[threadIdx.x]) atomicAdd(&S.bins[threadIdx.x], h[threadIdx.x]);
}

// one thread: counts -> first slot of every bin.  Unless `force`, a batch whose mean leg count is within
// kSortKeepOrder of its longest track's is left in its own order (bins[] = -1 tells the scatter kernel to write the
// identity): there the sort has nothing to win and its gathered per-track loads and stores only cost (measured on
// BASELINE.json configs[3], efficiency 0.95: 6.20 ms unsorted, 6.44 ms sorted; configs[4]: 13.9 -> 7.4 ms).
constexpr double kSortKeepOrder = 0.85;
__global__ void kf_sort_scan_kernel(int* bins, int lmax, int force) {
  if (threadIdx.x == 0) {
    const int top = min(lmax, kSortBins - 1);  // bin b holds quantised length top - b
    long long n = 0, sum = 0;
    int longest = 0;
    for (int b = kSortBins - 1; b >= 0; --b) {
      const int c = bins[b];
      if (c > 0) longest = top - b;
      n += c;
      sum += (long long)c * (top - b);
    }
    const bool keep = !force && (double)sum >= kSortKeepOrder * (double)longest * (double)n;
    int run = 0;
    for (int b = 0; b < kSortBins; ++b) {
      const int c = bins[b];
      bins[b] = keep ? -1 : run;
      run += c;
    }
  }
}

// a block takes its slots of a bin with ONE atomic per bin and hands them out in thread order, so that the
// tracks of a block that share a bin stay in ascending order (neighbouring slots read neighbouring tracks)
__global__ void __launch_bounds__(kSortBlock) kf_sort_scatter_kernel(const __grid_constant__ SortParams S) {
  __shared__ int cnt[kSortBins], base[kSortBins];
  const long long i = (long long)blockIdx.x * kSortBlock + threadIdx.x;
  if (S.bins[0] < 0) {  // the scan kernel decided to keep the batch's own order
    if (i < S.N) S.perm[i] = (int)i;
    return;
  }
  if (threadIdx.x < kSortBins) cnt[threadIdx.x] = 0;
  __syncthreads();
  int b = -1, rank = 0;
  if (i < S.N) b = sort_bin_of(S, i);
  // rank of this thread among the block's threads of the same bin, in thread order: warp by warp
  const unsigned lane = threadIdx.x & 31u;
  const unsigned peers = __match_any_sync(0xffffffffu, b);
  const int before = __popc(peers & ((1u << lane) - 1u));
  const int leader = __ffs(peers) - 1;
  for (int w = 0; w < kSortBlock / 32; ++w) {  // warps take their turn, so ranks follow thread order
    if ((int)(threadIdx.x >> 5) == w && b >= 0) {
      int first = 0;
      if ((int)lane == leader) first = atomicAdd(&cnt[b], __popc(peers));
      first = __shfl_sync(peers, first, leader);
      rank = first + before;
    }
    __syncthreads();
  }
  if (threadIdx.x < kSortBins && cnt[threadIdx.x]) base[threadIdx.x] = atomicAdd(&S.bins[threadIdx.x], cnt[threadIdx.x]);
  __syncthreads();
  if (b >= 0) S.perm[base[b] + rank] = (int)i;
}

}  // namespace kf
