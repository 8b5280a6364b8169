// kf_bwd.cu -- everything that follows the forward filter: the backward pass that matches the records (RTS thread
// per track in FP64 or MIXED precision, RTS lanes per track, Bryson-Frazier), and the small kernels around the fit
// (length sort of ragged batches, perigee extrapolation, DFMA probe).
#include "kf_host.h"
#include "kf_rts.cuh"
#include "kf_mbf.cuh"
#include "kf_perigee.cuh"
#include "kf_sort.cuh"

namespace kfh {

int launch_backward(const kf::FitParams& P, bool lanes, cudaStream_t stream) {
  if (P.mbf) return launch(kf::kf_mbf_kernel, P, KF_TILE, kf::kMbfSmem, stream, "kf_mbf_kernel");
  // two record stages + mbarriers
  const size_t rts_smem = 2 * (P.mixed ? kf::leg_bytes<float>() : kf::leg_bytes<double>()) + 2 * sizeof(unsigned long long);
  const bool plain = !P.var && !(P.output_states & kf::OUT_SMOOTH);
  if (P.mixed)
    return plain ? launch(kf::kf_rts_kernel<true, float>, P, KF_TILE, rts_smem, stream, "kf_rts_kernel (mixed precision)")
                 : launch(kf::kf_rts_kernel<false, float>, P, KF_TILE, rts_smem, stream, "kf_rts_kernel (mixed precision)");
  if (lanes)
    return launch(kf::kf_rts_lanes_kernel, P, kf::kRtsLanesBlock, kf::kRtsLanesSmem, stream, "kf_rts_lanes_kernel", kf::kLanes);
  return plain ? launch(kf::kf_rts_kernel<true>, P, KF_TILE, rts_smem, stream, "kf_rts_kernel")
               : launch(kf::kf_rts_kernel<false>, P, KF_TILE, rts_smem, stream, "kf_rts_kernel");
}

// kf_sort.cuh: zero the bin counters, histogram, scan, scatter
int launch_length_sort(const kf::FitParams& P, int* perm, int* bins, int force, cudaStream_t stream) {
  kf::SortParams S{};
  S.N = P.N; S.M = P.M; S.offsets = P.offsets; S.surf_idx = P.surf_idx; S.start = P.start;
  S.lmax = P.n_surfaces - 1 - P.start;
  S.bins = bins; S.perm = perm; S.force = force;
  if (set_cuda_error(cudaMemsetAsync(bins, 0, kf::kSortBins * sizeof(int), stream), "length sort")) return KF_ERR_CUDA;
  const unsigned grid = (unsigned)((P.N + kf::kSortBlock - 1) / kf::kSortBlock);
  kf::kf_sort_hist_kernel<<<grid, kf::kSortBlock, 0, stream>>>(S);
  kf::kf_sort_scan_kernel<<<1, 32, 0, stream>>>(bins, S.lmax, S.force);
  kf::kf_sort_scatter_kernel<<<grid, kf::kSortBlock, 0, stream>>>(S);
  if (set_cuda_error(cudaGetLastError(), "length sort")) return KF_ERR_CUDA;
  g_launches += 3;
  return KF_OK;
}

int launch_perigee(const kf::FitParams& P, const PerigeeLine& line, bool grid3, bool any_kind, cudaStream_t stream) {
  kf::PerigeeParams G{};
  G.any_kind = any_kind ? 1 : 0;
  for (int a = 0; a < 3; ++a) { G.line.c[a] = line.c[a]; G.line.a[a] = line.a[a]; }
  G.params = line.params;
  G.cov = line.cov;
  const unsigned grid = (unsigned)((P.N + kf::kPerigeeBlock - 1) / kf::kPerigeeBlock);
  if (grid3) kf::kf_perigee_kernel<kf::FIELD_GRID3><<<grid, kf::kPerigeeBlock, 0, stream>>>(P, G);
  else kf::kf_perigee_kernel<kf::FIELD_CONST><<<grid, kf::kPerigeeBlock, 0, stream>>>(P, G);
  if (set_cuda_error(cudaGetLastError(), "kf_perigee_kernel")) return KF_ERR_CUDA;
  g_launches++;
  return KF_OK;
}

double probe_fp64_tflops(int iters, cudaStream_t stream) {
  int dev = 0, sms = 0;
  if (set_cuda_error(cudaGetDevice(&dev), "cudaGetDevice")) return (double)KF_ERR_CUDA;
  if (set_cuda_error(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute"))
    return (double)KF_ERR_CUDA;
  const int block = 256, grid = sms * 8;
  cudaEvent_t e0, e1;
  if (set_cuda_error(cudaEventCreate(&e0), "cudaEventCreate")) return (double)KF_ERR_CUDA;
  if (set_cuda_error(cudaEventCreate(&e1), "cudaEventCreate")) { cudaEventDestroy(e0); return (double)KF_ERR_CUDA; }
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {  // first repetition is the warm-up
    cudaEventRecord(e0, stream);
    kf::kf_dfma_probe_kernel<<<grid, block, 0, stream>>>(nullptr, iters, 1.0000001, 1e-9);
    cudaEventRecord(e1, stream);
    if (set_cuda_error(cudaEventSynchronize(e1), "kf_dfma_probe_kernel")) { best = (double)KF_ERR_CUDA; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = 2.0 * 8.0 * (double)iters * (double)block * (double)grid;
    const double tf = flops / ((double)ms * 1e-3) * 1e-12;
    if (rep > 0 && tf > best) best = tf;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return best;
}

}  // namespace kfh
