// kf_fwd_grid.cu -- kf_forward_kernel instantiations for a 3-D grid field (trilinear), FP64, one thread per track.
// Always KF_FWD_BLOCK_SMALL threads per CTA (measured: the 256-thread CTA is slower for this kernel).
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

namespace {
template <bool MATERIAL, bool MBF, bool PLAIN>
int go(const kf::FitParams& P, cudaStream_t stream) {
  constexpr int BLOCK = KF_FWD_BLOCK_SMALL;
  const char* nm = "kf_forward_kernel (grid field)";
  if (P.geom_in_smem) {
    // the table is gathered through L1: ask for just the shared memory two resident CTAs use (+ 1 KB each that the
    // system reserves), leaving the rest of the SM's 256 KB to L1 (CFG4 forward 1.256 -> 1.224 ms per 262,144 tracks)
    const size_t smem = kf::geom_smem_bytes<double>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK) + kf::cov_park_bytes<double>(BLOCK);
    const int pct = carveout_for(smem, 2);
    return launch(kf::kf_forward_kernel<kf::FIELD_GRID3, MATERIAL, true, 1, BLOCK, MBF, PLAIN>, P, BLOCK, smem, stream, nm, 1, pct);
  }
  return launch(kf::kf_forward_kernel<kf::FIELD_GRID3, MATERIAL, false, 1, BLOCK, MBF, false>, P, BLOCK,
                kf::hit_stage_bytes(BLOCK) + kf::cov_park_bytes<double>(BLOCK), stream, nm);
}
template <bool MATERIAL, bool MBF>
int pick(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  return c.plain ? go<MATERIAL, MBF, true>(P, stream) : go<MATERIAL, MBF, false>(P, stream);
}
}  // namespace

int launch_forward_grid(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.mbf) return c.material ? pick<true, true>(P, c, stream) : pick<false, true>(P, c, stream);
  return c.material ? pick<true, false>(P, c, stream) : pick<false, false>(P, c, stream);
}

}  // namespace kfh
