// kf_fwd_const.cu -- kf_forward_kernel instantiations for a constant field, FP64, one thread per track.
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

namespace {
template <bool MATERIAL, int BLOCK, bool MBF, bool PLAIN>
int go(const kf::FitParams& P, cudaStream_t stream) {
  const char* nm = "kf_forward_kernel (constant field)";
  if (P.geom_in_smem)
    return launch(kf::kf_forward_kernel<kf::FIELD_CONST, MATERIAL, true, 1, BLOCK, MBF, PLAIN>, P, BLOCK,
                  kf::geom_smem_bytes<double>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK), stream, nm);
  // a geometry table too large to stage (> 1024 surfaces): the general instantiation reads it from global memory
  return launch(kf::kf_forward_kernel<kf::FIELD_CONST, MATERIAL, false, 1, KF_FWD_BLOCK_SMALL, MBF, false>, P,
                KF_FWD_BLOCK_SMALL, kf::hit_stage_bytes(KF_FWD_BLOCK_SMALL), stream, nm);
}
template <bool MATERIAL, bool MBF>
int pick(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.big) return c.plain ? go<MATERIAL, KF_FWD_BLOCK, MBF, true>(P, stream) : go<MATERIAL, KF_FWD_BLOCK, MBF, false>(P, stream);
  return c.plain ? go<MATERIAL, KF_FWD_BLOCK_SMALL, MBF, true>(P, stream) : go<MATERIAL, KF_FWD_BLOCK_SMALL, MBF, false>(P, stream);
}
}  // namespace

int launch_forward_const(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.mbf) return c.material ? pick<true, true>(P, c, stream) : pick<false, true>(P, c, stream);
  return c.material ? pick<true, false>(P, c, stream) : pick<false, false>(P, c, stream);
}

}  // namespace kfh
