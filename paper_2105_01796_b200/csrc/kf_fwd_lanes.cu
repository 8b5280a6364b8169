// kf_fwd_lanes.cu -- kf_forward_kernel instantiations of the lanes-per-track variant (8 lanes fit one track), FP64.
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

namespace {
template <int FIELD, bool MATERIAL>
int go(const kf::FitParams& P, cudaStream_t stream) {
  constexpr int BLOCK = KF_FWD_BLOCK_SMALL;
  const char* nm = "kf_forward_kernel (lanes per track)";
  if (P.geom_in_smem)
    return launch(kf::kf_forward_kernel<FIELD, MATERIAL, true, kf::kLanes, BLOCK, false, false>, P, BLOCK,
                  kf::geom_smem_bytes<double>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK), stream, nm, kf::kLanes);
  return launch(kf::kf_forward_kernel<FIELD, MATERIAL, false, kf::kLanes, BLOCK, false, false>, P, BLOCK,
                kf::hit_stage_bytes(BLOCK), stream, nm, kf::kLanes);
}
}  // namespace

int launch_forward_lanes(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.grid3) return c.material ? go<kf::FIELD_GRID3, true>(P, stream) : go<kf::FIELD_GRID3, false>(P, stream);
  return c.material ? go<kf::FIELD_CONST, true>(P, stream) : go<kf::FIELD_CONST, false>(P, stream);
}

}  // namespace kfh
