// kf_fwd_general.cu -- kf_forward_kernel instantiations of the general path (MODE 1: surfaces of any kind, planes,
// cylinders and discs, kf_geometry.surface_kinds; MODE 2: the same with the field-gradient terms of the step Jacobian,
// kf_options.field_gradient): FP64, one thread per track, RTS records, geometry in shared memory.
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

namespace {
template <int FIELD, bool MATERIAL, int MODE>
int go(const kf::FitParams& P, cudaStream_t stream) {
  constexpr int BLOCK = KF_FWD_BLOCK_SMALL;
  return launch(kf::kf_forward_kernel<FIELD, MATERIAL, true, 1, BLOCK, false, false, double, MODE>, P, BLOCK,
                kf::geom_smem_bytes<double>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK), stream,
                MODE == 2 ? "kf_forward_kernel (general surfaces, field-gradient terms)" : "kf_forward_kernel (general surfaces)");
}
}  // namespace

int launch_forward_general(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.mode == 2) return c.material ? go<kf::FIELD_GRID3, true, 2>(P, stream) : go<kf::FIELD_GRID3, false, 2>(P, stream);
  if (c.grid3) return c.material ? go<kf::FIELD_GRID3, true, 1>(P, stream) : go<kf::FIELD_GRID3, false, 1>(P, stream);
  return c.material ? go<kf::FIELD_CONST, true, 1>(P, stream) : go<kf::FIELD_CONST, false, 1>(P, stream);
}

}  // namespace kfh
