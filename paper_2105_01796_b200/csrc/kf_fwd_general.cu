// kf_fwd_general.cu -- kf_forward_kernel instantiations of the general path (MODE 1: surfaces of any kind, planes,
// cylinders and discs, kf_geometry.surface_kinds: the hot path's steps with the surfaces' own charts; MODE 2: any kind with
// the field-gradient terms of the step Jacobian, kf_options.field_gradient): FP64, one thread per track, RTS records,
// geometry in shared memory.
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

namespace {
template <int FIELD, bool MATERIAL, int MODE, int BLOCK, bool PLAIN, typename R = double>
int go(const kf::FitParams& P, cudaStream_t stream) {
  const size_t smem = kf::geom_smem_bytes<R>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK) +
                      (FIELD == kf::FIELD_GRID3 && MODE == 1 && sizeof(R) == 8 ? kf::cov_park_bytes<double>(BLOCK) : 0);
  const int pct = FIELD == kf::FIELD_GRID3 ? carveout_for(smem, 256 / BLOCK) : -1;   // grid field: the rest of the SM to L1
  return launch(kf::kf_forward_kernel<FIELD, MATERIAL, true, 1, BLOCK, false, PLAIN, R, MODE>, P, BLOCK, smem, stream,
                MODE == 2 ? "kf_forward_kernel (general surfaces, field-gradient terms)" : "kf_forward_kernel (general surfaces)",
                1, pct);
}
// MODE 1 follows the plane-only kernels' choices: 256-thread CTAs for large constant-field batches, PLAIN when the call
// asks for nothing optional
template <int FIELD, bool MATERIAL>
int pick1(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (P.mixed)   // MIXED precision (float operands and records): the 128-thread CTA, the general instantiation
    return go<FIELD, MATERIAL, 1, KF_FWD_BLOCK_SMALL, false, float>(P, stream);
  if (FIELD == kf::FIELD_CONST && c.big)
    return c.plain ? go<FIELD, MATERIAL, 1, KF_FWD_BLOCK, true>(P, stream) : go<FIELD, MATERIAL, 1, KF_FWD_BLOCK, false>(P, stream);
  return c.plain ? go<FIELD, MATERIAL, 1, KF_FWD_BLOCK_SMALL, true>(P, stream) : go<FIELD, MATERIAL, 1, KF_FWD_BLOCK_SMALL, false>(P, stream);
}
}  // namespace

int launch_forward_general(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.mode == 2)
    return c.material ? go<kf::FIELD_GRID3, true, 2, KF_FWD_BLOCK_SMALL, false>(P, stream)
                      : go<kf::FIELD_GRID3, false, 2, KF_FWD_BLOCK_SMALL, false>(P, stream);
  if (c.grid3) return c.material ? pick1<kf::FIELD_GRID3, true>(P, c, stream) : pick1<kf::FIELD_GRID3, false>(P, c, stream);
  return c.material ? pick1<kf::FIELD_CONST, true>(P, c, stream) : pick1<kf::FIELD_CONST, false>(P, c, stream);
}

}  // namespace kfh
