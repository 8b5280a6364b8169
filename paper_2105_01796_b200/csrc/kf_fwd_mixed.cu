// kf_fwd_mixed.cu -- kf_forward_kernel instantiations of the MIXED-precision path (kf_options.precision; PAPER.md:160-164,
// 272): float operands and records, one thread per track, geometry in shared memory (validate() refuses tables too
// large to stage).
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

namespace {
template <int FIELD, bool MATERIAL, int BLOCK, bool PLAIN>
int go(const kf::FitParams& P, cudaStream_t stream) {
  const size_t smem = kf::geom_smem_bytes<float>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK);
  // grid field: the table is gathered through L1 -- leave it all the SM's memory the resident CTAs do not use
  // (224-236 registers: 256 threads per SM)
  const int pct = FIELD == kf::FIELD_GRID3 ? carveout_for(smem, 256 / BLOCK) : -1;
  return launch(kf::kf_forward_kernel<FIELD, MATERIAL, true, 1, BLOCK, false, PLAIN, float>, P, BLOCK, smem, stream,
                "kf_forward_kernel (mixed precision)", 1, pct);
}
template <int FIELD, bool MATERIAL>
int pick(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.big) return c.plain ? go<FIELD, MATERIAL, KF_FWD_BLOCK, true>(P, stream) : go<FIELD, MATERIAL, KF_FWD_BLOCK, false>(P, stream);
  return c.plain ? go<FIELD, MATERIAL, KF_FWD_BLOCK_SMALL, true>(P, stream) : go<FIELD, MATERIAL, KF_FWD_BLOCK_SMALL, false>(P, stream);
}
}  // namespace

int launch_forward_mixed(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (c.grid3) return c.material ? pick<kf::FIELD_GRID3, true>(P, c, stream) : pick<kf::FIELD_GRID3, false>(P, c, stream);
  return c.material ? pick<kf::FIELD_CONST, true>(P, c, stream) : pick<kf::FIELD_CONST, false>(P, c, stream);
}

}  // namespace kfh
