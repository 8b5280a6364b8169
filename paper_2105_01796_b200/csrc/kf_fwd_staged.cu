// kf_fwd_staged.cu -- kf_forward_kernel instantiations for a grid field with a box of the table staged in shared
// memory (FIELD_GRID3S; kf_field.stage_*), FP64 and MIXED precision, one thread per track, RTS records.
// Dynamic shared memory: [geometry table][hit staging][box: box_n[0] x box_n[1] x box_n[2] x 3 values of type R].
#include "kf_host.h"
#include "kf_forward.cuh"

namespace kfh {

// two CTAs of KF_FWD_BLOCK_SMALL threads per SM while two boxes (+ tables) fit in the SM's shared memory, else one of
// KF_FWD_BLOCK threads: the same eight warps per SM the 255-register FP64 kernel has without the box
int staged_block(size_t box_bytes) { return box_bytes <= 100 * 1024 ? KF_FWD_BLOCK_SMALL : KF_FWD_BLOCK; }

namespace {
template <typename R, bool MATERIAL, int BLOCK, bool PLAIN>
int go(const kf::FitParams& P, size_t box_bytes, cudaStream_t stream) {
  return launch(kf::kf_forward_kernel<kf::FIELD_GRID3S, MATERIAL, true, 1, BLOCK, false, PLAIN, R>, P, BLOCK,
                kf::geom_smem_bytes<R>(P.n_surfaces) + kf::hit_stage_bytes(BLOCK) + box_bytes, stream,
                "kf_forward_kernel (grid field, staged box)");
}
template <typename R, bool MATERIAL>
int pick(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  const int* bn = P.mixed ? P.field_f.box_n : P.field.box_n;
  const size_t box_bytes = ((size_t)bn[0] * bn[1] * bn[2] * 3 * sizeof(R) + 15) / 16 * 16;
  if (staged_block(box_bytes) == KF_FWD_BLOCK)
    return c.plain ? go<R, MATERIAL, KF_FWD_BLOCK, true>(P, box_bytes, stream) : go<R, MATERIAL, KF_FWD_BLOCK, false>(P, box_bytes, stream);
  return c.plain ? go<R, MATERIAL, KF_FWD_BLOCK_SMALL, true>(P, box_bytes, stream)
                 : go<R, MATERIAL, KF_FWD_BLOCK_SMALL, false>(P, box_bytes, stream);
}
}  // namespace

int launch_forward_staged(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream) {
  if (P.mixed) return c.material ? pick<float, true>(P, c, stream) : pick<float, false>(P, c, stream);
  return c.material ? pick<double, true>(P, c, stream) : pick<double, false>(P, c, stream);
}

}  // namespace kfh
