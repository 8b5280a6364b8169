// kf_host.h -- host-side glue shared by the translation units of libkf_fit.so (internal; the C ABI is include/kf_fit.h).
//
// The library is built from several .cu files compiled side by side (build.py): kf_fit.cu holds the C ABI and every
// host decision (validation, workspace layout, which kernel a call takes); each of the others instantiates one family
// of kernels and exposes it through ONE plain launcher declared here, so that no kernel template crosses a
// translation-unit boundary.
#pragma once

#include <cuda_runtime.h>

#include "kf_fit.h"
#include "kf_common.cuh"

namespace kfh {

// per calling thread: text of the last CUDA error, kernels enqueued by the last call
extern thread_local char g_cuda_error[256];
extern thread_local int g_launches;

bool set_cuda_error(cudaError_t e, const char* where);  // true when e is an error (text kept)
// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (device, kernel): raised once, not per launch
bool raise_smem_limit(const void* kernel, size_t smem, const char* name);
// cudaFuncAttributePreferredSharedMemoryCarveout (per cent of the SM's 256 KB unified L1 / shared memory), set once per
// (device, kernel): a kernel that gathers from a table through L1 asks for no more shared memory than its CTAs use
bool prefer_carveout(const void* kernel, int percent, const char* name);

// one launch over the tracks of P: thread per track (block tracks per CTA) or lanes per track (block / lanes)
template <typename K>
int launch(K kernel, const kf::FitParams& P, int block, size_t smem, cudaStream_t stream, const char* name,
           int lanes_per_track = 1, int carveout_pct = -1) {
  if (smem > 48 * 1024 && !raise_smem_limit(reinterpret_cast<const void*>(kernel), smem, name)) return KF_ERR_CUDA;
  if (carveout_pct >= 0 && !prefer_carveout(reinterpret_cast<const void*>(kernel), carveout_pct, name)) return KF_ERR_CUDA;
  const unsigned grid = (unsigned)((P.N * lanes_per_track + block - 1) / block);
  kernel<<<grid, block, smem, stream>>>(P);
  if (set_cuda_error(cudaGetLastError(), name)) return KF_ERR_CUDA;
  g_launches++;
  return KF_OK;
}

// carve-out (per cent of the SM's 256 KB) that `ctas` resident CTAs of `smem` dynamic bytes (+ 1 KB each reserved by the
// system) need: what the kernels that gather the field table through L1 ask for, leaving the rest to L1
inline int carveout_for(size_t smem, int ctas) {
  const size_t need = (size_t)ctas * (smem + 1024);
  const size_t pct = (need * 100 + 256 * 1024 - 1) / (256 * 1024);
  return (int)(pct > 100 ? 100 : pct);
}

// which forward-kernel instantiation a call takes (decided in kf_fit.cu: enqueue_fit)
struct ForwardChoice {
  bool grid3;     // field kind
  bool material;
  bool big;       // KF_FWD_BLOCK threads per CTA instead of KF_FWD_BLOCK_SMALL
  bool plain;     // default stepping, per-surface resolutions, no per-leg PRED/FILT states, no RKN estimate
  bool mbf;       // Bryson-Frazier records
  bool staged;    // grid field with a box of the table in shared memory (FIELD_GRID3S; P.field.box_* set)
  int mode;       // 0 planes only, gradient neglected; 1 surfaces of any kind; 2 any kind + field-gradient terms
};

// kf_fwd_const.cu / kf_fwd_grid.cu: FP64, one thread per track
int launch_forward_const(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream);
int launch_forward_grid(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream);
// kf_fwd_staged.cu: grid field with the staged box, FP64 and MIXED, one thread per track.  smem_box = bytes of the box
int launch_forward_staged(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream);
// threads per CTA the staged kernels take for a box of `box_bytes` (two 128-thread CTAs per SM while two boxes fit)
int staged_block(size_t box_bytes);
// kf_fwd_general.cu: surfaces of any kind and / or the field-gradient terms (c.mode 1, 2), FP64, one thread per track
int launch_forward_general(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream);
// kf_fwd_lanes.cu: FP64, 8 lanes per track
int launch_forward_lanes(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream);
// kf_fwd_mixed.cu: float operands and records (kf_options.precision MIXED)
int launch_forward_mixed(const kf::FitParams& P, const ForwardChoice& c, cudaStream_t stream);

// kf_bwd.cu: the backward pass that matches the records (RTS thread/lanes, FP64/MIXED, Bryson-Frazier), the length
// sort, the perigee extrapolation, the DFMA probe
struct PerigeeLine {
  double c[3], a[3];
  double* params;  // [6][N] or nullptr
  double* cov;     // [21][N]
};
int launch_backward(const kf::FitParams& P, bool lanes, cudaStream_t stream);
int launch_length_sort(const kf::FitParams& P, int* perm, int* bins, int force, cudaStream_t stream);
// any_kind: the geometry table may hold cylinders / discs (kf_geometry.surface_kinds > 1); false: entry [18] is not read
int launch_perigee(const kf::FitParams& P, const PerigeeLine& line, bool grid3, bool any_kind, cudaStream_t stream);
double probe_fp64_tflops(int iters, cudaStream_t stream);

}  // namespace kfh
