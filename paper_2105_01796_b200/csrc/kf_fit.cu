// kf_fit.cu -- host side of libkf_fit.so: the C ABI declared in include/kf_fit.h.
//
// Validates the descriptors, lays out the workspace, decides which kernel family a call takes and enqueues it on the
// caller's stream through the launchers of kf_host.h (one translation unit per family: kf_fwd_*.cu, kf_bwd.cu).  No allocation, no synchronisation, no global state
// (apart from thread-local error text / launch counter).  There is no CPU fallback: every compute
// entry point ends in a kernel launch and reports KF_ERR_CUDA if that fails.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "kf_fit.h"
#include "kf_host.h"

namespace kfh {
thread_local char g_cuda_error[256] = "";
thread_local int g_launches = 0;

bool set_cuda_error(cudaError_t e, const char* where) {
  if (e == cudaSuccess) return false;
  snprintf(g_cuda_error, sizeof(g_cuda_error), "%s: %s", where, cudaGetErrorString(e));
  return true;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (device, kernel): set it the first time a kernel
// asks for more than 48 KB on a device (or for more than it asked before), not on every launch
bool raise_smem_limit(const void* kernel, size_t smem, const char* name) {
  struct Entry { const void* fn; int dev; size_t bytes; };
  static std::mutex mu;
  static std::vector<Entry> seen;
  int dev = 0;
  if (set_cuda_error(cudaGetDevice(&dev), name)) return false;
  std::lock_guard<std::mutex> lock(mu);
  for (Entry& e : seen)
    if (e.fn == kernel && e.dev == dev) {
      if (e.bytes >= smem) return true;
      if (set_cuda_error(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), name)) return false;
      e.bytes = smem;
      return true;
    }
  if (set_cuda_error(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), name)) return false;
  seen.push_back(Entry{kernel, dev, smem});
  return true;
}
bool prefer_carveout(const void* kernel, int percent, const char* name) {
  struct Entry { const void* fn; int dev; int pct; };
  static std::mutex mu;
  static std::vector<Entry> seen;
  int dev = 0;
  if (set_cuda_error(cudaGetDevice(&dev), name)) return false;
  std::lock_guard<std::mutex> lock(mu);
  for (Entry& e : seen)
    if (e.fn == kernel && e.dev == dev) {
      if (e.pct == percent) return true;
      if (set_cuda_error(cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, percent), name)) return false;
      e.pct = percent;
      return true;
    }
  if (set_cuda_error(cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, percent), name)) return false;
  seen.push_back(Entry{kernel, dev, percent});
  return true;
}
}  // namespace kfh

namespace {

using kfh::g_cuda_error;
using kfh::g_launches;
using kfh::set_cuda_error;

// batches of more tracks than this take the 256-thread forward CTA (148 SMs x 2 CTAs x 128 threads = one wave)
constexpr long long KF_FWD_BIG_MIN_TRACKS = 148LL * 2 * 128;

thread_local cudaEvent_t g_stage_events[3] = {nullptr, nullptr, nullptr};
thread_local bool g_stage_events_on = false;

inline void record_stage(int k, cudaStream_t stream) {
  if (g_stage_events_on && g_stage_events[k]) cudaEventRecord(g_stage_events[k], stream);
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Workspace: tile-major RTS records and the per-slot leg counts (both only
// when smoothing), then the length sort's slot -> track permutation and its bin counters (one set of
// kSortBins counters per 128 tracks, so that every pipeline chunk has its own).
// pipeline chunks are whole multiples of this many tracks (two record tiles); one set of sort counters per unit
constexpr int kChunkTracks = 128;
static_assert(kChunkTracks % KF_TILE == 0, "a chunk covers whole record tiles");

struct WorkspaceLayout {
  size_t rec_off, nleg_off, perm_off, bins_off, total;
  size_t rec_total;   // bytes up to the end of the leg counts: what the fit cannot run without
  size_t tile_stride;
  long long n_tiles;
};

WorkspaceLayout workspace_layout(long long N, int n_legs_max, int smooth, int mbf = 0, int mixed = 0) {
  WorkspaceLayout w{};
  w.n_tiles = N > 0 ? (N + KF_TILE - 1) / KF_TILE : 0;
  if (N <= 0 || n_legs_max <= 0) return w;
  size_t off = 0;
  if (smooth) {
    w.rec_off = off;
    // RTS: Lmax tile-legs of kLegBytes; Bryson-Frazier: Lmax tile-legs of kMbfLegBytes + the first-leg block
    w.tile_stride = mbf ? (size_t)n_legs_max * kf::kMbfLegBytes + (size_t)kf::kMbfFirstDoubles * KF_TILE * sizeof(double)
                        : (size_t)n_legs_max * (mixed ? kf::leg_bytes<float>() : kf::leg_bytes<double>());
    off += align_up((size_t)w.n_tiles * w.tile_stride, 256);
    w.nleg_off = off;
    off += align_up((size_t)w.n_tiles * KF_TILE * sizeof(int), 256);
  }
  w.rec_total = off;
  w.perm_off = off;
  off += align_up((size_t)w.n_tiles * KF_TILE * sizeof(int), 256);
  w.bins_off = off;
  off += align_up((size_t)((N + kChunkTracks - 1) / kChunkTracks) * kf::kSortBins * sizeof(int), 256);
  w.total = off;
  return w;
}

// where the length sort of a launch keeps its permutation and counters; perm == nullptr: no sort
struct SortPlan {
  int* perm;
  int* bins;
  int force;  // KF_SORT_ON: sort even when the lengths hardly differ
};

int validate(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge, const kf_field* fl,
             const kf_options* op, const kf_outputs* out) {
  if (!tr || !ms || !ge || !fl || !op || !out) return KF_ERR_ARG;
  if (tr->n_tracks < 0 || ms->n_meas < 0 || ms->n_meas > 2147483647LL) return KF_ERR_ARG;
  if (ge->n_surfaces < 1 || !ge->surfaces) return KF_ERR_ARG;
  if (tr->start_surface < 0 || tr->start_surface >= ge->n_surfaces) return KF_ERR_ARG;
  if (tr->n_tracks > 0) {
    if (!tr->params || !tr->cov || !ms->offsets) return KF_ERR_ARG;
    if (ms->n_meas > 0 && (!ms->surf_idx || !ms->loc)) return KF_ERR_ARG;
    if (ms->cov01 && !ms->var) return KF_ERR_ARG;
    if (!out->first_params || !out->first_cov || !out->last_params || !out->last_cov || !out->chi2 ||
        !out->ndf || !out->status || !out->n_used || !out->n_outliers || !out->n_holes)
      return KF_ERR_ARG;
  }
  if (fl->kind == KF_FIELD_GRID3) {
    if (!fl->grid) return KF_ERR_ARG;
    for (int a = 0; a < 3; ++a)
      if (fl->n[a] < 2 || !(fl->spacing[a] > 0.0)) return KF_ERR_ARG;
  } else if (fl->kind != KF_FIELD_CONST) {
    return KF_ERR_ARG;
  }
  if (op->n_corr_steps < 0 || op->n_corr_steps > 8) return KF_ERR_ARG;
  if (!(op->mass_gev > 0.0) || !(op->cov_inflation > 0.0)) return KF_ERR_ARG;
  if (op->output_states & ~7) return KF_ERR_ARG;
  if (op->material && !(ge->mat_A > 0.0 && ge->mat_Z > 0.0 && ge->mat_rho > 0.0 && ge->mat_I_eV > 0.0))
    return KF_ERR_ARG;
  for (int b = 0; b < 3; ++b)
    if ((op->output_states >> b) & 1)
      if (tr->n_tracks > 0 && (!out->state_params[b] || !out->state_cov[b])) return KF_ERR_ARG;
  if ((op->output_states & KF_STATES_SMOOTH) && !op->smooth) return KF_ERR_UNSUPPORTED;
  if ((out->perigee_params != nullptr) != (out->perigee_cov != nullptr)) return KF_ERR_ARG;
  if (out->perigee_params) {
    const double* a = op->perigee_axis;
    const double n2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2];
    if (!(std::fabs(n2 - 1.0) < 1e-9)) return KF_ERR_ARG;
  }
  if (op->length_sort < KF_SORT_AUTO || op->length_sort > KF_SORT_ON) return KF_ERR_ARG;
  if (op->smoother != KF_SMOOTHER_RTS && op->smoother != KF_SMOOTHER_BRYSON_FRAZIER) return KF_ERR_ARG;
  if (op->smooth && op->smoother == KF_SMOOTHER_BRYSON_FRAZIER &&
      ((op->output_states & KF_STATES_SMOOTH) || op->variant == KF_VARIANT_LANES_PER_TRACK))
    return KF_ERR_UNSUPPORTED;
  if (op->precision != KF_PRECISION_FP64 && op->precision != KF_PRECISION_MIXED) return KF_ERR_ARG;
  if (op->precision == KF_PRECISION_MIXED &&
      (op->variant == KF_VARIANT_LANES_PER_TRACK || (op->smooth && op->smoother == KF_SMOOTHER_BRYSON_FRAZIER) ||
       ge->n_surfaces > 1024))
    return KF_ERR_UNSUPPORTED;
  if (op->field_gradient != 0 && op->field_gradient != 1) return KF_ERR_ARG;
  if (ge->surface_kinds < 0 || ge->surface_kinds > 7) return KF_ERR_ARG;
  // the general kernels (surfaces of any kind, field-gradient terms): thread per track, RTS, staged geometry; the
  // field-gradient terms in FP64 only
  if (ge->surface_kinds > 1 || (op->field_gradient && fl->kind == KF_FIELD_GRID3))
    if (op->variant == KF_VARIANT_LANES_PER_TRACK || (op->smooth && op->smoother == KF_SMOOTHER_BRYSON_FRAZIER) ||
        ge->n_surfaces > 1024 ||
        (op->precision != KF_PRECISION_FP64 && op->field_gradient && fl->kind == KF_FIELD_GRID3))
      return KF_ERR_UNSUPPORTED;
  if (op->variant != KF_VARIANT_AUTO && op->variant != KF_VARIANT_THREAD_PER_TRACK &&
      op->variant != KF_VARIANT_LANES_PER_TRACK)
    return KF_ERR_ARG;
  return KF_OK;
}

}  // namespace

extern "C" {

void kf_default_options(kf_options* opt) {
  if (!opt) return;
  memset(opt, 0, sizeof(*opt));
  opt->smooth = 1;
  opt->material = 0;
  opt->outlier_chi2 = 0.0;
  opt->n_corr_steps = 2;
  opt->max_step_mm = INFINITY;
  opt->mass_gev = 0.1056583755;
  opt->cov_inflation = 1.0;
  opt->output_states = 0;
  opt->variant = KF_VARIANT_AUTO;
  opt->perigee_axis[2] = 1.0;
  opt->length_sort = KF_SORT_AUTO;
  opt->smoother = KF_SMOOTHER_RTS;
  opt->precision = KF_PRECISION_FP64;
}

size_t kf_workspace_bytes(int64_t n_tracks, int32_t n_legs_max, const kf_options* opt) {
  const int smooth = opt ? opt->smooth : 1;
  const int mbf = smooth && opt && opt->smoother == KF_SMOOTHER_BRYSON_FRAZIER;
  const int mixed = opt && opt->precision == KF_PRECISION_MIXED;
  return workspace_layout(n_tracks, n_legs_max, smooth, mbf, mixed).total;
}

int kf_last_launch_count(void) { return g_launches; }

void kf_set_stage_events(void* const* events3) {
  g_stage_events_on = events3 != nullptr;
  for (int k = 0; k < 3; ++k) g_stage_events[k] = events3 ? static_cast<cudaEvent_t>(events3[k]) : nullptr;
}
const char* kf_last_cuda_error(void) { return g_cuda_error; }
int kf_version(void) { return KF_VERSION; }

const char* kf_status_string(int rc) {
  switch (rc) {
    case KF_OK: return "ok";
    case KF_ERR_ARG: return "null or ill-formed descriptor";
    case KF_ERR_UNSUPPORTED: return "unsupported option combination";
    case KF_ERR_WORKSPACE: return "workspace too small";
    case KF_ERR_CUDA: return "CUDA error (see kf_last_cuda_error)";
    case KF_ERR_STATIC_LIMIT:
      return "batch needs more scratch than the 64 MiB static workspace of kf_fit_batch_static holds "
             "(kf_workspace_bytes > KF_STATIC_WORKSPACE_BYTES): split the batch or use kf_fit_batch with a workspace";
    default: return "unknown return code";
  }
}

}  // extern "C"

namespace {

// Kernel parameter block of the whole batch (host-side descriptor -> device-side view).
int build_params(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge, const kf_field* fl,
                 const kf_options* op, const kf_outputs* out, void* workspace, size_t workspace_bytes,
                 kf::FitParams& P, SortPlan& sort) {
  const long long N = tr->n_tracks;
  const int Lmax = ge->n_surfaces - 1 - tr->start_surface;
  const int mbf = op->smooth && op->smoother == KF_SMOOTHER_BRYSON_FRAZIER;
  const int mixed = op->precision == KF_PRECISION_MIXED;
  const WorkspaceLayout w = workspace_layout(N, Lmax, op->smooth, mbf, mixed);
  if (w.rec_total > 0 && (!workspace || workspace_bytes < w.rec_total)) return KF_ERR_WORKSPACE;
  // the sort's arrays come after the records: a workspace sized by kf_workspace_bytes always holds them; a
  // shorter one (records only) runs unsorted under AUTO and is refused under ON
  const bool sort_room = w.total > 0 && workspace && workspace_bytes >= w.total;
  sort = SortPlan{nullptr, nullptr, 0};
  if (op->length_sort == KF_SORT_ON && !sort_room && w.total > 0) return KF_ERR_WORKSPACE;
  if (op->length_sort != KF_SORT_OFF && sort_room) {
    char* base = static_cast<char*>(workspace);
    sort.perm = reinterpret_cast<int*>(base + w.perm_off);
    sort.bins = reinterpret_cast<int*>(base + w.bins_off);
  }

  P = kf::FitParams{};
  P.N = N; P.M = ms->n_meas; P.ldn = N; P.ldm = ms->n_meas;
  P.params = tr->params; P.cov = tr->cov; P.start = tr->start_surface;
  P.offsets = ms->offsets; P.surf_idx = ms->surf_idx; P.loc = ms->loc; P.var = ms->var; P.cov01 = ms->cov01;
  P.n_surfaces = ge->n_surfaces; P.geom = ge->surfaces;
  P.geom_in_smem = ge->n_surfaces <= 1024 ? 1 : 0;
  if (fl->kind == KF_FIELD_CONST) {
    for (int a = 0; a < 3; ++a) P.field.b[a] = fl->b[a] * 2.99792458e-4;  // tesla -> GeV/(e mm)
    P.field.b2 = P.field.b[0] * P.field.b[0] + P.field.b[1] * P.field.b[1] + P.field.b[2] * P.field.b[2];
  } else {
    for (int a = 0; a < 3; ++a) {
      P.field.n[a] = fl->n[a];
      P.field.origin[a] = fl->origin[a];
      P.field.spacing[a] = fl->spacing[a];
      P.field.inv_spacing[a] = 1.0 / fl->spacing[a];
    }
    P.field.grid = fl->grid;
    // the staging hint, when well-formed (else ignored: results do not depend on it)
    bool ok = true;
    for (int a = 0; a < 3; ++a)
      ok = ok && fl->stage_lo[a] >= 0 && fl->stage_n[a] >= 2 && fl->stage_lo[a] + fl->stage_n[a] <= fl->n[a];
    if (ok && (size_t)fl->stage_n[0] * fl->stage_n[1] * fl->stage_n[2] * 3 * sizeof(double) <= KF_FIELD_STAGE_MAX_BYTES)
      for (int a = 0; a < 3; ++a) { P.field.box_lo[a] = fl->stage_lo[a]; P.field.box_n[a] = fl->stage_n[a]; }
  }
  P.mat.mass = op->mass_gev;
  P.mat.inv_mass = 1.0 / op->mass_gev;
  P.mat.rme = 0.51099895e-3 / op->mass_gev;
  if (op->material) {
    P.mat.ZA = ge->mat_Z / ge->mat_A;
    P.mat.rho = ge->mat_rho;
    P.mat.I_gev = ge->mat_I_eV * 1e-9;
    P.mat.inv_I2 = 1.0 / (P.mat.I_gev * P.mat.I_gev);
    P.mat.log_hwp_I = log(28.816e-9 * sqrt(ge->mat_rho * P.mat.ZA) / P.mat.I_gev);
  }
  // the same two descriptors rounded to float (the MIXED path's kernels read these)
  for (int a = 0; a < 3; ++a) {
    P.field_f.b[a] = (float)P.field.b[a];
    P.field_f.inv_spacing[a] = (float)P.field.inv_spacing[a];
    P.field_f.n[a] = P.field.n[a];
    P.field_f.origin[a] = (float)P.field.origin[a];
    P.field_f.spacing[a] = (float)P.field.spacing[a];
    P.field_f.box_lo[a] = P.field.box_lo[a];
    P.field_f.box_n[a] = P.field.box_n[a];
  }
  P.field_f.b2 = P.field_f.b[0] * P.field_f.b[0] + P.field_f.b[1] * P.field_f.b[1] + P.field_f.b[2] * P.field_f.b[2];
  P.field_f.grid = P.field.grid;
  P.mat_f.mass = (float)P.mat.mass; P.mat_f.inv_mass = (float)P.mat.inv_mass; P.mat_f.rme = (float)P.mat.rme;
  P.mat_f.inv_I2 = (float)P.mat.inv_I2; P.mat_f.ZA = (float)P.mat.ZA; P.mat_f.rho = (float)P.mat.rho;
  P.mat_f.I_gev = (float)P.mat.I_gev; P.mat_f.log_hwp_I = (float)P.mat.log_hwp_I;
  P.mixed = mixed;
  P.smooth = op->smooth ? 1 : 0;
  P.n_corr = op->n_corr_steps;
  P.output_states = op->output_states;
  P.outlier_chi2 = op->outlier_chi2;
  P.max_step = (op->max_step_mm > 0.0 && std::isfinite(op->max_step_mm)) ? op->max_step_mm : 0.0;
  P.step_tol = (op->step_tolerance_mm > 0.0 && std::isfinite(op->step_tolerance_mm)) ? op->step_tolerance_mm : 0.0;
  P.inflation = op->cov_inflation;
  P.first_params = out->first_params; P.first_cov = out->first_cov;
  P.last_params = out->last_params; P.last_cov = out->last_cov;
  P.chi2 = out->chi2; P.ndf = out->ndf; P.status = out->status;
  P.n_used = out->n_used; P.n_outliers = out->n_outliers; P.n_holes = out->n_holes;
  for (int b = 0; b < 3; ++b) { P.state_params[b] = out->state_params[b]; P.state_cov[b] = out->state_cov[b]; }
  P.hit_chi2 = out->hit_chi2; P.hit_flags = out->hit_flags; P.rk_err_max = out->rk_err_max;
  if (w.rec_total > 0) {
    char* base = static_cast<char*>(workspace);
    P.rec = base + w.rec_off;
    P.leg_stride = mbf ? kf::kMbfLegBytes : (mixed ? kf::leg_bytes<float>() : kf::leg_bytes<double>());
    P.tile_stride = w.tile_stride;
    P.mbf = mbf;
    P.first_off = (size_t)Lmax * kf::kMbfLegBytes;
    P.nleg = reinterpret_cast<int*>(base + w.nleg_off);
  } else {
    P.smooth = 0;  // no legs to smooth (Lmax == 0)
  }
  return KF_OK;
}

// The same block restricted to tracks [t0, t0 + n): every per-track base pointer advances by t0 (t0 is a
// multiple of kChunkTracks, so tiles stay whole); hit arrays keep their absolute indexing through `offsets`.
kf::FitParams sub_range(const kf::FitParams& F, long long t0, long long n) {
  kf::FitParams P = F;
  P.N = n;
  P.params += t0; P.cov += t0; P.offsets += t0;
  P.first_params += t0; P.first_cov += t0; P.last_params += t0; P.last_cov += t0;
  P.chi2 += t0; P.ndf += t0; P.status += t0; P.n_used += t0; P.n_outliers += t0; P.n_holes += t0;
  for (int b = 0; b < 3; ++b) {
    if (P.state_params[b]) P.state_params[b] += t0;
    if (P.state_cov[b]) P.state_cov[b] += t0;
  }
  if (P.rk_err_max) P.rk_err_max += t0;
  if (P.rec) {
    P.rec += (size_t)(t0 / KF_TILE) * P.tile_stride;
    P.nleg += t0;
  }
  return P;
}

// variant: KF_VARIANT_*.  AUTO is the measured choice: 8 lanes
// per track while the batch is so small that every warp of either variant has an SM sub-partition to itself
// (<= KF_AUTO_LANES_MAX_TRACKS: 6-9 % shorter latency), one thread per track above (up to 6.5x the throughput).
//
// sort.perm != nullptr: first the length sort of the range (kf_sort.cuh: zero the bin counters, histogram, scan,
// scatter), then both kernels go through the slot -> track permutation.
int enqueue_fit(const kf::FitParams& P0, const kfh::PerigeeLine& G, bool grid3, bool material, int variant,
                SortPlan sort, cudaStream_t stream, int mode = 0) {
  kf::FitParams P = P0;
  P.perm = nullptr;
  int rc;
  if (sort.perm) {
    rc = kfh::launch_length_sort(P, sort.perm, sort.bins, sort.force, stream);
    if (rc != KF_OK) return rc;
    P.perm = sort.perm;
  }
  const bool lanes = mode == 0 && !P.mbf && !P.mixed && (variant == KF_VARIANT_LANES_PER_TRACK ||
                                            (variant == KF_VARIANT_AUTO && P.N <= KF_AUTO_LANES_MAX_TRACKS));
  record_stage(0, stream);
  kfh::ForwardChoice fc{};
  fc.grid3 = grid3;
  fc.material = material;
  // 256-thread forward CTAs once a batch is more than one wave of 128-thread CTAs at two per SM (CFG2 3.47 -> 3.40 ms;
  // the FP64 grid-field kernel is slower that way, CFG4 5.87 -> 6.11 ms, and always takes the small CTA)
  fc.big = P.N > KF_FWD_BIG_MIN_TRACKS;
  // the plain instantiation: default stepping, per-surface resolutions, no per-leg PRED/FILT states, no RKN estimate
  fc.plain = P.n_corr == 2 && P.max_step == 0.0 && P.step_tol == 0.0 && !P.var && !P.rk_err_max &&
             !(P.output_states & (kf::OUT_PRED | kf::OUT_FILT));
  fc.mbf = P.mbf != 0;
  fc.mode = mode;
  // grid field with the caller's box of the table in shared memory (kf_field.stage_*): thread per track, RTS records,
  // when [geometry][hit slots][box] fit the CTA's shared memory
  if (mode == 0 && grid3 && !lanes && !P.mbf && P.geom_in_smem && P.field.box_n[0] >= 2) {
    const size_t elem = P.mixed ? sizeof(float) : sizeof(double);
    const size_t box = ((size_t)P.field.box_n[0] * P.field.box_n[1] * P.field.box_n[2] * 3 * elem + 15) / 16 * 16;
    const size_t off = (P.mixed ? kf::geom_smem_bytes<float>(P.n_surfaces) : kf::geom_smem_bytes<double>(P.n_surfaces)) +
                       kf::hit_stage_bytes(kfh::staged_block(box));
    if (off + box <= 226 * 1024) {
      fc.staged = true;
      P.field.box_off = P.field_f.box_off = (int)off;
    }
  }
  if (mode != 0) rc = kfh::launch_forward_general(P, fc, stream);
  else if (fc.staged) rc = kfh::launch_forward_staged(P, fc, stream);
  else if (P.mixed) rc = kfh::launch_forward_mixed(P, fc, stream);
  else if (lanes) rc = kfh::launch_forward_lanes(P, fc, stream);
  else if (grid3) rc = kfh::launch_forward_grid(P, fc, stream);
  else rc = kfh::launch_forward_const(P, fc, stream);
  if (rc != KF_OK) return rc;
  record_stage(1, stream);
  if (P.smooth) rc = kfh::launch_backward(P, lanes, stream);
  record_stage(2, stream);
  // fitted parameters on the perigee surface: one more (small) kernel
  // (the perigee kernel reads the chart of the first surface the way the forward kernel did: entry [18] only when the
  // general kernels ran)
  if (rc == KF_OK && G.params) rc = kfh::launch_perigee(P, G, grid3, mode != 0, stream);
  return rc;
}

// which forward path a call takes: 0 = the plane-only kernels; 1 = surfaces of any kind; 2 = + field-gradient terms
int general_mode(const kf_geometry* ge, const kf_field* fl, const kf_options* op) {
  if (op->field_gradient && fl->kind == KF_FIELD_GRID3) return 2;
  return ge->surface_kinds > 1 ? 1 : 0;
}

// Does the range [t0, t0 + n) with n_hits hits get the length sort?  ON: yes.  AUTO: when its hit lists are not
// dense (some track has fewer hits than there are surfaces, so leg counts may differ) and it is large enough for
// the three extra launches not to matter.
SortPlan sort_for_range(const SortPlan& whole, const kf_options* op, long long t0, long long n, long long n_hits,
                        int lmax) {
  SortPlan r{nullptr, nullptr, op->length_sort == KF_SORT_ON ? 1 : 0};
  if (!whole.perm) return r;
  const bool ragged = n_hits != n * (long long)lmax;
  if (op->length_sort == KF_SORT_ON || (op->length_sort == KF_SORT_AUTO && ragged && n >= KF_AUTO_SORT_MIN_TRACKS)) {
    r.perm = whole.perm + t0;
    r.bins = whole.bins + (t0 / kChunkTracks) * kf::kSortBins;
  }
  return r;
}

kfh::PerigeeLine perigee_params(const kf_options* op, const kf_outputs* out, long long t0) {
  kfh::PerigeeLine G{};
  for (int a = 0; a < 3; ++a) { G.c[a] = op->perigee_center[a]; G.a[a] = op->perigee_axis[a]; }
  G.params = out->perigee_params ? out->perigee_params + t0 : nullptr;
  G.cov = out->perigee_cov ? out->perigee_cov + t0 : nullptr;
  return G;
}

}  // namespace

extern "C" {

int kf_fit_batch(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge,
                 const kf_field* fl, const kf_options* op, const kf_outputs* out, void* workspace,
                 size_t workspace_bytes, void* cuda_stream) {
  g_launches = 0;
  int rc = validate(tr, ms, ge, fl, op, out);
  if (rc != KF_OK) return rc;
  if (tr->n_tracks == 0) return KF_OK;
  kf::FitParams P;
  SortPlan sort;
  rc = build_params(tr, ms, ge, fl, op, out, workspace, workspace_bytes, P, sort);
  if (rc != KF_OK) return rc;
  const int lmax = ge->n_surfaces - 1 - tr->start_surface;
  return enqueue_fit(P, perigee_params(op, out, 0), fl->kind == KF_FIELD_GRID3, op->material != 0, op->variant,
                     sort_for_range(sort, op, 0, tr->n_tracks, ms->n_meas, lmax), static_cast<cudaStream_t>(cuda_stream),
                     general_mode(ge, fl, op));
}

// ---- kf_fit_batch_static: the fit for callers that may not allocate (include/kf_fit.h) ----------------------
}  // extern "C"

namespace {

// The workspace of kf_fit_batch_static.  It is part of the library image: each GPU gets its own copy when the module
// of this file is loaded there and keeps it until the process ends.  In HOST code the name below is only a handle
// for cudaGetSymbolAddress -- it is not a device address and must never be handed to a kernel.
static __device__ __align__(256) unsigned char g_static_workspace[KF_STATIC_WORKSPACE_BYTES];

constexpr int kMaxStaticDevices = 64;

// Device address of g_static_workspace on the CURRENT device, looked up once per device and kept.  The look-up is
// the set-up step that the header asks callers to get out of the way before any stream capture.
int static_workspace_on_current_device(void** ptr) {
  static std::mutex mu;
  static void* addr[kMaxStaticDevices] = {};
  int dev = 0;
  if (set_cuda_error(cudaGetDevice(&dev), "kf_fit_batch_static: cudaGetDevice")) return KF_ERR_CUDA;
  if (dev < 0 || dev >= kMaxStaticDevices) {
    snprintf(g_cuda_error, sizeof(g_cuda_error), "kf_fit_batch_static: device ordinal %d beyond the %d supported", dev,
             kMaxStaticDevices);
    return KF_ERR_CUDA;
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    if (set_cuda_error(cudaGetSymbolAddress(&p, g_static_workspace), "kf_fit_batch_static: cudaGetSymbolAddress"))
      return KF_ERR_CUDA;
    if (!p) {
      snprintf(g_cuda_error, sizeof(g_cuda_error), "kf_fit_batch_static: cudaGetSymbolAddress returned a null address");
      return KF_ERR_CUDA;
    }
    addr[dev] = p;
  }
  *ptr = addr[dev];
  return KF_OK;
}

}  // namespace

extern "C" {

int kf_fit_batch_static(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge, const kf_field* fl,
                        const kf_options* op, const kf_outputs* out, void* cuda_stream) {
  g_launches = 0;
  int rc = validate(tr, ms, ge, fl, op, out);
  if (rc != KF_OK) return rc;
  // the size test is host arithmetic and comes before any CUDA call: a batch that does not fit changes nothing
  const int lmax = ge->n_surfaces - 1 - tr->start_surface;
  const size_t need = kf_workspace_bytes(tr->n_tracks, lmax, op);
  if (need > (size_t)KF_STATIC_WORKSPACE_BYTES) return KF_ERR_STATIC_LIMIT;
  void* workspace = nullptr;
  rc = static_workspace_on_current_device(&workspace);  // first call on this device: the one-time address look-up
  if (rc != KF_OK) return rc;
  if (tr->n_tracks == 0) return KF_OK;
  // from here on this is kf_fit_batch with the static array as a full-size workspace.  What must start at zero in
  // it (the length sort's counters) is cleared on the stream by launch_length_sort; the rest of the last call's
  // contents is overwritten by the forward kernel before anything reads it.
  kf::FitParams P;
  SortPlan sort;
  rc = build_params(tr, ms, ge, fl, op, out, workspace, (size_t)KF_STATIC_WORKSPACE_BYTES, P, sort);
  if (rc != KF_OK) return rc;
  return enqueue_fit(P, perigee_params(op, out, 0), fl->kind == KF_FIELD_GRID3, op->material != 0, op->variant,
                     sort_for_range(sort, op, 0, tr->n_tracks, ms->n_meas, lmax), static_cast<cudaStream_t>(cuda_stream),
                     general_mode(ge, fl, op));
}

int kf_field_stage_box(const double* g, int32_t n_surfaces, kf_field* fl) {
  if (!fl) return KF_ERR_ARG;
  for (int a = 0; a < 3; ++a) fl->stage_lo[a] = fl->stage_n[a] = 0;
  if (fl->kind != KF_FIELD_GRID3) return KF_OK;
  if (!g || n_surfaces < 1) return KF_ERR_ARG;
  for (int a = 0; a < 3; ++a)
    if (fl->n[a] < 2 || !(fl->spacing[a] > 0.0)) return KF_ERR_ARG;
  double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int s = 0; s < n_surfaces; ++s) {
    const double* r = g + (size_t)s * KF_GEOM_STRIDE;
    if (!(r[12] > 0.0 && r[13] > 0.0 && std::isfinite(r[12]) && std::isfinite(r[13]))) return KF_OK;  // no acceptance known
    for (int a = 0; a < 3; ++a) {
      const double e = std::fabs(r[3 + a]) * r[12] + std::fabs(r[6 + a]) * r[13];  // extent of the rectangle along axis a
      lo[a] = std::min(lo[a], r[a] - e);
      hi[a] = std::max(hi[a], r[a] + e);
    }
  }
  int32_t blo[3], bn[3];
  for (int a = 0; a < 3; ++a) {
    // cells floor(f) - 1 .. floor(f) + 1 around both ends, clamped like the lookup clamps them
    const double f0 = std::floor((lo[a] - fl->origin[a]) / fl->spacing[a]) - 1.0;
    const double f1 = std::floor((hi[a] - fl->origin[a]) / fl->spacing[a]) + 1.0;
    const int c0 = (int)std::min(std::max(f0, 0.0), (double)(fl->n[a] - 2));
    const int c1 = (int)std::min(std::max(f1, 0.0), (double)(fl->n[a] - 2));
    blo[a] = c0;
    bn[a] = c1 - c0 + 2;  // nodes of cells c0 .. c1
  }
  if ((size_t)bn[0] * bn[1] * bn[2] * 3 * sizeof(double) > KF_FIELD_STAGE_MAX_BYTES) return KF_OK;
  for (int a = 0; a < 3; ++a) { fl->stage_lo[a] = blo[a]; fl->stage_n[a] = bn[a]; }
  return KF_OK;
}

double kf_probe_fp64_tflops(int iters, void* cuda_stream) {
  if (iters <= 0) return (double)KF_ERR_ARG;
  return kfh::probe_fp64_tflops(iters, static_cast<cudaStream_t>(cuda_stream));
}


// ---- end-to-end variant for HOST buffers (pinned per-track blocks, H2D copy,
// kernel, D2H copy) ------------------------------------------------------------------------
namespace {
struct Bump {
  size_t off = 0;
  size_t take(size_t bytes) {
    const size_t o = off;
    off += align_up(bytes, 256);
    return o;
  }
};
struct ArenaLayout {
  size_t params, cov, offsets, surf_idx, loc, var, cov01, geom, grid;
  size_t first_params, first_cov, last_params, last_cov, chi2, ndf, status, n_used, n_outliers, n_holes;
  size_t state_params[3], state_cov[3], hit_chi2, hit_flags, rk_err, perigee_params, perigee_cov, workspace, workspace_bytes, total;
};
ArenaLayout arena_layout(long long N, long long M, int nS, int start, const kf_field* fl, const kf_options* op,
                         int has_var, int has_cov01) {
  ArenaLayout a{};
  Bump b;
  const size_t D = sizeof(double), I = sizeof(int32_t);
  const int Lmax = nS - 1 - start;
  a.params = b.take(6 * N * D);
  a.cov = b.take(21 * N * D);
  a.offsets = b.take((N + 1) * I);
  a.surf_idx = b.take(M * I);
  a.loc = b.take(2 * M * D);
  a.var = has_var ? b.take(2 * M * D) : 0;
  a.cov01 = has_cov01 ? b.take(M * D) : 0;
  a.geom = b.take((size_t)nS * KF_GEOM_STRIDE * D);
  a.grid = 0;
  if (fl && fl->kind == KF_FIELD_GRID3) a.grid = b.take((size_t)fl->n[0] * fl->n[1] * fl->n[2] * 3 * D);
  a.first_params = b.take(6 * N * D);
  a.first_cov = b.take(21 * N * D);
  a.last_params = b.take(6 * N * D);
  a.last_cov = b.take(21 * N * D);
  a.chi2 = b.take(N * D);
  a.ndf = b.take(N * I);
  a.status = b.take(N * I);
  a.n_used = b.take(N * I);
  a.n_outliers = b.take(N * I);
  a.n_holes = b.take(N * I);
  for (int k = 0; k < 3; ++k) {
    const bool on = op && ((op->output_states >> k) & 1);
    a.state_params[k] = on ? b.take((size_t)Lmax * 6 * N * D) : 0;
    a.state_cov[k] = on ? b.take((size_t)Lmax * 21 * N * D) : 0;
  }
  a.hit_chi2 = b.take(M * D);
  a.hit_flags = b.take(M);
  a.rk_err = b.take(N * D);
  a.perigee_params = b.take(6 * N * D);
  a.perigee_cov = b.take(21 * N * D);
  a.workspace_bytes = workspace_layout(N, Lmax, op ? op->smooth : 1,
                                       op && op->smooth && op->smoother == KF_SMOOTHER_BRYSON_FRAZIER,
                                       op && op->precision == KF_PRECISION_MIXED).total;
  a.workspace = b.take(a.workspace_bytes);
  a.total = b.off;
  return a;
}
}  // namespace

size_t kf_host_arena_bytes(int64_t n_tracks, int64_t n_meas, int32_t n_surfaces, int32_t start_surface,
                           const kf_field* field, const kf_options* opt, int has_var, int has_cov01) {
  if (n_tracks < 0 || n_meas < 0 || n_surfaces < 1 || start_surface < 0 || start_surface >= n_surfaces) return 0;
  return arena_layout(n_tracks, n_meas, n_surfaces, start_surface, field, opt, has_var, has_cov01).total;
}

}  // extern "C"

namespace {

// Host-buffer path.  With pipe == nullptr: one chunk on `main` (H2D, forward, RTS, D2H in
// order).  With a pipeline: the tracks are cut into chunks of whole tiles; chunk c runs H2D -> fit -> D2H on
// pipe->streams[c % n_streams], so that the copy engines and the SMs work on different chunks at the same time
// (the paper's multi-stream offload).  Chunks address slices of the same full-size arena arrays.
int host_impl(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge, const kf_field* fl,
              const kf_options* op, const kf_outputs* out, void* device_arena, size_t arena_bytes,
              cudaStream_t main, const kf_pipeline* pipe) {
  g_launches = 0;
  int rc = validate(tr, ms, ge, fl, op, out);
  if (rc != KF_OK) return rc;
  int S = 0;
  if (pipe) {
    S = pipe->n_streams;
    if (S < 1 || S > KF_MAX_STREAMS || pipe->chunk_tracks < 0 || !pipe->events[S]) return KF_ERR_ARG;
    for (int k = 0; k < S; ++k)
      if (!pipe->events[k]) return KF_ERR_ARG;
  }
  const long long N = tr->n_tracks, M = ms->n_meas;
  if (N == 0) return KF_OK;
  const int nS = ge->n_surfaces;
  const ArenaLayout a = arena_layout(N, M, nS, tr->start_surface, fl, op, ms->var != nullptr, ms->cov01 != nullptr);
  if (!device_arena || arena_bytes < a.total) return KF_ERR_WORKSPACE;
  char* base = static_cast<char*>(device_arena);
  const size_t D = sizeof(double), I = sizeof(int32_t);
  const int Lmax = nS - 1 - tr->start_surface;

  // device-side descriptors: the arena's arrays
  kf_tracks_in dtr = *tr;
  dtr.params = reinterpret_cast<const double*>(base + a.params);
  dtr.cov = reinterpret_cast<const double*>(base + a.cov);
  kf_measurements dms = *ms;
  dms.offsets = reinterpret_cast<const int32_t*>(base + a.offsets);
  dms.surf_idx = reinterpret_cast<const int32_t*>(base + a.surf_idx);
  dms.loc = reinterpret_cast<const double*>(base + a.loc);
  dms.var = ms->var ? reinterpret_cast<const double*>(base + a.var) : nullptr;
  dms.cov01 = ms->cov01 ? reinterpret_cast<const double*>(base + a.cov01) : nullptr;
  kf_geometry dge = *ge;
  dge.surfaces = reinterpret_cast<const double*>(base + a.geom);
  kf_field dfl = *fl;
  if (fl->kind == KF_FIELD_GRID3) dfl.grid = reinterpret_cast<const double*>(base + a.grid);
  kf_outputs dout{};
  dout.first_params = reinterpret_cast<double*>(base + a.first_params);
  dout.first_cov = reinterpret_cast<double*>(base + a.first_cov);
  dout.last_params = reinterpret_cast<double*>(base + a.last_params);
  dout.last_cov = reinterpret_cast<double*>(base + a.last_cov);
  dout.chi2 = reinterpret_cast<double*>(base + a.chi2);
  dout.ndf = reinterpret_cast<int32_t*>(base + a.ndf);
  dout.status = reinterpret_cast<uint32_t*>(base + a.status);
  dout.n_used = reinterpret_cast<int32_t*>(base + a.n_used);
  dout.n_outliers = reinterpret_cast<int32_t*>(base + a.n_outliers);
  dout.n_holes = reinterpret_cast<int32_t*>(base + a.n_holes);
  for (int k = 0; k < 3; ++k)
    if ((op->output_states >> k) & 1) {
      dout.state_params[k] = reinterpret_cast<double*>(base + a.state_params[k]);
      dout.state_cov[k] = reinterpret_cast<double*>(base + a.state_cov[k]);
    }
  if (out->hit_chi2) dout.hit_chi2 = reinterpret_cast<double*>(base + a.hit_chi2);
  if (out->hit_flags) dout.hit_flags = reinterpret_cast<uint8_t*>(base + a.hit_flags);
  if (out->rk_err_max) dout.rk_err_max = reinterpret_cast<double*>(base + a.rk_err);
  if (out->perigee_params) {
    dout.perigee_params = reinterpret_cast<double*>(base + a.perigee_params);
    dout.perigee_cov = reinterpret_cast<double*>(base + a.perigee_cov);
  }
  kf::FitParams F;
  SortPlan sort;
  rc = build_params(&dtr, &dms, &dge, &dfl, op, &dout, base + a.workspace, a.workspace_bytes, F, sort);
  if (rc != KF_OK) return rc;

#define KF_TRY(call, what)                                 \
  do {                                                     \
    if (set_cuda_error((call), (what))) return KF_ERR_CUDA; \
  } while (0)
  // `rows` rows of `n` elements of `elem` bytes starting at element e0 of every row; row pitch `ld` elements
  auto h2d = [&](size_t dst_off, const void* src, size_t ld, size_t e0, size_t n, size_t rows, size_t elem,
                 cudaStream_t st) -> cudaError_t {
    if (!src || n == 0 || rows == 0) return cudaSuccess;
    return cudaMemcpy2DAsync(base + dst_off + e0 * elem, ld * elem, static_cast<const char*>(src) + e0 * elem,
                             ld * elem, n * elem, rows, cudaMemcpyHostToDevice, st);
  };
  auto d2h = [&](void* dst, size_t src_off, size_t ld, size_t e0, size_t n, size_t rows, size_t elem,
                 cudaStream_t st) -> cudaError_t {
    if (!dst || n == 0 || rows == 0) return cudaSuccess;
    return cudaMemcpy2DAsync(static_cast<char*>(dst) + e0 * elem, ld * elem, base + src_off + e0 * elem, ld * elem,
                             n * elem, rows, cudaMemcpyDeviceToHost, st);
  };

  // shared global data first, on the caller's stream
  KF_TRY(h2d(a.geom, ge->surfaces, (size_t)nS * KF_GEOM_STRIDE, 0, (size_t)nS * KF_GEOM_STRIDE, 1, D, main), "H2D geometry");
  if (fl->kind == KF_FIELD_GRID3) {
    const size_t g = (size_t)fl->n[0] * fl->n[1] * fl->n[2] * 3;
    KF_TRY(h2d(a.grid, fl->grid, g, 0, g, 1, D, main), "H2D field grid");
  }

  long long chunk = N;
  if (pipe) {
    chunk = pipe->chunk_tracks > 0 ? pipe->chunk_tracks : std::max<long long>(16384, N / (4LL * S));
    chunk = (chunk + kChunkTracks - 1) / kChunkTracks * kChunkTracks;  // whole record tiles
  }
  // every chunk boundary of the HOST offsets array is checked before anything of the chunks is enqueued
  for (long long t0 = 0; t0 < N; t0 += chunk) {
    const long long m0 = ms->offsets[t0], m1 = ms->offsets[std::min(t0 + chunk, N)];
    if (m0 < 0 || m1 < m0 || m1 > M) return KF_ERR_ARG;
  }
  // the whole CSR offsets array goes over once, on the caller's stream, ahead of the fork (chunks share their
  // boundary elements)
  KF_TRY(h2d(a.offsets, ms->offsets, N + 1, 0, N + 1, 1, I, main), "H2D offsets");
  if (pipe) {
    KF_TRY(cudaEventRecord(static_cast<cudaEvent_t>(pipe->events[S]), main), "pipeline fork");
    for (int k = 0; k < S; ++k)
      KF_TRY(cudaStreamWaitEvent(static_cast<cudaStream_t>(pipe->streams[k]), static_cast<cudaEvent_t>(pipe->events[S]), 0),
             "pipeline fork");
  }
  const bool grid3 = fl->kind == KF_FIELD_GRID3;
  int c = 0;
  // From here on an error must not leave the worker streams un-joined: the loop body reports through `rc`, and the
  // join below runs whatever it says (chunks enqueued before the failure still run; see kf_fit.h "Errors").
  auto enqueue_chunk = [&](long long t0, long long n, cudaStream_t st) -> int {
    const long long m0 = ms->offsets[t0], m1 = ms->offsets[t0 + n];  // HOST array in this entry point
    const size_t nm = (size_t)(m1 - m0);
    KF_TRY(h2d(a.params, tr->params, N, t0, n, 6, D, st), "H2D params");
    KF_TRY(h2d(a.cov, tr->cov, N, t0, n, 21, D, st), "H2D cov");
    KF_TRY(h2d(a.surf_idx, ms->surf_idx, M, m0, nm, 1, I, st), "H2D surf_idx");
    KF_TRY(h2d(a.loc, ms->loc, M, m0, nm, 2, D, st), "H2D loc");
    KF_TRY(h2d(a.var, ms->var, M, m0, nm, 2, D, st), "H2D var");
    KF_TRY(h2d(a.cov01, ms->cov01, M, m0, nm, 1, D, st), "H2D cov01");

    const int frc = enqueue_fit(sub_range(F, t0, n), perigee_params(op, &dout, t0), grid3, op->material != 0, op->variant,
                                sort_for_range(sort, op, t0, n, (long long)nm, Lmax), st, general_mode(ge, fl, op));
    if (frc != KF_OK) return frc;

    KF_TRY(d2h(out->first_params, a.first_params, N, t0, n, 6, D, st), "D2H first_params");
    KF_TRY(d2h(out->first_cov, a.first_cov, N, t0, n, 21, D, st), "D2H first_cov");
    KF_TRY(d2h(out->last_params, a.last_params, N, t0, n, 6, D, st), "D2H last_params");
    KF_TRY(d2h(out->last_cov, a.last_cov, N, t0, n, 21, D, st), "D2H last_cov");
    KF_TRY(d2h(out->chi2, a.chi2, N, t0, n, 1, D, st), "D2H chi2");
    KF_TRY(d2h(out->ndf, a.ndf, N, t0, n, 1, I, st), "D2H ndf");
    KF_TRY(d2h(out->status, a.status, N, t0, n, 1, I, st), "D2H status");
    KF_TRY(d2h(out->n_used, a.n_used, N, t0, n, 1, I, st), "D2H n_used");
    KF_TRY(d2h(out->n_outliers, a.n_outliers, N, t0, n, 1, I, st), "D2H n_outliers");
    KF_TRY(d2h(out->n_holes, a.n_holes, N, t0, n, 1, I, st), "D2H n_holes");
    for (int k = 0; k < 3; ++k)
      if ((op->output_states >> k) & 1) {
        KF_TRY(d2h(out->state_params[k], a.state_params[k], N, t0, n, (size_t)Lmax * 6, D, st), "D2H state_params");
        KF_TRY(d2h(out->state_cov[k], a.state_cov[k], N, t0, n, (size_t)Lmax * 21, D, st), "D2H state_cov");
      }
    KF_TRY(d2h(out->hit_chi2, a.hit_chi2, M, m0, nm, 1, D, st), "D2H hit_chi2");
    KF_TRY(d2h(out->hit_flags, a.hit_flags, M, m0, nm, 1, 1, st), "D2H hit_flags");
    KF_TRY(d2h(out->rk_err_max, a.rk_err, N, t0, n, 1, D, st), "D2H rk_err_max");
    KF_TRY(d2h(out->perigee_params, a.perigee_params, N, t0, n, 6, D, st), "D2H perigee_params");
    KF_TRY(d2h(out->perigee_cov, a.perigee_cov, N, t0, n, 21, D, st), "D2H perigee_cov");
    return KF_OK;
  };
  rc = KF_OK;
  for (long long t0 = 0; t0 < N && rc == KF_OK; t0 += chunk, ++c)
    rc = enqueue_chunk(t0, std::min(chunk, N - t0), pipe ? static_cast<cudaStream_t>(pipe->streams[c % S]) : main);
  if (pipe) {  // join: the caller's stream continues after every chunk stream, also when a chunk failed to enqueue
    for (int k = 0; k < S && k < c; ++k) {
      const bool bad = set_cuda_error(cudaEventRecord(static_cast<cudaEvent_t>(pipe->events[k]),
                                                      static_cast<cudaStream_t>(pipe->streams[k])), "pipeline join") ||
                       set_cuda_error(cudaStreamWaitEvent(main, static_cast<cudaEvent_t>(pipe->events[k]), 0), "pipeline join");
      if (bad && rc == KF_OK) rc = KF_ERR_CUDA;
    }
  }
  if (rc != KF_OK) return rc;
#undef KF_TRY
  return KF_OK;
}

}  // namespace

extern "C" {

int kf_fit_batch_host(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge,
                      const kf_field* fl, const kf_options* op, const kf_outputs* out, void* device_arena,
                      size_t arena_bytes, void* cuda_stream) {
  return host_impl(tr, ms, ge, fl, op, out, device_arena, arena_bytes, static_cast<cudaStream_t>(cuda_stream), nullptr);
}

int kf_fit_batch_host_pipelined(const kf_tracks_in* tr, const kf_measurements* ms, const kf_geometry* ge,
                                const kf_field* fl, const kf_options* op, const kf_outputs* out, void* device_arena,
                                size_t arena_bytes, void* cuda_stream, const kf_pipeline* pipe) {
  if (!pipe) return KF_ERR_ARG;
  return host_impl(tr, ms, ge, fl, op, out, device_arena, arena_bytes, static_cast<cudaStream_t>(cuda_stream), pipe);
}

}  // extern "C"
