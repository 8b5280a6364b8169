"""Thin Python binding of libkf_fit.so (include/kf_fit.h): argument marshalling only.

Every step of the fit runs in the CUDA kernels behind `kf_fit_batch`; this module converts
layouts (natural AoS numpy arrays <-> the library's component-major SoA, 6x6 <-> packed 21),
holds device memory in torch tensors, and passes raw pointers.  It never imports `oracle/` and
has no CPU fallback: if the library cannot be loaded, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from dataclasses import dataclass, field as _dc_field
from types import SimpleNamespace
from typing import Optional

import numpy as np

from . import build as _build

GEOM_STRIDE = 20
REC_DOUBLES = 55  # x-(6) C-(21) F(26) hit(2): doubles per (leg, track) in the RTS workspace
TILE = 64          # tracks per workspace tile (= threads per RTS CTA)
STATES_PRED, STATES_FILT, STATES_SMOOTH = 1, 2, 4
VARIANT_AUTO, VARIANT_THREAD_PER_TRACK, VARIANT_LANES_PER_TRACK = 0, 1, 2
SORT_AUTO, SORT_OFF, SORT_ON = 0, 1, 2
SMOOTHER_RTS, SMOOTHER_BRYSON_FRAZIER = 0, 1
PRECISION_FP64, PRECISION_MIXED = 0, 1
_TRIU = np.triu_indices(6)  # packed upper triangle, row-major: 00 01 .. 05 11 .. 55

EXPORTS = ("kf_default_options", "kf_workspace_bytes", "kf_fit_batch", "kf_host_arena_bytes",
           "kf_fit_batch_host", "kf_fit_batch_host_pipelined", "kf_last_launch_count", "kf_set_stage_events", "kf_probe_fp64_tflops", "kf_status_string",
           "kf_last_cuda_error", "kf_version", "kf_field_stage_box", "kf_fit_batch_static")
STATIC_WORKSPACE_BYTES = 64 * 1024 * 1024  # KF_STATIC_WORKSPACE_BYTES


class KfTracksIn(C.Structure):
    _fields_ = [("n_tracks", C.c_int64), ("params", C.c_void_p), ("cov", C.c_void_p),
                ("start_surface", C.c_int32)]


class KfMeasurements(C.Structure):
    _fields_ = [("n_meas", C.c_int64), ("offsets", C.c_void_p), ("surf_idx", C.c_void_p),
                ("loc", C.c_void_p), ("var", C.c_void_p), ("cov01", C.c_void_p)]


class KfGeometry(C.Structure):
    _fields_ = [("n_surfaces", C.c_int32), ("surfaces", C.c_void_p), ("mat_Z", C.c_double),
                ("mat_A", C.c_double), ("mat_rho", C.c_double), ("mat_I_eV", C.c_double), ("surface_kinds", C.c_int32)]


class KfField(C.Structure):
    _fields_ = [("kind", C.c_int32), ("b", C.c_double * 3), ("n", C.c_int32 * 3),
                ("origin", C.c_double * 3), ("spacing", C.c_double * 3), ("grid", C.c_void_p),
                ("stage_lo", C.c_int32 * 3), ("stage_n", C.c_int32 * 3)]


class KfOptions(C.Structure):
    _fields_ = [("smooth", C.c_int32), ("material", C.c_int32), ("outlier_chi2", C.c_double),
                ("n_corr_steps", C.c_int32), ("max_step_mm", C.c_double), ("mass_gev", C.c_double),
                ("cov_inflation", C.c_double), ("output_states", C.c_int32), ("variant", C.c_int32),
                ("length_sort", C.c_int32), ("smoother", C.c_int32), ("step_tolerance_mm", C.c_double),
                ("perigee_center", C.c_double * 3), ("perigee_axis", C.c_double * 3), ("precision", C.c_int32),
                ("field_gradient", C.c_int32)]


KF_MAX_STREAMS = 8


class KfPipeline(C.Structure):
    _fields_ = [("n_streams", C.c_int32), ("streams", C.c_void_p * KF_MAX_STREAMS),
                ("events", C.c_void_p * (KF_MAX_STREAMS + 1)), ("chunk_tracks", C.c_int64)]


class KfOutputs(C.Structure):
    _fields_ = [("first_params", C.c_void_p), ("first_cov", C.c_void_p), ("last_params", C.c_void_p),
                ("last_cov", C.c_void_p), ("chi2", C.c_void_p), ("ndf", C.c_void_p),
                ("status", C.c_void_p), ("n_used", C.c_void_p), ("n_outliers", C.c_void_p),
                ("n_holes", C.c_void_p), ("state_params", C.c_void_p * 3),
                ("state_cov", C.c_void_p * 3), ("hit_chi2", C.c_void_p), ("hit_flags", C.c_void_p),
                ("rk_err_max", C.c_void_p), ("perigee_params", C.c_void_p), ("perigee_cov", C.c_void_p)]


_lib = None


def lib():
    """Load libkf_fit.so (building it with nvcc if it is missing or stale). Raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if _build.is_stale():
        path = _build.build_library()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing and could not be built: there is no CPU fallback")
    L = C.CDLL(path)
    L.kf_default_options.restype = None
    L.kf_default_options.argtypes = [C.POINTER(KfOptions)]
    L.kf_workspace_bytes.restype = C.c_size_t
    L.kf_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.POINTER(KfOptions)]
    L.kf_field_stage_box.restype = C.c_int
    L.kf_field_stage_box.argtypes = [C.c_void_p, C.c_int32, C.POINTER(KfField)]
    L.kf_fit_batch.restype = C.c_int
    L.kf_fit_batch.argtypes = [C.POINTER(KfTracksIn), C.POINTER(KfMeasurements), C.POINTER(KfGeometry),
                               C.POINTER(KfField), C.POINTER(KfOptions), C.POINTER(KfOutputs),
                               C.c_void_p, C.c_size_t, C.c_void_p]
    L.kf_fit_batch_static.restype = C.c_int
    L.kf_fit_batch_static.argtypes = L.kf_fit_batch.argtypes[:6] + [C.c_void_p]
    L.kf_host_arena_bytes.restype = C.c_size_t
    L.kf_host_arena_bytes.argtypes = [C.c_int64, C.c_int64, C.c_int32, C.c_int32, C.POINTER(KfField),
                                      C.POINTER(KfOptions), C.c_int, C.c_int]
    L.kf_fit_batch_host.restype = C.c_int
    L.kf_fit_batch_host.argtypes = L.kf_fit_batch.argtypes
    L.kf_fit_batch_host_pipelined.restype = C.c_int
    L.kf_fit_batch_host_pipelined.argtypes = L.kf_fit_batch.argtypes + [C.POINTER(KfPipeline)]
    L.kf_last_launch_count.restype = C.c_int
    L.kf_set_stage_events.restype = None
    L.kf_set_stage_events.argtypes = [C.POINTER(C.c_void_p)]
    L.kf_probe_fp64_tflops.restype = C.c_double
    L.kf_probe_fp64_tflops.argtypes = [C.c_int, C.c_void_p]
    L.kf_status_string.restype = C.c_char_p
    L.kf_status_string.argtypes = [C.c_int]
    L.kf_last_cuda_error.restype = C.c_char_p
    L.kf_version.restype = C.c_int
    _lib = L
    return L


class KfError(RuntimeError):
    def __init__(self, rc):
        L = lib()
        msg = L.kf_status_string(rc).decode()
        if rc == -4:
            msg += ": " + L.kf_last_cuda_error().decode()
        super().__init__(f"kf_fit_batch rejected the call (rc={rc}): {msg}")
        self.rc = rc


def default_options() -> KfOptions:
    o = KfOptions()
    lib().kf_default_options(C.byref(o))
    return o


def make_options(smooth=1, material=0, outlier_chi2=0.0, n_corr_steps=2, max_step_mm=float("inf"),
                 mass_gev=0.1056583755, cov_inflation=1.0, output_states=0, variant=0,
                 perigee_center=(0.0, 0.0, 0.0), perigee_axis=(0.0, 0.0, 1.0), length_sort=0, step_tolerance_mm=0.0, smoother=0, precision=0, field_gradient=0,
                 **_ignored) -> KfOptions:
    o = KfOptions()
    o.field_gradient = int(field_gradient)
    o.smoother, o.precision = int(smoother), int(precision)
    o.length_sort, o.step_tolerance_mm = int(length_sort), float(step_tolerance_mm)
    for k in range(3):
        o.perigee_center[k], o.perigee_axis[k] = float(perigee_center[k]), float(perigee_axis[k])
    o.smooth, o.material, o.outlier_chi2 = int(smooth), int(material), float(outlier_chi2)
    o.n_corr_steps, o.max_step_mm, o.mass_gev = int(n_corr_steps), float(max_step_mm), float(mass_gev)
    o.cov_inflation, o.output_states, o.variant = float(cov_inflation), int(output_states), int(variant)
    return o


# ---- layout conversion (host side, numpy) -------------------------------------------------------------
def pack_cov(cov66: np.ndarray) -> np.ndarray:
    """(N, 6, 6) symmetric -> (21, N) packed upper triangle, component-major."""
    return np.ascontiguousarray(cov66[:, _TRIU[0], _TRIU[1]].T)


def unpack_cov(cov21: np.ndarray) -> np.ndarray:
    """(21, N) -> (N, 6, 6) symmetric."""
    n = cov21.shape[1]
    out = np.empty((n, 6, 6), dtype=np.float64)
    out[:, _TRIU[0], _TRIU[1]] = cov21.T
    out[:, _TRIU[1], _TRIU[0]] = cov21.T
    return out


@dataclass
class HostBatch:
    """One batch in the library's SoA layouts, as numpy arrays on the host."""
    n_tracks: int
    n_meas: int
    n_surfaces: int
    start_surface: int
    params: np.ndarray    # (6, N)
    cov: np.ndarray       # (21, N)
    offsets: np.ndarray   # (N+1,) int32
    surf_idx: np.ndarray  # (M,) int32
    loc: np.ndarray       # (2, M)
    var: Optional[np.ndarray]    # (2, M) or None
    cov01: Optional[np.ndarray]  # (M,) or None
    geometry: np.ndarray  # (n_surfaces, 20)
    field_kind: str
    field_b: np.ndarray
    grid_n: Optional[np.ndarray]
    grid_origin: Optional[np.ndarray]
    grid_spacing: Optional[np.ndarray]
    grid: Optional[np.ndarray]   # (nz, ny, nx, 3)
    material: dict = _dc_field(default_factory=dict)
    options: dict = _dc_field(default_factory=dict)

    @property
    def n_legs_max(self) -> int:
        return self.n_surfaces - 1 - self.start_surface

    @staticmethod
    def from_arrays(params0, cov0, start_surface, offsets, surf_idx, loc, geometry, field_kind="const",
                    field_b=(0.0, 0.0, 2.0), grid_n=None, grid_origin=None, grid_spacing=None, grid=None,
                    var=None, cov01=None, material=None, options=None) -> "HostBatch":
        params0 = np.asarray(params0, dtype=np.float64).reshape(-1, 6)
        cov0 = np.asarray(cov0, dtype=np.float64).reshape(-1, 6, 6)
        loc = np.asarray(loc, dtype=np.float64).reshape(-1, 2)
        geometry = np.ascontiguousarray(geometry, dtype=np.float64).reshape(-1, GEOM_STRIDE)
        return HostBatch(
            n_tracks=params0.shape[0], n_meas=loc.shape[0], n_surfaces=geometry.shape[0],
            start_surface=int(start_surface),
            params=np.ascontiguousarray(params0.T), cov=pack_cov(cov0),
            offsets=np.ascontiguousarray(offsets, dtype=np.int32),
            surf_idx=np.ascontiguousarray(surf_idx, dtype=np.int32),
            loc=np.ascontiguousarray(loc.T),
            var=None if var is None else np.ascontiguousarray(np.asarray(var, dtype=np.float64).reshape(-1, 2).T),
            cov01=None if cov01 is None else np.ascontiguousarray(cov01, dtype=np.float64),
            geometry=geometry, field_kind=field_kind, field_b=np.asarray(field_b, dtype=np.float64),
            grid_n=None if grid_n is None else np.asarray(grid_n, dtype=np.int32),
            grid_origin=None if grid_origin is None else np.asarray(grid_origin, dtype=np.float64),
            grid_spacing=None if grid_spacing is None else np.asarray(grid_spacing, dtype=np.float64),
            grid=None if grid is None else np.ascontiguousarray(grid, dtype=np.float64),
            material=dict(material or dict(Z=14.0, A=28.0855, rho=2.329, I_eV=173.0)),
            options=dict(options or {}))

    @staticmethod
    def from_workload(wl) -> "HostBatch":
        return HostBatch.from_arrays(
            wl.params0, wl.cov0, wl.start_surface, wl.offsets, wl.surf_idx, wl.loc, wl.geometry,
            wl.field_kind, wl.field_b, wl.grid_n, wl.grid_origin, wl.grid_spacing, wl.grid,
            material=wl.material, options=wl.options)


def _field_struct(hb: HostBatch, grid_ptr: int, stage: bool = False) -> KfField:
    """stage: let the library derive the shared-memory staging hint (kf_field.stage_*) from the host geometry table."""
    f = KfField()
    if hb.field_kind == "const":
        f.kind = 0
        f.b[:] = [float(v) for v in hb.field_b]
    else:
        f.kind = 1
        f.n[:] = [int(v) for v in hb.grid_n]
        f.origin[:] = [float(v) for v in hb.grid_origin]
        f.spacing[:] = [float(v) for v in hb.grid_spacing]
        f.grid = grid_ptr
        if stage:
            g = np.ascontiguousarray(hb.geometry, dtype=np.float64)
            rc = lib().kf_field_stage_box(g.ctypes.data_as(C.c_void_p), int(hb.n_surfaces), C.byref(f))
            if rc != 0:
                raise KfError(rc)
    return f


def _geom_struct(hb: HostBatch, ptr: int) -> KfGeometry:
    g = KfGeometry()
    g.n_surfaces, g.surfaces = hb.n_surfaces, ptr
    m = hb.material
    g.mat_Z, g.mat_A, g.mat_rho, g.mat_I_eV = float(m["Z"]), float(m["A"]), float(m["rho"]), float(m["I_eV"])
    # which surface kinds the (host copy of the) table holds: the library's dispatch cannot read device memory
    kinds = 0
    for k in np.unique(np.asarray(hb.geometry)[:, 18]).astype(np.int64):
        kinds |= 1 << int(k)
    g.surface_kinds = int(kinds)
    return g


def _options_for(hb: HostBatch, over: dict) -> KfOptions:
    kw = dict(hb.options)
    kw.update(over)
    return make_options(**kw)


# ---- device side: torch holds the memory and the stream, nothing else ----------------------------------
def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: the Kalman fit runs only in the sm_100a kernels (no CPU fallback)")
    return torch


def _ptr(t) -> int:
    return 0 if t is None else int(t.data_ptr())


class DeviceBatch:
    """A HostBatch uploaded to HBM (torch tensors in the library's SoA layouts)."""

    def __init__(self, hb: HostBatch, device="cuda:0"):
        torch = _torch()
        self.host = hb
        self.device = torch.device(device)
        up = lambda a: None if a is None else torch.from_numpy(a).to(self.device)
        self.params, self.cov = up(hb.params), up(hb.cov)
        self.offsets, self.surf_idx, self.loc = up(hb.offsets), up(hb.surf_idx), up(hb.loc)
        self.var, self.cov01 = up(hb.var), up(hb.cov01)
        self.geometry = up(hb.geometry)
        self.grid = up(hb.grid) if hb.field_kind != "const" else None

    @property
    def input_bytes(self) -> int:
        ts = (self.params, self.cov, self.offsets, self.surf_idx, self.loc, self.var, self.cov01,
              self.geometry, self.grid)
        return sum(t.numel() * t.element_size() for t in ts if t is not None)


class DeviceOutputs:
    """Output buffers of one kf_fit_batch call, allocated once and reusable across calls."""

    def __init__(self, n_tracks, n_meas, n_legs_max, output_states=0, per_hit=True, rk_err=True,
                 device="cuda:0", perigee=False):
        torch = _torch()
        N, M, L = int(n_tracks), int(n_meas), int(n_legs_max)
        dev = torch.device(device)
        f64 = dict(dtype=torch.float64, device=dev)
        i32 = dict(dtype=torch.int32, device=dev)
        self.n_tracks, self.n_meas, self.n_legs_max, self.output_states = N, M, L, int(output_states)
        self.first_params, self.first_cov = torch.zeros((6, N), **f64), torch.zeros((21, N), **f64)
        self.last_params, self.last_cov = torch.zeros((6, N), **f64), torch.zeros((21, N), **f64)
        self.chi2 = torch.zeros(N, **f64)
        self.ndf, self.status = torch.zeros(N, **i32), torch.zeros(N, **i32)
        self.n_used, self.n_outliers, self.n_holes = (torch.zeros(N, **i32) for _ in range(3))
        self.state_params, self.state_cov = [None] * 3, [None] * 3
        for b in range(3):
            if (self.output_states >> b) & 1:  # legs a track did not visit stay NaN
                self.state_params[b] = torch.full((L, 6, N), float("nan"), **f64)
                self.state_cov[b] = torch.full((L, 21, N), float("nan"), **f64)
        self.hit_chi2 = torch.zeros(M, **f64) if per_hit else None
        self.hit_flags = torch.zeros(M, dtype=torch.uint8, device=dev) if per_hit else None
        self.rk_err_max = torch.zeros(N, **f64) if rk_err else None
        self.perigee_params = torch.zeros((6, N), **f64) if perigee else None
        self.perigee_cov = torch.zeros((21, N), **f64) if perigee else None

    def struct(self) -> KfOutputs:
        o = KfOutputs()
        for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "ndf", "status",
                     "n_used", "n_outliers", "n_holes", "hit_chi2", "hit_flags", "rk_err_max", "perigee_params",
                     "perigee_cov"):
            setattr(o, name, _ptr(getattr(self, name)) or None)
        for b in range(3):
            o.state_params[b] = _ptr(self.state_params[b]) or None
            o.state_cov[b] = _ptr(self.state_cov[b]) or None
        return o

    @property
    def minimal_output_bytes(self) -> int:
        return self.n_tracks * (2 * 27 * 8 + 8 + 5 * 4)

    def to_host(self) -> SimpleNamespace:
        """Copy back and convert to the natural AoS layouts (params (N,6), cov (N,6,6), states (N,L,..))."""
        cpu = lambda t: None if t is None else t.cpu().numpy()
        r = SimpleNamespace(
            first_params=cpu(self.first_params).T.copy(), first_cov=unpack_cov(cpu(self.first_cov)),
            last_params=cpu(self.last_params).T.copy(), last_cov=unpack_cov(cpu(self.last_cov)),
            chi2=cpu(self.chi2), ndf=cpu(self.ndf), status=cpu(self.status).astype(np.uint32),
            n_used=cpu(self.n_used), n_outliers=cpu(self.n_outliers), n_holes=cpu(self.n_holes),
            hit_chi2=cpu(self.hit_chi2), hit_flags=cpu(self.hit_flags), rk_err_max=cpu(self.rk_err_max),
            perigee_params=None if self.perigee_params is None else cpu(self.perigee_params).T.copy(),
            perigee_cov=None if self.perigee_cov is None else unpack_cov(cpu(self.perigee_cov)))
        for b, name in enumerate(("pred", "filt", "smooth")):
            sp, sc = cpu(self.state_params[b]), cpu(self.state_cov[b])
            if sp is None:
                setattr(r, name + "_params", None)
                setattr(r, name + "_cov", None)
            else:
                L, _, N = sp.shape
                setattr(r, name + "_params", np.ascontiguousarray(sp.transpose(2, 0, 1)))
                c = unpack_cov(sc.transpose(1, 0, 2).reshape(21, L * N)).reshape(L, N, 6, 6)
                setattr(r, name + "_cov", np.ascontiguousarray(c.transpose(1, 0, 2, 3)))
        return r


def workspace_bytes(n_tracks, n_legs_max, opt: KfOptions) -> int:
    return int(lib().kf_workspace_bytes(int(n_tracks), int(n_legs_max), C.byref(opt)))


def alloc_workspace(n_tracks, n_legs_max, opt: KfOptions, device="cuda:0"):
    torch = _torch()
    nbytes = workspace_bytes(n_tracks, n_legs_max, opt)
    return torch.empty(max(nbytes, 1), dtype=torch.uint8, device=torch.device(device))


class FitCall:
    """A prepared kf_fit_batch call: descriptors built once, `run()` only enqueues.
    This is what bench.py times; `fit_batch` below is the one-shot convenience."""

    def __init__(self, batch: DeviceBatch, out: Optional[DeviceOutputs] = None, workspace=None, perigee=None,
                 field_stage=False, **opt_over):
        """perigee = (centre, unit axis): also return the fitted parameters on that line surface.
        field_stage: pass the staging hint for a grid field (kf_field_stage_box): the acceptance box of the table is then
        kept in shared memory.  Results do not depend on it; measured slower than the L1/L2 path on CFG4, so off."""
        hb = batch.host
        self.batch = batch
        if perigee is not None:
            opt_over = dict(opt_over, perigee_center=perigee[0], perigee_axis=perigee[1])
        self.opt = _options_for(hb, opt_over)
        self.out = out or DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, self.opt.output_states,
                                        device=batch.device, perigee=perigee is not None)
        self.workspace = workspace if workspace is not None else alloc_workspace(
            hb.n_tracks, hb.n_legs_max, self.opt, batch.device)
        self.tracks = KfTracksIn(hb.n_tracks, _ptr(batch.params), _ptr(batch.cov), hb.start_surface)
        self.meas = KfMeasurements(hb.n_meas, _ptr(batch.offsets), _ptr(batch.surf_idx), _ptr(batch.loc),
                                   _ptr(batch.var) or None, _ptr(batch.cov01) or None)
        self.geom = _geom_struct(hb, _ptr(batch.geometry))
        self.field = _field_struct(hb, _ptr(batch.grid), stage=field_stage)
        self.outs = self.out.struct()
        self.launches = 0

    def run(self, stream=None):
        torch = _torch()
        s = stream if stream is not None else torch.cuda.current_stream(self.batch.device)
        rc = lib().kf_fit_batch(C.byref(self.tracks), C.byref(self.meas), C.byref(self.geom),
                                C.byref(self.field), C.byref(self.opt), C.byref(self.outs),
                                _ptr(self.workspace), self.workspace.numel(), C.c_void_p(s.cuda_stream))
        if rc != 0:
            raise KfError(rc)
        self.launches = lib().kf_last_launch_count()
        return self.out


class StaticFitCall(FitCall):
    """A prepared kf_fit_batch_static call: the fit for callers that cannot allocate device memory for a workspace.

    Meant for code that receives its input and output buffers from somebody else's memory pool and is not allowed
    to call the CUDA allocator itself (a plug-in inside an event-processing framework), or that must not allocate
    once its latency-critical loop runs (cudaMalloc / cudaFree take driver-wide locks; cudaFree waits for the device).
    The RTS records and sort arrays then live in a 64 MiB array inside the library image (STATIC_WORKSPACE_BYTES)
    instead of a caller-owned workspace, so the batch must need no more than that (about 5,000 tracks x 30 legs in
    FP64): a larger one raises KfError with rc = -5 and nothing is enqueued.  Results are those of FitCall, bit for
    bit.  All calls on one GPU share that array: calls that could overlap on the GPU (two streams with no ordering
    between them) corrupt each other, so keep them on one stream or order them with events.  The first run() on a
    device also looks up the array's address there; do it once at start-up, outside any stream capture.

    Here torch still allocates the inputs and outputs (this is a test and example harness); the library call
    itself allocates nothing."""

    def __init__(self, batch: DeviceBatch, out: Optional[DeviceOutputs] = None, perigee=None, **opt_over):
        torch = _torch()
        # an empty tensor stands in for FitCall's workspace so that none is allocated
        super().__init__(batch, out=out, workspace=torch.empty(0, dtype=torch.uint8, device=batch.device),
                         perigee=perigee, **opt_over)

    def run(self, stream=None):
        torch = _torch()
        s = stream if stream is not None else torch.cuda.current_stream(self.batch.device)
        with torch.cuda.device(self.batch.device):  # the static array is looked up on the CURRENT device
            rc = lib().kf_fit_batch_static(C.byref(self.tracks), C.byref(self.meas), C.byref(self.geom),
                                           C.byref(self.field), C.byref(self.opt), C.byref(self.outs),
                                           C.c_void_p(s.cuda_stream))
        if rc != 0:
            raise KfError(rc)
        self.launches = lib().kf_last_launch_count()
        return self.out


def fit_batch(batch, device="cuda:0", **opt_over) -> DeviceOutputs:
    """Fit one batch (a Workload, HostBatch or DeviceBatch) on the GPU; returns device outputs."""
    if not isinstance(batch, (DeviceBatch, HostBatch)):
        batch = HostBatch.from_workload(batch)
    if isinstance(batch, HostBatch):
        batch = DeviceBatch(batch, device)
    return FitCall(batch, **opt_over).run()


def fit_workload(wl, device="cuda:0", states=False, **opt_over) -> SimpleNamespace:
    """Fit a Workload and return host arrays in the oracle's natural layouts (for the parity tests).
    perigee=(centre, unit axis) adds perigee_params / perigee_cov."""
    torch = _torch()
    if states:
        smooth = opt_over.get("smooth", wl.options.get("smooth", 1))
        opt_over.setdefault("output_states", STATES_PRED | STATES_FILT | (STATES_SMOOTH if smooth else 0))
    out = fit_batch(wl, device=device, **opt_over)
    torch.cuda.synchronize()
    return out.to_host()


# ---- end-to-end call with HOST buffers (kf_fit_batch_host) ---------------------------------------------
class HostCall:
    """kf_fit_batch_host on pinned host memory: inputs are copied H2D, fitted, results copied D2H,
    all enqueued on one stream by the library.  Pinned tensors are allocated once here; `run()` only
    enqueues.  h2d_bytes / d2h_bytes count the tensors the library copies per call."""

    def __init__(self, hb: HostBatch, device="cuda:0", per_hit=False, n_streams=0, chunk_tracks=0, perigee=None,
                 field_stage=False, **opt_over):
        torch = _torch()
        self.hb, self.device = hb, torch.device(device)
        if perigee is not None:
            opt_over = dict(opt_over, perigee_center=perigee[0], perigee_axis=perigee[1])
        self.opt = _options_for(hb, opt_over)
        # n_streams >= 1: kf_fit_batch_host_pipelined over that many caller-owned streams (+ fork/join events)
        self.pipe = None
        if n_streams:
            if not 1 <= n_streams <= KF_MAX_STREAMS:
                raise ValueError("n_streams must be in 1..%d" % KF_MAX_STREAMS)
            self.streams = [torch.cuda.Stream(self.device) for _ in range(n_streams)]
            self.events = [torch.cuda.Event(enable_timing=False) for _ in range(n_streams + 1)]
            with torch.cuda.device(self.device):
                for e in self.events:
                    e.record()  # torch creates the handle lazily: make it exist
            self.pipe = KfPipeline()
            self.pipe.n_streams, self.pipe.chunk_tracks = n_streams, int(chunk_tracks)
            for k, st in enumerate(self.streams):
                self.pipe.streams[k] = st.cuda_stream
            for k, e in enumerate(self.events):
                self.pipe.events[k] = e.cuda_event
        if self.opt.output_states:
            raise ValueError("HostCall returns the per-track results only (output_states must be 0)")
        pin = lambda a: None if a is None else torch.from_numpy(a).pin_memory()
        self.h_params, self.h_cov = pin(hb.params), pin(hb.cov)
        self.h_offsets, self.h_surf_idx, self.h_loc = pin(hb.offsets), pin(hb.surf_idx), pin(hb.loc)
        self.h_var, self.h_cov01 = pin(hb.var), pin(hb.cov01)
        self.h_geometry = pin(hb.geometry)
        self.h_grid = pin(hb.grid) if hb.field_kind != "const" else None
        N, M = hb.n_tracks, hb.n_meas
        hz = lambda shape, dt: torch.zeros(shape, dtype=dt).pin_memory()
        self.first_params, self.first_cov = hz((6, N), torch.float64), hz((21, N), torch.float64)
        self.last_params, self.last_cov = hz((6, N), torch.float64), hz((21, N), torch.float64)
        self.chi2 = hz(N, torch.float64)
        self.ndf, self.status = hz(N, torch.int32), hz(N, torch.int32)
        self.n_used, self.n_outliers, self.n_holes = (hz(N, torch.int32) for _ in range(3))
        self.hit_chi2 = hz(M, torch.float64) if per_hit else None
        self.hit_flags = hz(M, torch.uint8) if per_hit else None
        self.perigee_params = hz((6, N), torch.float64) if perigee is not None else None
        self.perigee_cov = hz((21, N), torch.float64) if perigee is not None else None
        self.tracks = KfTracksIn(N, _ptr(self.h_params), _ptr(self.h_cov), hb.start_surface)
        self.meas = KfMeasurements(M, _ptr(self.h_offsets), _ptr(self.h_surf_idx), _ptr(self.h_loc),
                                   _ptr(self.h_var) or None, _ptr(self.h_cov01) or None)
        self.geom = _geom_struct(hb, _ptr(self.h_geometry))
        self.field = _field_struct(hb, _ptr(self.h_grid), stage=field_stage)
        o = KfOutputs()
        for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "ndf", "status",
                     "n_used", "n_outliers", "n_holes", "hit_chi2", "hit_flags", "perigee_params", "perigee_cov"):
            setattr(o, name, _ptr(getattr(self, name)) or None)
        self.outs = o
        nbytes = int(lib().kf_host_arena_bytes(N, M, hb.n_surfaces, hb.start_surface, C.byref(self.field),
                                               C.byref(self.opt), int(hb.var is not None),
                                               int(hb.cov01 is not None)))
        self.arena = torch.empty(max(nbytes, 1), dtype=torch.uint8, device=self.device)
        nb = lambda t: 0 if t is None else t.numel() * t.element_size()
        self.h2d_bytes = sum(nb(t) for t in (self.h_params, self.h_cov, self.h_offsets, self.h_surf_idx,
                                             self.h_loc, self.h_var, self.h_cov01, self.h_geometry, self.h_grid))
        self.d2h_bytes = sum(nb(t) for t in (self.first_params, self.first_cov, self.last_params,
                                             self.last_cov, self.chi2, self.ndf, self.status, self.n_used,
                                             self.n_outliers, self.n_holes, self.hit_chi2, self.hit_flags,
                                             self.perigee_params, self.perigee_cov))
        self.launches = 0

    def run(self, stream=None):
        torch = _torch()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        args = (C.byref(self.tracks), C.byref(self.meas), C.byref(self.geom), C.byref(self.field), C.byref(self.opt),
                C.byref(self.outs), _ptr(self.arena), self.arena.numel(), C.c_void_p(s.cuda_stream))
        if self.pipe is not None:
            rc = lib().kf_fit_batch_host_pipelined(*args, C.byref(self.pipe))
        else:
            rc = lib().kf_fit_batch_host(*args)
        if rc != 0:
            raise KfError(rc)
        self.launches = lib().kf_last_launch_count()
        return self

    def to_host(self) -> SimpleNamespace:
        n = lambda t: None if t is None else t.numpy()
        return SimpleNamespace(
            first_params=n(self.first_params).T.copy(), first_cov=unpack_cov(n(self.first_cov)),
            last_params=n(self.last_params).T.copy(), last_cov=unpack_cov(n(self.last_cov)),
            chi2=n(self.chi2).copy(), ndf=n(self.ndf).copy(), status=n(self.status).astype(np.uint32),
            n_used=n(self.n_used).copy(), n_outliers=n(self.n_outliers).copy(), n_holes=n(self.n_holes).copy(),
            hit_chi2=None if self.hit_chi2 is None else n(self.hit_chi2).copy(),
            hit_flags=None if self.hit_flags is None else n(self.hit_flags).copy(),
            perigee_params=None if self.perigee_params is None else n(self.perigee_params).T.copy(),
            perigee_cov=None if self.perigee_cov is None else unpack_cov(n(self.perigee_cov)))


def probe_fp64_tflops(iters=20000, device="cuda:0") -> float:
    """Sustained DFMA throughput of the device in TFLOP/s (the FP64 roofline denominator)."""
    torch = _torch()
    with torch.cuda.device(torch.device(device)):
        v = float(lib().kf_probe_fp64_tflops(int(iters), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    if v < 0:
        raise KfError(int(v))
    return v


class StageTimer:
    """Per-kernel device times of kf_fit_batch calls via kf_set_stage_events: three CUDA events per
    call that the library records around its forward and RTS kernels, on the launching stream.
    prepare(K) creates the events, arm(k) points the library at set k before call k (no
    synchronisation), finish() reads all of them after the caller has synchronised."""

    def __init__(self, device="cuda:0"):
        torch = _torch()
        self.device = torch.device(device)
        self._sets, self._arrs = [], []

    def prepare(self, n_calls: int):
        torch = _torch()
        s = torch.cuda.current_stream(self.device)
        self._sets, self._arrs = [], []
        for _ in range(n_calls):
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            for e in ev:
                e.record(s)  # creates the cudaEvent_t handle
            self._sets.append(ev)
            self._arrs.append((C.c_void_p * 3)(*[C.c_void_p(int(e.cuda_event)) for e in ev]))

    def arm(self, k: int):
        lib().kf_set_stage_events(self._arrs[k])

    def disarm(self):
        lib().kf_set_stage_events(None)

    def finish(self):
        """-> (forward_ms list, rts_ms list); call after torch.cuda.synchronize()."""
        self.disarm()
        fwd = [ev[0].elapsed_time(ev[1]) for ev in self._sets]
        rts = [ev[1].elapsed_time(ev[2]) for ev in self._sets]
        return fwd, rts
