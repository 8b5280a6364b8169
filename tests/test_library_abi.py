"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol include/kf_fit.h
declares, and its host logic (defaults, workspace size, argument validation) behaves as the header
says.  No kernel runs here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2105_01796_b200 import binding as B
from paper_2105_01796_b200 import build as kbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    hdr = open(os.path.join(ROOT, "include", "kf_fit.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = re.findall(r"\b(kf_[a-z0-9_]+)\s*\(", hdr)
    return sorted(set(names))


def test_library_builds_and_exports_every_declared_symbol():
    path = kbuild.build_library()
    assert os.path.exists(path)
    lib = C.CDLL(path)
    names = declared_functions()
    assert set(names) == set(B.EXPORTS), (names, B.EXPORTS)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/kf_fit.h but not exported"


def test_a_build_with_other_flags_is_stale_for_the_default_build():
    """build.py: a tuning build (`python build.py -DKF_FWD_MIN_BLOCKS=2`) must not be picked up silently by a later default
    call (lib(), tests, bench): staleness compares the flag stamp of the library that is there, not only file times."""
    kbuild.build_library()
    assert not kbuild.is_stale()
    assert kbuild.built_flags() == kbuild.flag_stamp() and kbuild.built_defines() == []
    assert kbuild.is_stale(extra_flags=("-DKF_FWD_MIN_BLOCKS=2",))
    assert "-DKF_FWD_MIN_BLOCKS=2" in kbuild.flag_stamp(("-DKF_FWD_MIN_BLOCKS=2",))
    assert ROOT not in kbuild.flag_stamp()   # path-free: the repository sits elsewhere on the GPU box
    saved = kbuild.built_flags()
    try:
        with open(kbuild.STAMP, "w") as f:
            f.write(saved + " -DKF_FWD_MIN_BLOCKS=2")   # as a tuning build would leave it
        assert kbuild.is_stale() and kbuild.built_defines() == ["-DKF_FWD_MIN_BLOCKS=2"]
    finally:
        with open(kbuild.STAMP, "w") as f:
            f.write(saved)
    assert not kbuild.is_stale()


def test_struct_sizes_match_the_header_layout():
    # natural C layout of include/kf_fit.h on x86-64 / aarch64 (8-byte pointers and doubles)
    assert C.sizeof(B.KfTracksIn) == 32
    assert C.sizeof(B.KfMeasurements) == 48
    assert C.sizeof(B.KfGeometry) == 48 + 8   # ... surface_kinds (int32 + padding)
    assert C.sizeof(B.KfField) == 4 + 4 + 24 + 12 + 4 + 24 + 24 + 8 + 12 + 12
    assert C.sizeof(B.KfOptions) == 56 + 8 + 8 + 48 + 8  # ... perigee line (48), precision + field_gradient (2 x int32)
    assert C.sizeof(B.KfOutputs) == 10 * 8 + 6 * 8 + 3 * 8 + 2 * 8
    assert C.sizeof(B.KfPipeline) == 8 + 8 * 8 + 9 * 8 + 8


def test_defaults_and_version():
    L = B.lib()
    assert L.kf_version() == 109
    o = B.default_options()
    assert (o.smooth, o.material, o.n_corr_steps, o.output_states, o.variant, o.length_sort, o.precision) == (1, 0, 2, 0, 0, 0, 0)
    assert o.outlier_chi2 == 0.0 and np.isinf(o.max_step_mm) and o.cov_inflation == 1.0
    assert o.mass_gev == pytest.approx(0.1056583755)
    assert L.kf_status_string(0) == b"ok"
    assert b"workspace" in L.kf_status_string(-3)


def test_workspace_bytes():
    o = B.default_options()
    # tile-major records: tiles * Lmax * (55 doubles + 1 flag byte) * TILE, then nleg int32 per slot,
    # each block rounded to 256 B (include/kf_fit.h "workspace")
    up = lambda v: (v + 255) // 256 * 256
    # then the length sort's arrays: slot -> track permutation (int32 per slot), 64 counters per 128 tracks
    sort = lambda n: up((n + B.TILE - 1) // B.TILE * B.TILE * 4) + up((n + 127) // 128 * 64 * 4)
    for n, L in ((1000, 6), (50, 3), (65, 30)):
        tiles = (n + B.TILE - 1) // B.TILE
        assert B.workspace_bytes(n, L, o) == (up(tiles * L * (B.REC_DOUBLES * 8 + 1) * B.TILE) + up(tiles * B.TILE * 4)
                                              + sort(n))
    n, L = 1000, 6
    o.smooth = 0
    assert B.workspace_bytes(n, L, o) == sort(n)
    o.smooth = 1
    # MIXED precision: float records (55 floats + 1 flag byte per leg and track)
    o.precision = B.PRECISION_MIXED
    tiles = (n + B.TILE - 1) // B.TILE
    assert B.workspace_bytes(n, L, o) == up(tiles * L * (B.REC_DOUBLES * 4 + 1) * B.TILE) + up(tiles * B.TILE * 4) + sort(n)
    o.precision = B.PRECISION_FP64
    assert B.workspace_bytes(0, L, o) == 0
    # 1e6 tracks x 30 legs fits comfortably in 180 GB
    assert B.workspace_bytes(1_000_000, 30, o) < 14e9


def _dummy_call(**over):
    """A structurally valid call on HOST dummy pointers; only used for calls that must be rejected
    before anything is enqueued."""
    n = 4
    buf = np.zeros(4096)
    p = buf.ctypes.data
    tr = B.KfTracksIn(n, p, p, 0)
    ms = B.KfMeasurements(0, p, p, p, None, None)
    ge = B.KfGeometry(3, p, 14.0, 28.0855, 2.329, 173.0)
    fl = B.KfField()
    fl.kind = 0
    op = B.default_options()
    out = B.KfOutputs()
    for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "ndf", "status", "n_used",
                 "n_outliers", "n_holes"):
        setattr(out, name, p)
    d = dict(tr=tr, ms=ms, ge=ge, fl=fl, op=op, out=out, ws=p, ws_bytes=0, keep=buf)
    d.update(over)
    return d


def _call(d):
    return B.lib().kf_fit_batch(C.byref(d["tr"]), C.byref(d["ms"]), C.byref(d["ge"]), C.byref(d["fl"]),
                                C.byref(d["op"]), C.byref(d["out"]), d["ws"], d["ws_bytes"], None)


def test_argument_validation_rejects_before_any_launch():
    d = _dummy_call()
    assert _call(d) == -3  # smoothing needs a workspace
    d = _dummy_call()
    d["tr"].start_surface = 3
    assert _call(d) == -1
    d = _dummy_call()
    d["op"].n_corr_steps = 9
    assert _call(d) == -1
    d = _dummy_call()
    d["op"].mass_gev = 0.0
    assert _call(d) == -1
    d = _dummy_call()
    d["fl"].kind = 7
    assert _call(d) == -1
    d = _dummy_call()
    d["fl"].kind = 1  # GRID3 without a grid
    assert _call(d) == -1
    d = _dummy_call()
    d["out"].chi2 = None
    assert _call(d) == -1
    d = _dummy_call()
    d["op"].output_states = B.STATES_FILT  # requested but no buffers
    assert _call(d) == -1
    d = _dummy_call()
    d["op"].smooth = 0
    d["op"].output_states = B.STATES_SMOOTH
    d["out"].state_params[2] = d["ws"]
    d["out"].state_cov[2] = d["ws"]
    assert _call(d) == -2
    d = _dummy_call()
    d["op"].variant = 99
    assert _call(d) == -1
    # precision: FP64 | MIXED; MIXED is thread-per-track + RTS only
    d = _dummy_call()
    d["op"].precision = 5
    assert _call(d) == -1
    for bad in (dict(variant=B.VARIANT_LANES_PER_TRACK), dict(smoother=B.SMOOTHER_BRYSON_FRAZIER)):
        d = _dummy_call()
        d["op"].precision = B.PRECISION_MIXED
        for k, v in bad.items():
            setattr(d["op"], k, v)
        assert _call(d) == -2
    # null descriptor
    assert B.lib().kf_fit_batch(None, None, None, None, None, None, None, 0, None) == -1
    # zero tracks: accepted, nothing enqueued
    d = _dummy_call()
    d["tr"].n_tracks = 0
    assert _call(d) == 0
    assert B.lib().kf_last_launch_count() == 0


def test_layout_round_trip():
    rng = np.random.default_rng(0)
    a = rng.standard_normal((7, 6, 6))
    cov = a @ a.transpose(0, 2, 1)
    packed = B.pack_cov(cov)
    assert packed.shape == (21, 7)
    # packed order 00 01 .. 05 11 .. 55
    assert packed[1, 3] == cov[3, 0, 1] and packed[6, 2] == cov[2, 1, 1] and packed[20, 5] == cov[5, 5, 5]
    np.testing.assert_array_equal(B.unpack_cov(packed), 0.5 * (cov + cov.transpose(0, 2, 1)) * 0 + np.where(
        np.triu(np.ones((6, 6), bool)), cov, cov.transpose(0, 2, 1)))


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2105_01796_b200 import workloads as W
    import paper_2105_01796_b200 as kf
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        kf.fit_workload(W.make_config(0, n_tracks=8))


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2105_01796_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "kf_oracle" not in src, f


def test_field_stage_box_from_the_host_geometry():
    """kf_field_stage_box (host arithmetic only): the node box around every surface's rectangle plus one cell of margin,
    clipped to the grid; cleared for a constant field, for a table without half lengths, for a box that does not fit."""
    from paper_2105_01796_b200 import workloads as W
    L = B.lib()
    wl = W.make_config(4, n_tracks=16)
    hb = B.HostBatch.from_workload(wl)
    f = B._field_struct(hb, 0, stage=True)
    # planes x = 0..900 mm, 100 x 100 mm; grid 41 x 21 x 21 nodes from (0, -100, -100), 10 mm: x is clipped to the whole
    # axis, y and z cover cells 4..15 (-60..60 mm) -> nodes 4..17
    assert list(f.stage_lo) == [0, 4, 4] and list(f.stage_n) == [41, 14, 14]
    assert 41 * 14 * 14 * 3 * 8 <= 200 * 1024
    g = np.ascontiguousarray(hb.geometry, dtype=np.float64)
    # every corner of every rectangle lies in a cell whose nodes are all inside the box
    for s in range(hb.n_surfaces):
        c, u, v, hu, hv = g[s, 0:3], g[s, 3:6], g[s, 6:9], g[s, 12], g[s, 13]
        for su in (-1, 1):
            for sv in (-1, 1):
                p = c + su * hu * u + sv * hv * v
                for a in range(3):
                    cell = int(np.clip(np.floor((p[a] - f.origin[a]) / f.spacing[a]), 0, f.n[a] - 2))
                    assert f.stage_lo[a] <= cell and cell + 1 < f.stage_lo[a] + f.stage_n[a]
    # no half lengths -> no hint; a finer grid -> the box no longer fits -> no hint; constant field -> no hint
    g2 = g.copy(); g2[:, 12:14] = 0.0
    assert L.kf_field_stage_box(g2.ctypes.data_as(C.c_void_p), hb.n_surfaces, C.byref(f)) == 0 and list(f.stage_n) == [0, 0, 0]
    f.spacing[:] = [2.0, 2.0, 2.0]; f.n[:] = [201, 101, 101]
    assert L.kf_field_stage_box(g.ctypes.data_as(C.c_void_p), hb.n_surfaces, C.byref(f)) == 0 and list(f.stage_n) == [0, 0, 0]
    fc = B._field_struct(B.HostBatch.from_workload(W.make_config(0, n_tracks=4)), 0, stage=True)
    assert fc.kind == 0 and list(fc.stage_n) == [0, 0, 0]
    assert L.kf_field_stage_box(None, 3, None) == -1
