"""kf_fit_batch_static: the fit for callers that cannot allocate device memory.

Why the entry point exists.  kf_fit_batch wants a caller-owned workspace for its RTS records, leg counts and
length-sort arrays.  Some users of the library have no way to get one: a reconstruction module that runs inside
an event-processing framework is handed its input and output buffers from the framework's own device-memory pool
and is not allowed to call cudaMalloc; a latency-bound trigger thread must not allocate after start-up, because
cudaMalloc and cudaFree take driver-wide locks and cudaFree waits for every stream of the device.  For them the
library keeps one 64 MiB array inside its own image (KF_STATIC_WORKSPACE_BYTES) and kf_fit_batch_static fits
with that as the workspace; batches that need more are refused.

What is checked here.  The static-workspace call must give what kf_fit_batch gives on the same inputs -- it runs
the same kernels, so the comparison holds the floating-point results to the parity bars of tests/parity.py
(1e-10 / 1e-8 / 1e-9) and the integers exactly, and in fact expects equal bits.  Two calls are made in a row on
purpose: the array is shared by every call and still holds what the call before left in it, so the second call
(a different, shorter and ragged batch, length-sorted) runs on top of the first one's records and sort counters.
The file is named so that pytest collects it last: a failure here cannot hide another test behind `-x`.  It does
not depend on what ran before it in the process (the first call on a device does its own set-up).
"""
import ctypes as C

import numpy as np
import pytest

import parity
import paper_2105_01796_b200 as kf
from paper_2105_01796_b200 import binding as B
from paper_2105_01796_b200 import workloads as W


def _pair(wl, **over):
    """The same batch through kf_fit_batch (torch-allocated workspace) and through kf_fit_batch_static."""
    import torch
    db = B.DeviceBatch(B.HostBatch.from_workload(wl))
    ref = B.FitCall(db, **over).run().to_host()
    got = B.StaticFitCall(db, **over).run().to_host()
    torch.cuda.synchronize()
    return got, ref


def _assert_same(got, ref, label, states=False):
    rep = parity.assert_parity(got, ref, states=states, label=label)  # integers, flags, status: exact
    assert max(rep.values()) <= 1.0, rep
    # same kernels on the same inputs: the bits agree, not only the bars
    for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "hit_chi2"):
        np.testing.assert_array_equal(getattr(got, name), getattr(ref, name), err_msg=f"{label}: {name}")


@pytest.mark.gpu
def test_static_workspace_matches_the_caller_workspace_path_on_two_calls_in_a_row():
    # call 1: the headline kind of batch (30 surfaces, material, filter + RTS), dense hit lists, near the size limit
    wl1 = W.make_config(2, n_tracks=4099, seed=901)
    opt = B.make_options(**wl1.options)
    assert B.workspace_bytes(wl1.n_tracks, wl1.geometry.shape[0] - 1 - wl1.start_surface, opt) <= B.STATIC_WORKSPACE_BYTES
    got1, ref1 = _pair(wl1)
    _assert_same(got1, ref1, "static call 1 (cfg2)")
    assert np.all(got1.n_used >= 3)

    # call 2, straight after: a ragged batch with outliers and a grid field, forced through the length sort, all
    # per-leg states out -- it finds call 1's records, leg counts and sort counters in the array
    wl2 = W.make_config(4, n_tracks=1531, seed=902)
    over = dict(length_sort=B.SORT_ON, output_states=B.STATES_PRED | B.STATES_FILT | B.STATES_SMOOTH)
    got2, ref2 = _pair(wl2, **over)
    _assert_same(got2, ref2, "static call 2 (cfg4, sorted)", states=True)
    assert len(np.unique(np.diff(wl2.offsets))) > 1  # really ragged

    # and call 1's batch once more on top of call 2's leftovers, in the paper's mixed precision (float records)
    got3, ref3 = _pair(wl1, precision=B.PRECISION_MIXED)
    _assert_same(got3, ref3, "static call 3 (cfg2, mixed)")


@pytest.mark.gpu
def test_static_workspace_empty_batch_is_the_set_up_call():
    import torch
    wl = W.make_config(0, n_tracks=64, seed=903)
    db = B.DeviceBatch(B.HostBatch.from_workload(wl))
    call = B.StaticFitCall(db)
    call.tracks.n_tracks = 0
    call.meas.n_meas = 0
    call.run()
    assert call.launches == 0
    torch.cuda.synchronize()


def test_static_workspace_refuses_a_batch_beyond_its_size_before_touching_the_gpu():
    """Host arithmetic only (runs without a GPU): HOST dummy pointers, the call must return before any CUDA call."""
    n = 6000  # x 30 legs of FP64 records = 79 MB > 64 MiB
    buf = np.zeros(64)
    p = buf.ctypes.data
    tr = B.KfTracksIn(n, p, p, 0)
    ms = B.KfMeasurements(0, p, p, p, None, None)
    ge = B.KfGeometry(31, p, 14.0, 28.0855, 2.329, 173.0)
    fl = B.KfField()
    op = B.default_options()
    out = B.KfOutputs()
    for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "ndf", "status", "n_used",
                 "n_outliers", "n_holes"):
        setattr(out, name, p)
    L = B.lib()
    assert B.workspace_bytes(n, 30, op) > B.STATIC_WORKSPACE_BYTES
    rc = L.kf_fit_batch_static(C.byref(tr), C.byref(ms), C.byref(ge), C.byref(fl), C.byref(op), C.byref(out), None)
    assert rc == -5
    msg = L.kf_status_string(rc).decode()
    assert "64 MiB" in msg and "kf_fit_batch" in msg
    assert np.all(buf == 0.0)
    # the ordinary argument checks come first and are those of kf_fit_batch
    op.n_corr_steps = 9
    assert L.kf_fit_batch_static(C.byref(tr), C.byref(ms), C.byref(ge), C.byref(fl), C.byref(op), C.byref(out), None) == -1
    with pytest.raises(kf.KfError):
        raise kf.KfError(-5)
