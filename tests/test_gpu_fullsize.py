"""Full-size runs in the launch configuration bench.py times (FitCall on resident inputs, minimal
outputs): EVERY track is re-fitted by the oracle (first_*, last_*, chi2, ndf, counters, status, per-hit flags and
chi2 of all 1e6 tracks, north_star "1,000,000 tracks x 30 surfaces ... matches the CPU oracle"),
the per-leg states on a 1 % sample (tracks are independent, so a subset reproduces the per-track
results), and properties that hold at any size are checked on all tracks.  parity.whole_population prints the worst
factor of the bars and its 99.99th percentile per quantity and lists any track whose discrete decisions differ."""
import numpy as np
import pytest

import oracle
import parity
import paper_2105_01796_b200 as kf
from paper_2105_01796_b200 import workloads as W

pytestmark = pytest.mark.gpu


def run_full(wl):
    import torch
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    # the launch configuration bench.py times: minimal outputs (no RKN error diagnostic) -> the PLAIN forward kernel
    hb = db.host
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False)
    call = kf.FitCall(db, out=out)
    call.run()
    torch.cuda.synchronize()
    ragged = wl.n_meas != wl.n_tracks * (wl.geometry.shape[0] - 1 - wl.start_surface)
    sort = 3 if (ragged and wl.n_tracks >= 8192) else 0  # the length sort's three kernels (AUTO)
    assert call.launches == (2 if wl.options["smooth"] else 1) + sort
    return call.out.to_host()


def full_parity(wl, got, seed):
    """all tracks against the oracle; per-leg states of a 1 % sample"""
    rep, _ = parity.whole_population(wl, got, wl.name)
    parity.state_sample(wl, wl.name, fraction=0.01, seed=seed)
    return rep


def common_properties(wl, got):
    ok = (got.status & 7) == 0
    assert ok.mean() > 0.999
    d_first = np.einsum("nii->ni", got.first_cov)
    d_last = np.einsum("nii->ni", got.last_cov)
    assert np.all(d_first[ok] > 0) and np.all(d_last[ok] > 0)
    assert np.all(np.isfinite(got.chi2[ok])) and np.all(got.chi2 >= 0)
    np.testing.assert_array_equal(got.ndf, 2 * got.n_used - 5)
    counts = np.diff(wl.offsets)
    np.testing.assert_array_equal((got.n_used + got.n_outliers)[ok], counts[ok])


def test_cfg1_full_size():
    wl = W.make_config(1)
    got = run_full(wl)
    full_parity(wl, got, 1)
    common_properties(wl, got)
    assert np.all(got.status == 0) and np.all(got.n_used == 10)
    # consistent informative prior: E[chi2] = 2n (reading U10)
    assert abs(got.chi2.mean() - 20.0) < 4 * np.sqrt(40.0 / wl.n_tracks)


def test_cfg2_full_size_bench_configuration():
    wl = W.make_config(2)
    assert wl.n_tracks == 1_000_000 and wl.n_meas == 30_000_000
    got = run_full(wl)
    full_parity(wl, got, 2)
    common_properties(wl, got)
    assert np.all(got.status == 0) and np.all(got.n_used == 30) and np.all(got.n_holes == 0)
    assert abs(got.chi2.mean() - 60.0) < 4 * np.sqrt(120.0 / wl.n_tracks)
    # pulls of the filtered state at the last layer against truth entering that layer: unit width
    pull = (got.last_params - wl.truth[:, -1, :]) / np.sqrt(np.einsum("nii->ni", got.last_cov))
    assert np.all(np.abs(pull[:, :5].mean(0)) < 0.01)
    assert np.all(np.abs(pull[:, :5].std(0) - 1.0) < 0.01)
    spull = (got.first_params - wl.truth[:, 0, :]) / np.sqrt(np.einsum("nii->ni", got.first_cov))
    assert np.all(np.abs(spull[:, :5].std(0) - 1.0) < 0.01)


def test_cfg3_full_size_ragged_with_outliers():
    wl = W.make_config(3)
    got = run_full(wl)
    full_parity(wl, got, 3)
    common_properties(wl, got)
    # nearly all injected noise hits are far from the track and must be flagged
    n_true = int(wl.is_outlier.sum())
    assert got.n_outliers.sum() > 0.97 * n_true
    assert got.n_outliers.sum() < 1.02 * n_true + 3e-3 * wl.n_meas


def test_cfg4_full_size_field_map():
    """BASELINE.json configs[4] at its full size (1,000,000 ragged tracks in the grid field, length-sorted): all
    tracks against the oracle, properties on all; then the same batch with the field's acceptance box staged in shared
    memory (kf_field.stage_*): integers and flags identical, every value within 1 % of the parity bars of the unstaged
    run (another instantiation of the same arithmetic: the compiler's FMA contraction differs in places)."""
    import torch
    wl = W.make_config(4)
    assert wl.n_tracks == 1_000_000
    got = run_full(wl)
    full_parity(wl, got, 4)
    common_properties(wl, got)
    assert np.any(got.status & 32)   # the planes beyond x = 400 mm lie outside the table: clamped lookups
    lengths = got.n_used + got.n_outliers + got.n_holes
    assert lengths.min() >= 0 and lengths.max() == 30 and 10 < lengths.mean() < 16
    # pulls of the filtered state at the last visited layer against truth entering that layer: unit width
    ok = ((got.status & 7) == 0) & (got.n_used >= 5)
    last = np.clip(lengths - 1, 0, 29)
    truth_last = wl.truth[np.arange(wl.n_tracks), last, :]
    pull = (got.last_params - truth_last) / np.sqrt(np.einsum("nii->ni", got.last_cov))
    assert np.all(np.abs(pull[ok][:, :5].mean(0)) < 0.02)
    assert np.all(np.abs(pull[ok][:, :5].std(0) - 1.0) < 0.02)
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    hb = db.host
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False)
    call = kf.FitCall(db, out=out, field_stage=True)
    assert call.field.stage_n[0] >= 2   # the hint was derived from the geometry's half lengths
    call.run()
    torch.cuda.synchronize()
    staged = call.out.to_host()
    rep = parity.compare(staged, got)   # exact on ndf, counters, flags, status
    assert max(rep.values()) < 0.01, rep
