"""The MIXED-precision path (kf_options.precision; the paper's operating point: single precision
except the matrix inversion) against the FLOAT build of the oracle and against the double oracle.

Bars: float arithmetic (eps = 6e-8) on coordinates that reach 1e3 mm against resolutions
of 1e-2 mm moves a fitted parameter by up to a few per cent of its own standard deviation; two float evaluations that
order their operations differently (the oracle's dense loops, the kernel's closed-form step and FMA chains) are each
that far from the double fit and up to twice that from one another.  So, in units of the reference's sigma:
    against the double oracle   |dx| <= 0.05 sigma, |dC_ii/C_ii| <= 1e-3 (the bounds the float ORACLE is pinned to in
                                tests/test_oracle_precision.py), |dchi2| <= 0.1: chi2 = sum of (r/sigma)^2 over up to 30 hits
                                moves by 2 sum |r/sigma| (d/sigma) with d/sigma ~ 0.02 per hit and random signs, i.e.
                                ~ 2 sqrt(30) 0.02 = 0.2 at worst, 0.03 measured with the default stepping, 0.065 with five
                                primary steps per leg (max_step_mm = 7: five times the roundings of the position)
    against the float oracle    twice those.
Integers, flags and status are exact except on tracks where a hit's chi2 lies within 0.1 of the outlier cut (counted,
at most a handful per batch).  `pytest -m gpu`."""
import numpy as np
import pytest

import oracle
import parity
import paper_2105_01796_b200 as kf
from paper_2105_01796_b200 import binding as B
from paper_2105_01796_b200 import workloads as W

pytestmark = pytest.mark.gpu
MIXED = B.PRECISION_MIXED


BARS = dict(params_sigma=0.05, var_rel=1e-3, chi2_abs=0.1)


def check(got, ref64, ref32, wl_offsets, cut=0.0, label=""):
    """The bars above hold for the configs' own options.  Options that worsen the conditioning of the fit (an inflated
    prior: kappa = C-_ii / C+_ii grows with it and float loses kappa * 6e-8; a fit without the process noise its hits were
    generated with) move the FLOAT ORACLE itself beyond them; there a bar is widened to twice the float oracle's own
    distance from the double fit, and no further (the same rule as parity.arbitrated)."""
    a = parity.resolution_loss(got, ref64, wl_offsets, cut=cut)
    b = parity.resolution_loss(got, ref32, wl_offsets, cut=cut)
    o = parity.resolution_loss(ref32, ref64, wl_offsets, cut=cut)
    assert a["flipped_tracks"] <= 3 and b["flipped_tracks"] <= 3, (label, a, b)
    for k, bar in BARS.items():
        lim = max(bar, 2.0 * o[k])
        assert a[k] < lim, (label, "vs double", k, a[k], lim, "float oracle:", o[k])
        assert b[k] < 2.0 * lim, (label, "vs float oracle", k, b[k], 2.0 * lim)
    return a, b, o


def per_leg_states(got, ref64, kinds=("pred", "filt", "smooth")):
    ok = (ref64.status & 7) == 0
    worst = 0.0
    for kind in kinds:
        g, r = getattr(got, kind + "_params"), getattr(ref64, kind + "_params")
        if g is None or r is None:
            continue
        np.testing.assert_array_equal(np.isnan(g[ok]), np.isnan(r[ok]))
        sig = np.sqrt(np.einsum("nlii->nli", getattr(ref64, kind + "_cov")))
        d = g - r
        d[..., 2] = (d[..., 2] + np.pi) % (2 * np.pi) - np.pi
        with np.errstate(invalid="ignore"):
            worst = max(worst, float(np.nanmax(np.abs(d[ok]) / sig[ok])))
            vr = np.einsum("nlii->nli", getattr(got, kind + "_cov"))[ok] / np.einsum("nlii->nli", getattr(ref64, kind + "_cov"))[ok]
        assert np.nanmax(np.abs(vr - 1.0)) < 1e-3, kind
    return worst


@pytest.mark.parametrize("cfg,n", [(0, 1000), (0, 3001), (1, 20003), (2, 5003), (3, 5003), (4, 5003)])
def test_mixed_precision_config_parity_all_states(cfg, n):
    wl = W.make_config(cfg, n_tracks=n)
    ref64 = oracle.fit_workload(wl, states=True)
    ref32 = oracle.fit_workload(wl, states=True, precision="f32")
    got = kf.fit_workload(wl, states=True, precision=MIXED)
    assert B.lib().kf_last_launch_count() == (2 if wl.options.get("smooth", 1) else 1) + (3 if (cfg == 4 and n >= 8192) else 0)
    a, b, o = check(got, ref64, ref32, wl.offsets, cut=float(wl.options.get("outlier_chi2", 0.0)), label=f"cfg{cfg}")
    assert all(o[k] < BARS[k] for k in BARS), o      # nothing was widened on the configs themselves
    assert per_leg_states(got, ref64) < 0.05
    # the outputs are float values widened to double
    np.testing.assert_array_equal(got.first_cov, got.first_cov.astype(np.float32).astype(np.float64))
    np.testing.assert_array_equal(got.chi2, got.chi2.astype(np.float32).astype(np.float64))


def test_mixed_precision_plain_and_general_instantiations_agree():
    """minimal outputs -> the PLAIN instantiation (what bench.py --precision mixed times); all states -> the general one."""
    wl = W.make_config(2, n_tracks=45000, seed=8)
    hb = kf.HostBatch.from_workload(wl)
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False)
    plain = kf.FitCall(kf.DeviceBatch(hb), out=out, precision=MIXED).run().to_host()
    gen = kf.fit_workload(wl, states=True, precision=MIXED)
    ref64 = oracle.fit_workload(wl)
    a = parity.resolution_loss(plain, ref64, wl.offsets)
    assert a["flipped_tracks"] == 0 and a["params_sigma"] < 0.05 and a["var_rel"] < 1e-3 and a["chi2_abs"] < 0.05, a
    b = parity.resolution_loss(plain, gen, wl.offsets)
    assert b["params_sigma"] < 0.05 and b["chi2_abs"] < 0.05, b


@pytest.mark.parametrize("over", [
    dict(n_corr_steps=1), dict(max_step_mm=7.0), dict(step_tolerance_mm=1e-4), dict(smooth=0), dict(material=0),
    dict(outlier_chi2=6.0), dict(mass_gev=0.13957), dict(cov_inflation=10.0),
])
def test_mixed_precision_options(over):
    wl = W.make_config(3, n_tracks=2051, seed=77)
    ref64 = oracle.fit_workload(wl, states=True, **over)
    ref32 = oracle.fit_workload(wl, states=True, precision="f32", **over)
    got = kf.fit_workload(wl, states=True, precision=MIXED, **over)
    cut = float(over.get("outlier_chi2", wl.options.get("outlier_chi2", 0.0)))
    check(got, ref64, ref32, wl.offsets, cut=cut, label=str(over))


def test_mixed_precision_per_hit_variances_sorted_and_perigee():
    wl = W.make_config(4, n_tracks=9001, seed=5)
    rng = np.random.default_rng(3)
    M = wl.n_meas
    var = np.stack([rng.uniform(0.5e-4, 4e-4, M), rng.uniform(4e-4, 16e-4, M)], axis=1)
    line = ((0.0, 0.0, 0.0), (0.0, 0.0, 1.0))
    fld, opt = oracle.field_of(wl), oracle.options_of(wl)
    refs = {}
    for prec in ("f64", "f32"):
        r = oracle.fit_batch(wl.params0, wl.cov0, 0, wl.offsets, wl.surf_idx, wl.loc, wl.geometry, fld, opt, var=var,
                             precision=prec)
        refs[prec] = oracle.perigee_batch(r, wl.geometry, 0, fld, opt, *line, precision=prec)
    hb = kf.HostBatch.from_arrays(wl.params0, wl.cov0, 0, wl.offsets, wl.surf_idx, wl.loc, wl.geometry, field_kind="grid3",
                                  grid_n=wl.grid_n, grid_origin=wl.grid_origin, grid_spacing=wl.grid_spacing, grid=wl.grid,
                                  var=var, options=wl.options)
    for sort in (B.SORT_OFF, B.SORT_ON):
        call = kf.FitCall(kf.DeviceBatch(hb), perigee=line, precision=MIXED, length_sort=sort)
        got = call.run().to_host()
        check(got, refs["f64"], refs["f32"], wl.offsets, label=f"sort {sort}")
        ok = (refs["f64"].status == 0) & (got.status == 0)
        sig = np.sqrt(np.einsum("nii->ni", refs["f64"].perigee_cov))[ok]
        assert np.max(np.abs(got.perigee_params - refs["f64"].perigee_params)[ok] / sig) < 0.05


def test_mixed_precision_status_bits_and_degenerate_tracks():
    wl = W.make_config(2, n_tracks=600, seed=31)
    N = wl.n_tracks
    params0, cov0 = wl.params0.copy(), wl.cov0.copy()
    surf = [wl.surf_idx[wl.offsets[i]:wl.offsets[i + 1]].copy() for i in range(N)]
    locs = [wl.loc[wl.offsets[i]:wl.offsets[i + 1]].copy() for i in range(N)]
    surf[3], locs[3] = surf[3][:0], locs[3][:0]                  # no hits
    surf[4], locs[4] = surf[4][:1], locs[4][:1]                  # one hit: ndf <= 0
    surf[5] = surf[5][::-1].copy()                               # descending: BAD_HITS
    params0[8, 4] = 1.0 / 0.03                                   # 30 MeV: curls up, surface unreachable
    params0[10, 2] = np.pi / 2                                   # moving parallel to the planes
    params0[11, 0] = np.nan                                      # NaN input
    surf[13], locs[13] = surf[13][5:9], locs[13][5:9]            # leading holes
    cov0[14] = -cov0[14]                                         # negative covariance
    params0[15, 4] = 1.0 / 0.0601                                # stops by energy loss somewhere
    offsets = np.zeros(N + 1, np.int32)
    np.cumsum([len(s) for s in surf], out=offsets[1:])
    surf_idx, loc = np.concatenate(surf).astype(np.int32), np.concatenate(locs)
    fld = oracle.make_field("const", (0, 0, 2.0))
    opt = oracle.make_options(material=1, smooth=1, outlier_chi2=15.0)
    ref32 = oracle.fit_batch(params0, cov0, 0, offsets, surf_idx, loc, wl.geometry, fld, opt, precision="f32")
    hb = kf.HostBatch.from_arrays(params0, cov0, 0, offsets, surf_idx, loc, wl.geometry, options=dict(material=1, smooth=1, outlier_chi2=15.0))
    got = kf.fit_batch(hb, precision=MIXED).to_host()
    np.testing.assert_array_equal(got.status, ref32.status)
    np.testing.assert_array_equal(got.n_used, ref32.n_used)
    np.testing.assert_array_equal(got.hit_flags, ref32.hit_flags)
    assert ref32.status[3] == 8 and ref32.status[5] & 64 and ref32.status[8] & 1 and ref32.status[11] & 1 and ref32.status[14] & 2


def test_mixed_precision_through_the_host_entry_points():
    import torch
    wl = W.make_config(3, n_tracks=3001, seed=43)
    ref64 = oracle.fit_workload(wl)
    ref32 = oracle.fit_workload(wl, precision="f32")
    for ns, chunk in ((0, 0), (3, 256)):
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True, n_streams=ns, chunk_tracks=chunk, precision=MIXED)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        check(got, ref64, ref32, wl.offsets, cut=15.0, label=f"host S={ns}")


def test_mixed_precision_option_rules():
    wl = W.make_config(1, n_tracks=300)
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    for over in (dict(variant=B.VARIANT_LANES_PER_TRACK), dict(smoother=B.SMOOTHER_BRYSON_FRAZIER)):
        with pytest.raises(kf.KfError) as e:
            kf.FitCall(db, precision=MIXED, **over).run()
        assert e.value.rc == -2
    # AUTO on a small batch takes the thread-per-track kernels (the lanes variant is FP64 only)
    got = kf.fit_workload(wl, precision=MIXED)
    ref64 = oracle.fit_workload(wl)
    a = parity.resolution_loss(got, ref64, wl.offsets)
    assert a["params_sigma"] < 0.05


def test_mixed_precision_full_size_cfg2_pulls():
    """BASELINE.json configs[2] at full size in the launch configuration bench.py --precision mixed times: unit-width
    pulls (the paper's own validation of its single-precision fit), E[chi2] = 2n, and all tracks
    re-fitted by the double oracle."""
    import torch
    wl = W.make_config(2)
    hb = kf.HostBatch.from_workload(wl)
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False)
    call = kf.FitCall(kf.DeviceBatch(hb), out=out, precision=MIXED)
    call.run()
    torch.cuda.synchronize()
    assert call.launches == 2
    got = call.out.to_host()
    assert np.all(got.status == 0) and np.all(got.n_used == 30)
    assert abs(got.chi2.mean() - 60.0) < 4 * np.sqrt(120.0 / wl.n_tracks) + 0.01
    pull = (got.last_params - wl.truth[:, -1, :]) / np.sqrt(np.einsum("nii->ni", got.last_cov))
    assert np.all(np.abs(pull[:, :5].mean(0)) < 0.01) and np.all(np.abs(pull[:, :5].std(0) - 1.0) < 0.01)
    spull = (got.first_params - wl.truth[:, 0, :]) / np.sqrt(np.einsum("nii->ni", got.first_cov))
    assert np.all(np.abs(spull[:, :5].std(0) - 1.0) < 0.01)
    ref64 = oracle.fit_workload(wl)   # every track, not a sample
    g, sub = got, wl
    a = parity.resolution_loss(g, ref64, sub.offsets)
    print("\n[mixed, all 1e6 tracks of cfg2 against the double oracle]", a)
    assert a["flipped_tracks"] == 0 and a["params_sigma"] < 0.05 and a["var_rel"] < 1e-3 and a["chi2_abs"] < 0.05, a
