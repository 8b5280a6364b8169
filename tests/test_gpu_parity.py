"""Parity of the CUDA path (through the C ABI, kf_fit_batch) with the CPU oracle, element by element
on the same seeded inputs.  Tolerances: tests/parity.py (north_star: 1e-10 / 1e-8 / 1e-9; integers,
flags and status exact).  All tests here need a B200: `pytest -m gpu`."""
import numpy as np
import pytest

import oracle
import parity
import paper_2105_01796_b200 as kf
from paper_2105_01796_b200 import binding as B
from paper_2105_01796_b200 import workloads as W

pytestmark = pytest.mark.gpu


def both(wl, states=True, **over):
    ref = oracle.fit_workload(wl, states=states, **over)
    got = kf.fit_workload(wl, states=states, **over)
    return got, ref


# ---- the five configs at sizes the oracle finishes in seconds: several CTAs and a ragged tail ----------
@pytest.mark.parametrize("cfg,n", [(0, 1000), (0, 3001), (1, 20003), (2, 5003), (3, 5003), (4, 5003)])
def test_config_parity_all_states(cfg, n):
    wl = W.make_config(cfg, n_tracks=n)
    got, ref = both(wl, states=True)
    rep = parity.assert_parity(got, ref, states=True, label=f"cfg{cfg}")
    assert np.all(ref.status[ref.n_used >= 3] & 7 == 0)
    # head-room: round-off alone leaves >= 50x margin
    assert max(rep.values()) < 0.02, rep
    np.testing.assert_allclose(got.rk_err_max, ref.rk_err_max, rtol=1e-6, atol=1e-18)


# ---- fitted parameters on the perigee surface -------------------------------
Z_AXIS = ((0.0, 0.0, 0.0), (0.0, 0.0, 1.0))
_ax = np.array([0.12, -0.2, 1.0])
TILTED_AXIS = ((1.5, -2.0, 4.0), tuple(_ax / np.linalg.norm(_ax)))


@pytest.mark.parametrize("cfg,n,line", [(1, 6001, Z_AXIS), (2, 3001, Z_AXIS), (3, 3001, TILTED_AXIS), (4, 3001, Z_AXIS),
                                        (4, 1001, TILTED_AXIS), (0, 1000, Z_AXIS)])
def test_perigee_parameters_parity(cfg, n, line):
    wl = W.make_config(cfg, n_tracks=n, seed=80 + cfg)
    ref = oracle.fit_workload(wl, perigee=line)
    got = kf.fit_workload(wl, perigee=line)
    rep = parity.assert_parity(got, ref, label=f"perigee cfg{cfg}")
    assert rep["perigee_params"] < 0.05 and rep["perigee_cov"] < 0.05, rep
    smooth = wl.options.get("smooth", 1)
    assert B.lib().kf_last_launch_count() == (3 if smooth else 2)
    ok = (got.status & 128) == 0
    assert ok.mean() > 0.99 and np.all(np.isfinite(got.perigee_params[ok]))
    if line is Z_AXIS and cfg in (1, 2):
        # the truth starts ON the axis: its perigee is (0, 0, phi, theta, q/p, 0); Fig. 5 pulls
        truth = wl.truth_start.copy()
        truth[:, [0, 1, 5]] = 0.0
        pull = (got.perigee_params - truth) / np.sqrt(np.diagonal(got.perigee_cov, axis1=1, axis2=2))
        assert np.all(np.abs(pull.mean(axis=0)) < 4.5 / np.sqrt(n)) and np.all(np.abs(pull.std(axis=0) - 1.0) < 0.05)


def test_planes_only_table_ignores_the_kind_entry_also_in_the_perigee_extrapolation():
    """include/kf_fit.h, kf_geometry.surface_kinds: with 0 or 1 the plane-only kernels run and record entry [18] is
    ignored -- by the fit and by the perigee kernel alike (it once took the first surface's chart from [18] whatever
    the dispatch said).  Junk in [18..19] must not change a bit of the result."""
    import dataclasses
    wl = W.make_config(2, n_tracks=700, seed=61)
    hb = kf.HostBatch.from_workload(wl)
    ref = kf.FitCall(kf.DeviceBatch(hb), perigee=TILTED_AXIS).run().to_host()
    geo = hb.geometry.copy()
    geo[:, 18] = np.where(np.arange(geo.shape[0]) % 2 == 0, 1.0, 2.0)   # "cylinder", "disc"
    geo[:, 19] = 12345.0
    call = kf.FitCall(kf.DeviceBatch(dataclasses.replace(hb, geometry=geo)), perigee=TILTED_AXIS)
    assert call.geom.surface_kinds > 1      # what the binding derives from the host copy of the table ...
    call.geom.surface_kinds = 1             # ... and what this caller declares instead: planes only
    got = call.run().to_host()
    assert np.all(np.isfinite(got.perigee_params[(got.status & 128) == 0]))
    for name in ("perigee_params", "perigee_cov", "first_params", "first_cov", "last_params", "last_cov", "chi2", "status"):
        np.testing.assert_array_equal(getattr(got, name), getattr(ref, name), err_msg=name)


def test_perigee_failing_tracks_and_options(variant):
    """tracks that never start (bad hit lists, NaN input), moving along the axis, stepping options."""
    wl = W.make_config(2, n_tracks=400, seed=33)
    params0 = wl.params0.copy()
    params0[5, 0] = np.nan                       # NaN input: perigee NaN, bit 128
    params0[6, 3] = 1e-13                        # along +z = along the axis: never reaches the planes, no closest approach
    surf_idx = wl.surf_idx.copy()
    surf_idx[wl.offsets[7] + 2] = 99             # malformed list: not fitted; perigee of the start state
    for over in (dict(), dict(max_step_mm=6.0, n_corr_steps=1), dict(smooth=0), dict(material=0, n_corr_steps=3)):
        hb = kf.HostBatch.from_arrays(params0, wl.cov0, 0, wl.offsets, surf_idx, wl.loc, wl.geometry, field_kind="const",
                                      field_b=(0, 0, 2.0), options=dict(wl.options, **over))
        db = kf.DeviceBatch(hb)
        call = kf.FitCall(db, perigee=Z_AXIS, variant=variant)
        got = call.run().to_host()
        fld, opt = oracle.make_field("const", (0, 0, 2.0)), oracle.make_options(**dict(wl.options, **over))
        ref = oracle.fit_batch(params0, wl.cov0, 0, wl.offsets, surf_idx, wl.loc, wl.geometry, fld, opt)
        oracle.perigee_batch(ref, wl.geometry, 0, fld, opt, *Z_AXIS)
        assert ref.status[5] & 128 and ref.status[6] & 128 and ref.status[7] & 64 and not (ref.status[7] & 128)
        healthy = np.ones(400, bool)
        healthy[5] = False
        parity.assert_parity(got, ref, sel=healthy, label=f"perigee {over}")
        np.testing.assert_array_equal(got.status, ref.status)
        assert np.all(np.isnan(got.perigee_params[5])) and np.all(np.isnan(got.perigee_cov[6]))


def test_perigee_through_the_host_entry_points():
    import torch
    wl = W.make_config(3, n_tracks=2501, seed=47)
    ref = oracle.fit_workload(wl, perigee=TILTED_AXIS)
    for ns in (0, 3):
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True, n_streams=ns, chunk_tracks=512, perigee=TILTED_AXIS)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        got.rk_err_max = None
        rep = parity.assert_parity(got, ref, label=f"host perigee S={ns}")
        assert "perigee_cov" in rep


def test_perigee_axis_must_be_a_unit_vector():
    wl = W.make_config(1, n_tracks=64)
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    with pytest.raises(kf.KfError) as e:
        kf.FitCall(db, perigee=((0, 0, 0), (0, 0, 2.0))).run()
    assert e.value.rc == -1


# ---- adaptive step count (kf_options.step_tolerance_mm, U31) ----------------------------------------
@pytest.mark.parametrize("cfg,n,tol", [(1, 4001, 1e-5), (1, 4001, 1e-8), (4, 3001, 1e-6), (2, 2001, 1e-9)])
def test_adaptive_step_count_parity(cfg, n, tol, variant):
    """tracks of one warp take different numbers of primary steps (0.5-10 GeV: 1 to 4 at 1e-5); constant field
    (closed-form estimate in the kernel) and grid field (trial step), both variants."""
    wl = W.make_config(cfg, n_tracks=n, seed=70 + cfg)
    ref = oracle.fit_workload(wl, states=True, step_tolerance_mm=tol)
    got = kf.fit_workload(wl, states=True, step_tolerance_mm=tol, variant=variant)
    parity.assert_parity(got, ref, states=True, label=f"adaptive cfg{cfg} tol={tol}")
    np.testing.assert_allclose(got.rk_err_max, ref.rk_err_max, rtol=1e-6, atol=1e-18)
    base = oracle.fit_workload(wl)
    assert ref.rk_err_max.max() < 0.2 * base.rk_err_max.max()  # the option did change the stepping


# ---- the PLAIN forward instantiation (default stepping, no optional per-leg outputs: what bench.py times) -------
@pytest.mark.parametrize("cfg,n", [(0, 3001), (1, 5001), (2, 3001), (3, 3001), (4, 3001), (2, 45000)])
@pytest.mark.parametrize("smoother", [B.SMOOTHER_RTS, B.SMOOTHER_BRYSON_FRAZIER])
def test_plain_forward_kernel_parity(cfg, n, smoother):
    wl = W.make_config(cfg, n_tracks=n, seed=30 + cfg)
    ref = oracle.fit_workload(wl, states=True)
    hb = kf.HostBatch.from_workload(wl)
    smooth = wl.options.get("smooth", 1)
    states = B.STATES_SMOOTH if (smooth and smoother == B.SMOOTHER_RTS) else 0
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, states, per_hit=True, rk_err=False)
    got = kf.FitCall(kf.DeviceBatch(hb), out=out, output_states=states, smoother=smoother,
                     variant=B.VARIANT_THREAD_PER_TRACK).run().to_host()
    ref.pred_params = ref.filt_params = None
    rep = parity.assert_parity(got, ref, states=True, label=f"plain cfg{cfg}")
    assert max(rep.values()) < 0.1, rep
    # and the general instantiation's results to round-off (another instantiation is another instruction order)
    gen = kf.fit_workload(wl, smoother=smoother, variant=B.VARIANT_THREAD_PER_TRACK)
    for name in ("status", "hit_flags", "ndf"):
        np.testing.assert_array_equal(getattr(got, name), getattr(gen, name), err_msg=name)
    gen.hit_chi2 = got.hit_chi2 = gen.hit_flags = got.hit_flags = None
    rep = parity.compare(got, gen)
    assert max(rep.values()) < 0.1, rep


# ---- backward pass in Bryson-Frazier form (kf_options.smoother): the RTS result at the first surface ----------
@pytest.mark.parametrize("cfg,n,sort", [(1, 6001, 1), (2, 3001, 1), (3, 3001, 2), (4, 3001, 2), (3, 129, 1), (2, 40000, 0)])
def test_bryson_frazier_backward_pass_matches_the_rts_oracle(cfg, n, sort):
    wl = W.make_config(cfg, n_tracks=n, seed=95 + cfg)
    ref = oracle.fit_workload(wl, perigee=Z_AXIS)
    got = kf.fit_workload(wl, perigee=Z_AXIS, smoother=B.SMOOTHER_BRYSON_FRAZIER, length_sort=sort)
    rep = parity.assert_parity(got, ref, label=f"bryson-frazier cfg{cfg}")
    assert rep["first_params"] < 0.1 and rep["first_cov"] < 0.1, rep
    # the forward pass is the same code: last_*, chi2 and flags are bit-identical to the RTS run
    rts = kf.fit_workload(wl, perigee=Z_AXIS, length_sort=sort, variant=B.VARIANT_THREAD_PER_TRACK)
    for name in ("last_params", "last_cov", "chi2", "hit_flags", "status"):
        np.testing.assert_array_equal(getattr(got, name), getattr(rts, name), err_msg=name)


def test_bryson_frazier_flags_a_cancelling_first_state():
    """a 1e4-inflated prior: C- at the first leg is ~1e7 times the smoothed covariance, the subtraction
    C- - C- Lam C- cannot hold the 1e-8 bar, and the kernel says so (status bit 256) instead of staying silent."""
    wl = W.make_config(1, n_tracks=2000, seed=17)
    got = kf.fit_workload(wl, smoother=B.SMOOTHER_BRYSON_FRAZIER, cov_inflation=1e4)
    ref = oracle.fit_workload(wl, cov_inflation=1e4)
    assert np.mean((got.status & 256) != 0) > 0.9 and np.all((got.status & ~np.uint32(256)) == ref.status)
    np.testing.assert_allclose(got.first_params, ref.first_params, rtol=1e-6, atol=1e-6)  # still the same state
    plain = kf.fit_workload(wl, smoother=B.SMOOTHER_BRYSON_FRAZIER)
    assert not np.any(plain.status & 256)


def test_bryson_frazier_through_the_host_entry_points():
    import torch
    wl = W.make_config(3, n_tracks=2501, seed=48)
    ref = oracle.fit_workload(wl, perigee=TILTED_AXIS)
    for ns, sort in ((0, B.SORT_OFF), (3, B.SORT_ON)):
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True, n_streams=ns, chunk_tracks=512, perigee=TILTED_AXIS,
                           smoother=B.SMOOTHER_BRYSON_FRAZIER, length_sort=sort, variant=B.VARIANT_THREAD_PER_TRACK)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        got.rk_err_max = None
        parity.assert_parity(got, ref, label=f"host bryson-frazier S={ns}")


def test_bryson_frazier_option_rules():
    wl = W.make_config(1, n_tracks=300)
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    for over in (dict(output_states=B.STATES_SMOOTH), dict(variant=B.VARIANT_LANES_PER_TRACK)):
        with pytest.raises(kf.KfError) as e:
            kf.FitCall(db, smoother=B.SMOOTHER_BRYSON_FRAZIER, **over).run()
        assert e.value.rc == -2
    # filter only: the option is ignored; one leg: the first-leg block still fits the workspace
    a = kf.fit_workload(wl, smooth=0, smoother=B.SMOOTHER_BRYSON_FRAZIER)
    b = kf.fit_workload(wl, smooth=0)
    np.testing.assert_array_equal(a.first_cov, b.first_cov)
    short = W.make_config(0, n_tracks=200)
    geom1 = short.geometry[:2].copy()
    keep = short.surf_idx == 1
    offs = np.arange(201, dtype=np.int32)
    hb = kf.HostBatch.from_arrays(short.params0, short.cov0, 0, offs, short.surf_idx[keep], short.loc[keep], geom1,
                                  options=dict(smooth=1, smoother=B.SMOOTHER_BRYSON_FRAZIER))
    got = kf.fit_batch(hb).to_host()
    fld, opt = oracle.make_field("const", (0, 0, 2.0)), oracle.make_options(smooth=1)
    ref = oracle.fit_batch(short.params0, short.cov0, 0, offs, short.surf_idx[keep], short.loc[keep], geom1, fld, opt)
    parity.assert_parity(got, ref, label="one leg")


# ---- length sort of ragged batches (kf_sort.cuh): same results, track by track -------------------------------
@pytest.mark.parametrize("cfg,n", [(3, 5003), (4, 5003), (4, 129), (2, 1000), (4, 9001)])
def test_length_sort_parity_all_states(cfg, n, variant):
    wl = W.make_config(cfg, n_tracks=n, seed=90 + cfg)
    ref = oracle.fit_workload(wl, states=True, perigee=Z_AXIS)
    sort = B.SORT_AUTO if n == 9001 else B.SORT_ON   # 9001 ragged tracks: AUTO sorts on its own
    got = kf.fit_workload(wl, states=True, perigee=Z_AXIS, length_sort=sort, variant=variant)
    parity.assert_parity(got, ref, states=True, label=f"sorted cfg{cfg}")
    smooth = wl.options.get("smooth", 1)
    assert B.lib().kf_last_launch_count() == 3 + (2 if smooth else 1) + 1
    off = kf.fit_workload(wl, states=True, perigee=Z_AXIS, length_sort=B.SORT_OFF, variant=variant)
    assert B.lib().kf_last_launch_count() == (2 if smooth else 1) + 1
    # a track's fit does not depend on the slot it ran in: bit for bit the unsorted run
    for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "smooth_params", "smooth_cov",
                 "perigee_params", "status", "hit_flags"):
        np.testing.assert_array_equal(getattr(got, name), getattr(off, name), err_msg=name)


def test_length_sort_degenerate_lists_and_host_chunks():
    """pipeline chunks sort independently (each has its own counters); malformed and empty lists are covered by
    test_status_bits_and_degenerate_tracks, which runs sorted."""
    import torch
    wl = W.make_config(4, n_tracks=2600, seed=12)
    ref = oracle.fit_workload(wl)
    for ns, chunk in ((0, 0), (3, 384), (2, 128)):
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True, n_streams=ns, chunk_tracks=chunk,
                           length_sort=B.SORT_ON)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        got.rk_err_max = None
        parity.assert_parity(got, ref, label=f"sorted host S={ns}")
        n_chunks = 1 if ns == 0 else (2600 + chunk - 1) // chunk
        assert call.launches == 5 * n_chunks


# ---- lanes-per-track variant (8 lanes of a warp per track): same results ------------------
@pytest.mark.parametrize("cfg,n", [(0, 1000), (1, 3001), (2, 2003), (3, 2003), (4, 2003)])
def test_lanes_per_track_variant_parity(cfg, n):
    wl = W.make_config(cfg, n_tracks=n, seed=60 + cfg)
    ref = oracle.fit_workload(wl, states=True)
    got = kf.fit_workload(wl, states=True, variant=B.VARIANT_LANES_PER_TRACK)
    rep = parity.assert_parity(got, ref, states=True, label=f"lanes cfg{cfg}")
    assert max(rep.values()) < 0.02, rep
    assert B.lib().kf_last_launch_count() == (2 if wl.options.get("smooth", 1) else 1)


@pytest.mark.parametrize("n", [1, 3, 4, 5, 15, 16, 17, 67])
def test_lanes_per_track_ragged_group_counts(n):
    """Group counts that leave warps and CTAs partly filled (4 groups per warp, 16 per CTA), failing tracks included."""
    wl = W.make_config(3, n_tracks=n, seed=200 + n)
    ref = oracle.fit_workload(wl, states=True)
    got = kf.fit_workload(wl, states=True, variant=B.VARIANT_LANES_PER_TRACK)
    parity.assert_parity(got, ref, states=True, label=f"lanes n={n}")


def test_lanes_variant_with_inflated_prior_and_options():
    wl = W.make_config(3, n_tracks=1031, seed=78)
    for over in (dict(outlier_chi2=6.0), dict(max_step_mm=7.0, n_corr_steps=1), dict(smooth=0)):
        ref = oracle.fit_workload(wl, states=True, **over)
        got = kf.fit_workload(wl, states=True, variant=B.VARIANT_LANES_PER_TRACK, **over)
        parity.assert_parity(got, ref, states=True, label=f"lanes {over}")


@pytest.mark.parametrize("n", [1, 31, 32, 33, 127, 128, 129, 257])
def test_ragged_tail_sizes(n):
    wl = W.make_config(3, n_tracks=n, seed=100 + n)
    ref = oracle.fit_workload(wl, states=True)
    for variant in (B.VARIANT_THREAD_PER_TRACK, B.VARIANT_AUTO):  # AUTO takes the lanes variant at these sizes
        got = kf.fit_workload(wl, states=True, variant=variant)
        parity.assert_parity(got, ref, states=True, label=f"n={n} variant={variant}")


def test_runs_are_bitwise_deterministic():
    wl = W.make_config(3, n_tracks=4099)
    a = kf.fit_workload(wl, states=True)
    b = kf.fit_workload(wl, states=True)
    for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "smooth_params", "smooth_cov"):
        np.testing.assert_array_equal(getattr(a, name), getattr(b, name))


# ---- option plumbing ------------------------------------------------------------------------------------
@pytest.mark.parametrize("over", [
    dict(n_corr_steps=0), dict(n_corr_steps=1), dict(n_corr_steps=3), dict(max_step_mm=7.0),
    dict(max_step_mm=11.0, n_corr_steps=1), dict(cov_inflation=10.0), dict(smooth=0), dict(material=0),
    dict(outlier_chi2=6.0), dict(mass_gev=0.13957), dict(outlier_chi2=0.0), dict(step_tolerance_mm=1e-7),
    dict(step_tolerance_mm=1e-5, max_step_mm=20.0, n_corr_steps=1),
])
def test_options_parity(over):
    wl = W.make_config(3, n_tracks=2051, seed=77)
    got, ref = both(wl, states=True, **over)
    parity.assert_parity(got, ref, states=True, label=str(over))


@pytest.mark.parametrize("cfg,n", [(1, 2000), (3, 2051)])
@pytest.mark.parametrize("inflation", [1e2, 1e4])
def test_inflated_prior_against_the_long_double_arbiter(cfg, n, inflation, variant):
    """cov_inflation = 1e4 is the uninformative-prior variant of reading U10.  The gain-form update C+ = (I - KH) C-
    cancels a 25 mm^2 prior against 1e-4 mm^2 hits and the RTS recursion cancels a prior-sized C+ against a 1e6
    times smaller C^s: kappa ~ 1e6 digits are lost in ANY double-precision evaluation, the oracle's included
    (tests/test_oracle_precision.py: the double oracle is up to 5x over the covariance bar there).  So the CUDA path
    is compared with the LONG-DOUBLE evaluation of the algorithm, and a bar is widened only as far as the double
    oracle itself is from that result (parity.arbitrated, slack 2).  At inflation 1e2 nothing is widened."""
    wl = W.make_config(cfg, n_tracks=n, seed=77)
    ref = oracle.fit_workload(wl, states=True, cov_inflation=inflation)
    ref_ld = oracle.fit_workload(wl, states=True, cov_inflation=inflation, precision="ld")
    got = kf.fit_workload(wl, states=True, cov_inflation=inflation, variant=variant)
    rep, e64 = parity.arbitrated(got, ref, ref_ld, states=True, label=f"cfg{cfg} inflation {inflation}")
    if inflation <= 1e2:
        assert max(rep.values()) < 0.05 and max(e64.values()) < 0.05, (rep, e64)
    else:
        assert max(e64.values()) < 10.0 and max(rep.values()) < 10.0, (rep, e64)


def test_filter_only_with_material_and_grid_field():
    wl = W.make_config(4, n_tracks=3001, seed=9)
    got, ref = both(wl, states=True, smooth=0)
    parity.assert_parity(got, ref, states=True)
    assert np.any(ref.status & 32)  # some tracks leave the 400 mm grid: clamped lookups (U13)
    assert got.smooth_params is None


# ---- custom inputs (each test runs once per kernel variant) ----------------------------------------------------
_VARIANT = [B.VARIANT_AUTO]


@pytest.fixture(params=[B.VARIANT_THREAD_PER_TRACK, B.VARIANT_LANES_PER_TRACK], ids=["thread", "lanes"])
def variant(request):
    _VARIANT[0] = request.param
    yield request.param
    _VARIANT[0] = B.VARIANT_AUTO


def run_arrays(params0, cov0, start, offsets, surf_idx, loc, geom, var=None, cov01=None, field=("const", (0, 0, 2.0)),
               states=True, **opts):
    fld = oracle.make_field(field[0], field[1]) if field[0] == "const" else oracle.make_field(*field)
    opt = oracle.make_options(**opts)
    ref = oracle.fit_batch(params0, cov0, start, offsets, surf_idx, loc, geom, fld, opt, var=var, cov01=cov01,
                           states=states)
    hb = kf.HostBatch.from_arrays(params0, cov0, start, offsets, surf_idx, loc, geom, field_kind=field[0],
                                  field_b=field[1] if field[0] == "const" else (0, 0, 0), var=var, cov01=cov01,
                                  options=opts)
    smooth = opts.get("smooth", 1)
    os_ = (B.STATES_PRED | B.STATES_FILT | (B.STATES_SMOOTH if smooth else 0)) if states else 0
    out = kf.fit_batch(hb, output_states=os_, variant=_VARIANT[0])
    import torch
    torch.cuda.synchronize()
    return out.to_host(), ref


def test_per_hit_variances_and_correlation(variant):
    wl = W.make_config(2, n_tracks=1500, seed=5)
    rng = np.random.default_rng(3)
    M = wl.n_meas
    var = np.stack([rng.uniform(0.5e-4, 4e-4, M), rng.uniform(4e-4, 16e-4, M)], axis=1)
    rho = rng.uniform(-0.6, 0.6, M)
    cov01 = rho * np.sqrt(var[:, 0] * var[:, 1])
    for c01 in (None, cov01):
        got, ref = run_arrays(wl.params0, wl.cov0, 0, wl.offsets, wl.surf_idx, wl.loc, wl.geometry, var=var,
                              cov01=c01, material=1, smooth=1)
        parity.assert_parity(got, ref, states=True)


def tilted_geometry(L):
    g = W.telescope_geometry(L, 30.0, 50.0, 0.0032, 0.3, (0.01, 0.03))
    rng = np.random.default_rng(8)
    for k in range(L + 1):
        a, b = rng.uniform(-0.25, 0.25, 2)
        n = np.array([np.cos(a) * np.cos(b), np.sin(a) * np.cos(b), np.sin(b)])
        u = np.cross([0.0, 0.0, 1.0], n)
        u /= np.linalg.norm(u)
        v = np.cross(n, u)
        g[k, 3:6], g[k, 6:9], g[k, 9:12] = u, v, n
    return g


def test_tilted_planes_general_field_direction_and_start_surface(variant):
    L, N = 12, 1200
    geom = tilted_geometry(L)
    rng = np.random.default_rng(12)
    start = 2
    p = np.exp(rng.uniform(np.log(0.4), np.log(20), N))
    params0 = np.stack([rng.uniform(-5, 5, N), rng.uniform(-5, 5, N), rng.uniform(-0.1, 0.1, N),
                        np.pi / 2 + rng.uniform(-0.1, 0.1, N), rng.choice([-1.0, 1.0], N) / p,
                        rng.uniform(0, 100, N)], axis=1)
    cov0 = np.zeros((N, 6, 6))
    cov0[:, range(6), range(6)] = np.array([0.5, 0.5, 5e-3, 5e-3, 0.05, 300.0]) ** 2
    cov0[:, 4, 4] = (0.05 * np.abs(params0[:, 4])) ** 2
    cov0[:, 0, 2] = cov0[:, 2, 0] = 0.3 * 0.5 * 5e-3  # a correlated start covariance
    # hits: the start parameters transported plane to plane (step-level oracle call: an input
    # generator here, never the CUDA path), smeared by the measurement resolution
    nh = L - start
    offsets = (np.arange(N + 1) * nh).astype(np.int32)
    surf_idx = np.tile(np.arange(start + 1, L + 1, dtype=np.int32), N)
    fld = oracle.make_field("const", (0.3, -0.4, 1.7))
    opt = oracle.make_options()
    loc = np.zeros((N, nh, 2))
    for i in range(N):
        x = params0[i].copy()
        for k in range(nh):
            pr = oracle.propagate(fld, opt, x, geom[start + k], geom[start + k + 1])
            assert pr.rc == 0
            x = pr.x
            loc[i, k] = x[:2]
    loc = loc.reshape(-1, 2) + rng.standard_normal((N * nh, 2)) * np.array([0.01, 0.03])
    params0 = params0 + rng.standard_normal((N, 6)) * np.sqrt(cov0[:, range(6), range(6)]) * 0.5
    got, ref = run_arrays(params0, cov0, start, offsets, surf_idx, loc, geom, field=("const", (0.3, -0.4, 1.7)),
                          material=1, smooth=1)
    parity.assert_parity(got, ref, states=True)
    assert got.pred_params.shape == (N, L - start, 6)


def test_status_bits_and_degenerate_tracks(variant):
    """empty hit lists, malformed lists, unreachable surfaces, exhausted energy, NaN input,
    one-hit tracks -- all in one batch, next to healthy tracks."""
    wl = W.make_config(2, n_tracks=600, seed=31)
    N = wl.n_tracks
    params0, cov0 = wl.params0.copy(), wl.cov0.copy()
    counts = np.diff(wl.offsets).astype(np.int64)
    surf = [wl.surf_idx[wl.offsets[i]:wl.offsets[i + 1]].copy() for i in range(N)]
    locs = [wl.loc[wl.offsets[i]:wl.offsets[i + 1]].copy() for i in range(N)]
    surf[3], locs[3] = surf[3][:0], locs[3][:0]                  # no hits
    surf[4], locs[4] = surf[4][:1], locs[4][:1]                  # one hit: ndf <= 0
    surf[5] = surf[5][::-1].copy()                               # descending: BAD_HITS
    surf[6][2] = 31                                              # out of range: BAD_HITS
    surf[7][4] = surf[7][3]                                      # repeated surface: BAD_HITS
    params0[8, 4] = 1.0 / 0.03                                   # 30 MeV: curls up, surface unreachable
    params0[9, 4] = -1.0 / 0.12                                  # 120 MeV: loses its energy in silicon? (bit 4 or 1)
    params0[10, 2] = np.pi / 2                                   # moving parallel to the planes: n.T = 0
    params0[11, 0] = np.nan                                      # NaN input
    params0[12, 3] = 1e-14                                       # theta ~ 0: along z, never reaches x planes
    surf[13], locs[13] = surf[13][5:9], locs[13][5:9]            # first hits missing: leading holes
    cov0[14] = -cov0[14]                                         # negative covariance: S not positive
    params0[15, 4] = 1.0 / 0.0601                                # stops by energy loss somewhere
    offsets = np.zeros(N + 1, np.int32)
    np.cumsum([len(s) for s in surf], out=offsets[1:])
    surf_idx = np.concatenate(surf).astype(np.int32)
    loc = np.concatenate(locs)
    got, ref = run_arrays(params0, cov0, 0, offsets, surf_idx, loc, wl.geometry, material=1, smooth=1,
                          outlier_chi2=15.0, length_sort=B.SORT_ON)
    assert ref.status[3] == 8 and ref.status[4] & 8
    assert ref.status[5] & 64 and ref.status[6] & 64 and ref.status[7] & 64
    assert ref.status[8] & 1 and ref.status[10] & 1 and ref.status[11] & 1
    assert ref.status[14] & 2
    healthy = np.ones(N, bool)
    healthy[11] = False  # NaN inputs: compare status only (NaN payloads)
    parity.assert_parity(got, ref, states=True, sel=healthy)
    np.testing.assert_array_equal(got.status, ref.status)
    np.testing.assert_array_equal(got.hit_flags, ref.hit_flags)


def test_corrupted_csr_offsets_in_device_memory(variant):
    """The CSR offsets are device data the host validation cannot see: a range that runs backwards or past n_meas
    must not be dereferenced.  Such a track gets status bit 64, keeps its start state and none of its per-hit outputs
    is written; its neighbours are fitted as if nothing had happened."""
    import torch
    wl = W.make_config(3, n_tracks=700, seed=21)
    hb = kf.HostBatch.from_workload(wl)
    for sort in (B.SORT_OFF, B.SORT_ON):
        good = kf.FitCall(kf.DeviceBatch(hb), variant=variant, length_sort=sort).run().to_host()
        db = kf.DeviceBatch(hb)
        off = hb.offsets.copy()
        off[11] = off[10] - 3             # track 10 runs backwards; track 11 starts inside track 10's hits
        off[20] = hb.n_meas + 1000        # track 19 ends past the hit arrays; track 20 starts there
        off[300] = -7                     # track 299 ends below zero; track 300 starts there
        db.offsets.copy_(torch.from_numpy(off))
        call = kf.FitCall(db, variant=variant, length_sort=sort)
        call.out.hit_chi2.fill_(-1.0)
        call.out.hit_flags.fill_(77)
        got = call.run().to_host()
        bad = np.array([10, 19, 20, 299, 300])
        assert np.all(got.status[bad] == 64 | 8), got.status[bad]
        np.testing.assert_array_equal(got.first_params[bad], wl.params0[bad])
        np.testing.assert_array_equal(got.last_cov[bad], wl.cov0[bad])
        assert np.all(got.n_used[bad] == 0)
        ok = np.ones(700, bool)
        ok[[10, 11, 19, 20, 299, 300]] = False   # track 11's list is valid CSR but not its own hits any more
        for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "status", "ndf"):
            np.testing.assert_array_equal(getattr(got, name)[ok], getattr(good, name)[ok], err_msg=name)
        ok[9] = False                            # track 11's range now overlaps track 9's last hits (their per-hit outputs)
        hits_ok = np.repeat(ok, np.diff(hb.offsets))
        np.testing.assert_array_equal(got.hit_flags[hits_ok], good.hit_flags[hits_ok])
        np.testing.assert_array_equal(got.hit_chi2[hits_ok], good.hit_chi2[hits_ok])
        for t in (19, 20, 299, 300):             # hits that belong to no well-formed range: never written
            assert np.all(got.hit_flags[hb.offsets[t]:hb.offsets[t + 1]] == 77)
            assert np.all(got.hit_chi2[hb.offsets[t]:hb.offsets[t + 1]] == -1.0)


def test_energy_exhausted_in_material(variant):
    """slow muons in zero field lose all their kinetic energy in the silicon: status bit 4, track stops,
    last_* holds the filtered state of the layer where it stopped."""
    L, N = 30, 257
    geom = W.telescope_geometry(L, 30.0, 50.0, 0.0032, 0.3, (0.01, 0.03))
    rng = np.random.default_rng(4)
    p = np.linspace(0.03, 0.09, N)
    params0 = np.stack([np.zeros(N), np.zeros(N), rng.uniform(-0.02, 0.02, N),
                        np.pi / 2 + rng.uniform(-0.02, 0.02, N), rng.choice([-1.0, 1.0], N) / p, np.zeros(N)], axis=1)
    cov0 = np.zeros((N, 6, 6))
    cov0[:, range(6), range(6)] = np.array([0.05, 0.05, 1e-3, 1e-3, 0.1, 300.0]) ** 2
    xs = 30.0 * np.arange(1, L + 1)
    Y = np.tan(params0[:, 2])[:, None] * xs[None, :] + rng.standard_normal((N, L)) * 0.01
    Z = (1.0 / np.tan(params0[:, 3]) / np.cos(params0[:, 2]))[:, None] * xs[None, :] + rng.standard_normal((N, L)) * 0.03
    offsets = (np.arange(N + 1) * L).astype(np.int32)
    surf_idx = np.tile(np.arange(1, L + 1, dtype=np.int32), N)
    loc = np.stack([Y.ravel(), Z.ravel()], axis=1)
    got, ref = run_arrays(params0, cov0, 0, offsets, surf_idx, loc, geom, field=("const", (0.0, 0.0, 0.0)),
                          material=1, smooth=1)
    assert np.sum(ref.status & 4) > 20 and np.sum(ref.status == 0) > 20
    parity.assert_parity(got, ref, states=True)


def test_empty_batch_and_small_workspace():
    import ctypes as C
    import torch
    wl = W.make_config(1, n_tracks=64)
    hb = kf.HostBatch.from_workload(wl)
    db = kf.DeviceBatch(hb)
    call = kf.FitCall(db)
    call.workspace = torch.empty(16, dtype=torch.uint8, device="cuda:0")
    with pytest.raises(kf.KfError) as e:
        call.run()
    assert e.value.rc == -3
    # zero tracks
    empty = wl.subset(np.zeros(0, dtype=np.int64))
    out = kf.fit_batch(empty)
    assert out.chi2.numel() == 0 and B.lib().kf_last_launch_count() == 0


def test_host_buffer_entry_point_matches_oracle():
    """kf_fit_batch_host: pinned host buffers in, H2D + fit + D2H enqueued by the library."""
    import torch
    for cfg, n in ((2, 3001), (4, 2001)):
        wl = W.make_config(cfg, n_tracks=n, seed=41)
        ref = oracle.fit_workload(wl)
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        got.rk_err_max = None
        parity.assert_parity(got, ref, label=f"host cfg{cfg}")
        assert call.h2d_bytes > 0 and call.d2h_bytes >= n * (54 * 8 + 8 + 20)
        assert call.launches == 2


@pytest.mark.parametrize("n_streams,chunk", [(1, 0), (3, 256), (4, 1000), (8, 128)])
def test_pipelined_host_entry_point_matches_oracle(n_streams, chunk):
    """kf_fit_batch_host_pipelined: chunks of whole 128-track CTAs over several streams, ragged
    hit lists (CFG3) and a ragged last chunk; every chunk writes its slice of the same host arrays."""
    import torch
    for cfg, n in ((3, 3001), (4, 1501)):
        wl = W.make_config(cfg, n_tracks=n, seed=43)
        ref = oracle.fit_workload(wl)
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True, n_streams=n_streams, chunk_tracks=chunk)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        got.rk_err_max = None
        parity.assert_parity(got, ref, label=f"pipelined host cfg{cfg} S={n_streams}")
        step = n if chunk == 0 and n <= 16384 else ((chunk or max(16384, n // (4 * n_streams))) + 127) // 128 * 128
        assert call.launches == 2 * ((n + step - 1) // step)
        # a second call on the same buffers is ordered after the first (fork/join on the caller's stream)
        call.run()
        torch.cuda.synchronize()
        again = call.to_host()
        assert np.array_equal(again.chi2, got.chi2) and np.array_equal(again.first_cov, got.first_cov)


def test_cuda_graph_capture_of_the_fit_replays_to_the_same_bits():
    """kf_fit_batch only enqueues (no allocation, no synchronisation, no host-side state of a fit): a call captured in a
    CUDA graph replays the whole fit -- length sort, forward, RTS, perigee -- with results identical bit for bit to the
    direct call, also after the inputs changed in place (the event-at-a-time regime)."""
    import torch
    wl = W.make_config(3, n_tracks=20_001, seed=77)
    hb = kf.HostBatch.from_workload(wl)
    db = kf.DeviceBatch(hb)
    direct = kf.FitCall(db, perigee=Z_AXIS)
    direct.run()
    torch.cuda.synchronize()
    ref = direct.out.to_host()
    call = kf.FitCall(db, perigee=Z_AXIS)
    call.run()                       # warm-up outside the capture (one-time attribute calls)
    torch.cuda.synchronize()
    for t in (call.out.first_params, call.out.first_cov, call.out.chi2, call.out.perigee_params):
        t.zero_()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        call.run(stream=torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert float(call.out.chi2.abs().sum()) == 0.0        # capture enqueued nothing
    graph.replay()
    torch.cuda.synchronize()
    got = call.out.to_host()
    for name in ("first_params", "first_cov", "last_params", "last_cov", "chi2", "ndf", "status", "n_used", "n_outliers",
                 "n_holes", "perigee_params", "perigee_cov"):
        np.testing.assert_array_equal(getattr(got, name), getattr(ref, name), err_msg=name)
    # new hits in the same buffers, same graph
    db.loc += 0.001
    graph.replay()
    torch.cuda.synchronize()
    got2 = call.out.to_host()
    direct.run()
    torch.cuda.synchronize()
    ref2 = direct.out.to_host()
    assert not np.array_equal(ref2.chi2, ref.chi2)
    for name in ("first_params", "first_cov", "chi2", "status", "perigee_params"):
        np.testing.assert_array_equal(getattr(got2, name), getattr(ref2, name), err_msg=name)
