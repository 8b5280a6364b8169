"""Parity of the general path of the CUDA library with the oracle: surfaces of any kind (planes, cylinders, discs;
kf_geometry.surface_kinds, U33) and the field-gradient terms of the transported Jacobian
(kf_options.field_gradient, U32).  Same bars as everywhere (tests/parity.py)."""
import dataclasses

import numpy as np
import pytest

import oracle
import parity
import paper_2105_01796_b200 as kf
from paper_2105_01796_b200 import binding as B
from paper_2105_01796_b200 import workloads as W

pytestmark = pytest.mark.gpu

Z_AXIS = ((0.0, 0.0, 0.0), (0.0, 0.0, 1.0))


def both(wl, states=True, **over):
    ref = oracle.fit_workload(wl, states=states, **over)
    got = kf.fit_workload(wl, states=states, **over)
    return got, ref


def in_cfg4_grid(wl):
    n, origin, spacing, grid = W.cfg4_field_grid()
    return dataclasses.replace(wl, field_kind="grid3", grid_n=n, grid_origin=origin, grid_spacing=spacing, grid=grid)


@pytest.mark.parametrize("kind,n", [("barrel", 5003), ("endcap", 5003), ("barrel", 130), ("endcap", 1)])
def test_cylinders_and_discs_parity_all_states(kind, n):
    wl = W.make_tracker(kind, n_tracks=n)
    got, ref = both(wl, states=True)
    rep = parity.assert_parity(got, ref, states=True, label=kind)
    assert np.all(ref.status == 0)
    assert max(rep.values()) < 0.05, rep
    np.testing.assert_allclose(got.rk_err_max, ref.rk_err_max, rtol=1e-6, atol=1e-18)
    if n > 1000:   # the GPU fit's own pulls against the truth on the last cylinder / disc
        pull = (got.last_params - wl.truth[:, -1, :]) / np.sqrt(np.einsum("nii->ni", got.last_cov))
        assert np.all(np.abs(pull.std(0) - 1.0) < 0.05)
        assert abs(got.chi2.mean() - 20.0) < 0.5


@pytest.mark.parametrize("kind", ["barrel", "endcap"])
def test_general_surfaces_options_and_filter_only(kind):
    wl = W.make_tracker(kind, n_tracks=1501, seed=21)
    for over in (dict(smooth=0), dict(material=0), dict(max_step_mm=7.0), dict(step_tolerance_mm=1e-7), dict(n_corr_steps=3),
                 dict(cov_inflation=100.0, outlier_chi2=12.0)):
        got, ref = both(wl, states=True, **over)
        loosen = 1.0
        if "cov_inflation" in over:   # conditioning of the inflated prior: bars from the long-double arbiter
            ld = oracle.fit_workload(wl, states=True, precision="ld", **over)
            parity.arbitrated(got, ref, ld, states=True, label=f"{kind} {over}")
            continue
        rep = parity.assert_parity(got, ref, states=True, label=f"{kind} {over}", loosen=loosen)
        assert max(rep.values()) < 0.1, (over, rep)


def test_mixed_kinds_in_a_grid_field_with_holes_and_perigee():
    """plane -> cylinders in the CFG4 table (lookups clamped beyond x = 400 mm... the barrel reaches 300 mm), hits missing
    on random layers (CSR lists of different lengths, length sort under AUTO), perigee of the smoothed first state."""
    wl = in_cfg4_grid(W.make_tracker("barrel", n_tracks=9001, seed=33))
    rng = np.random.default_rng(5)
    keep = rng.random(wl.n_meas) < 0.9
    counts = np.add.reduceat(keep.astype(np.int64), wl.offsets[:-1])
    off = np.zeros(wl.n_tracks + 1, np.int32)
    np.cumsum(counts, out=off[1:])
    wl = dataclasses.replace(wl, offsets=off, surf_idx=wl.surf_idx[keep].copy(), loc=wl.loc[keep].copy())
    for over in (dict(), dict(field_gradient=1)):
        ref = oracle.fit_workload(wl, states=True, perigee=Z_AXIS, **over)
        got = kf.fit_workload(wl, states=True, perigee=Z_AXIS, **over)
        rep = parity.assert_parity(got, ref, states=True, label=f"barrel in grid {over}")
        assert max(rep.values()) < 0.1, rep
        assert np.any(got.n_holes > 0)


@pytest.mark.parametrize("cfg,n", [(4, 5003), (4, 257)])
def test_field_gradient_terms_parity(cfg, n):
    wl = W.make_config(cfg, n_tracks=n)
    got, ref = both(wl, states=True, field_gradient=1)
    rep = parity.assert_parity(got, ref, states=True, label="cfg4 with gradient terms")
    assert max(rep.values()) < 0.05, rep
    # the terms change the covariances (and through the gain the states), not the bookkeeping
    plain = kf.fit_workload(wl, states=True)
    np.testing.assert_array_equal(plain.n_used, got.n_used)
    np.testing.assert_allclose(plain.pred_params[:, 0, :], got.pred_params[:, 0, :], rtol=1e-12, atol=1e-12)  # first leg: same state
    assert np.nanmax(np.abs(plain.pred_cov[:, 0] - got.pred_cov[:, 0])) > 0
    sig = np.sqrt(np.einsum("nii->ni", plain.first_cov))
    ok = (plain.status & 7) == 0
    assert 0 < np.max(np.abs(plain.first_params - got.first_params)[ok] / sig[ok]) < 0.05


def test_field_gradient_in_a_strongly_non_uniform_table_and_constant_field():
    wl = W.make_config(4, n_tracks=2001, seed=9)
    n, origin, spacing, grid = W.cfg4_field_grid()
    rng = np.random.default_rng(3)
    grid = grid.copy()
    grid[..., 0] = 0.3 * rng.standard_normal(grid.shape[:-1])     # node-to-node noise: kinks everywhere
    grid[..., 1] = 0.3 * rng.standard_normal(grid.shape[:-1])
    grid[..., 2] *= 1.0 + 0.2 * rng.standard_normal(grid.shape[:-1])
    wl2 = dataclasses.replace(wl, grid=grid)
    got, ref = both(wl2, states=True, field_gradient=1)
    rep = parity.assert_parity(got, ref, states=True, label="noisy table with gradient terms")
    assert max(rep.values()) < 0.2, rep
    # constant field: the option is accepted and changes nothing (the plane-only kernels run)
    wl1 = W.make_config(2, n_tracks=1001)
    a = kf.fit_workload(wl1, field_gradient=1)
    b = kf.fit_workload(wl1)
    for name in ("first_params", "first_cov", "last_cov", "chi2"):
        np.testing.assert_array_equal(getattr(a, name), getattr(b, name))


def test_general_path_through_the_host_entry_points():
    import torch
    wl = W.make_tracker("barrel", n_tracks=3001, seed=12)
    ref = oracle.fit_workload(wl, perigee=Z_AXIS)
    for kw in (dict(), dict(n_streams=3, chunk_tracks=512)):
        call = kf.HostCall(kf.HostBatch.from_workload(wl), per_hit=True, perigee=Z_AXIS, **kw)
        call.run()
        torch.cuda.synchronize()
        got = call.to_host()
        got.rk_err_max = None
        parity.assert_parity(got, ref, label=f"host barrel {kw}")
    wl4 = W.make_config(4, n_tracks=2001, seed=13)
    ref = oracle.fit_workload(wl4, field_gradient=1)
    call = kf.HostCall(kf.HostBatch.from_workload(wl4), per_hit=True, field_gradient=1)
    call.run()
    torch.cuda.synchronize()
    got = call.to_host()
    got.rk_err_max = None
    parity.assert_parity(got, ref, label="host cfg4 gradient")


def test_general_path_option_rules():
    wl = W.make_tracker("endcap", n_tracks=300)
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    for over in (dict(variant=2), dict(smoother=1)):
        with pytest.raises(kf.KfError) as e:
            kf.FitCall(db, **over).run()
        assert e.value.rc == -2, over
    with pytest.raises(kf.KfError) as e:
        kf.FitCall(db, field_gradient=2).run()
    assert e.value.rc == -1
    wl4 = W.make_config(4, n_tracks=300)
    db4 = kf.DeviceBatch(kf.HostBatch.from_workload(wl4))
    for over in (dict(precision=B.PRECISION_MIXED), dict(variant=2), dict(smoother=1)):
        with pytest.raises(kf.KfError) as e:
            kf.FitCall(db4, field_gradient=1, **over).run()
        assert e.value.rc == -2, over
    # a small batch under AUTO takes the thread-per-track general kernels (not the lanes variant)
    kf.FitCall(db).run()
    assert B.lib().kf_last_launch_count() == 2
    # a track that cannot reach the next cylinder (moving along the axis): stopped with bit 1, same on both sides
    wlb = W.make_tracker("barrel", n_tracks=64, seed=3)
    wlb.params0[5, 3] = 1e-9          # theta -> 0: along z, the cylinder axis
    wlb.params0[9, 2] = np.pi         # heading back through the start plane: n.T < 0 ... the cylinder is still ahead
    got, ref = both(wlb, states=False)
    parity.assert_parity(got, ref, label="degenerate barrel")
    assert got.status[5] & 1


# ---- randomised trackers: mixed kinds, tilted axes, random fields, holes, options -------------------------------------
def _frame(u, v):
    u = np.asarray(u, float) / np.linalg.norm(u)
    v = np.asarray(v, float)
    v = v - u * (u @ v)
    v /= np.linalg.norm(v)
    return u, v, np.cross(u, v)


def random_tracker(seed):
    """Start plane near x = 0, then surfaces of random kinds ordered so that a track along +x meets them in index order:
    cylinders of growing radius around a slightly tilted, slightly off-origin axis ~ z; planes and discs with normal ~ x
    at growing x (the disc's centre far off in -y so that rho stays well above zero and alpha away from +-pi)."""
    rng = np.random.default_rng(7000 + seed)
    L = int(rng.integers(3, 12))
    g = np.zeros((L + 1, 20))
    reach = 0.0
    for k in range(L + 1):
        kind = 0 if k == 0 else int(rng.choice([0, 1, 2], p=[0.25, 0.45, 0.3]))
        reach += rng.uniform(15.0, 40.0) if k else 0.0
        t1, t2 = rng.uniform(-0.08, 0.08, 2)
        if kind == 1:      # cylinder: axis ~ z, azimuth zero along ~ x
            u, v, n = _frame((t1, 1.0, t2), (t2, -t1, 1.0))
            g[k, 0:3] = (rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-1, 1))
            g[k, 12:14] = (reach, 500.0)
        elif kind == 2:    # disc: normal ~ x, centre displaced along -y: rho ~ 150 mm, alpha ~ +pi/2
            u, v, n = _frame((t1, 1.0, 0.0), (t2, 0.0, 1.0))
            g[k, 0:3] = (reach, -150.0 + rng.uniform(-5, 5), rng.uniform(-2, 2))
            g[k, 12:14] = 300.0
        else:
            u, v, n = _frame((t1, 1.0, 0.0), (t2, 0.0, 1.0))
            g[k, 0:3] = (reach, rng.uniform(-2, 2), rng.uniform(-2, 2))
            g[k, 12:14] = 50.0
        g[k, 3:6], g[k, 6:9], g[k, 9:12], g[k, 18] = u, v, n, kind
        if k and rng.random() < 0.7:
            g[k, 14] = rng.uniform(5e-4, 1e-2)
            g[k, 15] = g[k, 14] * 93.7
        g[k, 16:18] = (rng.uniform(0.005, 0.05) ** 2, (rng.uniform(0.005, 0.05) if kind != 2 else rng.uniform(5e-5, 3e-4)) ** 2)
    fkind = rng.choice(["const", "grid3"], p=[0.6, 0.4])
    if fkind == "grid3":
        n = np.array([int(rng.integers(8, 16)), int(rng.integers(5, 9)), int(rng.integers(5, 9))])
        origin = np.array([-30.0, -70.0, -70.0])
        spacing = np.array([(reach + 80.0) / (n[0] - 1), 140.0 / (n[1] - 1), 140.0 / (n[2] - 1)])
        grid = rng.uniform(-0.2, 0.2, (n[2], n[1], n[0], 3))
        grid[..., 2] += rng.uniform(1.0, 2.5)
        field = dict(field_kind="grid3", grid_n=n, grid_origin=origin, grid_spacing=spacing, grid=grid)
        fld = oracle.make_field("grid3", grid_n=n, grid_origin=origin, grid_spacing=spacing, grid=grid)
    else:
        b = tuple(rng.uniform(-0.4, 0.4, 2)) + (rng.choice([-1, 1]) * rng.uniform(0.5, 3.0),)
        field = dict(field_kind="const", field_b=b)
        fld = oracle.make_field("const", b)
    N = int(rng.integers(40, 400))
    p = np.exp(rng.uniform(np.log(0.6), np.log(40.0), N))
    x0 = np.stack([rng.uniform(-3, 3, N), rng.uniform(-3, 3, N), rng.uniform(-0.15, 0.15, N),
                   np.pi / 2 + rng.uniform(-0.15, 0.15, N), rng.choice([-1.0, 1.0], N) / p, rng.uniform(0, 50, N)], axis=1)
    sig = np.array([0.1, 0.1, 2e-3, 2e-3, 0.0, 300.0])[None, :].repeat(N, 0)
    sig[:, 4] = 0.03 * np.abs(x0[:, 4])
    cov0 = np.zeros((N, 6, 6))
    for a in range(6):
        cov0[:, a, a] = sig[:, a] ** 2
    opts = dict(smooth=int(rng.random() < 0.8), material=int(rng.random() < 0.7), outlier_chi2=float(rng.choice([0.0, 15.0])),
                n_corr_steps=int(rng.integers(1, 4)), max_step_mm=float(rng.choice([np.inf, np.inf, 11.0])),
                step_tolerance_mm=float(rng.choice([0.0, 0.0, 1e-6])), mass_gev=0.1056583755, cov_inflation=float(rng.choice([1.0, 4.0])),
                field_gradient=int(fkind == "grid3" and rng.random() < 0.5))
    opt0 = oracle.make_options()
    offsets, surf, loc = [0], [], []
    eff = rng.uniform(0.8, 1.0)
    for i in range(N):
        x = x0[i].copy()
        for k in range(0, L):
            pr = oracle.propagate(fld, opt0, x, g[k], g[k + 1])     # truth hits: input generation only
            if pr.rc != 0:
                break
            x = pr.x
            if rng.random() < eff:
                surf.append(k + 1)
                loc.append(x[:2] + rng.standard_normal(2) * np.sqrt(g[k + 1, 16:18]))
        offsets.append(len(surf))
    params0 = x0 + rng.standard_normal((N, 6)) * sig * 0.7
    return dict(params0=params0, cov0=cov0, offsets=np.array(offsets, np.int32), surf_idx=np.array(surf, np.int32),
                loc=np.array(loc).reshape(-1, 2), geom=g, field=field, fld=fld, opts=opts, kinds=sorted(set(g[:, 18].astype(int))))


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("KF_TRACKER_SEEDS", "16"))))
def test_random_tracker_parity(seed):
    c = random_tracker(seed)
    opt = oracle.make_options(**c["opts"])
    ref = oracle.fit_batch(c["params0"], c["cov0"], 0, c["offsets"], c["surf_idx"], c["loc"], c["geom"], c["fld"], opt, states=True)
    oracle.perigee_batch(ref, c["geom"], 0, c["fld"], opt, *Z_AXIS)
    hb = kf.HostBatch.from_arrays(c["params0"], c["cov0"], 0, c["offsets"], c["surf_idx"], c["loc"], c["geom"],
                                  options=c["opts"], **c["field"])
    smooth = c["opts"]["smooth"]
    states = B.STATES_PRED | B.STATES_FILT | (B.STATES_SMOOTH if smooth else 0)
    for sort in (B.SORT_OFF, B.SORT_ON):
        out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, states, perigee=True)
        call = kf.FitCall(kf.DeviceBatch(hb), out=out, perigee=Z_AXIS, length_sort=sort, output_states=states)
        got = call.run().to_host()
        label = f"tracker seed {seed} kinds {c['kinds']} sort {sort} opts {c['opts']}"
        # tracks whose fit ran away (a hit list that stops constraining a low-momentum track) carry no digits
        with np.errstate(invalid="ignore"):
            wide = np.nan_to_num(np.einsum("nlii->nli", ref.pred_cov)[..., :2], nan=0.0, posinf=1e99).max(axis=(1, 2)) > 1e4
        ok = ~wide
        rep = parity.assert_parity(got, ref, states=True, sel=ok, label=label, offsets=c["offsets"])
        assert max(rep.values()) < 0.5, (label, rep)
    assert (ref.status[ok] & 7 == 0).mean() > 0.9


@pytest.mark.parametrize("kind", ["barrel", "endcap"])
def test_cylinders_and_discs_in_mixed_precision(kind):
    """kf_options.precision = MIXED on surfaces of other kinds: against the float build of the oracle and the double oracle,
    with the bars of tests/test_gpu_mixed.py (sigma units; widened only as far as the float oracle itself is from the
    double fit)."""
    import test_gpu_mixed as TM
    wl = W.make_tracker(kind, n_tracks=5003, seed=5)
    ref64 = oracle.fit_workload(wl, states=True)
    ref32 = oracle.fit_workload(wl, states=True, precision="f32")
    got = kf.fit_workload(wl, states=True, precision=B.PRECISION_MIXED)
    assert B.lib().kf_last_launch_count() == 2
    a, b, o = TM.check(got, ref64, ref32, wl.offsets, label=kind)

    def per_leg(x):   # worst |dx| / sigma and worst relative change of a variance over all per-leg states, against the double fit
        wp, wv = 0.0, 0.0
        for nm in ("pred", "filt", "smooth"):
            d = getattr(x, nm + "_params") - getattr(ref64, nm + "_params")
            d[..., 2] = (d[..., 2] + np.pi) % (2 * np.pi) - np.pi
            va = np.einsum("nlii->nli", getattr(ref64, nm + "_cov"))
            wp = max(wp, float(np.nanmax(np.abs(d) / np.sqrt(va))))
            wv = max(wv, float(np.nanmax(np.abs(np.einsum("nlii->nli", getattr(x, nm + "_cov")) / va - 1.0))))
        return wp, wv

    (gp, gv), (op_, ov) = per_leg(got), per_leg(ref32)
    # the same rule as TM.check: the fixed bars, widened only as far as twice the float ORACLE's own distance from the double
    # fit (the polar chart of a disc divides by rho: its alpha variance is the most sensitive entry)
    assert gp < max(0.05, 2.0 * op_) and gv < max(1e-3, 2.0 * ov), (gp, gv, op_, ov)
    np.testing.assert_array_equal(got.first_cov, got.first_cov.astype(np.float32).astype(np.float64))
    pull = (got.last_params - wl.truth[:, -1, :]) / np.sqrt(np.einsum("nii->ni", got.last_cov))
    assert np.all(np.abs(pull.std(0) - 1.0) < 0.05)


@pytest.mark.parametrize("kind", ["barrel", "endcap"])
def test_tracker_workloads_at_a_million_tracks(kind):
    """the launch configuration `bench.py --config 5|6` times: all tracks re-fitted by the oracle, per-leg states of a 1 % sample, properties on all"""
    import torch
    wl = W.make_tracker(kind, n_tracks=1_000_000)
    db = kf.DeviceBatch(kf.HostBatch.from_workload(wl))
    hb = db.host
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False)
    call = kf.FitCall(db, out=out)
    call.run()
    torch.cuda.synchronize()
    assert call.launches == 2
    got = call.out.to_host()
    parity.whole_population(wl, got, kind + " 1e6")        # every track against the oracle
    parity.state_sample(wl, kind + " 1e6", fraction=0.01, seed=8)
    assert np.all(got.status == 0) and np.all(got.n_used == 10)
    assert abs(got.chi2.mean() - 20.0) < 4 * np.sqrt(40.0 / wl.n_tracks)
    pull = (got.last_params - wl.truth[:, -1, :]) / np.sqrt(np.einsum("nii->ni", got.last_cov))
    assert np.all(np.abs(pull[:, :5].mean(0)) < 0.01) and np.all(np.abs(pull[:, :5].std(0) - 1.0) < 0.01)


@pytest.mark.parametrize("kind", ["barrel", "endcap"])
def test_hits_across_the_branch_cut_of_an_angular_coordinate(kind):
    """U33: a hit is taken on the branch of its periodic coordinate nearest the prediction, in the forward kernel and -- through
    the record, which keeps the hit as used -- in the RTS kernel's re-filtering.  The chart turned by pi (tracks cross at
    alpha ~ +-pi) with a third of the hits given a whole period off, against the oracle and against the original chart."""
    from test_oracle_surfaces import across_the_branch_cut
    wl = W.make_tracker(kind, n_tracks=3001, seed=17)
    wl2 = across_the_branch_cut(wl, kind)
    ang = 0 if kind == "barrel" else 1
    shift = (2 * np.pi * wl.geometry[wl2.surf_idx, 12]) if kind == "barrel" else np.full(wl2.n_meas, 2 * np.pi)
    wl2.loc[::3, ang] += shift[::3]
    wl2.loc[1::7, ang] -= 2 * shift[1::7]
    got, ref = both(wl2, states=True)
    rep = parity.assert_parity(got, ref, states=True, label=kind + " across the cut")
    assert max(rep.values()) < 0.1, rep
    assert np.all(got.status == 0) and np.all(got.n_used == 10)
    base = kf.fit_workload(wl, states=True)
    np.testing.assert_allclose(got.chi2, base.chi2, rtol=1e-8, atol=1e-8)
    other = [k for k in range(6) if k != ang]
    np.testing.assert_allclose(got.first_params[:, other], base.first_params[:, other], rtol=1e-8, atol=1e-9)


def test_cylinder_behind_the_start_point_stops_the_track_like_the_oracle():
    """kf_fit.h KF_SURFACE_CYLINDER "reached ... from inside" (pin PS11 on the oracle side): tracks that start outside the
    first cylinder -- moving away, moving inwards, missing it -- stop with KF_ST_PROPAGATION on both sides instead of
    stepping backwards; the tracks that start inside are fitted as before.  Status and counters exact, values at the bars."""
    rng = np.random.default_rng(77)
    def rec(kind, radius):
        s = np.zeros(20)
        s[3:6], s[6:9], s[9:12] = (0, 1, 0), (0, 0, 1), (1, 0, 0)   # plane x = 0: loc0 = y, loc1 = z; cylinders: axis z
        s[12:14], s[16:18], s[18] = (radius, 500.0), (1e-4, 1e-4), kind
        return s
    geom = np.stack([rec(0, 50.0), rec(1, 60.0), rec(1, 80.0)])
    n = 640
    y0 = np.where(np.arange(n) % 4 == 0, rng.uniform(-20, 20, n), rng.uniform(90, 120, n))      # a quarter starts inside
    phi = np.choose(np.arange(n) % 4, [rng.uniform(-0.3, 0.3, n), np.full(n, np.pi / 2), np.full(n, -np.pi / 2),
                                       rng.uniform(-0.05, 0.05, n)])                           # ahead, away, inwards, missing
    params0 = np.stack([y0, rng.uniform(-5, 5, n), phi, np.pi / 2 + rng.uniform(-0.1, 0.1, n),
                        rng.choice([-1.0, 1.0], n) / rng.uniform(0.5, 5.0, n), np.zeros(n)], axis=1)
    cov0 = np.tile(np.diag([0.05, 0.05, 1e-3, 1e-3, 0.01 * 0.5, 1.0]) ** 2, (n, 1, 1))
    offsets = np.arange(0, 2 * n + 1, 2, dtype=np.int32)
    surf_idx = np.tile(np.array([1, 2], np.int32), n)
    loc = rng.normal(0.0, 5.0, (2 * n, 2))
    opts = dict(smooth=1, material=0)
    hb = kf.HostBatch.from_arrays(params0, cov0, 0, offsets, surf_idx, loc, geom, field_kind="const", field_b=(0, 0, 2.0),
                                  options=opts)
    got = kf.FitCall(kf.DeviceBatch(hb)).run().to_host()
    ref = oracle.fit_batch(params0, cov0, 0, offsets, surf_idx, loc, geom, oracle.make_field("const", (0, 0, 2.0)),
                           oracle.make_options(**opts))
    outside = np.arange(n) % 4 != 0
    assert np.all(ref.status[outside] & 1) and np.all(ref.n_used[outside] == 0)
    assert np.all(ref.status[~outside] & 1 == 0) and np.all(ref.n_used[~outside] == 2)
    parity.assert_parity(got, ref, label="cylinder behind the start point")


def test_gpu_helix_to_cylinder_closed_form_without_the_oracle():
    """A pin of the CUDA path's cylinder chart, crossing and landing that does not go through the oracle (whose surface
    helpers follow the same decomposition as the kernel's): in B = (0, 0, 2 T) the per-leg PRED state on a cylinder
    around z must be the closed-form helix from the previous state, with the crossing found here by bisection on
    |r_T(s)| = R.  Leg 0 starts from the start parameters on a plane; leg 1 starts from the kernel's own FILTERED state on
    the first cylinder, mapped to space with the chart's definition written out below (include/kf_fit.h KF_SURFACE_CYLINDER)."""
    TESLA, M_MU, BZ = 2.99792458e-4, 0.1056583755, 2.0
    rng = np.random.default_rng(5)
    n = 3000
    def rec(kind, radius):
        s = np.zeros(20)
        s[3:6], s[6:9], s[9:12] = (0, 1, 0), (0, 0, 1), (1, 0, 0)   # plane x = 0: loc0 = y, loc1 = z; cylinders: axis z
        s[12:14], s[16:18], s[18] = (radius, 500.0), (1e-4, 1e-4), kind
        return s
    R1, R2 = 40.0, 75.0
    geom = np.stack([rec(0, 50.0), rec(1, R1), rec(1, R2)])

    def helix(x0, y0, z0, phi, theta, lam, s):
        kappa = -lam * BZ * TESLA / np.sin(theta)
        half = 0.5 * kappa * s
        chord = s * np.sinc(half / np.pi)
        return x0 + chord * np.cos(phi + half), y0 + chord * np.sin(phi + half), z0 + s / np.tan(theta), phi + kappa * s

    def to_cylinder(x0, y0, z0, phi, theta, lam, t, R):
        lo, hi = np.zeros_like(x0), np.full_like(x0, 300.0)
        for _ in range(80):
            mid = 0.5 * (lo + hi)
            x, y, _, _ = helix(x0, y0, z0, phi, theta, lam, mid)
            inside = x * x + y * y < R * R
            lo, hi = np.where(inside, mid, lo), np.where(inside, hi, mid)
        s = 0.5 * (lo + hi)
        x, y, z, phi1 = helix(x0, y0, z0, phi, theta, lam, s)
        t1 = t + s / np.sin(theta) * np.sqrt(1.0 + (M_MU * lam) ** 2)
        return np.stack([R * np.arctan2(y, x), z, phi1, theta, lam, t1], axis=1)

    y0, z0 = rng.uniform(-10, 10, n), rng.uniform(-5, 5, n)
    phi, theta = rng.uniform(-0.5, 0.5, n), rng.uniform(1.2, 1.9, n)
    lam = rng.choice([-1.0, 1.0], n) / np.exp(rng.uniform(np.log(0.5), np.log(10.0), n))
    params0 = np.stack([y0, z0, phi, theta, lam, np.full(n, 1.5)], axis=1)
    want0 = to_cylinder(np.zeros(n), y0, z0, phi, theta, lam, params0[:, 5], R1)
    hit1 = want0[:, :2] + rng.normal(0, 0.01, (n, 2))
    hit2 = to_cylinder(np.zeros(n), y0, z0, phi, theta, lam, params0[:, 5], R2)[:, :2] + rng.normal(0, 0.01, (n, 2))
    cov0 = np.tile(np.diag([0.05, 0.05, 1e-3, 1e-3, 0.01 * 0.5, 1.0]) ** 2, (n, 1, 1))
    offsets = np.arange(0, 2 * n + 1, 2, dtype=np.int32)
    loc = np.stack([hit1, hit2], axis=1).reshape(-1, 2)
    hb = kf.HostBatch.from_arrays(params0, cov0, 0, offsets, np.tile(np.array([1, 2], np.int32), n), loc, geom,
                                  field_kind="const", field_b=(0, 0, BZ), options=dict(smooth=1, material=0, max_step_mm=2.0))
    call = kf.FitCall(kf.DeviceBatch(hb), output_states=B.STATES_PRED | B.STATES_FILT)
    assert call.geom.surface_kinds == 0b11
    got = call.run().to_host()
    assert np.all(got.status & 7 == 0)
    tol = np.array([2e-9, 2e-9, 1e-10, 1e-12, 1e-15, 1e-8])
    d0 = np.abs(got.pred_params[:, 0, :] - want0)
    assert np.all(d0 <= tol), d0.max(axis=0)
    # leg 1: from the kernel's filtered state on cylinder 1 (chart: alpha = loc0 / R from n = x towards u = y)
    f = got.filt_params[:, 0, :]
    a = f[:, 0] / R1
    want1 = to_cylinder(R1 * np.cos(a), R1 * np.sin(a), f[:, 1], f[:, 2], f[:, 3], f[:, 4], f[:, 5], R2)
    d1 = np.abs(got.pred_params[:, 1, :] - want1)
    assert np.all(d1 <= tol), d1.max(axis=0)
