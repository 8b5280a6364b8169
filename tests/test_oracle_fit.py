"""Pins for the oracle's whole-track fit (P5-P9, P12) and its edge cases.

Nothing here compares the oracle with itself: truth comes from the generator's closed-form
helix, least-squares references are solved with numpy, statistics are fixed by theory.  CPU only.
"""
import numpy as np
import pytest

import oracle
from paper_2105_01796_b200 import workloads as W

M_MU = 0.1056583755


def diag_of(C):
    return np.einsum("...ii->...i", C)


# ---- P5: noiseless recovery ------------------------------------------------------------------------
def test_p5_noiseless_recovery():
    wl = W.make_config(1, n_tracks=300, sig=(0.0, 0.0))
    wl.params0 = wl.truth_start.copy()  # start = truth
    wl.geometry[:, 16:18] = (0.01 ** 2, 0.01 ** 2)  # the fitter still assumes 10 um
    r = oracle.fit_workload(wl, states=True)
    assert np.all(r.status == 0)
    # residuals are the stepper's landing error (<= 5e-7 mm at 0.5 GeV, P1) over 10 um: chi2 <~ 1e-8
    assert np.max(r.chi2) <= 1e-8
    for arr in (r.pred_params, r.filt_params, r.smooth_params):
        d = np.abs(arr - wl.truth)
        assert np.max(d[..., 0:2]) < 1e-6  # limited by the stepper (P1): <= 5e-7 mm at 0.5 GeV
        assert np.max(d[..., 2:4]) < 5e-9  # <= 6e-10 per leg at 0.5 GeV, accumulated over 10 legs
        assert np.max(d[..., 4]) < 2e-8  # the ~1e-7 mm residuals feed back into q/p through the gain
        assert np.max(d[..., 5]) < 1e-5  # path-length error <= 5e-7 mm per leg, accumulated
    np.testing.assert_array_equal(r.first_params, r.smooth_params[:, 0])
    np.testing.assert_array_equal(r.last_params, r.filt_params[:, -1])


# ---- P6: straight tracks at zero field == brute-force weighted least squares -------------------------
def test_p6_zero_field_weighted_least_squares():
    # The extended filter linearises y' = y + dx tan(phi) at its current estimate, so it equals the
    # exact linear regression only up to ~ dx * slope * (angle error)^2.  Hit noise of 0.1 / 0.3 um
    # and a 1e-5 rad start error keep that below 1e-9 mm, which makes the comparison sharp.
    # The prior is made uninformative (0.5 mm / 10 mrad against 0.1 um hits: weight ratio 2.5e7)
    # but not astronomically wide: C+ = (I - KH) C- loses eps * (prior var / hit var) relative
    # accuracy by cancellation, so a 1e8 inflation would itself cost 1e-3 in the covariance.
    rng = np.random.default_rng(21)
    L, N = 8, 200
    S0, S1 = 1e-4, 3e-4
    geom = W.telescope_geometry(L, 30.0, 50.0, 0.0, 0.0, (S0, S1))
    xs = 30.0 * np.arange(1, L + 1)
    y0, z0 = rng.uniform(-1, 1, N), rng.uniform(-1, 1, N)
    ty, tz = rng.uniform(-0.1, 0.1, N), rng.uniform(-0.1, 0.1, N)
    Y = y0[:, None] + ty[:, None] * xs[None, :] + rng.standard_normal((N, L)) * S0
    Z = z0[:, None] + tz[:, None] * xs[None, :] + rng.standard_normal((N, L)) * S1
    phi = np.arctan2(ty, 1.0)
    theta = np.arccos(tz / np.sqrt(1 + ty ** 2 + tz ** 2))
    params0 = np.stack([y0, z0, phi, theta, np.full(N, 0.5), np.zeros(N)], axis=1)
    params0[:, :4] += rng.standard_normal((N, 4)) * np.array([1e-4, 1e-4, 1e-5, 1e-5])
    cov0 = np.zeros((N, 6, 6))
    cov0[:, range(6), range(6)] = np.array([0.05, 0.05, 1e-3, 1e-3, 5e-3, 300.0]) ** 2
    offsets = (np.arange(N + 1) * L).astype(np.int32)
    surf_idx = np.tile(np.arange(1, L + 1, dtype=np.int32), N)
    loc = np.stack([Y.ravel(), Z.ravel()], axis=1)
    fld = oracle.make_field("const", (0, 0, 0))
    opt = oracle.make_options(smooth=1, cov_inflation=1e2)
    r = oracle.fit_batch(params0, cov0, 0, offsets, surf_idx, loc, geom, fld, opt, states=True)
    assert np.all(r.status == 0)
    # direct linear regression per projection: parameters (value at the last plane, slope)
    xl = xs[-1]
    A = np.stack([np.ones(L), xs - xl], axis=1)
    for proj, data, sig, ip in ((0, Y, S0, 0), (1, Z, S1, 1)):
        cov_ls = np.linalg.inv(A.T @ A) * sig ** 2
        sol = (np.linalg.inv(A.T @ A) @ A.T @ data.T).T  # (N, 2): value at last plane, slope
        np.testing.assert_allclose(r.last_params[:, ip], sol[:, 0], rtol=0, atol=1e-9)
        # slopes from the fitted angles: T ~ (1, ty, tz)
        ph, th = r.last_params[:, 2], r.last_params[:, 3]
        slope = np.tan(ph) if proj == 0 else np.cos(th) / (np.sin(th) * np.cos(ph))
        np.testing.assert_allclose(slope, sol[:, 1], rtol=0, atol=1e-10)
        np.testing.assert_allclose(r.last_cov[:, ip, ip], cov_ls[0, 0], rtol=1e-6)
        # slope variance through the angle Jacobian
        if proj == 0:
            var_slope = r.last_cov[:, 2, 2] / np.cos(ph) ** 4
            np.testing.assert_allclose(var_slope, cov_ls[1, 1], rtol=2e-4)
            np.testing.assert_allclose(r.last_cov[:, 0, 2] / np.cos(ph) ** 2, cov_ls[0, 1], rtol=2e-4)
    # chi2 == residual sum of squares of the regression (prior is uninformative)
    rss = np.zeros(N)
    for data, sig in ((Y, S0), (Z, S1)):
        sol = (np.linalg.inv(A.T @ A) @ A.T @ data.T).T
        rss += (((data - sol @ A.T) / sig) ** 2).sum(axis=1)
    np.testing.assert_allclose(r.chi2, rss, rtol=2e-5)
    # the smoothed state at the first plane equals the regression evaluated there
    A1 = np.stack([np.ones(L), xs - xs[0]], axis=1)
    sol1 = (np.linalg.inv(A1.T @ A1) @ A1.T @ Y.T).T
    np.testing.assert_allclose(r.first_params[:, 0], sol1[:, 0], rtol=0, atol=1e-9)
    np.testing.assert_allclose(r.first_cov[:, 0, 0], (np.linalg.inv(A1.T @ A1) * S0 ** 2)[0, 0], rtol=1e-6)


# ---- P7: KF + RTS == global linear least squares on the affine model the filter used ------------------
def _global_lsq(wl, i, r, material):
    """Solve, with numpy, the least-squares problem over z = (x_0, w_1 .. w_{n-1}) whose recursive
    solution is the Kalman filter + RTS smoother: prior on x_0, one 2-D residual per hit, one 2-D
    scattering pseudo-measurement w_k ~ N(0, Q_k) per layer; states are affine in z through the
    linearisation points the filter used (x+_k) and the step functions' Jacobians."""
    fld, opt = oracle.field_of(wl), oracle.options_of(wl)
    n = wl.n_layers
    nz = 6 + 2 * (n - 1)
    x0, C0 = wl.params0[i], wl.cov0[i]
    a = np.zeros((n, 6))
    B = np.zeros((n, 6, nz))
    pr = oracle.propagate(fld, opt, x0, wl.geometry[0], wl.geometry[1])
    a[0] = pr.x - pr.J @ x0
    B[0][:, :6] = pr.J
    Qs = []
    for k in range(1, n):
        xf = r.filt_params[i, k - 1]
        surf = wl.geometry[k]
        if material:
            mt = oracle.material(opt, surf, xf, r.filt_cov[i, k - 1])
            x_after, g = mt.x, mt.g
            Qs.append(np.array([mt.theta0 ** 2 / np.sin(xf[3]) ** 2, mt.theta0 ** 2]))
        else:
            x_after, g = xf, 1.0
            Qs.append(None)
        G = np.diag([1, 1, 1, 1, g, 1.0])
        pr = oracle.propagate(fld, opt, x_after, wl.geometry[k], wl.geometry[k + 1])
        E = np.zeros((6, nz))
        E[2, 6 + 2 * (k - 1)] = 1.0
        E[3, 6 + 2 * (k - 1) + 1] = 1.0
        # x_{k+1} = x-_{k+1} + J [ G (x_k - x+_k) + E w_k ]
        a[k] = pr.x + pr.J @ G @ (a[k - 1] - xf)
        B[k] = pr.J @ (G @ B[k - 1] + (E if material else 0.0))
    rows, rhs = [], []
    s0 = np.sqrt(np.diag(C0))
    P = np.zeros((6, nz))
    P[:, :6] = np.diag(1 / s0)
    rows.append(P)
    rhs.append(x0 / s0)
    sig = np.sqrt(wl.geometry[1, 16:18])
    o = wl.offsets[i]
    for k in range(n):
        rows.append(B[k][:2] / sig[:, None])
        rhs.append((wl.loc[o + k] - a[k][:2]) / sig)
    scale = np.ones(nz)
    scale[:6] = s0
    for k in range(1, n):
        Rw = np.zeros((2, nz))
        if material:
            sd = np.sqrt(Qs[k - 1])
            Rw[0, 6 + 2 * (k - 1)] = 1 / sd[0]
            Rw[1, 6 + 2 * (k - 1) + 1] = 1 / sd[1]
            scale[6 + 2 * (k - 1): 6 + 2 * k] = sd
        else:
            Rw[0, 6 + 2 * (k - 1)] = Rw[1, 6 + 2 * (k - 1) + 1] = 1.0  # pins w = 0
        rows.append(Rw)
        rhs.append(np.zeros(2))
    A = np.vstack(rows) * scale[None, :]
    b = np.concatenate(rhs)
    Q_, R_ = np.linalg.qr(A)
    zs = np.linalg.solve(R_, Q_.T @ b)
    Rinv = np.linalg.inv(R_)
    cov_z = (Rinv @ Rinv.T) * np.outer(scale, scale)
    z = zs * scale
    xs_ = np.array([a[k] + B[k] @ z for k in range(n)])
    Cs_ = np.array([B[k] @ cov_z @ B[k].T for k in range(n)])
    return xs_, Cs_


@pytest.mark.parametrize("cfg,material", [(1, False), (2, True)])
def test_p7_kf_rts_equals_global_least_squares(cfg, material):
    wl = W.make_config(cfg, n_tracks=12, layers=8) if cfg == 2 else W.make_config(cfg, n_tracks=12)
    r = oracle.fit_workload(wl, states=True)
    assert np.all(r.status == 0)
    floors = np.array([1.0, 1.0, 0.1, 1.0, 0.01, 1.0])
    for i in range(wl.n_tracks):
        xs_, Cs_ = _global_lsq(wl, i, r, material)
        dx = np.abs(r.smooth_params[i] - xs_) / np.maximum(np.abs(xs_), floors)
        assert dx.max() < 1e-9, dx.max()
        sd = np.sqrt(diag_of(Cs_))
        dC = np.abs(r.smooth_cov[i] - Cs_) / (sd[:, :, None] * sd[:, None, :])
        assert dC.max() < 1e-7, dC.max()
        # the last filtered state is the last smoothed one
        np.testing.assert_array_equal(r.smooth_params[i, -1], r.filt_params[i, -1])


# ---- P8: invariants ---------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_p8_covariance_invariants(cfg):
    wl = W.make_config(cfg, n_tracks=400)
    r = oracle.fit_workload(wl, states=True)
    nleg = r.n_used + r.n_outliers + r.n_holes
    assert np.all((r.status & 7) == 0)
    assert np.all(r.hit_chi2 >= 0)
    for i in range(wl.n_tracks):
        n = nleg[i]
        if n == 0:
            continue
        Cp, Cf, Cs = r.pred_cov[i, :n], r.filt_cov[i, :n], r.smooth_cov[i, :n]
        for C in (Cp, Cf, Cs):
            assert np.array_equal(C, np.swapaxes(C, 1, 2))
            s = np.sqrt(diag_of(C))
            corr = C / (s[:, :, None] * s[:, None, :])
            assert np.linalg.eigvalsh(corr).min() > 0
        s = np.sqrt(diag_of(Cp))
        d1 = (Cp - Cf) / (s[:, :, None] * s[:, None, :])
        assert np.linalg.eigvalsh(d1).min() > -1e-10  # filtered <= predicted
        assert np.all(np.sum(np.linalg.eigvalsh(d1) > 1e-9, axis=1) <= 2)  # rank <= 2
        s = np.sqrt(diag_of(Cf))
        d2 = (Cf - Cs) / (s[:, :, None] * s[:, None, :])
        assert np.linalg.eigvalsh(d2).min() > -1e-9  # smoothed <= filtered
        assert np.array_equal(r.smooth_params[i, n - 1], r.filt_params[i, n - 1])
        assert np.all(np.isnan(r.pred_params[i, n:]))
    assert np.all(diag_of(r.first_cov) <= diag_of(r.filt_cov[:, 0]) * (1 + 1e-12))
    assert np.all(r.ndf == 2 * r.n_used - 5)


# ---- P9: statistics on smeared data -------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n_layers", [(0, 6), (1, 10), (2, 30)])
def test_p9_chi2_and_pulls(cfg, n_layers):
    N = 10000 if cfg < 2 else 6000
    wl = W.make_config(cfg, n_tracks=N)
    n = n_layers
    for infl, expect in ((1.0, 2 * n), (1e4, 2 * n - 5)):
        r = oracle.fit_workload(wl, smooth=1, cov_inflation=infl)
        assert np.all(r.status == 0)
        se = r.chi2.std() / np.sqrt(N)
        assert abs(r.chi2.mean() - expect) < 3.5 * se, (infl, r.chi2.mean(), expect, se)
        for fitted, cov, truth in ((r.last_params, r.last_cov, wl.truth[:, -1]),
                                   (r.first_params, r.first_cov, wl.truth[:, 0])):
            pull = (fitted - truth) / np.sqrt(diag_of(cov))
            npar = 6 if infl == 1.0 else 5  # the time pull equals the prior: unit width at inflation 1 only
            assert np.all(np.abs(pull[:, :npar].mean(axis=0)) < 4.0 / np.sqrt(N))
            assert np.all(np.abs(pull[:, :npar].std(axis=0) - 1.0) < 0.035), pull.std(axis=0)


def test_p9_per_hit_chi2_is_chi2_with_two_dof():
    wl = W.make_config(1, n_tracks=5000)
    r = oracle.fit_workload(wl)
    c = r.hit_chi2.reshape(5000, 10)[:, 3:]
    assert abs(c.mean() - 2.0) < 0.03
    assert abs(np.mean(c > 5.991) - 0.05) < 0.005  # 95 % quantile of chi2(2)


# ---- P12: option limits ----------------------------------------------------------------------------------
def test_p12_limits():
    wl = W.make_config(2, n_tracks=200)
    r2 = oracle.fit_workload(wl, states=True)
    r3 = oracle.fit_workload(wl, states=True, n_corr_steps=3)
    floors = np.array([1.0, 1.0, 0.1, 1.0, 0.01, 1.0])
    d = np.abs(r3.first_params - r2.first_params) / np.maximum(np.abs(r2.first_params), floors)
    assert d.max() < 1e-12
    assert np.max(np.abs(r3.chi2 - r2.chi2) / r2.chi2) < 1e-9
    # material with x/X0 = 0 == material off, bit for bit
    wl0 = W.make_config(1, n_tracks=200)
    a = oracle.fit_workload(wl0, material=0)
    b = oracle.fit_workload(wl0, material=1)
    np.testing.assert_array_equal(a.first_params, b.first_params)
    np.testing.assert_array_equal(a.first_cov, b.first_cov)
    # mass -> 0 only alters t
    c = oracle.fit_workload(wl0, mass_gev=1e-9)
    np.testing.assert_allclose(c.first_params[:, :5], a.first_params[:, :5], rtol=1e-12, atol=1e-13)
    assert np.max(np.abs(c.first_params[:, 5] - a.first_params[:, 5])) > 1e-6
    # an outlier-free ragged track == the same track through the dense path with the cut switched off
    wl3 = W.make_config(3, n_tracks=300)
    r_cut = oracle.fit_workload(wl3)
    r_nocut = oracle.fit_workload(wl3, outlier_chi2=0.0)
    clean = r_cut.n_outliers == 0
    assert clean.sum() > 100
    np.testing.assert_array_equal(r_cut.first_params[clean], r_nocut.first_params[clean])
    np.testing.assert_array_equal(r_cut.chi2[clean], r_nocut.chi2[clean])


def test_outliers_are_flagged():
    wl = W.make_config(3, n_tracks=3000)
    r = oracle.fit_workload(wl)
    flagged = r.hit_flags == 2
    first_layer = wl.surf_idx == 1
    true_out = wl.is_outlier
    # every far-off noise hit beyond the first layer is caught; few good hits are lost
    missed = true_out & ~flagged & ~first_layer
    assert missed.sum() <= 0.02 * true_out.sum()
    good_tracks = np.repeat(r.n_used > 20, np.diff(wl.offsets))
    assert (flagged & ~true_out & good_tracks).sum() <= 3e-3 * (~true_out).sum()
    assert np.all(r.n_outliers == np.add.reduceat(flagged.astype(int), wl.offsets[:-1]))
    assert np.all(r.hit_chi2[flagged] > 15.0)
    assert np.all(r.n_used + r.n_outliers == np.diff(wl.offsets))
    assert np.all(r.n_used + r.n_outliers + r.n_holes == wl.surf_idx[wl.offsets[1:] - 1])


# ---- edge cases ----------------------------------------------------------------------------------------------
def test_edge_cases_and_status_bits():
    wl = W.make_config(2, n_tracks=6)
    L = wl.n_layers
    # track 0: no hits; track 1: hit list not ascending; track 2: parallel to the planes;
    # track 3: start covariance not positive; track 4: stops in thick material; track 5: normal
    offs = wl.offsets.copy()
    surf = wl.surf_idx.copy()
    loc = wl.loc.copy()
    keep = np.ones(surf.size, bool)
    keep[offs[0]:offs[1]] = False
    surf[offs[1] + 3] = surf[offs[1] + 2]
    wl.params0[2, 2] = np.pi / 2  # phi = 90 deg: n.T = 0
    wl.cov0[3] = -wl.cov0[3]
    new_off = np.zeros_like(offs)
    np.cumsum([(keep[offs[i]:offs[i + 1]]).sum() for i in range(6)], out=new_off[1:])
    wl.offsets, wl.surf_idx, wl.loc = new_off, surf[keep], loc[keep]
    geom = wl.geometry.copy()
    r = oracle.fit_workload(wl, states=True)
    assert r.status[0] == 8 and r.ndf[0] == -5 and r.chi2[0] == 0
    np.testing.assert_array_equal(r.first_params[0], wl.params0[0])
    np.testing.assert_array_equal(r.last_cov[0], wl.cov0[0])
    assert r.status[1] == (64 | 8) and r.n_used[1] == 0
    assert r.status[2] == (1 | 8) and r.n_used[2] == 0
    np.testing.assert_array_equal(r.last_params[2], wl.params0[2])
    assert r.status[3] & 2
    assert r.status[5] == 0 and r.n_used[5] == L
    # energy exhausted: a very soft track in very thick layers
    wl.geometry = geom.copy()
    wl.geometry[1:, 14] = 1.0
    wl.geometry[1:, 15] = 93.7
    wl.params0[4, 4] = 1 / 0.12
    r = oracle.fit_workload(wl, states=True)
    assert r.status[4] & 4
    n4 = r.n_used[4] + r.n_holes[4] + r.n_outliers[4]
    assert 1 <= n4 < L
    np.testing.assert_array_equal(r.last_params[4], r.filt_params[4, n4 - 1])
    assert np.all(np.isnan(r.filt_params[4, n4:]))


def test_thread_count_does_not_change_results():
    wl = W.make_config(3, n_tracks=500)
    a = oracle.fit_workload(wl, n_threads=1)
    b = oracle.fit_workload(wl, n_threads=4)
    assert a.threads == 1 and b.threads == 4
    np.testing.assert_array_equal(a.first_params, b.first_params)
    np.testing.assert_array_equal(a.chi2, b.chi2)


def test_subset_reproduces_per_track_results():
    wl = W.make_config(4, n_tracks=600)
    idx = np.array([5, 17, 311, 599, 42])
    a = oracle.fit_workload(wl)
    b = oracle.fit_workload(wl.subset(idx))
    np.testing.assert_array_equal(a.first_params[idx], b.first_params)
    np.testing.assert_array_equal(a.chi2[idx], b.chi2)
    np.testing.assert_array_equal(a.status[idx], b.status)


def test_rts_phi_difference_is_wrapped_over_any_number_of_turns():
    """x^s_{k+1} - x^-_{k+1} in phi is an angle difference: taken into (-pi, pi] (DESIGN.md A.7), whatever the number
    of turns between the two representations (a far-off hit that is not cut can turn the filtered phi by more than
    one), and a non-finite state ends the step instead of hanging it."""
    rng = np.random.default_rng(3)
    A = rng.standard_normal((6, 6)) * 0.1
    Cf = A @ A.T + np.eye(6) * 0.05
    F = np.eye(6) + rng.standard_normal((6, 6)) * 0.05
    Cp1 = F @ Cf @ F.T + np.eye(6) * 0.01
    xf, xp1 = rng.standard_normal(6), rng.standard_normal(6)
    xs1 = xp1 + rng.standard_normal(6) * 0.1
    Cs1 = Cp1 * 0.9
    rc0, x0, C0 = oracle.rts_step(xf, Cf, F, xp1, Cp1, xs1, Cs1)
    assert rc0 == 0
    for turns in (1, -1, 3, -5, 1000):
        shifted = xs1.copy()
        shifted[2] += 2 * np.pi * turns
        rc, x, C = oracle.rts_step(xf, Cf, F, xp1, Cp1, shifted, Cs1)
        assert rc == 0
        np.testing.assert_allclose(x, x0, rtol=0, atol=1e-9 * abs(turns))
        np.testing.assert_array_equal(C, C0)
    bad = xs1.copy()
    bad[2] = np.inf
    rc, x, C = oracle.rts_step(xf, Cf, F, xp1, Cp1, bad, Cs1)
    assert rc != 0
    bad[2] = 1e300
    rc, x, C = oracle.rts_step(xf, Cf, F, xp1, Cp1, bad, Cs1)  # returns (the loop form never did)

