"""Pins for the oracle's perigee step (kfo_to_line / kfo_perigee_batch; PAPER.md:70, 85, 260-264;
DESIGN.md readings U27-U30).  Each check compares with something fixed independently of the oracle:
the closed-form closest approach of a helix / a straight line to the axis, central finite differences,
a composition identity, and the unit-width pulls of Fig. 5.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2105_01796_b200 import workloads as W
from test_oracle_steps import M_MU, TESLA, tilted, xplane


def helix_perigee(x0, y0, z0, phi, theta, lam, t, bz, mass):
    """Closest approach to the z axis of the helix through (x0, y0, z0) with direction (phi, theta) in
    B = (0, 0, bz): the transverse projection is a circle with dphi/ds_T = kappa = -lam Bz / sin(theta),
    centre c = (x0 - sin(phi)/kappa, y0 + cos(phi)/kappa); the closest point lies on the ray from the
    origin through c, where the tangent angle phi_p satisfies (sin phi_p, -cos phi_p) = -sign(kappa) c/|c|."""
    kappa = -lam * bz * TESLA / np.sin(theta)
    cx, cy = x0 - np.sin(phi) / kappa, y0 + np.cos(phi) / kappa
    cn = np.hypot(cx, cy)
    sg = np.sign(kappa)
    phi_p = np.arctan2(-sg * cx / cn, sg * cy / cn)
    dphi = (phi_p - phi + np.pi) % (2 * np.pi) - np.pi
    s_t = dphi / kappa
    px, py = cx + np.sin(phi_p) / kappa, cy - np.cos(phi_p) / kappa
    d0 = -px * np.sin(phi_p) + py * np.cos(phi_p)       # D . (z^ x T)/|z^ x T|
    assert abs(abs(d0) - abs(cn - 1.0 / abs(kappa))) < 1e-9 * max(1.0, cn)
    s = s_t / np.sin(theta)
    return np.array([d0, z0 + s_t / np.tan(theta), phi_p, theta, lam, t + s * np.sqrt(1 + (mass * lam) ** 2)])


@pytest.mark.parametrize("p", [0.5, 1.0, 10.0, 100.0])
@pytest.mark.parametrize("q", [-1.0, 1.0])
def test_pp1_helix_closest_approach_to_the_axis(p, q):
    fld = oracle.make_field("const", (0, 0, 2.0))
    opt = oracle.make_options()
    rng = np.random.default_rng(21)
    C = np.diag([1e-2, 1e-2, 1e-6, 1e-6, 1e-4, 1.0])
    for _ in range(20):
        x = np.array([rng.uniform(-8, 8), rng.uniform(-8, 8), rng.uniform(-0.3, 0.3),
                      np.pi / 2 + rng.uniform(-0.3, 0.3), q / p, 7.0])
        r = oracle.to_line(fld, opt, x, C, xplane(30.0))
        assert r.rc == 0
        ref = helix_perigee(30.0, x[0], x[1], x[2], x[3], x[4], x[5], 2.0, M_MU)
        assert abs(r.x[0] - ref[0]) <= 1e-6 and abs(r.x[1] - ref[1]) <= 1e-6, (r.x, ref)
        assert abs(r.x[2] - ref[2]) <= 1e-10 and abs(r.x[3] - ref[3]) <= 1e-10
        assert r.x[4] == x[4] and abs(r.x[5] - ref[5]) <= 1e-6
        assert r.x[5] < x[5]  # the perigee lies behind the plane: the time runs backwards


def test_pp1_error_falls_with_the_fourth_power_of_the_step():
    """the residual against the helix is the stepper's truncation error: capping the primary step at a quarter of
    the leg cuts it by 2^4 per halving (P2 for the line surface)."""
    fld = oracle.make_field("const", (0, 0, 2.0))
    x = np.array([4.0, -3.0, 0.25, np.pi / 2 - 0.2, -2.0, 7.0])
    ref = helix_perigee(30.0, x[0], x[1], x[2], x[3], x[4], x[5], 2.0, M_MU)
    err = []
    for cap in (16.0, 8.0, 4.0):
        r = oracle.to_line(fld, oracle.make_options(max_step_mm=cap), x, np.eye(6), xplane(30.0))
        assert r.rc == 0
        err.append(np.abs(r.x - ref)[[1, 5]])  # z0 and t carry the along-track error
    err = np.array(err)
    assert np.all(err[0] / err[1] > 12) and np.all(err[0] / err[1] < 20), err
    assert np.all(err[1] / err[2] > 12) and np.all(err[1] / err[2] < 20), err


def test_pp1_sign_convention_of_d0():
    """d0 = D . (a x T)/|a x T|: a track passing the z axis on its left (axis at +y of a track moving along
    +x ... i.e. the track is at y < 0) has D = (0, y, 0), a x T = (0, 1, 0) -> d0 = y."""
    fld = oracle.make_field("const", (0, 0, 0.0))
    opt = oracle.make_options()
    for y in (-3.0, 2.5):
        r = oracle.to_line(fld, opt, [y, 1.0, 0.0, np.pi / 2, 0.5, 0.0], np.eye(6), xplane(30.0))
        assert r.rc == 0 and abs(r.x[0] - y) < 1e-12 and abs(r.x[1] - 1.0) < 1e-12


def test_pp2_zero_field_straight_line_any_axis():
    """B = 0: the closest approach of the line r + s T to the axis (c, a) in closed form."""
    fld = oracle.make_field("const", (0, 0, 0.0))
    opt = oracle.make_options()
    rng = np.random.default_rng(5)
    for _ in range(50):
        sf = tilted(40.0, rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2))
        x = np.array([rng.uniform(-5, 5), rng.uniform(-5, 5), rng.uniform(-0.4, 0.4),
                      np.pi / 2 + rng.uniform(-0.4, 0.4), rng.choice([-1, 1]) / rng.uniform(0.5, 20), 2.0])
        c = rng.uniform(-3, 3, 3)
        a = np.array([rng.uniform(-0.3, 0.3), rng.uniform(-0.3, 0.3), 1.0])
        a /= np.linalg.norm(a)
        r = oracle.to_line(fld, opt, x, np.eye(6), sf, c, a)
        assert r.rc == 0
        pos = sf[0:3] + x[0] * sf[3:6] + x[1] * sf[6:9]
        T = np.array([np.cos(x[2]) * np.sin(x[3]), np.sin(x[2]) * np.sin(x[3]), np.cos(x[3])])
        D = pos - c
        s = -((D - (D @ a) * a) @ T) / (1 - (a @ T) ** 2)
        D1 = D + s * T
        ed = np.cross(a, T)
        ed /= np.linalg.norm(ed)
        ref = np.array([D1 @ ed, D1 @ a, x[2], x[3], x[4], x[5] + s * np.sqrt(1 + (M_MU * x[4]) ** 2)])
        np.testing.assert_allclose(r.x, ref, rtol=1e-13, atol=1e-12)
        # brute force: no other point of the line is closer to the axis
        ss = s + np.linspace(-1, 1, 201)
        dist = np.linalg.norm(np.cross((D[None, :] + ss[:, None] * T[None, :]), a), axis=1)
        assert np.argmin(dist) == 100 and abs(dist[100] - abs(ref[0])) < 1e-10


@pytest.mark.parametrize("p", [0.7, 5.0])
@pytest.mark.parametrize("axis", ["z", "tilted"])
def test_pp3_finite_difference_jacobian(p, axis):
    fld = oracle.make_field("const", (0.1, -0.05, 2.0))
    opt = oracle.make_options()
    sf = tilted(45.0, -0.1, 0.25)
    c, a = ((0.0, 0.0, 0.0), (0.0, 0.0, 1.0)) if axis == "z" else ((1.0, -2.0, 0.5), np.array([0.15, -0.1, 1.0]))
    a = np.asarray(a, float) / np.linalg.norm(a)
    x = np.array([1.5, -2.0, 0.15, np.pi / 2 + 0.12, -1.0 / p, 10.0])
    C = np.eye(6)
    r = oracle.to_line(fld, opt, x, C, sf, c, a)
    assert r.rc == 0
    steps = [1e-4, 1e-4, 1e-6, 1e-6, 1e-6, 1e-3]
    Jfd = np.zeros((6, 6))
    for k, h in enumerate(steps):
        xp, xm = x.copy(), x.copy()
        xp[k] += h
        xm[k] -= h
        Jfd[:, k] = (oracle.to_line(fld, opt, xp, C, sf, c, a).x - oracle.to_line(fld, opt, xm, C, sf, c, a).x) / (2 * h)
    scale = np.maximum(np.abs(Jfd), 1e-3)
    assert np.max(np.abs(r.J - Jfd) / scale) < 2e-6, np.abs(r.J - Jfd) / scale
    # a dropped path-length correction or a missing T-part of w shows up at the 1e-2 level
    np.testing.assert_allclose(r.C, r.J @ C @ r.J.T, rtol=1e-12, atol=1e-15)


def test_pp4_composition_plane_to_plane_to_line():
    """Taking a state to the line directly, or first to another plane (kfo_propagate, covariance transported with
    its Jacobian) and from there, must give the same perigee: the chain rule through two different surfaces."""
    fld = oracle.make_field("const", (0, 0, 2.0))
    opt = oracle.make_options(n_corr_steps=3, max_step_mm=4.0)  # truncation error of the stepper below 1e-9
    rng = np.random.default_rng(8)
    for _ in range(10):
        x = np.array([rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(-0.2, 0.2),
                      np.pi / 2 + rng.uniform(-0.2, 0.2), rng.choice([-1, 1]) / rng.uniform(0.5, 5), 1.0])
        A = rng.standard_normal((6, 6)) * np.array([0.05, 0.05, 1e-3, 1e-3, 1e-2, 1.0])[:, None]
        C = A @ A.T + np.diag([1e-4, 1e-4, 1e-8, 1e-8, 1e-6, 1e-2])
        direct = oracle.to_line(fld, opt, x, C, xplane(30.0))
        hop = oracle.propagate(fld, opt, x, xplane(30.0), xplane(60.0))
        via = oracle.to_line(fld, opt, hop.x, hop.J @ C @ hop.J.T, xplane(60.0))
        assert direct.rc == 0 and hop.rc == 0 and via.rc == 0
        np.testing.assert_allclose(via.x, direct.x, rtol=0, atol=2e-9)
        sd = np.sqrt(np.diag(direct.C))
        assert np.max(np.abs(via.C - direct.C) / np.outer(sd, sd)) < 1e-6


def test_pp5_failure_modes():
    fld = oracle.make_field("const", (0, 0, 2.0))
    opt = oracle.make_options()
    # moving along the axis: no closest approach
    r = oracle.to_line(fld, opt, [1.0, 1.0, 0.0, 1e-9, 1.0, 0.0], np.eye(6), xplane(30.0))
    assert r.rc == 1
    r = oracle.to_line(fld, opt, [1.0, 1.0, np.nan, 1.5, 1.0, 0.0], np.eye(6), xplane(30.0))
    assert r.rc == 1


@pytest.mark.parametrize("cfg", [1, 2])
def test_pp6_perigee_pulls_have_unit_width(cfg):
    """PAPER.md:260-264 (Fig. 5): pulls of the six fitted perigee parameters have mean 0 and width 1.  The truth
    starts at the origin with t = 0, i.e. ON the z axis: its perigee parameters are (0, 0, phi, theta, q/p, 0)."""
    N = 8000
    wl = W.make_config(cfg, n_tracks=N)
    r = oracle.fit_workload(wl, perigee=((0, 0, 0), (0, 0, 1)))
    assert np.all(r.status == 0)
    truth = wl.truth_start.copy()
    truth[:, 0] = truth[:, 1] = truth[:, 5] = 0.0
    # on the start plane x = 0 the truth is at y = z = 0 as well
    assert np.all(wl.truth_start[:, :2] == 0.0)
    sig = np.sqrt(np.diagonal(r.perigee_cov, axis1=1, axis2=2))
    pull = (r.perigee_params - truth) / sig
    assert np.all(np.abs(pull.mean(axis=0)) < 4.0 / np.sqrt(N)), pull.mean(axis=0)
    assert np.all(np.abs(pull.std(axis=0) - 1.0) < 0.035), pull.std(axis=0)
    # the perigee is behind the first plane: the back-extrapolation loses precision on d0 relative to the first layer
    assert np.median(sig[:, 0]) > np.median(np.sqrt(r.first_cov[:, 0, 0]))
