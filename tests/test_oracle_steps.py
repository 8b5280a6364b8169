"""Pins for the oracle's step-level functions (P1-P4, P10, P11, P13).

Each check compares the oracle with something fixed independently of it: a closed form, a
finite difference, an information-form identity, or the worked material table.  CPU only.
"""
import os

import numpy as np
import pytest

import oracle

TESLA = 2.99792458e-4
M_MU = 0.1056583755
HERE = os.path.dirname(os.path.abspath(__file__))


def surface(center, u, v, xX0=0.0, thick=0.0, var=(1e-4, 1e-4)):
    u = np.asarray(u, float) / np.linalg.norm(u)
    v = np.asarray(v, float)
    v = v - u * (u @ v)
    v /= np.linalg.norm(v)
    s = np.zeros(20)
    s[0:3], s[3:6], s[6:9], s[9:12] = center, u, v, np.cross(u, v)
    s[12:14] = 50.0
    s[14], s[15], s[16:18] = xX0, thick, var
    return s


def xplane(x):
    return surface((x, 0, 0), (0, 1, 0), (0, 0, 1))


def tilted(x, a=0.2, b=-0.15):
    """a plane through (x, 1, -2) whose normal is rotated away from the x axis"""
    u = np.array([-np.sin(a), np.cos(a), 0.0])
    v = np.array([-np.sin(b) * np.cos(a), -np.sin(b) * np.sin(a), np.cos(b)])
    s = surface((x, 1.0, -2.0), u, v)
    assert s[9] > 0.9
    return s


def helix_to_xplane(y, z, phi, theta, lam, t, x0, x1, bz, mass):
    """closed-form helix in B = (0, 0, bz): textbook circle in the transverse plane,
    dphi/ds_T = kappa = -lam Bz / sin(theta)."""
    kappa = -lam * bz * TESLA / np.sin(theta)
    phi1 = np.arcsin(np.sin(phi) + kappa * (x1 - x0))
    s_t = (phi1 - phi) / kappa
    y1 = y - (np.cos(phi1) - np.cos(phi)) / kappa
    z1 = z + s_t / np.tan(theta)
    s = s_t / np.sin(theta)
    return y1, z1, phi1, theta, lam, t + s * np.sqrt(1 + (mass * lam) ** 2)


# ---- P1: analytic helix ------------------------------------------------------------------------
@pytest.mark.parametrize("p", [0.5, 1.0, 10.0, 100.0])
@pytest.mark.parametrize("q", [-1.0, 1.0])
def test_p1_helix_closed_form(p, q):
    fld = oracle.make_field("const", (0, 0, 2.0))
    opt = oracle.make_options()
    rng = np.random.default_rng(11)
    for _ in range(20):
        x = np.array([rng.uniform(-5, 5), rng.uniform(-5, 5), rng.uniform(-0.2, 0.2),
                      np.pi / 2 + rng.uniform(-0.2, 0.2), q / p, 3.0])
        r = oracle.propagate(fld, opt, x, xplane(0.0), xplane(30.0))
        assert r.rc == 0
        ref = helix_to_xplane(x[0], x[1], x[2], x[3], x[4], x[5], 0.0, 30.0, 2.0, M_MU)
        assert abs(r.x[0] - ref[0]) <= 1e-6 and abs(r.x[1] - ref[1]) <= 1e-6
        assert abs(r.x[2] - ref[2]) <= 1e-9 and abs(r.x[3] - ref[3]) <= 1e-9
        assert r.x[4] == x[4]
        assert abs(r.x[5] - ref[5]) <= 1e-6
        assert abs(r.free[0] - 30.0) <= 1e-11  # landed on the plane


def test_p1_sign_of_charge_and_units():
    """positive charge in +z field bends towards -y (F = q v x B); radius = p / (0.29979 B)."""
    fld = oracle.make_field("const", (0, 0, 2.0))
    opt = oracle.make_options()
    x = np.array([0, 0, 0, np.pi / 2, 1.0, 0.0])
    r = oracle.propagate(fld, opt, x, xplane(0.0), xplane(30.0))
    R = 1.0 / (0.299792458e-3 * 2.0)  # mm
    sag = R - np.sqrt(R * R - 30.0 ** 2)
    assert r.x[0] < 0 and abs(r.x[0] + sag) < 1e-7
    x[4] = -1.0
    r = oracle.propagate(fld, opt, x, xplane(0.0), xplane(30.0))
    assert abs(r.x[0] - sag) < 1e-7


# ---- P2: the stepper is 4th order ---------------------------------------------------------------
def test_p2_fourth_order_convergence():
    fld = oracle.make_field("const", (0, 0, 2.0))
    x = np.array([0.3, -0.2, 0.15, np.pi / 2 + 0.12, 1.0 / 0.3, 0.0])
    ref = np.array(helix_to_xplane(x[0], x[1], x[2], x[3], x[4], x[5], 0.0, 60.0, 2.0, M_MU))
    errs, hs = [], []
    for max_step in (64.0, 32.0, 16.0, 8.0):
        opt = oracle.make_options(max_step_mm=max_step)
        r = oracle.propagate(fld, opt, x, xplane(0.0), xplane(60.0))
        errs.append(np.hypot(r.x[0] - ref[0], r.x[1] - ref[1]))
        hs.append(max_step)
    slope = np.polyfit(np.log(hs), np.log(errs), 1)[0]
    assert errs[0] > 1e-6 and errs[-1] > 1e-11  # above the round-off floor
    assert abs(slope - 4.0) < 0.35, (slope, errs)


def test_single_step_local_error_is_fifth_order():
    fld = oracle.make_field("const", (0, 0, 2.0))
    lam, th, ph = 1 / 0.3, np.pi / 2 + 0.1, 0.1
    f = np.array([0, 0, 0, 0, np.cos(ph) * np.sin(th), np.sin(ph) * np.sin(th), np.cos(th), lam])
    errs = []
    for h in (40.0, 20.0, 10.0):
        fo, _, _ = oracle.rkn4_step(fld, M_MU, f, h)
        kappa = -lam * 2.0 * TESLA / np.sin(th)
        s_t = h * np.sin(th)
        ph1 = ph + kappa * s_t
        ex = np.array([(np.sin(ph1) - np.sin(ph)) / kappa, -(np.cos(ph1) - np.cos(ph)) / kappa,
                       h * np.cos(th)])
        errs.append(np.linalg.norm(fo[:3] - ex))
    assert 20 < errs[0] / errs[1] < 45 and 20 < errs[1] / errs[2] < 45, errs


# ---- P3: zero field = exact straight line with a closed-form Jacobian ----------------------------
def straight_line_closed_form(x, sa, sb, mass):
    ca, ua, va = sa[0:3], sa[3:6], sa[6:9]
    cb, ub, vb, nb = sb[0:3], sb[3:6], sb[6:9], sb[9:12]
    l0, l1, ph, th, lam, t = x
    T = np.array([np.cos(ph) * np.sin(th), np.sin(ph) * np.sin(th), np.cos(th)])
    r = ca + l0 * ua + l1 * va
    s = nb @ (cb - r) / (nb @ T)
    r1 = r + s * T
    dtds = np.sqrt(1 + (mass * lam) ** 2)
    xo = np.array([ub @ (r1 - cb), vb @ (r1 - cb), ph, th, lam, t + s * dtds])
    dT = np.zeros((3, 6))
    dT[:, 2] = [-np.sin(ph) * np.sin(th), np.cos(ph) * np.sin(th), 0]
    dT[:, 3] = [np.cos(ph) * np.cos(th), np.sin(ph) * np.cos(th), -np.sin(th)]
    dr = np.zeros((3, 6))
    dr[:, 0], dr[:, 1] = ua, va
    ds = -(nb @ dr) / (nb @ T) - s * (nb @ dT) / (nb @ T)  # d s / d x
    dr1 = dr + s * dT + np.outer(T, ds)
    J = np.zeros((6, 6))
    J[0], J[1] = ub @ dr1, vb @ dr1
    J[2, 2] = J[3, 3] = J[4, 4] = J[5, 5] = 1.0
    J[5] += dtds * ds
    J[5, 4] += s * mass ** 2 * lam / dtds
    return xo, J


@pytest.mark.parametrize("planes", ["x", "tilted"])
def test_p3_zero_field_straight_line(planes):
    fld = oracle.make_field("const", (0, 0, 0.0))
    opt = oracle.make_options()
    sa, sb = (xplane(0.0), xplane(30.0)) if planes == "x" else (tilted(0.0), tilted(45.0, -0.1, 0.25))
    rng = np.random.default_rng(3)
    for _ in range(20):
        x = np.array([rng.uniform(-5, 5), rng.uniform(-5, 5), rng.uniform(-0.3, 0.3),
                      np.pi / 2 + rng.uniform(-0.3, 0.3), rng.choice([-1, 1]) / rng.uniform(0.3, 5),
                      rng.uniform(-10, 10)])
        r = oracle.propagate(fld, opt, x, sa, sb)
        xo, J = straight_line_closed_form(x, sa, sb, M_MU)
        assert r.rc == 0
        np.testing.assert_allclose(r.x, xo, rtol=1e-13, atol=1e-12)
        np.testing.assert_allclose(r.J, J, rtol=1e-12, atol=1e-12)


# ---- P4: finite-difference Jacobian ---------------------------------------------------------------
@pytest.mark.parametrize("planes", ["x", "tilted"])
@pytest.mark.parametrize("p", [0.7, 5.0])
def test_p4_finite_difference_jacobian(planes, p):
    fld = oracle.make_field("const", (0.1, -0.05, 2.0) if planes == "tilted" else (0, 0, 2.0))
    opt = oracle.make_options()
    sa, sb = (xplane(0.0), xplane(30.0)) if planes == "x" else (tilted(0.0), tilted(45.0, -0.1, 0.25))
    x = np.array([1.2, -0.7, 0.15, np.pi / 2 + 0.12, -1.0 / p, 2.0])
    r0 = oracle.propagate(fld, opt, x, sa, sb)
    assert r0.rc == 0
    steps = [1e-4, 1e-4, 1e-6, 1e-6, 1e-6, 1e-3]
    Jfd = np.zeros((6, 6))
    for j in range(6):
        xp_, xm_ = x.copy(), x.copy()
        xp_[j] += steps[j]
        xm_[j] -= steps[j]
        Jfd[:, j] = (oracle.propagate(fld, opt, xp_, sa, sb).x - oracle.propagate(fld, opt, xm_, sa, sb).x) / (2 * steps[j])
    scale = np.maximum(np.abs(r0.J), 1e-3)
    assert np.max(np.abs(Jfd - r0.J) / scale) < 1e-6, np.abs(Jfd - r0.J) / scale
    # structural facts of J: row q/p = e_qp, column t = e_t
    np.testing.assert_array_equal(r0.J[4], [0, 0, 0, 0, 1, 0])
    np.testing.assert_array_equal(r0.J[:, 5], [0, 0, 0, 0, 0, 1])


def test_p4_step_jacobian_finite_difference():
    """8x8 step Jacobian against central differences of the step itself (constant field, so the
    neglected field-gradient term is exactly zero).  The T-normalisation is not differentiated in
    Dstep, so compare on directions tangent to the unit sphere plus r, t, lam."""
    fld = oracle.make_field("const", (0.2, -0.1, 2.0))
    ph, th, lam = 0.2, 1.3, 1 / 0.8
    T = np.array([np.cos(ph) * np.sin(th), np.sin(ph) * np.sin(th), np.cos(th)])
    f = np.concatenate([[1.0, 2.0, 3.0, 0.5], T, [lam]])
    h = 25.0
    _, Ds, _ = oracle.rkn4_step(fld, M_MU, f, h)
    # lam column
    d = 1e-6
    fp, fm = f.copy(), f.copy()
    fp[7] += d
    fm[7] -= d
    col = (oracle.rkn4_step(fld, M_MU, fp, h)[0] - oracle.rkn4_step(fld, M_MU, fm, h)[0]) / (2 * d)
    # the step renormalises T: project the analytic column the same way, P = I - T' T'^T
    fo = oracle.rkn4_step(fld, M_MU, f, h)[0]
    P = np.eye(3) - np.outer(fo[4:7], fo[4:7])
    ana = Ds[:, 7].copy()
    ana[4:7] = P @ ana[4:7]
    np.testing.assert_allclose(col, ana, rtol=2e-7, atol=1e-9)
    # tangent direction columns
    for e in (np.array([-np.sin(ph), np.cos(ph), 0.0]),
              np.array([np.cos(ph) * np.cos(th), np.sin(ph) * np.cos(th), -np.sin(th)])):
        d = 1e-6
        fp, fm = f.copy(), f.copy()
        fp[4:7] = (T + d * e) / np.linalg.norm(T + d * e)
        fm[4:7] = (T - d * e) / np.linalg.norm(T - d * e)
        col = (oracle.rkn4_step(fld, M_MU, fp, h)[0] - oracle.rkn4_step(fld, M_MU, fm, h)[0]) / (2 * d)
        ana = Ds[:, 4:7] @ e
        ana[4:7] = P @ ana[4:7]
        np.testing.assert_allclose(col, ana, rtol=2e-7, atol=1e-9)
    # r and t columns are unit vectors
    for j in (0, 1, 2, 3):
        e = np.zeros(8)
        e[j] = 1.0
        np.testing.assert_array_equal(Ds[:, j], e)


# ---- P10: material formulas ----------------------------------------------------------------------
def _golden_material():
    rows = []
    with open(os.path.join(HERE, "golden", "material_table.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                rows.append([float(v) for v in line.split()])
    return rows


def test_p10_material_table():
    opt = oracle.make_options(material=1)
    s = surface((30, 0, 0), (0, 1, 0), (0, 0, 1), xX0=0.0032, thick=0.3)
    C = np.diag([1e-4, 1e-4, 1e-6, 1e-6, 1e-4, 1.0])
    for p, th0, dedx, dE, dhalf, g in _golden_material():
        x = np.array([0, 0, 0, np.pi / 2, 1.0 / p, 0])
        r = oracle.material(opt, s, x, C)
        assert r.rc == 0
        assert abs(r.theta0 / th0 - 1) < 2e-6
        assert abs(r.dE * 1e3 / dE - 1) < 5e-5
        assert abs(r.dE * 1e3 / (2.329 * 0.1 * 0.3) / dedx - 1) < 5e-5
        assert abs(r.g - g) < 2e-8


def test_p10_material_physics_anchors():
    """independent anchors: plasma energy of silicon 31.05 eV; minimum of the mean stopping power
    within 3 % of the tabulated 1.664 MeV cm^2/g near beta*gamma = 3-3.5; theta0 ~ 1/p at high p."""
    assert abs(28.816 * np.sqrt(2.329 * 14 / 28.0855) - 31.05) < 0.01
    opt = oracle.make_options(material=1)
    s = surface((30, 0, 0), (0, 1, 0), (0, 0, 1), xX0=0.0032, thick=0.3)
    C = np.eye(6) * 1e-6
    bgs = np.linspace(2.0, 5.0, 61)
    dedx = []
    for bg in bgs:
        r = oracle.material(opt, s, np.array([0, 0, 0, np.pi / 2, 1 / (bg * M_MU), 0]), C)
        dedx.append(r.dE * 1e3 / (2.329 * 0.03))
    dedx = np.array(dedx)
    assert abs(dedx.min() / 1.664 - 1) < 0.03
    assert 2.8 < bgs[dedx.argmin()] < 3.6
    r1 = oracle.material(opt, s, np.array([0, 0, 0, np.pi / 2, 1 / 50.0, 0]), C)
    r2 = oracle.material(opt, s, np.array([0, 0, 0, np.pi / 2, 1 / 100.0, 0]), C)
    assert abs(r1.theta0 / r2.theta0 - 2.0) < 1e-4


def test_material_covariance_and_energy_jacobian():
    opt = oracle.make_options(material=1)
    s = tilted(30.0)
    s[14], s[15] = 0.0032, 0.3
    rng = np.random.default_rng(5)
    A = rng.standard_normal((6, 6)) * np.array([1e-2, 1e-2, 1e-3, 1e-3, 1e-2, 1.0])[:, None]
    C = A @ A.T
    x = np.array([0.3, 0.1, 0.2, 1.4, -1 / 2.0, 5.0])
    r = oracle.material(opt, s, x, C)
    # path factor: inclined incidence lengthens the path
    T = np.array([np.cos(x[2]) * np.sin(x[3]), np.sin(x[2]) * np.sin(x[3]), np.cos(x[3])])
    cfac = 1 / abs(s[9:12] @ T)
    s0 = surface((30, 0, 0), (0, 1, 0), (0, 0, 1), xX0=0.0032 * cfac, thick=0.3 * cfac)
    x_n = np.array([0, 0, 0, np.pi / 2, x[4], 0])
    r0 = oracle.material(opt, s0, x_n, C)
    assert abs(r.theta0 / r0.theta0 - 1) < 1e-12 and abs(r.dE / r0.dE - 1) < 1e-12
    # q/p after the loss, and g = d lam'/d lam at constant dE by finite differences
    m = M_MU

    def lam_after(lam):
        E = np.sqrt(1 / lam ** 2 + m * m) - r.dE
        return np.sign(lam) / np.sqrt(E * E - m * m)

    assert abs(r.x[4] - lam_after(x[4])) < 1e-15
    d = 1e-6
    gfd = (lam_after(x[4] + d) - lam_after(x[4] - d)) / (2 * d)
    assert abs(gfd - r.g) < 1e-8
    G = np.diag([1, 1, 1, 1, r.g, 1.0])
    Q = np.zeros((6, 6))
    Q[2, 2], Q[3, 3] = r.theta0 ** 2 / np.sin(x[3]) ** 2, r.theta0 ** 2
    np.testing.assert_allclose(r.C, G @ C @ G.T + Q, rtol=1e-13, atol=0)
    assert np.all(np.delete(r.x, 4) == np.delete(x, 4))


def test_material_energy_exhausted():
    opt = oracle.make_options(material=1)
    s = surface((30, 0, 0), (0, 1, 0), (0, 0, 1), xX0=3.2, thick=300.0)  # 30 cm of silicon
    r = oracle.material(opt, s, np.array([0, 0, 0, np.pi / 2, 1 / 0.05, 0]), np.eye(6))
    assert r.rc == 4


# ---- P11: trilinear field -------------------------------------------------------------------------
def test_p11_trilinear_exact_on_linear_field():
    n = np.array([5, 4, 6])
    origin, spacing = np.array([-3.0, 2.0, 10.0]), np.array([2.0, 5.0, 1.5])
    a0 = np.array([0.3, -0.2, 1.1])
    Ax = np.array([[0.01, 0.02, -0.03], [0.04, -0.01, 0.02], [-0.02, 0.03, 0.05]])
    xs = origin[0] + spacing[0] * np.arange(n[0])
    ys = origin[1] + spacing[1] * np.arange(n[1])
    zs = origin[2] + spacing[2] * np.arange(n[2])
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    pos = np.stack([X, Y, Z], axis=-1)
    grid = a0 + pos @ Ax.T  # (nz, ny, nx, 3)
    fld = oracle.make_field("grid3", grid_n=n, grid_origin=origin, grid_spacing=spacing, grid=grid)
    rng = np.random.default_rng(7)
    for _ in range(50):
        r = origin + rng.uniform(0, 1, 3) * spacing * (n - 1)
        b, cl = oracle.field_at(fld, r)
        np.testing.assert_allclose(b, a0 + Ax @ r, rtol=1e-13, atol=1e-14)
        assert cl == 0
    # node values, including the last node of every axis
    for idx in [(0, 0, 0), (4, 3, 5), (2, 1, 3), (4, 0, 5)]:
        r = origin + spacing * np.array(idx)
        b, cl = oracle.field_at(fld, r)
        np.testing.assert_allclose(b, grid[idx[2], idx[1], idx[0]], rtol=1e-14)
        assert cl == 0
    # outside: constant extrapolation (clamped) and flagged
    r_out = np.array([origin[0] + spacing[0] * (n[0] - 1) + 7.0, ys[1] + 1.0, zs[2] + 0.3])
    r_edge = r_out.copy()
    r_edge[0] = xs[-1]
    b_out, cl = oracle.field_at(fld, r_out)
    b_edge, _ = oracle.field_at(fld, r_edge)
    np.testing.assert_allclose(b_out, b_edge, rtol=1e-14)
    assert cl == 1
    b_lo, cl = oracle.field_at(fld, np.array([origin[0] - 1.0, ys[0], zs[0]]))
    np.testing.assert_allclose(b_lo, grid[0, 0, 0], rtol=1e-14)
    assert cl == 1


def test_p11_cfg4_grid_error_bound():
    from paper_2105_01796_b200 import workloads as W
    n, origin, spacing, grid = W.cfg4_field_grid()
    fld = oracle.make_field("grid3", grid_n=n, grid_origin=origin, grid_spacing=spacing, grid=grid)
    worst = 0.0
    for x in np.linspace(0.0, 400.0, 173):
        b, _ = oracle.field_at(fld, np.array([x, 3.3, -7.7]))
        exact = 2.0 * (1 - 0.2 * (x / 400.0) ** 2)
        worst = max(worst, abs(b[2] - exact) / exact)
        assert b[0] == 0 and b[1] == 0
    assert worst <= 10.0 ** 2 / 8 * (2 * 0.4 / 400 ** 2) / 1.6 * 1.01  # (D^2/8) |f''| / f


# ---- P13: the update against the information (weighted-mean) form ---------------------------------
def test_p13_update_equals_weighted_mean():
    rng = np.random.default_rng(9)
    for _ in range(20):
        A = rng.standard_normal((6, 6)) * np.array([0.05, 0.05, 1e-3, 1e-3, 1e-2, 10.0])[:, None]
        Cp = A @ A.T
        xp = rng.standard_normal(6) * np.array([1, 1, 0.1, 0.1, 0.5, 10])
        Vh = rng.standard_normal((2, 2)) * 0.01
        V = Vh @ Vh.T + np.diag([1e-4, 9e-4])
        m = xp[:2] + rng.standard_normal(2) * 0.05
        rc, xf, Cf, chi2 = oracle.update(xp, Cp, m, V)
        assert rc == 0
        H = np.zeros((2, 6))
        H[0, 0] = H[1, 1] = 1
        # scale to unit diagonal for a well-conditioned inverse, then the weighted mean
        s = np.sqrt(np.diag(Cp))
        Cpi = np.linalg.inv(Cp / np.outer(s, s)) / np.outer(s, s)
        W = Cpi + H.T @ np.linalg.inv(V) @ H
        Cw = np.linalg.inv(W * np.outer(s, s)) * np.outer(s, s)
        xw = Cw @ (Cpi @ xp + H.T @ np.linalg.inv(V) @ m)
        np.testing.assert_allclose(Cf, Cw, rtol=1e-7, atol=0)
        np.testing.assert_allclose(xf, xw, rtol=1e-8, atol=1e-10)
        # chi2: predicted-residual form == filtered-residual form (reading U8)
        rf = m - xf[:2]
        chi2_f = rf @ np.linalg.inv(V - Cf[:2, :2]) @ rf
        assert abs(chi2 - chi2_f) < 1e-6 * max(chi2, 1)
        assert np.allclose(Cf, Cf.T, rtol=0, atol=0)
    rc, *_ = oracle.update(xp, -Cp, m, np.zeros((2, 2)))
    assert rc == 2


def test_p13_one_hit_by_hand():
    """diagonal C-, diagonal V: each measured coordinate is a 1-D weighted mean; the rest is untouched."""
    Cp = np.diag([4e-2, 9e-2, 1e-6, 1e-6, 1e-4, 1.0])
    xp = np.array([1.0, -2.0, 0.1, 1.5, 0.3, 7.0])
    m = np.array([1.3, -2.6])
    V = np.diag([1e-2, 1e-2])
    rc, xf, Cf, chi2 = oracle.update(xp, Cp, m, V)
    assert abs(xf[0] - (1.0 / 4e-2 + 1.3 / 1e-2) / (1 / 4e-2 + 1 / 1e-2)) < 1e-13
    assert abs(xf[1] - (-2.0 / 9e-2 - 2.6 / 1e-2) / (1 / 9e-2 + 1 / 1e-2)) < 1e-13
    np.testing.assert_allclose(xf[2:], xp[2:], rtol=0, atol=0)
    assert abs(Cf[0, 0] - 1 / (1 / 4e-2 + 1 / 1e-2)) < 1e-15
    assert abs(chi2 - (0.3 ** 2 / 5e-2 + 0.6 ** 2 / 1e-1)) < 1e-12


# ---- adaptive step count (reading U31; "adaptive") ---------------------------------
def _leg_state(x, sf):
    """free vector of a bound state on surface sf and the straight-line distance to the plane x = x1"""
    T = np.array([np.cos(x[2]) * np.sin(x[3]), np.sin(x[2]) * np.sin(x[3]), np.cos(x[3])])
    r = sf[0:3] + x[0] * sf[3:6] + x[1] * sf[6:9]
    return np.concatenate([r, [x[5]], T, [x[4]]]), T, r


@pytest.mark.parametrize("p", [0.15, 0.3, 1.0])
@pytest.mark.parametrize("tol", [1e-3, 1e-5, 1e-7])
def test_adaptive_step_count_is_the_quartic_rule_on_the_trial_estimate(p, tol):
    """The tolerance only selects the number of primary steps: n = ceil((eps0/tol)^(1/4)) with eps0 the embedded
    estimate of one trial step over the leg (taken from kfo_rkn4_step, pinned on its own).  The propagation must
    then equal, bit for bit, the one with the primary step capped at leg/n; and every step's estimate is ~tol or less."""
    fld = oracle.make_field("const", (0.05, -0.1, 2.0))
    sa, sb = xplane(0.0), xplane(60.0)
    x = np.array([0.3, -0.2, 0.15, np.pi / 2 + 0.12, -1.0 / p, 0.0])
    f, T, r = _leg_state(x, sa)
    s0 = (60.0 - r[0]) / T[0]
    _, _, eps0 = oracle.rkn4_step(fld, M_MU, f, s0)
    n = max(1, int(np.ceil(np.sqrt(np.sqrt(eps0 / tol)))))
    got = oracle.propagate(fld, oracle.make_options(step_tolerance_mm=tol), x, sa, sb)
    same = oracle.propagate(fld, oracle.make_options(max_step_mm=s0 / n * (1 + 1e-9)), x, sa, sb)
    more = oracle.propagate(fld, oracle.make_options(max_step_mm=s0 / (n + 1) * (1 + 1e-9)), x, sa, sb)
    assert got.rc == 0
    np.testing.assert_array_equal(got.x, same.x)
    np.testing.assert_array_equal(got.J, same.J)
    if n > 1:
        assert not np.array_equal(got.x, more.x)
    assert got.rk_err <= 1.5 * tol or n == 1024
    if n > 1:
        assert got.rk_err >= tol * ((n - 1) / n) ** 4 * 0.5  # not finer than the rule asks for


def test_adaptive_steps_track_the_helix_and_switch_off_cleanly():
    fld = oracle.make_field("const", (0, 0, 2.0))
    x = np.array([0.3, -0.2, 0.15, np.pi / 2 + 0.12, 1.0 / 0.3, 0.0])
    ref = np.array(helix_to_xplane(x[0], x[1], x[2], x[3], x[4], x[5], 0.0, 60.0, 2.0, M_MU))
    errs = []
    for tol in (1e-2, 1e-4, 1e-6, 1e-8):
        r = oracle.propagate(fld, oracle.make_options(step_tolerance_mm=tol), x, xplane(0.0), xplane(60.0))
        errs.append(np.hypot(r.x[0] - ref[0], r.x[1] - ref[1]))
    # the true error follows the tolerance (it is ~1000x below the pessimistic estimate) down to round-off
    assert errs[0] > errs[1] > errs[2] > errs[3] and errs[3] < 1e-10 and errs[0] / errs[2] > 1e3, errs
    # off: <= 0, inf, or so loose that one step suffices -> the default policy, bit for bit
    base = oracle.propagate(fld, oracle.make_options(), x, xplane(0.0), xplane(60.0))
    for tol in (0.0, -1.0, float("inf"), 1e6):
        r = oracle.propagate(fld, oracle.make_options(step_tolerance_mm=tol), x, xplane(0.0), xplane(60.0))
        np.testing.assert_array_equal(r.x, base.x)
        np.testing.assert_array_equal(r.J, base.J)


def test_adaptive_steps_in_the_batch_fit():
    """CFG4-like low-momentum tracks in the grid field: the tolerance changes the fit at the level of the stepper's
    truncation error and nothing else -- same hits used, and the chi2 of every track moves by no more than the shift of
    its predicted positions explains: with r -> r + d at a hit, r^T S^-1 r changes by 2 d^T S^-1 r + d^T S^-1 d
    <= 2 sqrt(chi2_k) |d|/sigma + (|d|/sigma)^2, sigma^2 = the smallest measurement variance (S = C- + V >= V); summed
    over the hits, with a factor 2 for the second-order change of S itself.  The largest per-step estimate drops by
    three orders of magnitude.  (The trilinear field has kinks at the cell faces, where the estimate falls more
    slowly than h^4: it ends within ~10x of the tolerance, not below it as in a smooth field.)"""
    from paper_2105_01796_b200 import workloads as W
    wl = W.make_config(4, n_tracks=300)
    a = oracle.fit_workload(wl, states=True)
    b = oracle.fit_workload(wl, states=True, step_tolerance_mm=1e-6)
    np.testing.assert_array_equal(a.n_used, b.n_used)
    np.testing.assert_array_equal(a.hit_flags, b.hit_flags)
    assert a.rk_err_max.max() > 1e-2 and b.rk_err_max.max() <= 2e-5 and np.median(b.rk_err_max) <= 2e-6
    sigma = np.sqrt(wl.geometry[1:, 16:18].min())
    bound = np.zeros(wl.n_tracks)
    for i in range(wl.n_tracks):
        for j in range(wl.offsets[i], wl.offsets[i + 1]):
            leg = wl.surf_idx[j] - wl.start_surface - 1
            d = np.linalg.norm(b.pred_params[i, leg, :2] - a.pred_params[i, leg, :2]) / sigma
            bound[i] += 2.0 * np.sqrt(a.hit_chi2[j]) * d + d * d
    shift = np.abs(a.chi2 - b.chi2)
    assert np.all(shift <= 2.0 * bound + 1e-9), (shift - 2.0 * bound).max()
    assert np.median(shift) < 1e-4 and np.any(a.first_params != b.first_params)
