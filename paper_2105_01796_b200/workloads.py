"""Seeded synthetic workloads (the five BASELINE.json configs) for the batched Kalman track fit.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2105_01796_b200/csrc`): it *simulates* particles (truth transport, multiple scattering
kicks, mean energy loss, hit smearing) and emits plain numpy arrays.  It contains none of the
fit's arithmetic (no Kalman update, no RKN stepper, no Jacobian, no smoother) and imports neither
the oracle nor the CUDA binding.  numpy only.

The Fatras-simulated single-muon sample the paper measured on is not available;
these inputs take its shape (planar telescope perpendicular to x, 30 mm pitch, 2 T along z,
mu+-, Gaussian-smeared 2-D hits, smeared-truth start -- PAPER.md:186, 206-210) and stand in for it.
Recipe: SURVEY.md section 8(d) D.1 / DESIGN.md "Input recipe".

Units: mm, GeV, q in e, q/p in 1/GeV, time as c*t in mm, field in tesla.
"""
from __future__ import annotations

from dataclasses import dataclass, field as _dc_field
from typing import Optional

import os

import numpy as np

# ---------------------------------------------------------------------------------------------
# constants of the *simulation* (the fitters carry their own copies; nothing is imported from here
# by oracle/ or csrc/)
# ---------------------------------------------------------------------------------------------
TESLA = 2.99792458e-4  # 1 T in GeV/(e mm)
C_MM_PER_NS = 299.792458
M_MU = 0.1056583755  # GeV
M_E = 0.51099895e-3  # GeV
SILICON = dict(Z=14.0, A=28.0855, rho=2.329, I_eV=173.0, X0_mm=93.7)
K_BETHE = 0.307075  # MeV mol^-1 cm^2

GEOM_STRIDE = 20  # doubles per surface in the packed geometry table
# packed surface record: center[3] u[3] v[3] n[3] half_len[2] x_over_X0 thickness_mm meas_var[2] pad[2]


@dataclass
class Workload:
    """Plain arrays describing one batch of tracks to fit (natural AoS layouts, float64/int32)."""

    name: str
    n_tracks: int
    n_layers: int
    geometry: np.ndarray  # (n_surfaces, GEOM_STRIDE)
    field_kind: str  # "const" | "grid3"
    field_b: np.ndarray  # (3,) tesla (const)
    grid_n: Optional[np.ndarray]  # (3,) int32 nodes per axis (x, y, z)
    grid_origin: Optional[np.ndarray]  # (3,) mm
    grid_spacing: Optional[np.ndarray]  # (3,) mm
    grid: Optional[np.ndarray]  # (nz, ny, nx, 3) tesla
    start_surface: int
    params0: np.ndarray  # (N, 6) start parameters (truth smeared)
    cov0: np.ndarray  # (N, 6, 6) start covariance
    offsets: np.ndarray  # (N+1,) int32 CSR offsets into the hit arrays
    surf_idx: np.ndarray  # (M,) int32 surface index of each hit (ascending per track)
    loc: np.ndarray  # (M, 2) measured local position
    options: dict  # smooth, material, outlier_chi2, mass_gev, ...
    material: dict  # Z, A, rho, I_eV, X0_mm
    truth_start: np.ndarray  # (N, 6) true bound parameters on the start surface
    truth: np.ndarray  # (N, L, 6) true bound parameters entering layer k (NaN if not reached)
    is_outlier: Optional[np.ndarray] = None  # (M,) bool, hits replaced by noise (CFG3)
    meta: dict = _dc_field(default_factory=dict)

    @property
    def n_meas(self) -> int:
        return int(self.surf_idx.shape[0])

    def subset(self, idx) -> "Workload":
        """The same workload restricted to tracks `idx` (CSR rebased). Tracks are independent
        (PAPER.md:119), so fitting a subset reproduces the same per-track results."""
        idx = np.asarray(idx, dtype=np.int64)
        lens = (self.offsets[1:] - self.offsets[:-1])[idx]
        new_off = np.zeros(idx.size + 1, dtype=np.int32)
        np.cumsum(lens, out=new_off[1:])
        take = np.concatenate(
            [np.arange(self.offsets[i], self.offsets[i + 1], dtype=np.int64) for i in idx]
        ) if idx.size else np.zeros(0, dtype=np.int64)
        return Workload(
            name=self.name + f"[subset {idx.size}]", n_tracks=int(idx.size), n_layers=self.n_layers,
            geometry=self.geometry, field_kind=self.field_kind, field_b=self.field_b,
            grid_n=self.grid_n, grid_origin=self.grid_origin, grid_spacing=self.grid_spacing,
            grid=self.grid, start_surface=self.start_surface,
            params0=self.params0[idx].copy(), cov0=self.cov0[idx].copy(), offsets=new_off,
            surf_idx=self.surf_idx[take].copy(), loc=self.loc[take].copy(),
            options=dict(self.options), material=dict(self.material),
            truth_start=self.truth_start[idx].copy(), truth=self.truth[idx].copy(),
            is_outlier=None if self.is_outlier is None else self.is_outlier[take].copy(),
            meta=dict(self.meta),
        )


# ---------------------------------------------------------------------------------------------
# geometry / field builders
# ---------------------------------------------------------------------------------------------
def telescope_geometry(n_layers: int, pitch_mm: float = 30.0, half_len_mm: float = 50.0,
                       x_over_X0: float = 0.0, thickness_mm: float = 0.0,
                       meas_sigma_mm=(0.010, 0.010)) -> np.ndarray:
    """Surface 0 = start plane at x = 0 (no hit, no material); surface k = plane at x = pitch*k.
    u = (0,1,0), v = (0,0,1), n = u x v = (1,0,0): loc0 = global y, loc1 = global z."""
    g = np.zeros((n_layers + 1, GEOM_STRIDE), dtype=np.float64)
    for k in range(n_layers + 1):
        g[k, 0:3] = (pitch_mm * k, 0.0, 0.0)
        g[k, 3:6] = (0.0, 1.0, 0.0)
        g[k, 6:9] = (0.0, 0.0, 1.0)
        g[k, 9:12] = (1.0, 0.0, 0.0)
        g[k, 12:14] = (half_len_mm, half_len_mm)
        if k > 0:
            g[k, 14] = x_over_X0
            g[k, 15] = thickness_mm
        g[k, 16:18] = (meas_sigma_mm[0] ** 2, meas_sigma_mm[1] ** 2)
    return g


def cfg4_field_grid():
    """3-D grid, 10 mm spacing over 400 x 200 x 200 mm: nodes 41 x 21 x 21 at x in [0, 400],
    y, z in [-100, 100]; B_z = 2 T (1 - 0.2 (x/400 mm)^2), B_x = B_y = 0 (BASELINE.json configs[4]).
    Layout (nz, ny, nx, 3): x fastest, component innermost."""
    n = np.array([41, 21, 21], dtype=np.int32)
    origin = np.array([0.0, -100.0, -100.0])
    spacing = np.array([10.0, 10.0, 10.0])
    xs = origin[0] + spacing[0] * np.arange(n[0])
    grid = np.zeros((n[2], n[1], n[0], 3), dtype=np.float64)
    grid[:, :, :, 2] = 2.0 * (1.0 - 0.2 * (xs / 400.0) ** 2)[None, None, :]
    return n, origin, spacing, grid


def _trilinear(grid, n, origin, spacing, pos):
    """Generator's own trilinear lookup (clamped outside the grid). pos: (N, 3) -> (N, 3) tesla."""
    idx = []
    w = []
    for a in range(3):
        f = (pos[:, a] - origin[a]) / spacing[a]
        i = np.clip(np.floor(f), 0, n[a] - 2).astype(np.int64)
        idx.append(i)
        w.append(np.clip(f - i, 0.0, 1.0))
    flat = grid.reshape(-1, 3)                      # node (k, j, i) at row (k * ny + j) * nx + i
    base = (idx[2] * n[1] + idx[1]) * n[0] + idx[0]
    out = np.zeros((pos.shape[0], 3))
    for dz in (0, 1):
        wz = w[2] if dz else 1.0 - w[2]
        for dy in (0, 1):
            wy = w[1] if dy else 1.0 - w[1]
            for dx in (0, 1):
                wx = w[0] if dx else 1.0 - w[0]
                out += (wz * wy * wx)[:, None] * np.take(flat, base + ((dz * n[1] + dy) * n[0] + dx), axis=0)
    return out


# ---------------------------------------------------------------------------------------------
# truth transport (simulation)
# ---------------------------------------------------------------------------------------------
class _Truth:
    """Global truth state of N particles: position, direction angles, q/p, time."""

    def __init__(self, n):
        self.x = np.zeros(n)
        self.y = np.zeros(n)
        self.z = np.zeros(n)
        self.phi = np.zeros(n)
        self.theta = np.zeros(n)
        self.lam = np.zeros(n)
        self.t = np.zeros(n)
        self.alive = np.ones(n, dtype=bool)

    def bound_on_x_plane(self):
        return np.stack([self.y, self.z, self.phi, self.theta, self.lam, self.t], axis=1)


def _helix_to_x_plane(st: _Truth, x_plane: float, bz_tesla: float, mass: float):
    """Closed-form helix in a constant field along z, from the current point to the plane
    x = x_plane. dT/ds = lam T x B  =>  dphi/ds_T = kappa = -lam Bz / sin(theta) along the
    transverse arc s_T;  x(s_T) = x0 + (sin(phi0 + kappa s_T) - sin(phi0)) / kappa."""
    sth = np.sin(st.theta)
    kappa = -st.lam * (bz_tesla * TESLA) / sth
    dx = x_plane - st.x
    small = np.abs(kappa * dx) < 1e-14
    arg = np.sin(st.phi) + kappa * dx
    ok = np.abs(arg) < 1.0
    arg = np.where(ok, arg, 0.0)
    phi1 = np.arcsin(arg)
    with np.errstate(divide="ignore", invalid="ignore"):
        s_t = np.where(small, dx / np.cos(st.phi), (phi1 - st.phi) / kappa)
        dy = np.where(small, dx * np.tan(st.phi), -(np.cos(phi1) - np.cos(st.phi)) / kappa)
    s = s_t / sth
    st.alive &= ok & (s > 0)
    st.x = np.full_like(st.x, x_plane)
    st.y = st.y + dy
    st.z = st.z + s_t * np.cos(st.theta) / sth
    st.phi = np.where(small, st.phi, phi1)
    st.t = st.t + s * np.sqrt(1.0 + (mass * st.lam) ** 2)


def _rk4_to_x_plane(st: _Truth, x_plane: float, grid_desc, mass: float, max_step=5.0):
    """Classical RK4 on (r, T) in the trilinear grid field with fixed steps <= max_step, then
    Newton-like landing steps onto x = x_plane (simulation only; U15 of SURVEY.md 8(c))."""
    n, origin, spacing, grid = grid_desc
    # only the particles still alive are transported (a stopped one makes no further hit); every operation below is
    # element-wise per particle, so the values of the live ones do not depend on who else is in the arrays
    live = np.flatnonzero(st.alive)
    if live.size == 0:
        st.x = np.full_like(st.x, x_plane)
        return
    r_all = np.stack([st.x[live], st.y[live], st.z[live]], axis=1)
    T_all = np.stack([np.cos(st.phi[live]) * np.sin(st.theta[live]), np.sin(st.phi[live]) * np.sin(st.theta[live]),
                      np.cos(st.theta[live])], axis=1)
    lam_all = st.lam[live]
    with np.errstate(divide="ignore", invalid="ignore"):
        n_big = int(np.ceil(np.nanmax((x_plane - r_all[:, 0]) / np.maximum(T_all[:, 0], 0.2)) / max_step))
    n_big = max(n_big, 1)

    def transport(sl):
        """The particles of one slice through the n_big + 3 steps (every operation is per particle)."""
        r, T, lam = r_all[sl], T_all[sl], lam_all[sl]
        path = np.zeros_like(lam)

        def acc(rr, TT):
            B = _trilinear(grid, n, origin, spacing, rr) * TESLA
            return lam[:, None] * np.cross(TT, B)

        def step(h):
            nonlocal r, T, path
            hh = h[:, None]
            k1r, k1t = T, acc(r, T)
            k2r, k2t = T + 0.5 * hh * k1t, acc(r + 0.5 * hh * k1r, T + 0.5 * hh * k1t)
            k3r, k3t = T + 0.5 * hh * k2t, acc(r + 0.5 * hh * k2r, T + 0.5 * hh * k2t)
            k4r, k4t = T + hh * k3t, acc(r + hh * k3r, T + hh * k3t)
            r = r + hh / 6.0 * (k1r + 2 * k2r + 2 * k3r + k4r)
            T = T + hh / 6.0 * (k1t + 2 * k2t + 2 * k3t + k4t)
            T = T / np.linalg.norm(T, axis=1, keepdims=True)
            path = path + h

        with np.errstate(divide="ignore", invalid="ignore"):
            for i in range(n_big):
                h = (x_plane - r[:, 0]) / T[:, 0] / (n_big - i)
                h = np.where(np.isfinite(h), h, 0.0)
                step(h)
            for _ in range(3):
                h = (x_plane - r[:, 0]) / T[:, 0]
                h = np.where(np.isfinite(h), h, 0.0)
                step(h)
        return r, T, path

    # slices of particles side by side on the host's cores (numpy releases the interpreter lock inside its loops)
    chunk = 16384
    slices = [slice(a, min(a + chunk, live.size)) for a in range(0, live.size, chunk)]
    if len(slices) > 1:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=min(len(slices), os.cpu_count() or 1)) as pool:
            parts = list(pool.map(transport, slices))
    else:
        parts = [transport(slices[0])]
    r = np.concatenate([p[0] for p in parts])
    T = np.concatenate([p[1] for p in parts])
    path = np.concatenate([p[2] for p in parts])
    lam = lam_all
    st.alive[live] &= T[:, 0] > 1e-3
    st.x = np.full_like(st.x, x_plane)
    st.y[live], st.z[live] = r[:, 1], r[:, 2]
    st.phi[live] = np.arctan2(T[:, 1], T[:, 0])
    st.theta[live] = np.arccos(np.clip(T[:, 2], -1.0, 1.0))
    st.t[live] = st.t[live] + path * np.sqrt(1.0 + (mass * lam) ** 2)


def highland_theta0(p, mass, x_over_X0_eff):
    """Highland / PDG multiple-scattering width (simulation copy)."""
    E = np.sqrt(p * p + mass * mass)
    beta = p / E
    return 0.0136 / (beta * p) * np.sqrt(x_over_X0_eff) * (1.0 + 0.038 * np.log(x_over_X0_eff / beta ** 2))


def bethe_mean_dedx_mass(p, mass, mat):
    """Mean mass stopping power in MeV cm^2/g, Bethe with the asymptotic density correction
    (simulation copy; formula stated in SURVEY.md 8(c) C.2.5)."""
    E = np.sqrt(p * p + mass * mass)
    beta = p / E
    gamma = E / mass
    bg = p / mass
    I = mat["I_eV"] * 1e-9  # GeV
    wmax = 2 * M_E * bg ** 2 / (1 + 2 * gamma * M_E / mass + (M_E / mass) ** 2)
    hwp = 28.816e-9 * np.sqrt(mat["rho"] * mat["Z"] / mat["A"])  # GeV
    dhalf = np.maximum(0.0, np.log(hwp / I) + np.log(bg) - 0.5)
    return K_BETHE * mat["Z"] / mat["A"] / beta ** 2 * (
        0.5 * np.log(2 * M_E * bg ** 2 * wmax / I ** 2) - beta ** 2 - dhalf)


def _apply_material(st: _Truth, rng, x_over_X0, thickness_mm, mass, mat, g1, g2, normal=None):
    """Gaussian multiple-scattering kick (two independent projected angles of width theta0 in the
    plane perpendicular to the direction) and mean energy loss, using the TRUE momentum before
    the layer and the path factor 1/|n.T| (n = x axis, or the per-particle unit normals `normal` (N, 3))."""
    sth, cth = np.sin(st.theta), np.cos(st.theta)
    sph, cph = np.sin(st.phi), np.cos(st.phi)
    T = np.stack([cph * sth, sph * sth, cth], axis=1)
    cfac = 1.0 / np.abs(T[:, 0] if normal is None else np.sum(T * normal, axis=1))
    p = 1.0 / np.abs(st.lam)
    th0 = highland_theta0(p, mass, x_over_X0 * cfac)
    e_th = np.stack([cph * cth, sph * cth, -sth], axis=1)
    e_ph = np.stack([-sph, cph, np.zeros_like(sph)], axis=1)
    Tn = T + (th0 * g1)[:, None] * e_th + (th0 * g2)[:, None] * e_ph
    Tn /= np.linalg.norm(Tn, axis=1, keepdims=True)
    st.phi = np.arctan2(Tn[:, 1], Tn[:, 0])
    st.theta = np.arccos(np.clip(Tn[:, 2], -1.0, 1.0))
    # mean energy loss
    E = np.sqrt(p * p + mass * mass)
    dE = bethe_mean_dedx_mass(p, mass, mat) * mat["rho"] * 1e-3 * 0.1 * thickness_mm * cfac  # GeV
    E2 = E - dE
    ok = E2 > mass
    st.alive &= ok
    p2 = np.sqrt(np.where(ok, E2 * E2 - mass * mass, 1.0))
    st.lam = np.sign(st.lam) / p2


# ---------------------------------------------------------------------------------------------
# the configs
# ---------------------------------------------------------------------------------------------
_CFG = {
    0: dict(seed=1, n=1_000, layers=6, p=("fixed", 1.0), ang=0.05, sig=(0.010, 0.010),
            material=False, smooth=False, ragged=None, field="const"),
    1: dict(seed=2, n=100_000, layers=10, p=("log", 0.5, 10.0), ang=0.1, sig=(0.010, 0.010),
            material=False, smooth=True, ragged=None, field="const"),
    2: dict(seed=3, n=1_000_000, layers=30, p=("log", 1.0, 100.0), ang=0.1, sig=(0.010, 0.030),
            material=True, smooth=True, ragged=None, field="const"),
    3: dict(seed=4, n=1_000_000, layers=30, p=("log", 1.0, 100.0), ang=0.1, sig=(0.010, 0.030),
            material=True, smooth=True, ragged="efficiency", field="const"),
    4: dict(seed=5, n=1_000_000, layers=30, p=("log", 0.5, 10.0), ang=0.2, sig=(0.010, 0.030),
            material=True, smooth=True, ragged="acceptance", field="grid3"),
}


def make_config(cfg: int, n_tracks: Optional[int] = None, seed: Optional[int] = None,
                **overrides) -> Workload:
    """Build BASELINE.json configs[cfg] (optionally with fewer/more tracks or another seed).

    Draw order (whole arrays over tracks, numpy Generator(PCG64(seed))): charge, |p|, phi, theta;
    then per layer: hit noise 2N, [material: kick angles 2N], [CFG3: efficiency uniforms N,
    outlier uniforms N, outlier positions 2N]; finally start smearing 6N.
    """
    c = dict(_CFG[cfg])
    c.update(overrides)
    N = int(n_tracks if n_tracks is not None else c["n"])
    L = int(c["layers"])
    rng = np.random.Generator(np.random.PCG64(c["seed"] if seed is None else seed))
    mass = M_MU
    mat = dict(SILICON)
    x_over_X0, thick = (0.0032, 0.3) if c["material"] else (0.0, 0.0)
    geom = telescope_geometry(L, 30.0, 50.0, x_over_X0, thick, c["sig"])
    bz = 2.0
    grid_desc = cfg4_field_grid() if c["field"] == "grid3" else None

    charge = np.where(rng.random(N) < 0.5, -1.0, 1.0)
    if c["p"][0] == "fixed":
        p = np.full(N, c["p"][1])
        rng.random(N)  # keep the draw order uniform across configs
    else:
        p = np.exp(rng.uniform(np.log(c["p"][1]), np.log(c["p"][2]), N))
    phi = rng.uniform(-c["ang"], c["ang"], N)
    theta = np.pi / 2 + rng.uniform(-c["ang"], c["ang"], N)

    st = _Truth(N)
    st.phi, st.theta, st.lam = phi.copy(), theta.copy(), charge / p
    truth_start = st.bound_on_x_plane()
    truth = np.full((N, L, 6), np.nan)
    hit_ok = np.zeros((N, L), dtype=bool)
    hit_loc = np.zeros((N, L, 2))
    hit_outl = np.zeros((N, L), dtype=bool)
    sig = np.asarray(c["sig"])

    for k in range(1, L + 1):
        xk = 30.0 * k
        if grid_desc is None:
            _helix_to_x_plane(st, xk, bz, mass)
        else:
            _rk4_to_x_plane(st, xk, grid_desc, mass)
        if c["ragged"] == "acceptance":
            st.alive &= (np.abs(st.y) <= 50.0) & (np.abs(st.z) <= 50.0)
        truth[:, k - 1, :] = np.where(st.alive[:, None], st.bound_on_x_plane(), np.nan)
        noise = rng.standard_normal((N, 2)) * sig[None, :]
        hit_loc[:, k - 1, 0] = st.y + noise[:, 0]
        hit_loc[:, k - 1, 1] = st.z + noise[:, 1]
        keep = st.alive.copy()
        if c["material"]:
            g = rng.standard_normal((N, 2))
            _apply_material(st, rng, x_over_X0, thick, mass, mat, g[:, 0], g[:, 1])
        if c["ragged"] == "efficiency":
            eff_u = rng.random(N)
            out_u = rng.random(N)
            out_pos = rng.uniform(-50.0, 50.0, (N, 2))
            keep &= eff_u < 0.95
            is_out = out_u < 0.01
            hit_loc[:, k - 1, :] = np.where(is_out[:, None], out_pos, hit_loc[:, k - 1, :])
            hit_outl[:, k - 1] = is_out
        hit_ok[:, k - 1] = keep

    # start parameters: truth at the origin smeared by the diagonal C0 that is handed to the fit
    sig0 = np.stack([np.full(N, 0.05), np.full(N, 0.05), np.full(N, 1e-3), np.full(N, 1e-3),
                     0.01 * np.abs(truth_start[:, 4]), np.full(N, C_MM_PER_NS)], axis=1)
    params0 = truth_start + rng.standard_normal((N, 6)) * sig0
    cov0 = np.zeros((N, 6, 6))
    for a in range(6):
        cov0[:, a, a] = sig0[:, a] ** 2

    # acceptance stop: hits end at the last layer reached in acceptance (alive is monotone)
    counts = hit_ok.sum(axis=1).astype(np.int32)
    offsets = np.zeros(N + 1, dtype=np.int32)
    np.cumsum(counts, out=offsets[1:])
    tr, ly = np.nonzero(hit_ok)  # row-major: ascending layer within each track
    surf_idx = (ly + 1).astype(np.int32)
    loc = hit_loc[tr, ly, :].copy()
    is_outlier = hit_outl[tr, ly].copy() if c["ragged"] == "efficiency" else None

    options = dict(smooth=int(c["smooth"]), material=int(c["material"]),
                   outlier_chi2=15.0 if c["ragged"] == "efficiency" else 0.0,
                   n_corr_steps=2, max_step_mm=float("inf"), mass_gev=mass, cov_inflation=1.0)
    if grid_desc is None:
        gn = go = gs = gg = None
    else:
        gn, go, gs, gg = grid_desc
    return Workload(
        name=f"cfg{cfg}", n_tracks=N, n_layers=L, geometry=geom,
        field_kind=c["field"], field_b=np.array([0.0, 0.0, bz]),
        grid_n=gn, grid_origin=go, grid_spacing=gs, grid=gg,
        start_surface=0, params0=params0, cov0=cov0, offsets=offsets, surf_idx=surf_idx, loc=loc,
        options=options, material=mat, truth_start=truth_start, truth=truth,
        is_outlier=is_outlier, meta=dict(cfg=cfg, seed=c["seed"] if seed is None else seed),
    )


# ---------------------------------------------------------------------------------------------
# non-planar surfaces ("surfaces of different concrete types"; U33): two small
# tracker-shaped workloads for the cylinder and disc surface kinds.  Not BASELINE.json configs: they exist so that
# the surface kinds are exercised by a whole fit (parity, pulls), not only step by step.
# ---------------------------------------------------------------------------------------------
SURF_PLANE, SURF_CYLINDER, SURF_DISC = 0, 1, 2


def _sinc(a):
    return np.sinc(a / np.pi)  # sin(a)/a, 1 at 0


def _helix_advance(st: _Truth, s_t, bz_tesla, mass):
    """Move every particle by the transverse arc length s_t along its helix in B = (0, 0, bz) (closed form, written with
    sin(a)/a so that it stays exact for straight tracks)."""
    sth = np.sin(st.theta)
    kappa = -st.lam * (bz_tesla * TESLA) / sth
    half = 0.5 * kappa * s_t
    chord = s_t * _sinc(half)
    st.x = st.x + chord * np.cos(st.phi + half)
    st.y = st.y + chord * np.sin(st.phi + half)
    st.z = st.z + s_t * np.cos(st.theta) / sth
    st.phi = st.phi + kappa * s_t
    st.t = st.t + (s_t / sth) * np.sqrt(1.0 + (mass * st.lam) ** 2)


def _helix_to_cylinder(st: _Truth, R, bz_tesla, mass):
    """To the cylinder of radius R around the z axis: Newton iteration on g(s_T) = x(s_T)^2 + y(s_T)^2 - R^2 with the
    closed-form helix, started from the straight-line crossing (outward going)."""
    sth = np.sin(st.theta)
    kappa = -st.lam * (bz_tesla * TESLA) / sth
    b = st.x * np.cos(st.phi) + st.y * np.sin(st.phi)
    c0 = st.x ** 2 + st.y ** 2 - R * R
    disc = b * b - c0
    ok = disc > 0
    s = np.where(ok, -c0 / (b + np.sqrt(np.where(ok, disc, 1.0))), 0.0)
    for _ in range(8):
        half = 0.5 * kappa * s
        chord = s * _sinc(half)
        x = st.x + chord * np.cos(st.phi + half)
        y = st.y + chord * np.sin(st.phi + half)
        ph = st.phi + kappa * s
        g = x * x + y * y - R * R
        dg = 2.0 * (x * np.cos(ph) + y * np.sin(ph))
        with np.errstate(divide="ignore", invalid="ignore"):
            s = np.where(ok & (dg > 0), s - g / dg, s)
    st.alive &= ok & (s > 0)
    _helix_advance(st, np.where(st.alive, s, 0.0), bz_tesla, mass)


def _helix_to_z_plane(st: _Truth, z_plane, bz_tesla, mass):
    cth = np.cos(st.theta)
    ok = cth > 1e-3
    s_t = np.where(ok, (z_plane - st.z) * np.sin(st.theta) / np.where(ok, cth, 1.0), 0.0)
    st.alive &= ok & (s_t > 0)
    _helix_advance(st, np.where(st.alive, s_t, 0.0), bz_tesla, mass)
    st.z = np.where(st.alive, z_plane, st.z)


def make_tracker(kind: str, n_tracks: int = 20_000, seed: Optional[int] = None, n_layers: int = 10, material: bool = True,
                 p_range=(0.5, 10.0), smooth: bool = True) -> Workload:
    """kind = "barrel": start plane x = 0, then n_layers cylinders around the z axis (radius 30 k mm, axis v = z,
    azimuth from n = x towards u = y): bound (R alpha, z, phi, theta, q/p, t).
    kind = "endcap": start plane z = 0 (u = x, v = y, n = z), then n_layers discs z = 30 k mm in polar coordinates:
    bound (rho, alpha, phi, theta, q/p, t).
    B = 2 T along z; truth = closed-form helix between surfaces, Highland kicks + Bethe mean loss per layer when
    `material`; hits = truth local position + N(0, sigma), sigma = (10 um, 30 um) on cylinders (arc length, z) and
    (10 um, 0.1 mrad) on discs (rho, alpha).  Start = truth on surface 0 smeared by the diagonal C0 of the configs."""
    assert kind in ("barrel", "endcap")
    N, L = int(n_tracks), int(n_layers)
    rng = np.random.Generator(np.random.PCG64((6 if kind == "barrel" else 7) if seed is None else seed))
    mass, mat, bz = M_MU, dict(SILICON), 2.0
    x_over_X0, thick = (0.0032, 0.3) if material else (0.0, 0.0)
    g = np.zeros((L + 1, GEOM_STRIDE), dtype=np.float64)
    if kind == "barrel":
        sig = np.array([0.010, 0.030])
        for k in range(L + 1):
            g[k, 0:3] = (0.0, 0.0, 0.0)
            g[k, 3:6], g[k, 6:9], g[k, 9:12] = (0.0, 1.0, 0.0), (0.0, 0.0, 1.0), (1.0, 0.0, 0.0)
            g[k, 12:14] = (30.0 * k, 500.0) if k > 0 else (50.0, 50.0)   # cylinder: radius, half length in z
            g[k, 18] = SURF_CYLINDER if k > 0 else SURF_PLANE
    else:
        sig = np.array([0.010, 1.0e-4])
        for k in range(L + 1):
            g[k, 0:3] = (0.0, 0.0, 30.0 * k)
            g[k, 3:6], g[k, 6:9], g[k, 9:12] = (1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0)
            g[k, 12:14] = (200.0, 200.0)
            g[k, 18] = SURF_DISC if k > 0 else SURF_PLANE
    g[1:, 14], g[1:, 15] = x_over_X0, thick
    g[:, 16:18] = sig[None, :] ** 2

    charge = np.where(rng.random(N) < 0.5, -1.0, 1.0)
    p = np.exp(rng.uniform(np.log(p_range[0]), np.log(p_range[1]), N))
    st = _Truth(N)
    if kind == "barrel":
        st.phi = rng.uniform(-0.3, 0.3, N)
        st.theta = np.pi / 2 + rng.uniform(-0.3, 0.3, N)
    else:
        st.phi = rng.uniform(-1.0, 1.0, N)
        st.theta = rng.uniform(0.2, 0.5, N)
    st.lam = charge / p

    def bound(k):
        if kind == "barrel":
            if k == 0:
                return np.stack([st.y, st.z, st.phi, st.theta, st.lam, st.t], axis=1)
            return np.stack([30.0 * k * np.arctan2(st.y, st.x), st.z, st.phi, st.theta, st.lam, st.t], axis=1)
        if k == 0:
            return np.stack([st.x, st.y, st.phi, st.theta, st.lam, st.t], axis=1)
        return np.stack([np.hypot(st.x, st.y), np.arctan2(st.y, st.x), st.phi, st.theta, st.lam, st.t], axis=1)

    truth_start = bound(0)
    truth = np.full((N, L, 6), np.nan)
    hit_ok = np.zeros((N, L), dtype=bool)
    hit_loc = np.zeros((N, L, 2))
    for k in range(1, L + 1):
        if kind == "barrel":
            _helix_to_cylinder(st, 30.0 * k, bz, mass)
        else:
            _helix_to_z_plane(st, 30.0 * k, bz, mass)
        b = bound(k)
        truth[:, k - 1, :] = np.where(st.alive[:, None], b, np.nan)
        hit_loc[:, k - 1, :] = b[:, :2] + rng.standard_normal((N, 2)) * sig[None, :]
        hit_ok[:, k - 1] = st.alive
        if material:
            kicks = rng.standard_normal((N, 2))
            if kind == "barrel":
                rho = np.hypot(st.x, st.y)
                nrm = np.stack([st.x / rho, st.y / rho, np.zeros(N)], axis=1)
            else:
                nrm = np.tile(np.array([0.0, 0.0, 1.0]), (N, 1))
            _apply_material(st, rng, x_over_X0, thick, mass, mat, kicks[:, 0], kicks[:, 1], normal=nrm)

    sig0 = np.stack([np.full(N, 0.05), np.full(N, 0.05), np.full(N, 1e-3), np.full(N, 1e-3),
                     0.01 * np.abs(truth_start[:, 4]), np.full(N, C_MM_PER_NS)], axis=1)
    params0 = truth_start + rng.standard_normal((N, 6)) * sig0
    cov0 = np.zeros((N, 6, 6))
    for a in range(6):
        cov0[:, a, a] = sig0[:, a] ** 2
    counts = hit_ok.sum(axis=1).astype(np.int32)
    offsets = np.zeros(N + 1, dtype=np.int32)
    np.cumsum(counts, out=offsets[1:])
    tr, ly = np.nonzero(hit_ok)
    options = dict(smooth=int(smooth), material=int(material), outlier_chi2=0.0, n_corr_steps=2,
                   max_step_mm=float("inf"), mass_gev=mass, cov_inflation=1.0)
    return Workload(
        name=kind, n_tracks=N, n_layers=L, geometry=g, field_kind="const", field_b=np.array([0.0, 0.0, bz]),
        grid_n=None, grid_origin=None, grid_spacing=None, grid=None, start_surface=0, params0=params0, cov0=cov0,
        offsets=offsets, surf_idx=(ly + 1).astype(np.int32), loc=hit_loc[tr, ly, :].copy(), options=options,
        material=mat, truth_start=truth_start, truth=truth, is_outlier=None,
        meta=dict(kind=kind, surface_kinds=(1 << SURF_PLANE) | (1 << (SURF_CYLINDER if kind == "barrel" else SURF_DISC))),
    )


WORKLOAD_NAMES = {
    0: "cfg0 telescope 6 layers, no material, filter only, 1e3 tracks",
    1: "cfg1 telescope 10 layers, no material, filter+RTS, 1e5 tracks",
    2: "cfg2 telescope 30 layers with material, filter+RTS, 1e6 tracks",
    3: "cfg3 ragged 100 events x 1e4 tracks, 30 layers material, eff 0.95, 1% outliers, filter+RTS",
    4: "cfg4 field-map 30 layers material, trilinear grid field, acceptance stop, filter+RTS",
    # not BASELINE.json configs: the two tracker-shaped workloads of the cylinder and disc surface kinds (make_tracker)
    5: "barrel: start plane + 10 cylinders around z, material, constant field, filter+RTS",
    6: "endcap: start plane + 10 discs in polar coordinates, material, constant field, filter+RTS",
}


def make_workload(cfg: int, n_tracks: Optional[int] = None, seed: Optional[int] = None) -> Workload:
    """BASELINE.json configs[cfg] for cfg 0..4; 5 / 6: the barrel / endcap workloads (default 1,000,000 tracks)."""
    if cfg in (5, 6):
        return make_tracker("barrel" if cfg == 5 else "endcap", n_tracks=n_tracks or 1_000_000, seed=seed)
    return make_config(cfg, n_tracks=n_tracks, seed=seed)
