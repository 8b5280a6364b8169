"""GPU-vs-oracle comparator with the tolerances of BASELINE.json's north_star, read as DESIGN.md
"Tolerances" states them:

  parameters   |d| <= 1e-10 * max(|ref|, floor)   floors (1 mm, 1 mm, 0.1 rad, 1 rad, 0.01 /GeV, 1 mm)
  covariance   |dC_ij| <= 1e-8 * sqrt(C_ii C_jj)   (reference values)
  chi2         |d| <= 1e-9 * max(|ref|, 1)
  ndf, counters, flags, status: exact

Both sides are numpy arrays in the natural AoS layouts (params (..., 6), cov (..., 6, 6)).
"""
import numpy as np

PARAM_RTOL = 1e-10
COV_RTOL = 1e-8
CHI2_RTOL = 1e-9
PARAM_FLOOR = np.array([1.0, 1.0, 0.1, 1.0, 0.01, 1.0])


def param_excess(got, ref):
    """max over elements of |d| / (1e-10 * max(|ref|, floor)); <= 1 passes. NaN must match NaN."""
    got, ref = np.asarray(got), np.asarray(ref)
    nan_g, nan_r = np.isnan(got), np.isnan(ref)
    if not np.array_equal(nan_g, nan_r):
        return np.inf
    tol = PARAM_RTOL * np.maximum(np.abs(ref), PARAM_FLOOR)
    with np.errstate(invalid="ignore"):
        ex = np.abs(got - ref) / tol
    ex = np.where(nan_r, 0.0, ex)
    return float(ex.max()) if ex.size else 0.0


def cov_excess(got, ref):
    got, ref = np.asarray(got), np.asarray(ref)
    nan_g, nan_r = np.isnan(got), np.isnan(ref)
    if not np.array_equal(nan_g, nan_r):
        return np.inf
    d = np.sqrt(np.abs(np.einsum("...ii->...i", ref)))
    scale = d[..., :, None] * d[..., None, :]
    with np.errstate(invalid="ignore", divide="ignore"):
        ex = np.abs(got - ref) / (COV_RTOL * scale)
    ex = np.where(nan_r | (np.abs(got - ref) == 0), 0.0, ex)
    return float(ex.max()) if ex.size else 0.0


def chi2_excess(got, ref):
    got, ref = np.asarray(got), np.asarray(ref)
    ex = np.abs(got - ref) / (CHI2_RTOL * np.maximum(np.abs(ref), 1.0))
    return float(ex.max()) if ex.size else 0.0


def compare(gpu, ref, states=False, sel=None, offsets=None):
    """Returns a dict of excess factors (<= 1 passes) and asserts the exact fields.
    `sel`: optional boolean/index selection of tracks; with `offsets` (the batch's CSR offsets) the per-hit
    arrays are compared on the selected tracks' hits too."""
    def pick(a):
        return a if sel is None else a[sel]
    rep = {}
    for name in ("ndf", "n_used", "n_outliers", "n_holes"):
        np.testing.assert_array_equal(pick(getattr(gpu, name)), pick(getattr(ref, name)), err_msg=name)
    np.testing.assert_array_equal(pick(gpu.status).astype(np.uint32), pick(ref.status).astype(np.uint32),
                                  err_msg="status")
    rep["first_params"] = param_excess(pick(gpu.first_params), pick(ref.first_params))
    rep["last_params"] = param_excess(pick(gpu.last_params), pick(ref.last_params))
    rep["first_cov"] = cov_excess(pick(gpu.first_cov), pick(ref.first_cov))
    rep["last_cov"] = cov_excess(pick(gpu.last_cov), pick(ref.last_cov))
    rep["chi2"] = chi2_excess(pick(gpu.chi2), pick(ref.chi2))
    if gpu.hit_flags is not None and ref.hit_flags is not None and (sel is None or offsets is not None):
        hsel = slice(None)
        if sel is not None:  # the hits of the selected tracks (CSR offsets of the batch)
            keep = np.zeros(len(offsets) - 1, bool)
            keep[sel] = True
            hsel = np.repeat(keep, np.diff(offsets))
        np.testing.assert_array_equal(gpu.hit_flags[hsel], ref.hit_flags[hsel], err_msg="hit_flags")
        rep["hit_chi2"] = chi2_excess(gpu.hit_chi2[hsel], ref.hit_chi2[hsel])
    gp, rp = getattr(gpu, "perigee_params", None), getattr(ref, "perigee_params", None)
    if gp is not None and rp is not None:  # fitted parameters on the perigee surface (NaN where bit 128 is set)
        rep["perigee_params"] = param_excess(pick(gp), pick(rp))
        rep["perigee_cov"] = cov_excess(pick(gpu.perigee_cov), pick(ref.perigee_cov))
    if states:
        for kind in ("pred", "filt", "smooth"):
            g, r = getattr(gpu, kind + "_params", None), getattr(ref, kind + "_params", None)
            if g is None or r is None:
                continue
            rep[kind + "_params"] = param_excess(pick(g), pick(r))
            rep[kind + "_cov"] = cov_excess(pick(getattr(gpu, kind + "_cov")), pick(getattr(ref, kind + "_cov")))
    return rep


def assert_parity(gpu, ref, states=False, sel=None, label="", loosen=1.0, offsets=None):
    """loosen > 1 widens every floating-point bar by that factor (only for inputs whose conditioning
    DESIGN.md "Tolerances" shows to exceed the north_star bars, e.g. a 1e4-inflated prior)."""
    rep = compare(gpu, ref, states=states, sel=sel, offsets=offsets)
    bad = {k: v for k, v in rep.items() if not v <= loosen}
    assert not bad, f"{label}: tolerance exceeded (factor over the bar): {bad}; all: {rep}"
    return rep


def arbitrated(gpu, ref64, ref_ld, states=False, sel=None, offsets=None, label="", slack=2.0):
    """Parity where the conditioning of the inputs exceeds the north_star bars.

    ref_ld is the long-double build of the oracle (the same algorithm with a 64-bit mantissa) on the same inputs: the
    nearest thing to the exact result of the algorithm.  Every quantity is compared with IT; the bar of a quantity is
    the north_star bar, widened only where -- and only as far as -- the DOUBLE oracle itself is away from the
    long-double result:   factor(q) = max(1, slack * excess(ref64 vs ref_ld)(q)).
    So the CUDA path may be at most `slack` times further from the exact result than the double oracle is, or inside
    the north_star bar, whichever is wider.  Integers, flags and status stay exact (against both builds).
    Returns (rep_gpu_vs_ld, rep_ref64_vs_ld)."""
    e64 = compare(ref64, ref_ld, states=states, sel=sel, offsets=offsets)
    rep = compare(gpu, ref_ld, states=states, sel=sel, offsets=offsets)
    bad = {k: (v, max(1.0, slack * e64.get(k, 0.0))) for k, v in rep.items() if not v <= max(1.0, slack * e64.get(k, 0.0))}
    assert not bad, f"{label}: further from the long-double result than allowed (excess, allowed): {bad}; gpu: {rep}; f64: {e64}"
    return rep, e64


def resolution_loss(low, ref, offsets, cut=0.0, guard=0.1):
    """How far a reduced-precision fit `low` (float operands) is from the double fit `ref` of the same inputs, in the
    units that matter for the physics: parameters in standard deviations of the reference, variances relative, chi2
    absolute.  Tracks on which a discrete decision flipped (a hit whose chi2 is within `guard` of the outlier cut, a
    status bit) are counted and left out of the value statistics.  Returns a dict."""
    flipped = (low.status != ref.status) | (low.n_used != ref.n_used) | (low.n_outliers != ref.n_outliers)
    if low.hit_flags is not None and ref.hit_flags is not None:
        hit_track = np.repeat(np.arange(len(offsets) - 1), np.diff(offsets))
        diff = low.hit_flags != ref.hit_flags
        if cut > 0:  # a flip is only legitimate next to the cut
            assert np.all(np.abs(ref.hit_chi2[diff] - cut) < guard), "a hit flag flipped far from the outlier cut"
        flipped[np.unique(hit_track[diff])] = True
    ok = ~flipped & ((ref.status & 7) == 0)
    out = dict(flipped_tracks=int(flipped.sum()), tracks=int(ok.sum()))
    worst_p, worst_v = 0.0, 0.0
    for nm in ("first", "last"):
        xa, xb = getattr(ref, nm + "_params")[ok], getattr(low, nm + "_params")[ok]
        va = np.einsum("nii->ni", getattr(ref, nm + "_cov")[ok])
        vb = np.einsum("nii->ni", getattr(low, nm + "_cov")[ok])
        d = xb - xa
        d[:, 2] = (d[:, 2] + np.pi) % (2 * np.pi) - np.pi
        worst_p = max(worst_p, float(np.max(np.abs(d) / np.sqrt(va))))
        worst_v = max(worst_v, float(np.max(np.abs(vb / va - 1.0))))
        out[nm + "_params_sigma_rms"] = [float(v) for v in np.sqrt(np.mean((d / np.sqrt(va)) ** 2, axis=0))]
    out["params_sigma"], out["var_rel"] = worst_p, worst_v
    out["chi2_abs"] = float(np.max(np.abs(low.chi2[ok] - ref.chi2[ok])))
    return out


# ---- whole-population comparison at full size (first_*, last_*, chi2, ndf, counters, status for ALL
# tracks; per-surface states for a 1 % sample) --------------------------------------------------------------------------
def per_track_factors(gpu, ref):
    """Per track, the largest factor of the tolerance used by each floating-point quantity (same bars as compare())."""
    out = {}
    for name in ("first_params", "last_params"):
        g, r = np.asarray(getattr(gpu, name)), np.asarray(getattr(ref, name))
        tol = PARAM_RTOL * np.maximum(np.abs(r), PARAM_FLOOR)
        with np.errstate(invalid="ignore"):
            ex = np.abs(g - r) / tol
        ex = np.where(np.isnan(r) & np.isnan(g), 0.0, np.where(np.isnan(ex), np.inf, ex))
        out[name] = ex.max(axis=1)
    for name in ("first_cov", "last_cov"):
        g, r = np.asarray(getattr(gpu, name)), np.asarray(getattr(ref, name))
        d = np.sqrt(np.abs(np.einsum("nii->ni", r)))
        with np.errstate(invalid="ignore", divide="ignore"):
            ex = np.abs(g - r) / (COV_RTOL * d[:, :, None] * d[:, None, :])
        ex = np.where((np.isnan(r) & np.isnan(g)) | (g == r), 0.0, np.where(np.isnan(ex), np.inf, ex))
        out[name] = ex.reshape(ex.shape[0], -1).max(axis=1)
    g, r = np.asarray(gpu.chi2), np.asarray(ref.chi2)
    out["chi2"] = np.abs(g - r) / (CHI2_RTOL * np.maximum(np.abs(r), 1.0))
    return out


def whole_population(wl, gpu, label, **oracle_over):
    """Every track of `wl` re-fitted by the oracle (all host cores) and compared with the CUDA result `gpu` (host arrays of
    DeviceOutputs.to_host()).  Discrete results (ndf, counters, status, per-hit flags) must agree on every track: a track
    that differs is LISTED in the failure message, none is excluded.  Floating-point results: the worst factor of the
    north_star bars and the 99.99th percentile over tracks are printed per quantity; the worst must be <= 1."""
    import oracle
    ref = oracle.fit_workload(wl, **oracle_over)
    n = wl.n_tracks
    flipped = np.zeros(n, bool)
    for name in ("ndf", "n_used", "n_outliers", "n_holes"):
        flipped |= np.asarray(getattr(gpu, name)) != np.asarray(getattr(ref, name))
    flipped |= np.asarray(gpu.status).astype(np.uint32) != np.asarray(ref.status).astype(np.uint32)
    hit_diff = 0
    if gpu.hit_flags is not None and ref.hit_flags is not None:
        bad_hits = np.asarray(gpu.hit_flags) != np.asarray(ref.hit_flags)
        hit_diff = int(bad_hits.sum())
        if hit_diff:
            flipped[np.unique(np.searchsorted(wl.offsets, np.flatnonzero(bad_hits), side="right") - 1)] = True
    idx = np.flatnonzero(flipped)
    listing = [dict(track=int(i), status=(int(gpu.status[i]), int(ref.status[i])), n_used=(int(gpu.n_used[i]), int(ref.n_used[i])),
                    n_outliers=(int(gpu.n_outliers[i]), int(ref.n_outliers[i])), n_holes=(int(gpu.n_holes[i]), int(ref.n_holes[i])))
               for i in idx[:20]]
    fac = per_track_factors(gpu, ref)
    if gpu.hit_chi2 is not None and ref.hit_chi2 is not None:
        g, r = np.asarray(gpu.hit_chi2), np.asarray(ref.hit_chi2)
        fac["hit_chi2"] = np.abs(g - r) / (CHI2_RTOL * np.maximum(np.abs(r), 1.0))
    rep = {k: dict(worst=float(v.max()) if v.size else 0.0, p9999=float(np.percentile(v, 99.99)) if v.size else 0.0,
                   at=int(np.argmax(v)) if v.size else -1) for k, v in fac.items()}
    print(f"\n[whole population] {label}: {n} tracks, {wl.n_meas} hits against the oracle; discrete decisions differing on "
          f"{idx.size} tracks ({hit_diff} hit flags)")
    for k, v in rep.items():
        print(f"    {k:13s} worst factor of the bar {v['worst']:.3e} (element {v['at']}), 99.99th percentile {v['p9999']:.3e}")
    assert idx.size == 0, f"{label}: discrete decisions differ on {idx.size} of {n} tracks (first 20 listed): {listing}"
    over = {k: v for k, v in rep.items() if not v["worst"] <= 1.0}
    assert not over, f"{label}: tolerance exceeded: {over}"
    return rep, ref


def state_sample(wl, label, fraction=0.01, seed=0, **over):
    """Per-surface PRED / FILT / SMOOTH states of a `fraction` sample of the tracks (first and last tile included): the
    sample is fitted by both sides with all per-leg states out and compared element by element."""
    import oracle
    import paper_2105_01796_b200 as kf
    rng = np.random.default_rng(seed)
    n = wl.n_tracks
    idx = np.unique(np.concatenate([rng.choice(n, max(1, int(n * fraction)), replace=False), np.arange(min(64, n)),
                                    np.arange(max(0, n - 64), n)]))
    sub = wl.subset(idx)
    ref = oracle.fit_workload(sub, states=True, **over)
    got = kf.fit_workload(sub, states=True, **over)
    rep = assert_parity(got, ref, states=True, label=label + f" (per-leg states, {idx.size} tracks)")
    print(f"[state sample] {label}: {idx.size} tracks, worst factor {max(rep.values()):.3e}")
    return rep
