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
