"""CPU ORACLE binding -- TEST INFRASTRUCTURE ONLY (see oracle/kf_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It builds oracle/kf_oracle.c with gcc and exposes it through ctypes with
numpy arrays in natural AoS layouts.  It imports nothing from the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kf_oracle.c")
_HDR = os.path.join(_HERE, "kf_oracle.h")
GEOM_STRIDE = 20

# The three builds of the one source file (kf_oracle.c "the arithmetic type"):
#   f64  the oracle proper (IEEE double)
#   ld   the arbiter: the same algorithm in x87 80-bit long double (64-bit mantissa), results rounded to double at the door
#   f32  the paper's operating point: every operand float, the 6x6 solve of the smoother in double
PRECISIONS = {
    "f64": dict(lib="libkf_oracle.so", flags=[]),
    "ld": dict(lib="libkf_oracle_ld.so", flags=['-DKFO_REAL=long double', '-DKFO_SOLVE_REAL=long double']),
    "f32": dict(lib="libkf_oracle_f32.so", flags=["-DKFO_REAL=float", "-fsingle-precision-constant"]),
}
_LIB = os.path.join(_HERE, PRECISIONS["f64"]["lib"])


def build(force: bool = False, precision: str = "f64") -> str:
    """gcc -O2 -ffp-contract=off -fopenmp (no fused multiply-add; -ffp-contract=off also keeps x87 out of the
    double and float builds: SSE arithmetic in the declared type throughout)."""
    spec = PRECISIONS[precision]
    out = os.path.join(_HERE, spec["lib"])
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(out) or os.path.getmtime(out) < newest:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c99", "-Wall", "-shared",
               "-fPIC", *spec["flags"], "-o", out, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return out


def build_all(force: bool = False) -> list:
    return [build(force, p) for p in PRECISIONS]


class _Field(C.Structure):
    _fields_ = [("kind", C.c_int32), ("b", C.c_double * 3), ("n", C.c_int32 * 3),
                ("origin", C.c_double * 3), ("spacing", C.c_double * 3),
                ("grid", C.POINTER(C.c_double))]


class _Options(C.Structure):
    _fields_ = [("smooth", C.c_int32), ("material", C.c_int32), ("outlier_chi2", C.c_double),
                ("n_corr_steps", C.c_int32), ("max_step_mm", C.c_double), ("mass_gev", C.c_double),
                ("cov_inflation", C.c_double), ("mat_Z", C.c_double), ("mat_A", C.c_double),
                ("mat_rho", C.c_double), ("mat_I_eV", C.c_double), ("step_tolerance_mm", C.c_double),
                ("field_gradient", C.c_int32)]


_libs = {}
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def lib(precision: str = "f64"):
    if precision not in _libs:
        L = C.CDLL(build(precision=precision))
        L.kfo_fit_batch.restype = C.c_int32
        L.kfo_propagate.restype = C.c_int32
        L.kfo_update.restype = C.c_int32
        L.kfo_material.restype = C.c_int32
        L.kfo_rts_step.restype = C.c_int32
        L.kfo_field_at.restype = None
        L.kfo_to_line.restype = C.c_int32
        L.kfo_perigee_batch.restype = C.c_int32
        L.kfo_rkn4_step.restype = None
        L.kfo_real_bytes.restype = C.c_int32
        L.kfo_solve_real_bytes.restype = C.c_int32
        _libs[precision] = L
    return _libs[precision]


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _arr(a, dtype=np.float64):
    return np.ascontiguousarray(a, dtype=dtype)


def make_field(kind="const", b=(0.0, 0.0, 2.0), grid_n=None, grid_origin=None, grid_spacing=None,
               grid=None):
    f = _Field()
    keep = None
    if kind == "const":
        f.kind = 0
        f.b[:] = [float(v) for v in b]
    else:
        f.kind = 1
        keep = _arr(grid)
        f.n[:] = [int(v) for v in grid_n]
        f.origin[:] = [float(v) for v in grid_origin]
        f.spacing[:] = [float(v) for v in grid_spacing]
        f.grid = keep.ctypes.data_as(_dp)
    f._keep = keep
    return f


def make_options(smooth=1, material=0, outlier_chi2=0.0, n_corr_steps=2, max_step_mm=float("inf"),
                 mass_gev=0.1056583755, cov_inflation=1.0, Z=14.0, A=28.0855, rho=2.329,
                 I_eV=173.0, step_tolerance_mm=0.0, field_gradient=0, **_ignored):
    o = _Options()
    o.step_tolerance_mm = float(step_tolerance_mm)
    o.field_gradient = int(field_gradient)
    o.smooth, o.material, o.outlier_chi2 = int(smooth), int(material), float(outlier_chi2)
    o.n_corr_steps, o.max_step_mm, o.mass_gev = int(n_corr_steps), float(max_step_mm), float(mass_gev)
    o.cov_inflation = float(cov_inflation)
    o.mat_Z, o.mat_A, o.mat_rho, o.mat_I_eV = float(Z), float(A), float(rho), float(I_eV)
    return o


def field_of(wl):
    return make_field(wl.field_kind, wl.field_b, wl.grid_n, wl.grid_origin, wl.grid_spacing, wl.grid)


def options_of(wl, **over):
    kw = dict(wl.options)
    kw.update(Z=wl.material["Z"], A=wl.material["A"], rho=wl.material["rho"], I_eV=wl.material["I_eV"])
    kw.update(over)
    return make_options(**kw)


# ---- step-level wrappers (used by the pin tests) ----------------------------------------------
def field_at(fld, r, precision="f64"):
    b = np.zeros(3)
    cl = C.c_int32(0)
    lib(precision).kfo_field_at(C.byref(fld), _d(_arr(r)), _d(b), C.byref(cl))
    return b, cl.value


def field_gradient_at(fld, r, precision="f64"):
    G = np.zeros((3, 3))
    L = lib(precision)
    L.kfo_field_gradient_at.restype = None
    L.kfo_field_gradient_at(C.byref(fld), _d(_arr(r)), _d(G))
    return G


def rkn4_step(fld, mass, f, h, precision="f64", field_gradient=0):
    fo, Ds = np.zeros(8), np.zeros((8, 8))
    eps, cl = C.c_double(0), C.c_int32(0)
    lib(precision).kfo_rkn4_step(C.byref(fld), C.c_double(mass), _d(_arr(f)), C.c_double(h), _d(fo), _d(Ds),
                        C.byref(eps), C.byref(cl), C.c_int32(int(field_gradient)))
    return fo, Ds, eps.value


def propagate(fld, opt, x, surf_from, surf_to, precision="f64"):
    xo, J, fo = np.zeros(6), np.zeros((6, 6)), np.zeros(8)
    err, cl = C.c_double(0), C.c_int32(0)
    rc = lib(precision).kfo_propagate(C.byref(fld), C.byref(opt), _d(_arr(x)), _d(_arr(surf_from)),
                             _d(_arr(surf_to)), _d(xo), _d(J), _d(fo), C.byref(err), C.byref(cl))
    return SimpleNamespace(rc=rc, x=xo, J=J, free=fo, rk_err=err.value, clamped=cl.value)


def update(xp, Cp, m, V, precision="f64"):
    xf, Cf, chi2 = np.zeros(6), np.zeros((6, 6)), C.c_double(0)
    rc = lib(precision).kfo_update(_d(_arr(xp)), _d(_arr(Cp)), _d(_arr(m)), _d(_arr(V)), _d(xf), _d(Cf),
                          C.byref(chi2))
    return rc, xf, Cf, chi2.value


def material(opt, surf, xf, Cf, precision="f64"):
    xo, Co = np.zeros(6), np.zeros((6, 6))
    g, th0, dE = C.c_double(0), C.c_double(0), C.c_double(0)
    rc = lib(precision).kfo_material(C.byref(opt), _d(_arr(surf)), _d(_arr(xf)), _d(_arr(Cf)), _d(xo), _d(Co),
                            C.byref(g), C.byref(th0), C.byref(dE))
    return SimpleNamespace(rc=rc, x=xo, C=Co, g=g.value, theta0=th0.value, dE=dE.value)


def rts_step(xf, Cf, F1, xp1, Cp1, xs1, Cs1, precision="f64"):
    xs, Cs = np.zeros(6), np.zeros((6, 6))
    rc = lib(precision).kfo_rts_step(_d(_arr(xf)), _d(_arr(Cf)), _d(_arr(F1)), _d(_arr(xp1)), _d(_arr(Cp1)),
                            _d(_arr(xs1)), _d(_arr(Cs1)), _d(xs), _d(Cs))
    return rc, xs, Cs


def to_line(fld, opt, x, Cm, surf_from, line_c=(0.0, 0.0, 0.0), line_a=(0.0, 0.0, 1.0), precision="f64"):
    """bound state on a plane -> perigee parameters on the line surface (kfo_to_line)."""
    xo, Co, J = np.zeros(6), np.zeros((6, 6)), np.zeros((6, 6))
    cl = C.c_int32(0)
    rc = lib(precision).kfo_to_line(C.byref(fld), C.byref(opt), _d(_arr(x)), _d(_arr(Cm)), _d(_arr(surf_from)),
                           _d(_arr(line_c)), _d(_arr(line_a)), _d(xo), _d(Co), _d(J), C.byref(cl))
    return SimpleNamespace(rc=rc, x=xo, C=Co, J=J, clamped=cl.value)


def perigee_batch(res, geometry, start_surface, fld, opt, line_c=(0.0, 0.0, 0.0), line_a=(0.0, 0.0, 1.0), precision="f64"):
    """Adds perigee_params (N,6), perigee_cov (N,6,6) to a fit result (and KFO_ST_PERIGEE = 128 to its
    status where the extrapolation stopped): first_* taken to the line surface."""
    N = res.first_params.shape[0]
    nleg = (res.n_used + res.n_outliers + res.n_holes).astype(np.int32)
    on = (int(start_surface) + (nleg > 0)).astype(np.int32)
    res.perigee_params, res.perigee_cov = np.zeros((N, 6)), np.zeros((N, 6, 6))
    rc = lib(precision).kfo_perigee_batch(C.c_int64(N), _d(_arr(res.first_params)), _d(_arr(res.first_cov)),
                                 on.ctypes.data_as(_ip), _d(_arr(geometry)), C.byref(fld), C.byref(opt),
                                 _d(_arr(line_c)), _d(_arr(line_a)), _d(res.perigee_params), _d(res.perigee_cov),
                                 res.status.ctypes.data_as(C.POINTER(C.c_uint32)))
    if rc < 0:
        raise ValueError("kfo_perigee_batch rejected the call")
    return res


# ---- the batch fit ----------------------------------------------------------------------------
def fit_batch(params0, cov0, start_surface, offsets, surf_idx, loc, geometry, fld, opt, var=None,
              cov01=None, states=False, n_threads=0, precision="f64"):
    """Fit N tracks; returns a namespace of numpy arrays (AoS: params (N,6), cov (N,6,6))."""
    params0, cov0 = _arr(params0), _arr(cov0)
    offsets, surf_idx = _arr(offsets, np.int32), _arr(surf_idx, np.int32)
    loc, geometry = _arr(loc), _arr(geometry)
    N, M, nS = params0.shape[0], surf_idx.shape[0], geometry.shape[0]
    Lmax = nS - 1 - int(start_surface)
    r = SimpleNamespace(
        first_params=np.zeros((N, 6)), first_cov=np.zeros((N, 6, 6)),
        last_params=np.zeros((N, 6)), last_cov=np.zeros((N, 6, 6)), chi2=np.zeros(N),
        ndf=np.zeros(N, np.int32), status=np.zeros(N, np.uint32), n_used=np.zeros(N, np.int32),
        n_outliers=np.zeros(N, np.int32), n_holes=np.zeros(N, np.int32),
        hit_chi2=np.zeros(M), hit_flags=np.zeros(M, np.uint8), rk_err_max=np.zeros(N))
    if states:
        r.pred_params, r.pred_cov = np.zeros((N, Lmax, 6)), np.zeros((N, Lmax, 6, 6))
        r.filt_params, r.filt_cov = np.zeros((N, Lmax, 6)), np.zeros((N, Lmax, 6, 6))
        r.smooth_params, r.smooth_cov = np.zeros((N, Lmax, 6)), np.zeros((N, Lmax, 6, 6))
    else:
        r.pred_params = r.pred_cov = r.filt_params = r.filt_cov = r.smooth_params = r.smooth_cov = None
    var_a = None if var is None else _arr(var)
    c01_a = None if cov01 is None else _arr(cov01)
    rc = lib(precision).kfo_fit_batch(
        C.c_int64(N), _d(params0), _d(cov0), C.c_int32(int(start_surface)),
        offsets.ctypes.data_as(_ip), surf_idx.ctypes.data_as(_ip), _d(loc), _d(var_a), _d(c01_a),
        C.c_int32(nS), _d(geometry), C.byref(fld), C.byref(opt),
        _d(r.first_params), _d(r.first_cov), _d(r.last_params), _d(r.last_cov), _d(r.chi2),
        r.ndf.ctypes.data_as(_ip), r.status.ctypes.data_as(C.POINTER(C.c_uint32)),
        r.n_used.ctypes.data_as(_ip), r.n_outliers.ctypes.data_as(_ip), r.n_holes.ctypes.data_as(_ip),
        _d(r.pred_params), _d(r.pred_cov), _d(r.filt_params), _d(r.filt_cov), _d(r.smooth_params),
        _d(r.smooth_cov), _d(r.hit_chi2), r.hit_flags.ctypes.data_as(C.POINTER(C.c_uint8)),
        _d(r.rk_err_max), C.c_int32(int(n_threads)))
    if rc < 0:
        raise ValueError(f"kfo_fit_batch rejected the call (rc={rc})")
    r.threads = rc
    return r


def fit_workload(wl, states=False, n_threads=0, perigee=None, precision="f64", **opt_over):
    """perigee = (line_centre, line_direction) adds perigee_params / perigee_cov (perigee_batch).
    precision: "f64" (the oracle), "ld" (the long-double arbiter) or "f32" (float operands, 6x6 solve in double)."""
    opt_over.pop("variant", None)  # a kernel-variant choice of the CUDA path means nothing here
    fld, opt = field_of(wl), options_of(wl, **opt_over)
    res = fit_batch(wl.params0, wl.cov0, wl.start_surface, wl.offsets, wl.surf_idx, wl.loc,
                    wl.geometry, fld, opt, states=states, n_threads=n_threads, precision=precision)
    if perigee is not None:
        perigee_batch(res, wl.geometry, wl.start_surface, fld, opt, perigee[0], perigee[1], precision=precision)
    return res
