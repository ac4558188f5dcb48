"""CPU oracle for the DISC hot path -- TEST INFRASTRUCTURE, NOT PRODUCT.

numpy-in / numpy-out ctypes wrapper around `disc_oracle.c` (plain C, fp64
arithmetic inside each step, naive per-voxel patch loops).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It shares nothing with
`paper_1204_6295_b200/` and neither imports the other.

Arrays are C-order ``[nz, ny, nx]`` float32; fields are ``[3, nz, ny, nx]``.
Defaults of the two regularisers are the readings of DESIGN.md (A5, A7):
``EPS_VAR = 1e-6 HU^2`` and ``EPS_DEN = 1e-3 HU^2``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

EPS_VAR = 1e-6
EPS_DEN = 1e-3

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "disc_oracle.c")
_LIB = os.path.join(_HERE, "libdisc_oracle.so")
_lib = None

_f32p = ctypes.POINTER(ctypes.c_float)
_f64p = ctypes.POINTER(ctypes.c_double)
_i64p = ctypes.POINTER(ctypes.c_longlong)


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2 -fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu99", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_num_threads.restype = ctypes.c_int
        _lib.oracle_gauss_radius.restype = ctypes.c_int
        _lib.oracle_gauss_radius.argtypes = [ctypes.c_double]
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(_f32p)


def _dims(vol):
    nz, ny, nx = vol.shape[-3:]
    return ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def warp(moving, disp):
    """m(x) = I_m(x + r(x)), trilinear, clamped (reading A11)."""
    L = _load()
    I, pI = _f32(moving)
    d, pd = _f32(disp)
    out = np.empty_like(I)
    L.oracle_warp(pI, pd, *_dims(I), out.ctypes.data_as(_f32p))
    return out


def box_moments(vol, R):
    """(mean, var) over the truncated cube of radius R, fp64 (PAPER.md:95 Eq. 3, :458 A.4; reading A4)."""
    L = _load()
    v, pv = _f32(vol)
    mean = np.empty(v.shape, dtype=np.float64)
    var = np.empty(v.shape, dtype=np.float64)
    L.oracle_box_moments(pv, *_dims(v), ctypes.c_int(R), mean.ctypes.data_as(_f64p), var.ctypes.data_as(_f64p))
    return mean, var


def box_moments_at(vol, R, idx):
    L = _load()
    v, pv = _f32(vol)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    mean = np.empty(idx.shape, dtype=np.float64)
    var = np.empty(idx.shape, dtype=np.float64)
    L.oracle_box_moments_at(pv, *_dims(v), ctypes.c_int(R), idx.ctypes.data_as(_i64p), ctypes.c_int(idx.size),
                            mean.ctypes.data_as(_f64p), var.ctypes.data_as(_f64p))
    return mean, var


def correct(cbct, ct_warped, R, eps_var=EPS_VAR):
    """I'_s = a (I_s - mu_s) + mu_m, a = STD(M)/STD(S) (reading A5)."""
    L = _load()
    s, ps = _f32(cbct)
    m, pm = _f32(ct_warped)
    out = np.empty_like(s)
    L.oracle_correct(ps, pm, *_dims(s), ctypes.c_int(R), ctypes.c_double(eps_var), out.ctypes.data_as(_f32p))
    return out


def correct_from_moments(cbct, mu_s, var_s, mu_m, var_m, eps_var=EPS_VAR):
    """Eqs. (5)-(6) applied with given patch moments (the driver computes the CBCT's once per level)."""
    L = _load()
    s, ps = _f32(cbct)
    arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (mu_s, var_s, mu_m, var_m)]
    out = np.empty_like(s)
    L.oracle_correct_from_moments(ps, *[a.ctypes.data_as(_f64p) for a in arrs], ctypes.c_size_t(s.size),
                                  ctypes.c_double(eps_var), out.ctypes.data_as(_f32p))
    return out


def correct_at(cbct, ct_warped, R, idx, eps_var=EPS_VAR):
    L = _load()
    s, ps = _f32(cbct)
    m, pm = _f32(ct_warped)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    out = np.empty(idx.shape, dtype=np.float64)
    L.oracle_correct_at(ps, pm, *_dims(s), ctypes.c_int(R), ctypes.c_double(eps_var), idx.ctypes.data_as(_i64p),
                        ctypes.c_int(idx.size), out.ctypes.data_as(_f64p))
    return out


def force_update(m, s, disp, eps_den=EPS_DEN, double_force=False):
    """r += (s'-m) grad s' / (|grad s'|^2 + (s'-m)^2 + eps) (PAPER.md:73 Eq. 1 first term, :192-193; readings A1, A7, A8);
    with double_force also the second term of Eq. 1, + (s'-m) grad m / (|grad m|^2 + (s'-m)^2 + eps)."""
    L = _load()
    m_, pm = _f32(m)
    s_, ps = _f32(s)
    d = np.array(disp, dtype=np.float32, order="C", copy=True)
    fn = L.oracle_force_update_double if double_force else L.oracle_force_update
    fn(pm, ps, *_dims(m_), ctypes.c_double(eps_den), d.ctypes.data_as(_f32p))
    return d


def gauss_weights(sigma):
    L = _load()
    K = int(L.oracle_gauss_radius(ctypes.c_double(sigma)))
    w = np.empty(2 * K + 1, dtype=np.float32)
    L.oracle_gauss_weights(ctypes.c_double(sigma), w.ctypes.data_as(_f32p))
    return w


def smooth_field(disp, sigma):
    """Separable Gaussian of the total field, replicate border (reading A10)."""
    L = _load()
    d = np.array(disp, dtype=np.float32, order="C", copy=True)
    L.oracle_smooth_field(d.ctypes.data_as(_f32p), *_dims(d), ctypes.c_double(sigma))
    return d


def downsample(vol):
    """2x2x2 block mean (reading A9)."""
    L = _load()
    v, pv = _f32(vol)
    nz, ny, nx = v.shape
    out = np.empty((nz // 2, ny // 2, nx // 2), dtype=np.float32)
    L.oracle_downsample(pv, *_dims(v), out.ctypes.data_as(_f32p))
    return out


def upsample_field(disp):
    """x2 trilinear up-sampling at i/2 - 1/4, values doubled (reading A9)."""
    L = _load()
    d, pd = _f32(disp)
    _, nz, ny, nx = d.shape
    out = np.empty((3, 2 * nz, 2 * ny, 2 * nx), dtype=np.float32)
    L.oracle_upsample_field(pd, ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz), out.ctypes.data_as(_f32p))
    return out


def demons_step(m, s, disp, sigma, eps_den=EPS_DEN, double_force=False):
    """Alg. A1 steps 4-6."""
    return smooth_field(force_update(m, s, disp, eps_den, double_force), sigma)


def register(ct, cbct, R, sigma, levels, iters, eps_var=EPS_VAR, eps_den=EPS_DEN, want_corr=True, want_trace=False,
             double_force=False):
    """Algorithm A1 with a fixed iteration count (readings A9, A12, A14)."""
    L = _load()
    a, pa = _f32(ct)
    b, pb = _f32(cbct)
    disp = np.empty((3,) + a.shape, dtype=np.float32)
    corr = np.empty_like(a) if want_corr else None
    trace = np.zeros(levels * iters, dtype=np.float64) if want_trace else None
    L.oracle_register_mode(pa, pb, *_dims(a), ctypes.c_int(R), ctypes.c_double(sigma), ctypes.c_int(levels),
                           ctypes.c_int(iters), ctypes.c_double(eps_var), ctypes.c_double(eps_den),
                           ctypes.c_int(1 if double_force else 0), disp.ctypes.data_as(_f32p), corr.ctypes.data_as(_f32p) if want_corr else None,
                      trace.ctypes.data_as(_f64p) if want_trace else None)
    out = (disp, corr)
    return out + (trace,) if want_trace else out


def force_norms(m, s, disp, eps_den=EPS_DEN, double_force=False):
    """(sum |dr|, sum |r|) of the paper's convergence measure l = sum|dr| / sum|r| (reading A16)."""
    L = _load()
    m_, pm = _f32(m)
    s_, ps = _f32(s)
    d, pd = _f32(disp)
    a, b = ctypes.c_double(0.0), ctypes.c_double(0.0)
    L.oracle_force_norms(pm, ps, pd, *_dims(m_), ctypes.c_double(eps_den), ctypes.c_int(1 if double_force else 0),
                         ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


def register_stop(ct, cbct, R, sigma, levels, iters, stop_eps=None, iters_per_level=None, double_force=False,
                  eps_var=EPS_VAR, eps_den=EPS_DEN):
    """Algorithm A1 with the paper's stopping criterion l(k-10) - l(k) <= stop_eps inside every level (PAPER.md:167,
    :187); `iters` is the per-level maximum.  Returns (disp, iterations run per level [0 = finest],
    l trace [levels, iters], coarsest level first, nan where not run)."""
    L = _load()
    a, pa = _f32(ct)
    b, pb = _f32(cbct)
    disp = np.empty((3,) + a.shape, dtype=np.float32)
    run = np.zeros(levels, dtype=np.int32)
    ltrace = np.full((levels, max(iters, 1)), np.nan, dtype=np.float64)
    ipl = None if iters_per_level is None else np.ascontiguousarray(iters_per_level, dtype=np.int32)
    if ipl is not None:
        assert ipl.size == levels and ipl.max() <= iters
    i32p = ctypes.POINTER(ctypes.c_int)
    L.oracle_register_full(pa, pb, *_dims(a), ctypes.c_int(R), ctypes.c_double(sigma), ctypes.c_int(levels),
                           ctypes.c_int(iters), ctypes.c_double(eps_var), ctypes.c_double(eps_den),
                           ctypes.c_int(1 if double_force else 0),
                           ctypes.c_double(-1.0 if stop_eps is None else float(stop_eps)),
                           ipl.ctypes.data_as(i32p) if ipl is not None else None, run.ctypes.data_as(i32p),
                           ltrace.ctypes.data_as(_f64p), disp.ctypes.data_as(_f32p), None, None)
    return disp, run, ltrace


# ------------------------------------------------------------------------------------------------
# SURVEY.md section 8(f) extensions: NEXT-4 (per-axis patch radius, per-axis pyramid factor), NEXT-1 (mask and
# interpolation of a, b), Fig.-9 diagnostics, summed-area moments.
# ------------------------------------------------------------------------------------------------
_i32p = ctypes.POINTER(ctypes.c_int)
_u8p = ctypes.POINTER(ctypes.c_ubyte)


def _r3(R):
    """patch radius as (Rx, Ry, Rz): an int means the cube of the hot path"""
    r = (R, R, R) if np.isscalar(R) else tuple(int(v) for v in R)
    assert len(r) == 3
    return (ctypes.c_int * 3)(*r)


def box_moments3(vol, R, sat=False):
    """(mean, var) over the truncated box of per-axis radius R = (Rx, Ry, Rz); sat=True uses the
    independently written fp64 summed-area routine."""
    L = _load()
    v, pv = _f32(vol)
    mean = np.empty(v.shape, dtype=np.float64)
    var = np.empty(v.shape, dtype=np.float64)
    if sat:
        L.oracle_box_moments_sat.restype = ctypes.c_int
        if L.oracle_box_moments_sat(pv, *_dims(v), _r3(R), mean.ctypes.data_as(_f64p), var.ctypes.data_as(_f64p)) != 0:
            raise ValueError("oracle_box_moments_sat: a value is not finite or |v| >= 2^14 HU (outside its fixed-point range)")
    else:
        L.oracle_box_moments3(pv, *_dims(v), _r3(R), mean.ctypes.data_as(_f64p), var.ctypes.data_as(_f64p))
    return mean, var


def correct3(cbct, ct_warped, R, eps_var=EPS_VAR):
    """correct() with a per-axis patch radius."""
    mus, vs = box_moments3(cbct, R)
    mum, vm = box_moments3(ct_warped, R)
    return correct_from_moments(cbct, mus, vs, mum, vm, eps_var)


def downsample3(vol, fac):
    """block mean over fac = (fx, fy, fz) voxels, each factor 1 or 2."""
    L = _load()
    v, pv = _f32(vol)
    nz, ny, nx = v.shape
    out = np.empty((nz // fac[2], ny // fac[1], nx // fac[0]), dtype=np.float32)
    L.oracle_downsample3(pv, *_dims(v), (ctypes.c_int * 3)(*fac), out.ctypes.data_as(_f32p))
    return out


def upsample_field3(disp, fac):
    """field up-sampling with a per-axis factor (reading A9)."""
    L = _load()
    d, pd = _f32(disp)
    _, nz, ny, nx = d.shape
    out = np.empty((3, fac[2] * nz, fac[1] * ny, fac[0] * nx), dtype=np.float32)
    L.oracle_upsample_field3(pd, ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz), (ctypes.c_int * 3)(*fac),
                             out.ctypes.data_as(_f32p))
    return out


def ab_from_moments(mu_s, var_s, mu_m, var_m, eps_var=EPS_VAR):
    """Eqs. (5), (6): a = STD(M)/STD(S), b = E(M) - a E(S)."""
    L = _load()
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (mu_s, var_s, mu_m, var_m)]
    a = np.empty(arrs[0].shape, dtype=np.float64)
    b = np.empty(arrs[0].shape, dtype=np.float64)
    L.oracle_ab_from_moments(*[x.ctypes.data_as(_f64p) for x in arrs], ctypes.c_size_t(a.size), ctypes.c_double(eps_var),
                             a.ctypes.data_as(_f64p), b.ctypes.data_as(_f64p))
    return a, b


def mask(m, cbct, a, hu0, a_min, a_max):
    """Eq. (7): xi = 1 where |I_m - I_s| > HU_0 or a outside [a_min, a_max]."""
    L = _load()
    m_, pm = _f32(m)
    s_, ps = _f32(cbct)
    a_ = np.ascontiguousarray(a, dtype=np.float64)
    xi = np.empty(m_.shape, dtype=np.uint8)
    L.oracle_mask(pm, ps, a_.ctypes.data_as(_f64p), ctypes.c_size_t(m_.size), ctypes.c_double(hu0), ctypes.c_double(a_min),
                  ctypes.c_double(a_max), xi.ctypes.data_as(_u8p))
    return xi


def fill_ab(cbct, xi, a, b, fill_radius, h, max_passes=64):
    """Eqs. (8)-(10): interpolate / extrapolate a, b into the xi = 1 voxels.  Returns
    (a, b, xi_left, passes)."""
    L = _load()
    s_, ps = _f32(cbct)
    x = np.array(xi, dtype=np.uint8, order="C", copy=True)
    a_ = np.array(a, dtype=np.float64, order="C", copy=True)
    b_ = np.array(b, dtype=np.float64, order="C", copy=True)
    L.oracle_fill_ab.restype = ctypes.c_int
    n = L.oracle_fill_ab(ps, *_dims(s_), x.ctypes.data_as(_u8p), a_.ctypes.data_as(_f64p), b_.ctypes.data_as(_f64p),
                         ctypes.c_int(fill_radius), ctypes.c_double(h), ctypes.c_int(max_passes))
    return a_, b_, x, int(n)


def apply_ab(cbct, a, b):
    """I'_s = a I_s + b."""
    L = _load()
    s_, ps = _f32(cbct)
    a_ = np.ascontiguousarray(a, dtype=np.float64)
    b_ = np.ascontiguousarray(b, dtype=np.float64)
    out = np.empty_like(s_)
    L.oracle_apply_ab(ps, a_.ctypes.data_as(_f64p), b_.ctypes.data_as(_f64p), ctypes.c_size_t(s_.size),
                      out.ctypes.data_as(_f32p))
    return out


def delta_hu(ct, cbct):
    """Delta HU = mean(CT) - mean(CBCT)."""
    L = _load()
    a, pa = _f32(ct)
    b, pb = _f32(cbct)
    L.oracle_delta_hu.restype = ctypes.c_double
    return float(L.oracle_delta_hu(pa, pb, ctypes.c_size_t(a.size)))


def median_a(a, var_s, var_m, eps_var=EPS_VAR):
    """a_m = median(A) before the DIR (reading A17)."""
    L = _load()
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (a, var_s, var_m)]
    L.oracle_median_a.restype = ctypes.c_double
    return float(L.oracle_median_a(*[x.ctypes.data_as(_f64p) for x in arrs], ctypes.c_size_t(arrs[0].size),
                                   ctypes.c_double(eps_var)))


class _Params(ctypes.Structure):
    _fields_ = [("R", ctypes.c_int * 3), ("fac", ctypes.c_int * 3), ("sigma", ctypes.c_double),
                ("levels", ctypes.c_int), ("iters", ctypes.c_int), ("eps_var", ctypes.c_double),
                ("eps_den", ctypes.c_double), ("double_force", ctypes.c_int), ("stop_eps", ctypes.c_double),
                ("moments_policy", ctypes.c_int), ("mask", ctypes.c_int), ("hu0", ctypes.c_double),
                ("a_min", ctypes.c_double), ("a_max", ctypes.c_double), ("fill_radius", ctypes.c_int),
                ("h", ctypes.c_double), ("max_fill_passes", ctypes.c_int)]


class _Info(ctypes.Structure):
    _fields_ = [("delta_hu", ctypes.c_double), ("hu0", ctypes.c_double), ("a_m", ctypes.c_double),
                ("a_min", ctypes.c_double), ("a_max", ctypes.c_double)]


def register_ex(ct, cbct, R, sigma, levels, iters, fac=(2, 2, 2), double_force=False, stop_eps=None, sat_between=False,
                mask=False, hu0=None, a_range=None, fill_radius=1, h=50.0, max_fill_passes=64, want_corr=True,
                eps_var=EPS_VAR, eps_den=EPS_DEN):
    """Algorithm A1 with every option of the oracle: per-axis patch radius R and pyramid factor
    `fac` (NEXT-4), double force (NEXT-2), stopping criterion (NEXT-3), mask + interpolation of a, b with the global
    Delta-HU shift (NEXT-1), and `sat_between` = summed-area moments in all but the first and last iteration of a
    level (config 4's whole-schedule check).  Returns a dict: disp, corr, iters_run [levels, 0 = finest], l, mean_a,
    mean_b [levels, iters] (coarsest level first, nan where not run), info."""
    L = _load()
    a, pa = _f32(ct)
    b, pb = _f32(cbct)
    prm = _Params()
    prm.R = _r3(R)
    prm.fac = (ctypes.c_int * 3)(*fac)
    prm.sigma, prm.levels, prm.iters = float(sigma), int(levels), int(iters)
    prm.eps_var, prm.eps_den = float(eps_var), float(eps_den)
    prm.double_force = 1 if double_force else 0
    prm.stop_eps = -1.0 if stop_eps is None else float(stop_eps)
    prm.moments_policy = 1 if sat_between else 0
    prm.mask = 1 if mask else 0
    prm.hu0 = -1.0 if hu0 is None else float(hu0)
    prm.a_min, prm.a_max = (-1.0, -1.0) if a_range is None else (float(a_range[0]), float(a_range[1]))
    prm.fill_radius, prm.h, prm.max_fill_passes = int(fill_radius), float(h), int(max_fill_passes)
    disp = np.empty((3,) + a.shape, dtype=np.float32)
    corr = np.empty_like(a) if want_corr else None
    run = np.zeros(levels, dtype=np.int32)
    shape = (levels, max(iters, 1))
    ltrace, mean_a, mean_b = (np.full(shape, np.nan, dtype=np.float64) for _ in range(3))
    info = _Info()
    L.oracle_register_ex(pa, pb, *_dims(a), ctypes.byref(prm), disp.ctypes.data_as(_f32p),
                         corr.ctypes.data_as(_f32p) if want_corr else None, run.ctypes.data_as(_i32p),
                         ltrace.ctypes.data_as(_f64p), mean_a.ctypes.data_as(_f64p), mean_b.ctypes.data_as(_f64p),
                         ctypes.byref(info))
    return {"disp": disp, "corr": corr, "iters_run": run, "l": ltrace, "mean_a": mean_a, "mean_b": mean_b,
            "info": {k: getattr(info, k) for k, _ in _Info._fields_}}
