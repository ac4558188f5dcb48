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
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"])
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
