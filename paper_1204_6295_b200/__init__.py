"""Python binding of the DISC C-ABI (`include/disc.h`): argument marshalling only.

Every function has the name and argument order of its C counterpart and does nothing but check tensor
device / dtype / contiguity / size and pass `data_ptr()` and the current CUDA stream.  Every step of the path
runs in the CUDA kernels of `libdisc.so`; there is no CPU or PyTorch fallback -- if the library is missing the
import fails, and without a B200 `disc_create` raises.

PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdisc.so")

DISC_OK, DISC_ERR_INVALID_ARG, DISC_ERR_UNSUPPORTED, DISC_ERR_ALLOC, DISC_ERR_CUDA = range(5)
DISC_MAX_PATCH_RADIUS = 12
DISC_MAX_GAUSS_RADIUS = 12
DISC_EPS_VAR = 1e-6
DISC_EPS_DEN = 1e-3
DISC_FORCE_THIRION, DISC_FORCE_DOUBLE = 1, 2
DISC_NOALLOC_MAX_VOXELS = 1 << 20

EXPORTS = (
    "disc_create", "disc_create_ex", "disc_destroy", "disc_last_error", "disc_launch_count", "disc_set_force", "disc_set_stop", "disc_iterations_run", "disc_set_mask", "disc_mask_params", "disc_get_ab", "disc_set_diagnostics", "disc_get_diagnostics", "disc_warp", "disc_correct_intensity",
    "disc_demons_step", "disc_register", "disc_register_host", "disc_iterate", "disc_box_moments",
    "disc_force_update", "disc_smooth_field", "disc_downsample", "disc_upsample_field", "disc_profile_iteration",
    "disc_smooth_field_noalloc",
)

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_1204_6295_b200.build` "
        "(or `__graft_entry__.build()`); there is no fallback path")

_lib = ctypes.CDLL(LIB_PATH)
_vp, _i = ctypes.c_void_p, ctypes.c_int
_lib.disc_create.restype = _i
_lib.disc_create.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(_i), ctypes.POINTER(ctypes.c_float), _i,
                             ctypes.c_float, _i, _i]
_lib.disc_create_ex.restype = _i
_lib.disc_create_ex.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(_i), ctypes.POINTER(ctypes.c_float), ctypes.POINTER(_i),
                                ctypes.c_float, _i, _i, ctypes.POINTER(_i)]
_lib.disc_destroy.restype = None
_lib.disc_destroy.argtypes = [_vp]
_lib.disc_last_error.restype = ctypes.c_char_p
_lib.disc_last_error.argtypes = [_vp]
_lib.disc_launch_count.restype = ctypes.c_ulonglong
_lib.disc_launch_count.argtypes = [_vp]
_lib.disc_set_force.restype = _i
_lib.disc_set_force.argtypes = [_vp, _i]
_lib.disc_set_stop.restype = _i
_lib.disc_set_stop.argtypes = [_vp, ctypes.c_float]
_lib.disc_iterations_run.restype = _i
_lib.disc_iterations_run.argtypes = [_vp, ctypes.POINTER(_i)]
_lib.disc_set_mask.restype = _i
_lib.disc_set_mask.argtypes = [_vp, _i, ctypes.c_float, ctypes.c_float, ctypes.c_float, _i, ctypes.c_float, _i]
_lib.disc_mask_params.restype = _i
_lib.disc_mask_params.argtypes = [_vp, _vp, _vp, ctypes.POINTER(ctypes.c_float), _vp]
_lib.disc_get_ab.restype = _i
_lib.disc_get_ab.argtypes = [_vp, _i, _vp, _vp, _vp, _vp]
_lib.disc_set_diagnostics.restype = _i
_lib.disc_set_diagnostics.argtypes = [_vp, _i]
_lib.disc_get_diagnostics.restype = _i
_lib.disc_get_diagnostics.argtypes = [_vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
for _name, _nptr in (("disc_warp", 3), ("disc_correct_intensity", 3), ("disc_demons_step", 3),
                     ("disc_box_moments", 3), ("disc_force_update", 3), ("disc_smooth_field", 1),
                     ("disc_downsample", 2), ("disc_upsample_field", 2)):
    _f = getattr(_lib, _name)
    _f.restype = _i
    _f.argtypes = [_vp, _i] + [_vp] * _nptr + [_vp]
_lib.disc_register.restype = _i
_lib.disc_register.argtypes = [_vp] * 6
_lib.disc_register_host.restype = _i
_lib.disc_register_host.argtypes = [_vp] * 6
_lib.disc_iterate.restype = _i
_lib.disc_iterate.argtypes = [_vp, _i, _vp, _vp, _vp, _i, _vp]
_lib.disc_profile_iteration.restype = _i
_lib.disc_profile_iteration.argtypes = [_vp, _i, _vp, _vp, _vp, _i, ctypes.POINTER(ctypes.c_float), _vp]
_lib.disc_smooth_field_noalloc.restype = _i
_lib.disc_smooth_field_noalloc.argtypes = [ctypes.POINTER(_i), ctypes.c_float, _vp, _vp]


class DiscError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"disc status {status}: {message}")
        self.status = status


def _check(ctx, status):
    if status != DISC_OK:
        msg = _lib.disc_last_error(ctx)
        raise DiscError(status, msg.decode() if msg else "")


def _dev(t, numel=None):
    """device pointer of a CUDA float32 contiguous tensor (None -> NULL)"""
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 CUDA tensor")
    if numel is not None and t.numel() != int(numel):
        raise ValueError(f"tensor has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def _x3(n):
    return None if n is None else 3 * n


def _host(a, numel=None):
    """host pointer of a float32 C-contiguous numpy array or CPU tensor with `numel` elements (None -> NULL)"""
    if a is None:
        return None
    if hasattr(a, "data_ptr"):
        import torch
        if a.is_cuda or not a.is_contiguous() or a.dtype != torch.float32:
            raise TypeError("expected a contiguous float32 CPU tensor")
        n, ptr = a.numel(), a.data_ptr()
    else:
        import numpy as np
        if a.dtype != np.float32 or not a.flags["C_CONTIGUOUS"]:
            raise TypeError("expected a C-contiguous float32 numpy array")
        n, ptr = a.size, a.ctypes.data
    if numel is not None and n != int(numel):
        raise ValueError(f"host buffer has {n} elements, expected {numel}")
    return ptr


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


class Ctx:
    """Opaque handle returned by disc_create (keeps the level sizes for argument checks)."""

    def __init__(self, handle, dims, levels, pyramid_factor=(2, 2, 2), iters=0):
        self.handle = handle
        self.iters = int(iters)
        self.dims = tuple(dims)
        self.levels = levels
        self.pyramid_factor = tuple(pyramid_factor)

    def level_dims(self, level):
        """(nx, ny, nz) at `level`"""
        return tuple(d // f ** level for d, f in zip(self.dims, self.pyramid_factor))

    def n(self, level):
        """voxels at `level`; None for a level the context does not have (the C layer reports that)"""
        if not 0 <= level < self.levels:
            return None
        nx, ny, nz = self.level_dims(level)
        return nx * ny * nz

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:     # at interpreter shutdown the module globals may already be gone
            _lib.disc_destroy(h)


def disc_create(dims, spacing, patch_radius, sigma_smooth, levels, iters) -> Ctx:
    out = _vp()
    d = (_i * 3)(*[int(v) for v in dims])
    s = (ctypes.c_float * 3)(*[float(v) for v in spacing])
    st = _lib.disc_create(ctypes.byref(out), d, s, int(patch_radius), float(sigma_smooth), int(levels), int(iters))
    _check(None, st)
    return Ctx(out.value, dims, levels, iters=iters)


def disc_create_ex(dims, spacing, patch_radius, sigma_smooth, levels, iters, pyramid_factor=(2, 2, 2)) -> Ctx:
    """patch_radius = (Rx, Ry, Rz), pyramid_factor = (fx, fy, fz) with each factor 1 or 2"""
    out = _vp()
    d = (_i * 3)(*[int(v) for v in dims])
    s = (ctypes.c_float * 3)(*[float(v) for v in spacing])
    r = (_i * 3)(*[int(v) for v in patch_radius])
    f = (_i * 3)(*[int(v) for v in pyramid_factor])
    st = _lib.disc_create_ex(ctypes.byref(out), d, s, r, float(sigma_smooth), int(levels), int(iters), f)
    _check(None, st)
    return Ctx(out.value, dims, levels, pyramid_factor, iters)


def disc_destroy(ctx: Ctx) -> None:
    h, ctx.handle = ctx.handle, None
    if h:
        _lib.disc_destroy(h)


def disc_last_error(ctx: Ctx | None) -> str:
    msg = _lib.disc_last_error(ctx.handle if ctx else None)
    return msg.decode() if msg else ""


def disc_launch_count(ctx: Ctx) -> int:
    return int(_lib.disc_launch_count(ctx.handle))


def disc_set_force(ctx, mode):
    _check(ctx.handle, _lib.disc_set_force(ctx.handle, int(mode)))


def disc_set_stop(ctx, eps):
    _check(ctx.handle, _lib.disc_set_stop(ctx.handle, float(eps)))


def disc_set_mask(ctx, enable, hu0=-1.0, a_min=-1.0, a_max=-1.0, fill_radius=1, h=50.0, max_fill_passes=64):
    _check(ctx.handle, _lib.disc_set_mask(ctx.handle, int(bool(enable)), float(hu0), float(a_min), float(a_max),
                                          int(fill_radius), float(h), int(max_fill_passes)))


def disc_mask_params(ctx, ct, cbct, stream=None):
    """(Delta HU, HU_0, a_m, a_min, a_max) from the full-resolution images; synchronises"""
    n = ctx.n(0)
    out = (ctypes.c_float * 5)()
    _check(ctx.handle, _lib.disc_mask_params(ctx.handle, _dev(ct, n), _dev(cbct, n), out, _stream(stream)))
    return [float(v) for v in out]


def disc_get_ab(ctx, level, out_a, out_b, out_xi, stream=None):
    n = ctx.n(level)
    xi_ptr = None
    if out_xi is not None:
        import torch
        if not (out_xi.is_cuda and out_xi.dtype == torch.uint8 and out_xi.is_contiguous() and out_xi.numel() == n):
            raise TypeError("out_xi: expected a contiguous uint8 CUDA tensor of the level's size")
        xi_ptr = out_xi.data_ptr()
    _check(ctx.handle, _lib.disc_get_ab(ctx.handle, level, _dev(out_a, n), _dev(out_b, n), xi_ptr, _stream(stream)))


def disc_set_diagnostics(ctx, enable):
    _check(ctx.handle, _lib.disc_set_diagnostics(ctx.handle, int(bool(enable))))


def disc_get_diagnostics(ctx):
    """(mean_a, mean_b), each a list of levels*iters floats, level-major from the coarsest level; synchronises"""
    n = ctx.levels * max(ctx.iters, 1)
    a, b = (ctypes.c_double * n)(), (ctypes.c_double * n)()
    _check(ctx.handle, _lib.disc_get_diagnostics(ctx.handle, a, b))
    return [float(v) for v in a], [float(v) for v in b]


def disc_iterations_run(ctx):
    """iterations run per level (index = level) by the last disc_register / disc_iterate; synchronises"""
    out = (_i * ctx.levels)()
    _check(ctx.handle, _lib.disc_iterations_run(ctx.handle, out))
    return [int(v) for v in out]


def disc_warp(ctx, level, moving, disp, out, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_warp(ctx.handle, level, _dev(moving, n), _dev(disp, _x3(n)), _dev(out, n), _stream(stream)))


def disc_correct_intensity(ctx, level, cbct, ct_warped, out_corrected, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_correct_intensity(ctx.handle, level, _dev(cbct, n), _dev(ct_warped, n),
                                                   _dev(out_corrected, n), _stream(stream)))


def disc_demons_step(ctx, level, m_warped, s_corrected, disp_inout, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_demons_step(ctx.handle, level, _dev(m_warped, n), _dev(s_corrected, n),
                                             _dev(disp_inout, _x3(n)), _stream(stream)))


def disc_register(ctx, ct, cbct, out_disp, out_corrected_cbct, stream=None):
    n = ctx.n(0)
    _check(ctx.handle, _lib.disc_register(ctx.handle, _dev(ct, n), _dev(cbct, n), _dev(out_disp, _x3(n)),
                                          _dev(out_corrected_cbct, n), _stream(stream)))


def disc_register_host(ctx, ct_host, cbct_host, out_disp_host, out_corrected_cbct_host, stream=None):
    n = ctx.n(0)
    _check(ctx.handle, _lib.disc_register_host(ctx.handle, _host(ct_host, n), _host(cbct_host, n), _host(out_disp_host, 3 * n),
                                               _host(out_corrected_cbct_host, n), _stream(stream)))


def disc_iterate(ctx, level, ct, cbct, disp_inout, n_iters, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_iterate(ctx.handle, level, _dev(ct, n), _dev(cbct, n), _dev(disp_inout, _x3(n)),
                                         int(n_iters), _stream(stream)))


def disc_profile_iteration(ctx, level, ct, cbct, disp_inout, n_iters, stream=None):
    """returns the three mean kernel durations in ms (host floats written by the C call)"""
    n = ctx.n(level)
    ms = (ctypes.c_float * 3)()
    _check(ctx.handle, _lib.disc_profile_iteration(ctx.handle, level, _dev(ct, n), _dev(cbct, n),
                                                   _dev(disp_inout, _x3(n)), int(n_iters), ms, _stream(stream)))
    return [float(v) for v in ms]


def disc_box_moments(ctx, level, vol, mean, var, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_box_moments(ctx.handle, level, _dev(vol, n), _dev(mean, n), _dev(var, n), _stream(stream)))


def disc_force_update(ctx, level, m, s, disp_inout, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_force_update(ctx.handle, level, _dev(m, n), _dev(s, n), _dev(disp_inout, _x3(n)),
                                              _stream(stream)))


def disc_smooth_field(ctx, level, disp_inout, stream=None):
    n = ctx.n(level)
    _check(ctx.handle, _lib.disc_smooth_field(ctx.handle, level, _dev(disp_inout, _x3(n)), _stream(stream)))


def disc_downsample(ctx, level_from, vol, out, stream=None):
    _check(ctx.handle, _lib.disc_downsample(ctx.handle, level_from, _dev(vol, ctx.n(level_from)),
                                            _dev(out, ctx.n(level_from + 1)), _stream(stream)))


def disc_upsample_field(ctx, level_from, disp, out, stream=None):
    _check(ctx.handle, _lib.disc_upsample_field(ctx.handle, level_from, _dev(disp, _x3(ctx.n(level_from))),
                                                _dev(out, _x3(ctx.n(level_from - 1))), _stream(stream)))


def disc_smooth_field_noalloc(dims, sigma_smooth, disp_inout, stream=None):
    """disc_smooth_field for callers that must not allocate device memory (an application that owns the GPU's memory
    pool, or a latency-bound loop that cannot afford the device-wide stall of cudaMalloc): no context, the buffer
    between the two kernels is a fixed 12 MiB array inside libdisc.so.  dims = (nx, ny, nz) with at most
    DISC_NOALLOC_MAX_VOXELS voxels (more raises DiscError); calls that may overlap on the GPU race on that array;
    make the first call on a device at start-up (it looks the array's address up).  See include/disc.h."""
    d = (_i * 3)(*[int(v) for v in dims])
    n = int(dims[0]) * int(dims[1]) * int(dims[2])
    _check(None, _lib.disc_smooth_field_noalloc(d, float(sigma_smooth), _dev(disp_inout, 3 * n), _stream(stream)))
