"""Thin ctypes binding of ``include/pyhst.h`` -- argument marshalling only.

Every step of the hot path runs in the CUDA library (``csrc/`` -> ``libpyhst_b200.so``).
PyTorch is used for device memory and streams only.  There is no CPU fallback: if the
library cannot be loaded, or a call fails, ``PyhstError`` is raised.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_double, c_float, c_int, c_int32, c_int64, c_void_p

import numpy as np

FILTER_RAMLAK = 0
FILTER_SHEPP_LOGAN = 1
FILTER_HANN = 2
FILTER_HAMMING = 3
FILTER_COSINE = 4
SCAN_180 = 0
SCAN_360 = 1
SCAN_360_HALF = 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBNAME = "libpyhst_b200.so"

# every symbol include/*.h declares
EXPORTS = ("pyhst_ramp_filter", "pyhst_backproject", "pyhst_forward_project", "pyhst_fbp",
           "pyhst_fista_tv", "pyhst_ista_tv", "pyhst_ring_filter", "pyhst_ring_filter_static", "pyhst_ecohe", "pyhst_cv_distance", "pyhst_patch_grid",
           "pyhst_patch_gradient", "pyhst_patch_fista", "pyhst_fbp_host", "pyhst_backproject_host", "pyhst_forward_project_host", "pyhst_halfacq_extent", "pyhst_profile_enable", "pyhst_profile_read", "pyhst_set_backproject_variant", "pyhst_set_forward_project_variant", "pyhst_last_forward_project_kernel", "pyhst_test_fd_plan", "pyhst_set_halfacq_stitch", "pyhst_set_filter_variant", "pyhst_set_patch_gemm_variant", "pyhst_test_set_workspace_limit",
           "pyhst_last_error", "pyhst_release_cache")


class PyhstError(RuntimeError):
    pass


class Geom(ctypes.Structure):
    _fields_ = [("n_slices", c_int32), ("n_angles", c_int32), ("n_bins", c_int32),
                ("sino_pitch", c_int64), ("angles_rad", POINTER(c_double)),
                ("axis_pos", POINTER(c_double)), ("nx", c_int32), ("ny", c_int32),
                ("pixel_size", c_double)]


_lib = None


def library_path() -> str:
    return os.path.join(_HERE, _LIBNAME)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise PyhstError("%s is not built (run `python -c 'import __graft_entry__ as g; g.build()'`); "
                         "there is no CPU fallback" % path)
    lib = ctypes.CDLL(path)
    lib.pyhst_ramp_filter.argtypes = [c_void_p, c_void_p, c_int64, c_int32, c_int32, c_int32, c_int64,
                                      c_int, c_void_p, c_void_p]
    lib.pyhst_backproject.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_float, c_void_p]
    lib.pyhst_forward_project.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_float, c_void_p]
    lib.pyhst_fbp.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_int, c_int, c_void_p]
    lib.pyhst_fbp_host.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_int, c_int, c_int32, c_void_p]
    lib.pyhst_backproject_host.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_float, c_int32, c_void_p]
    lib.pyhst_forward_project_host.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_float, c_int32, c_void_p]
    lib.pyhst_fista_tv.argtypes = [c_void_p, c_void_p, POINTER(Geom), c_float, c_int32, c_int32, c_int32,
                                   POINTER(c_double), POINTER(c_double), c_void_p]
    lib.pyhst_ista_tv.argtypes = lib.pyhst_fista_tv.argtypes
    lib.pyhst_ring_filter.argtypes = [c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int64, c_int32,
                                      c_void_p]
    lib.pyhst_ring_filter_static.argtypes = lib.pyhst_ring_filter.argtypes
    lib.pyhst_ecohe.argtypes = [c_void_p, c_void_p, c_int32, c_int64, POINTER(c_double), c_void_p]
    lib.pyhst_cv_distance.argtypes = [c_void_p, c_void_p, POINTER(Geom), POINTER(c_double), c_void_p]
    lib.pyhst_patch_grid.argtypes = [c_int32, c_int32, c_int32, c_int32, POINTER(c_int32), POINTER(c_int32)]
    lib.pyhst_patch_gradient.argtypes = [c_void_p, c_void_p, c_void_p, POINTER(Geom), POINTER(Patch), c_void_p,
                                         c_void_p, POINTER(c_double), c_void_p]
    lib.pyhst_patch_fista.argtypes = [c_void_p, c_void_p, POINTER(Geom), POINTER(Patch), c_float, c_int32, c_int32,
                                      c_void_p, c_void_p, POINTER(c_double), POINTER(c_double), c_void_p]
    lib.pyhst_halfacq_extent.argtypes = [c_int32, c_double, POINTER(c_int32), POINTER(c_int32)]
    lib.pyhst_set_backproject_variant.argtypes = [c_int]
    lib.pyhst_set_forward_project_variant.argtypes = [c_int]
    lib.pyhst_set_halfacq_stitch.argtypes = [c_int]
    lib.pyhst_set_filter_variant.argtypes = [c_int]
    lib.pyhst_test_set_workspace_limit.argtypes = [c_int64]
    lib.pyhst_test_set_workspace_limit.restype = c_int64
    lib.pyhst_set_patch_gemm_variant.argtypes = [c_int]
    lib.pyhst_profile_enable.argtypes = [c_int]
    lib.pyhst_profile_read.argtypes = [POINTER(c_double), POINTER(c_int64), POINTER(c_int64), c_int32]
    lib.pyhst_last_error.restype = c_char_p
    lib.pyhst_release_cache.restype = None
    _lib = lib
    return lib


def last_error() -> str:
    return _load().pyhst_last_error().decode()


def _check(rc, what):
    if rc != 0:
        raise PyhstError("%s failed (status %d): %s" % (what, rc, last_error()))


def _stream(stream):
    if stream is None:
        import torch
        return c_void_p(torch.cuda.current_stream().cuda_stream)
    return c_void_p(int(getattr(stream, "cuda_stream", stream)))


def _dev(t, name):
    """Device pointer of a contiguous float32 CUDA tensor."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise PyhstError("%s must be a contiguous float32 CUDA tensor" % name)
    return c_void_p(t.data_ptr())


def _dev_sino(t, name):
    """(device pointer, sino_pitch) of a float32 CUDA sinogram stack [S, P, B]: contiguous, or rows pitched
    (stride(2) == 1, stride(1) = pitch >= B, stride(0) == P * pitch -- e.g. a [:, :, :B] view of a wider stack)."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.dim() == 3):
        raise PyhstError("%s must be a float32 CUDA tensor [S, P, B]" % name)
    if t.is_contiguous():
        return c_void_p(t.data_ptr()), 0
    s, p, b = t.shape
    st = t.stride()
    if st[2] == 1 and st[1] >= b and (s == 1 or st[0] == p * st[1]):
        return c_void_p(t.data_ptr()), int(st[1])
    raise PyhstError("%s must be contiguous or have pitched rows" % name)


def _geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, pixel_size, sino_pitch=0):
    angles = np.ascontiguousarray(angles, dtype=np.float64)
    axis = np.ascontiguousarray(axis, dtype=np.float64)
    if angles.shape != (n_angles,) or axis.shape != (n_angles,):
        raise PyhstError("angles and axis must both have shape [n_angles]")
    g = Geom(n_slices, n_angles, n_bins, sino_pitch, angles.ctypes.data_as(POINTER(c_double)),
             axis.ctypes.data_as(POINTER(c_double)), nx, ny, float(pixel_size))
    g._keep = (angles, axis)
    return g


def ramp_filter(d_in, n_bins_out=None, pad_left=0, filter=FILTER_RAMLAK, col_weights=None, out=None,
                stream=None):
    """pyhst_ramp_filter: float32 CUDA [..., n_bins_in] -> [..., n_bins_out] (contiguous)."""
    import torch
    lib = _load()
    b_in = d_in.shape[-1]
    b_out = b_in if n_bins_out is None else int(n_bins_out)
    n_rows = d_in.numel() // b_in if b_in else 0
    if out is None:
        out = torch.empty(d_in.shape[:-1] + (b_out,), dtype=torch.float32, device=d_in.device)
    w = None if col_weights is None else _dev(col_weights, "col_weights")
    _check(lib.pyhst_ramp_filter(_dev(d_in, "d_in"), _dev(out, "out"), n_rows, b_in, b_out, pad_left,
                                 out.shape[-1], filter, w, _stream(stream)), "pyhst_ramp_filter")
    return out


def backproject(d_sino, angles, axis, nx, ny, pixel_size=1.0, scale=1.0, out=None, stream=None):
    """pyhst_backproject: float32 CUDA [S,P,B] -> [S,ny,nx]."""
    import torch
    lib = _load()
    s, p, b = d_sino.shape
    if out is None:
        out = torch.empty((s, ny, nx), dtype=torch.float32, device=d_sino.device)
    ptr, pitch = _dev_sino(d_sino, "d_sino")
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size, pitch)
    _check(lib.pyhst_backproject(ptr, _dev(out, "out"), ctypes.byref(g), scale,
                                 _stream(stream)), "pyhst_backproject")
    return out


def forward_project(d_img, angles, axis, n_bins, pixel_size=1.0, scale=1.0, out=None, stream=None):
    """pyhst_forward_project: float32 CUDA [S,ny,nx] -> [S,P,B]."""
    import torch
    lib = _load()
    s, ny, nx = d_img.shape
    p = len(angles)
    if out is None:
        out = torch.empty((s, p, n_bins), dtype=torch.float32, device=d_img.device)
    ptr, pitch = _dev_sino(out, "out")
    g = _geom(s, p, n_bins, angles, axis, nx, ny, pixel_size, pitch)
    _check(lib.pyhst_forward_project(_dev(d_img, "d_img"), ptr, ctypes.byref(g), scale,
                                     _stream(stream)), "pyhst_forward_project")
    return out


def fbp(d_sino_raw, angles, axis, nx, ny, pixel_size=1.0, filter=FILTER_RAMLAK, mode=SCAN_180, out=None,
        stream=None):
    """pyhst_fbp: float32 CUDA [S,P,B] -> [S,ny,nx]."""
    import torch
    lib = _load()
    s, p, b = d_sino_raw.shape
    if out is None:
        out = torch.empty((s, ny, nx), dtype=torch.float32, device=d_sino_raw.device)
    ptr, pitch = _dev_sino(d_sino_raw, "d_sino_raw")
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size, pitch)
    _check(lib.pyhst_fbp(ptr, _dev(out, "out"), ctypes.byref(g), filter, mode,
                         _stream(stream)), "pyhst_fbp")
    return out


def fista_tv(d_data, angles, axis, nx, ny, beta, n_iter, n_inner=20, n_power=8, pixel_size=1.0, out=None,
             want_energy=True, stream=None, accelerated=True):
    """pyhst_fista_tv (accelerated=False: pyhst_ista_tv): float32 CUDA data [S,P,B] ->
    (x [S,ny,nx] CUDA, energy float64 [n_iter], L).
    With want_energy=False nothing is copied back and the call does not synchronise."""
    import torch
    lib = _load()
    fn = lib.pyhst_fista_tv if accelerated else lib.pyhst_ista_tv
    s, p, b = d_data.shape
    if out is None:
        out = torch.empty((s, ny, nx), dtype=torch.float32, device=d_data.device)
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size)
    energy = np.zeros(max(int(n_iter), 1), dtype=np.float64)
    lip = c_double(0.0)
    _check(fn(_dev(d_data, "d_data"), _dev(out, "out"), ctypes.byref(g), float(beta),
              int(n_iter), int(n_inner), int(n_power),
              energy.ctypes.data_as(POINTER(c_double)) if want_energy else None,
              ctypes.byref(lip) if want_energy else None, _stream(stream)),
           "pyhst_fista_tv" if accelerated else "pyhst_ista_tv")
    return out, energy[:int(n_iter)], float(lip.value)


def ista_tv(*args, **kwargs):
    """pyhst_ista_tv: fista_tv without the momentum."""
    return fista_tv(*args, accelerated=False, **kwargs)


def ring_filter(d_sino, half_width, model=None, out=None, stream=None):
    """pyhst_ring_filter: float32 CUDA [S,P,B] (+ optional model of the same shape) -> [S,P,B]."""
    import torch
    lib = _load()
    s, p, b = d_sino.shape
    if out is None:
        out = torch.empty_like(d_sino)
    _check(lib.pyhst_ring_filter(_dev(d_sino, "d_sino"), None if model is None else _dev(model, "model"),
                                 _dev(out, "out"), s, p, b, c_int64(b), int(half_width), _stream(stream)),
           "pyhst_ring_filter")
    return out


RING_STATIC_MAX_CELLS = 32768   # PYHST_RING_STATIC_MAX_CELLS of include/pyhst.h


def ring_filter_static(d_sino, half_width, model=None, out=None, stream=None):
    """pyhst_ring_filter_static: ``ring_filter`` for programs in which the library may not allocate.

    ``ring_filter`` parks its column sums in a workspace the library grows with cudaMalloc on the first
    call of a shape.  Some programs cannot have that: they have given all device memory to their own
    pools, cannot afford the device-wide stall of cudaMalloc / cudaFree inside an acquisition loop, or
    have to go on after an out-of-memory condition.  This variant keeps the same intermediates in a fixed
    8.5 MB array inside the library, allocates nothing, and returns bit-identical output.

    Limit: ``S * B <= RING_STATIC_MAX_CELLS`` (32768), otherwise ``PyhstError`` -- split the stack by
    slices.  Pass ``out`` if this wrapper must not allocate either (without it the result tensor comes
    from torch's allocator).  All calls on a device share the one array: keep them ordered on one stream
    (or by events); calls that overlap on the GPU corrupt each other.  The first call on a device looks
    the array's address up -- make it during set-up, before any stream capture.
    """
    import torch
    lib = _load()
    s, p, b = d_sino.shape
    if out is None:
        out = torch.empty_like(d_sino)
    _check(lib.pyhst_ring_filter_static(_dev(d_sino, "d_sino"), None if model is None else _dev(model, "model"),
                                        _dev(out, "out"), s, p, b, c_int64(b), int(half_width), _stream(stream)),
           "pyhst_ring_filter_static")
    return out


def ecohe(d_img_beta, d_img_0, stream=None):
    """pyhst_ecohe: eq. 11 per slice of two float32 CUDA stacks [S, ...] -> float64 [S] (host)."""
    lib = _load()
    s = d_img_beta.shape[0]
    if tuple(d_img_beta.shape) != tuple(d_img_0.shape):
        raise PyhstError("stacks must have the same shape")
    out = np.zeros(s, dtype=np.float64)
    _check(lib.pyhst_ecohe(_dev(d_img_beta, "d_img_beta"), _dev(d_img_0, "d_img_0"), s,
                           c_int64(d_img_beta[0].numel()), out.ctypes.data_as(POINTER(c_double)), _stream(stream)),
           "pyhst_ecohe")
    return out


def cv_distance(d_img, d_data_excl, angles_excl, axis_excl, pixel_size=1.0, stream=None):
    """pyhst_cv_distance: sum over the excluded projections of ||P x - data||^2 per slice -> float64 [S]."""
    lib = _load()
    s, ny, nx = d_img.shape
    s2, e, b = d_data_excl.shape
    if s2 != s:
        raise PyhstError("d_img and d_data_excl must have the same number of slices")
    g = _geom(s, e, b, angles_excl, axis_excl, nx, ny, pixel_size)
    out = np.zeros(s, dtype=np.float64)
    _check(lib.pyhst_cv_distance(_dev(d_img, "d_img"), _dev(d_data_excl, "d_data_excl"), ctypes.byref(g),
                                 out.ctypes.data_as(POINTER(c_double)), _stream(stream)), "pyhst_cv_distance")
    return out


class Patch(ctypes.Structure):
    _fields_ = [("m", c_int32), ("stride", c_int32), ("n_atoms", c_int32), ("rho", c_float)]


def patch_grid(ny, nx, m, stride):
    na, nb = c_int32(0), c_int32(0)
    _check(_load().pyhst_patch_grid(ny, nx, m, stride, ctypes.byref(na), ctypes.byref(nb)), "pyhst_patch_grid")
    return int(na.value), int(nb.value)


def patch_gradient(d_W, d_D, d_data, angles, axis, nx, ny, m, stride, rho, pixel_size=1.0, want_f=True,
                   stream=None):
    """pyhst_patch_gradient (Algorithm 1): W [S,N,Nc], D [Nc,m*m], data [S,P,B] (float32 CUDA) ->
    (G [S,N,Nc], X [S,ny,nx], f)."""
    import torch
    lib = _load()
    s, p, b = d_data.shape
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size)
    pp = Patch(int(m), int(stride), int(d_D.shape[0]), float(rho))
    G = torch.empty_like(d_W)
    X = torch.empty((s, ny, nx), dtype=torch.float32, device=d_W.device)
    f = c_double(0.0)
    _check(lib.pyhst_patch_gradient(_dev(d_W, "d_W"), _dev(d_D, "d_D"), _dev(d_data, "d_data"), ctypes.byref(g),
                                    ctypes.byref(pp), _dev(G, "G"), _dev(X, "X"),
                                    ctypes.byref(f) if want_f else None, _stream(stream)), "pyhst_patch_gradient")
    return G, X, float(f.value)


def patch_fista(d_D, d_data, angles, axis, nx, ny, m, stride, rho, beta, n_iter, n_power=8, pixel_size=1.0,
                want_energy=True, stream=None):
    """pyhst_patch_fista -> (W [S,N,Nc] CUDA, X [S,ny,nx] CUDA, energy float64 [n_iter], Lw)."""
    import torch
    lib = _load()
    s, p, b = d_data.shape
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size)
    pp = Patch(int(m), int(stride), int(d_D.shape[0]), float(rho))
    na, nb = patch_grid(ny, nx, m, stride)
    W = torch.empty((s, na * nb, d_D.shape[0]), dtype=torch.float32, device=d_data.device)
    X = torch.empty((s, ny, nx), dtype=torch.float32, device=d_data.device)
    energy = np.zeros(max(int(n_iter), 1), dtype=np.float64)
    lip = c_double(0.0)
    _check(lib.pyhst_patch_fista(_dev(d_D, "d_D"), _dev(d_data, "d_data"), ctypes.byref(g), ctypes.byref(pp),
                                 float(beta), int(n_iter), int(n_power), _dev(W, "W"), _dev(X, "X"),
                                 energy.ctypes.data_as(POINTER(c_double)) if want_energy else None,
                                 ctypes.byref(lip) if want_energy else None, _stream(stream)), "pyhst_patch_fista")
    return W, X, energy[:int(n_iter)], float(lip.value)


def _host_ptr(a, name):
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous():
            raise PyhstError("%s must be a contiguous float32 host tensor" % name)
        return c_void_p(a.data_ptr())
    if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous):
        raise PyhstError("%s must be a contiguous float32 host array" % name)
    return c_void_p(a.ctypes.data)


def fbp_host(h_sino_raw, angles, axis, nx, ny, pixel_size=1.0, filter=FILTER_RAMLAK, mode=SCAN_180,
             out=None, max_slices_per_chunk=0, stream=None):
    """pyhst_fbp_host: HOST float32 [S,P,B] (numpy or pinned torch) -> HOST [S,ny,nx]."""
    lib = _load()
    s, p, b = h_sino_raw.shape
    if out is None:
        out = np.empty((s, ny, nx), dtype=np.float32)
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size)
    _check(lib.pyhst_fbp_host(_host_ptr(h_sino_raw, "h_sino_raw"), _host_ptr(out, "out"), ctypes.byref(g),
                              filter, mode, max_slices_per_chunk, _stream(stream)), "pyhst_fbp_host")
    return out


def backproject_host(h_sino, angles, axis, nx, ny, pixel_size=1.0, scale=1.0, out=None,
                     max_slices_per_chunk=0, stream=None):
    """pyhst_backproject_host: HOST float32 [S,P,B] -> HOST [S,ny,nx]."""
    lib = _load()
    s, p, b = h_sino.shape
    if out is None:
        out = np.empty((s, ny, nx), dtype=np.float32)
    g = _geom(s, p, b, angles, axis, nx, ny, pixel_size)
    _check(lib.pyhst_backproject_host(_host_ptr(h_sino, "h_sino"), _host_ptr(out, "out"), ctypes.byref(g),
                                      scale, max_slices_per_chunk, _stream(stream)), "pyhst_backproject_host")
    return out


def forward_project_host(h_img, angles, axis, n_bins, pixel_size=1.0, scale=1.0, out=None,
                         max_slices_per_chunk=0, stream=None):
    """pyhst_forward_project_host: HOST float32 [S,ny,nx] -> HOST [S,P,B]."""
    lib = _load()
    s, ny, nx = h_img.shape
    p = len(angles)
    if out is None:
        out = np.empty((s, p, n_bins), dtype=np.float32)
    g = _geom(s, p, n_bins, angles, axis, nx, ny, pixel_size)
    _check(lib.pyhst_forward_project_host(_host_ptr(h_img, "h_img"), _host_ptr(out, "out"), ctypes.byref(g),
                                          scale, max_slices_per_chunk, _stream(stream)),
           "pyhst_forward_project_host")
    return out


def halfacq_extent(n_bins, cbar):
    ext, pad = c_int32(0), c_int32(0)
    _check(_load().pyhst_halfacq_extent(n_bins, float(cbar), ctypes.byref(ext), ctypes.byref(pad)),
           "pyhst_halfacq_extent")
    return int(ext.value), int(pad.value)


def set_backproject_variant(variant: int) -> int:
    return int(_load().pyhst_set_backproject_variant(int(variant)))


def set_halfacq_stitch(enable: bool) -> int:
    return int(_load().pyhst_set_halfacq_stitch(1 if enable else 0))


def set_filter_variant(variant: int) -> int:
    """0 automatic, 1 cuFFT path, 2 fused shared-memory FFT kernel; returns the previous value."""
    return int(_load().pyhst_set_filter_variant(int(variant)))


def set_patch_gemm_variant(variant: int) -> int:
    """0 automatic, 1 FP32 SIMT GEMM, 2 tcgen05 3xTF32 GEMM; returns the previous value."""
    return int(_load().pyhst_set_patch_gemm_variant(int(variant)))


def set_forward_project_variant(variant: int) -> int:
    return int(_load().pyhst_set_forward_project_variant(int(variant)))


def test_fd_plan(angles, axis, n_bins, nx, ny, pixel_size=1.0, n_slices=1):
    """Host-only tables of the diagonal-line forward projector (pyhst_test.h): (info dict, chunk index per projection,
    line ranges [chunks][blocks][2])."""
    import numpy as np
    lib = _load()
    angles = np.ascontiguousarray(angles, dtype=np.float64)
    axis = np.ascontiguousarray(axis, dtype=np.float64)
    g = Geom(int(n_slices), int(angles.size), int(n_bins), 0, angles.ctypes.data_as(POINTER(c_double)),
             axis.ctypes.data_as(POINTER(c_double)), int(nx), int(ny), float(pixel_size))
    info = np.zeros(8, dtype=np.int32)
    chunk_of = np.zeros(angles.size, dtype=np.int32)
    lib.pyhst_test_fd_plan.argtypes = [POINTER(Geom), c_void_p, c_void_p, c_void_p]
    st = lib.pyhst_test_fd_plan(ctypes.byref(g), info.ctypes.data, chunk_of.ctypes.data, None)
    names = ("chunks", "left_out", "window", "blocks", "intervals_per_block", "projections_per_chunk", "zpad", "lines")
    d = dict(zip(names, (int(v) for v in info)))
    d["status"] = int(st)
    ranges = None
    if st == 0:
        ranges = np.zeros((d["chunks"], d["blocks"], 2), dtype=np.int32)
        lib.pyhst_test_fd_plan(ctypes.byref(g), info.ctypes.data, chunk_of.ctypes.data, ranges.ctypes.data)
    return d, chunk_of, ranges


test_fd_plan.__test__ = False   # not a pytest test


def set_test_workspace_limit(max_bytes: int) -> int:
    """pyhst_test_set_workspace_limit (pyhst_test.h): workspace growth beyond max_bytes fails with NOMEM; 0 = off."""
    return int(_load().pyhst_test_set_workspace_limit(int(max_bytes)))




def last_forward_project_kernel() -> int:
    return int(_load().pyhst_last_forward_project_kernel())


STAGES = ("ramp_filter", "repack", "backproject", "transpose", "forward_project", "tv_solver")


def profile_enable(enable: bool) -> bool:
    return bool(_load().pyhst_profile_enable(1 if enable else 0))


def profile_read(reset: bool = True):
    """{stage: (device ms, own kernel launches, cuFFT executions)} accumulated since the last reset."""
    n = len(STAGES)
    ms, k, f = (c_double * n)(), (c_int64 * n)(), (c_int64 * n)()
    _check(_load().pyhst_profile_read(ms, k, f, 1 if reset else 0), "pyhst_profile_read")
    return {STAGES[i]: (float(ms[i]), int(k[i]), int(f[i])) for i in range(n)}


def release_cache():
    _load().pyhst_release_cache()
