"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end of ``oracle/pyhst_oracle.c``: the plain double-precision CPU
statement of the ramp filter, backprojection, forward projection and FBP of
arxiv/paper_1306_1392 (readings R1-R15 of
SURVEY.md sec. 8(c), restated in DESIGN.md).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1306_1392_b200`` and the product imports nothing from here.

Arrays are numpy; float32 inputs are the very arrays the GPU path receives and
are widened exactly, all results are float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_float, c_int, c_int32, c_int64

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pyhst_oracle.c")
_LIB = os.path.join(_HERE, "libpyhst_oracle.so")

FILTER_RAMLAK = 0
FILTER_SHEPP_LOGAN = 1
FILTER_HANN = 2
FILTER_HAMMING = 3
SCAN_180 = 0
SCAN_360 = 1
SCAN_360_HALF = 2


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_ramp_kernel.restype = c_double
        lib.oracle_ramp_kernel.argtypes = [c_int, c_int64]
        lib.oracle_num_threads.restype = c_int
        _lib = lib
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a, ty):
    return a.ctypes.data_as(POINTER(ty))


def _check(rc, what):
    if rc != 0:
        raise ValueError("oracle %s failed with status %d" % (what, rc))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


class threads:
    """``with oracle.threads(1): ...`` -- run the enclosed oracle calls on ``n`` OpenMP threads."""

    def __init__(self, n: int):
        self.n = int(n)

    def __enter__(self):
        self.old = num_threads()
        _load().oracle_set_num_threads(c_int(self.n))
        return self

    def __exit__(self, *exc):
        _load().oracle_set_num_threads(c_int(self.old))
        return False


def ramp_kernel(filter: int, n) -> np.ndarray:
    """h[n] of R8 for integer lags ``n`` (array-like)."""
    lib = _load()
    n = np.asarray(n, dtype=np.int64)
    return np.array([lib.oracle_ramp_kernel(int(filter), int(v)) for v in n.ravel()],
                    dtype=np.float64).reshape(n.shape)


def halfacq_weights(n_bins: int, cbar: float) -> np.ndarray:
    w = np.empty(n_bins, dtype=np.float64)
    _check(_load().oracle_halfacq_weights(c_int32(n_bins), c_double(cbar), _p(w, c_double)),
           "halfacq_weights")
    return w


def halfacq_extent(n_bins: int, cbar: float):
    ext, pad = c_int32(0), c_int32(0)
    _load().oracle_halfacq_extent(c_int32(n_bins), c_double(cbar), ctypes.byref(ext),
                                  ctypes.byref(pad))
    return int(ext.value), int(pad.value)


def ramp_filter(rows, n_bins_out=None, pad_left=0, filter=FILTER_RAMLAK, col_weights=None):
    """rows: float32 [..., n_bins_in] -> float64 [..., n_bins_out] (direct convolution)."""
    rows = _f32(rows)
    b_in = rows.shape[-1]
    b_out = b_in if n_bins_out is None else int(n_bins_out)
    flat = rows.reshape(-1, b_in)
    out = np.empty((flat.shape[0], b_out), dtype=np.float64)
    w = None if col_weights is None else _f32(col_weights)
    _check(_load().oracle_ramp_filter(
        _p(flat, c_float), c_int64(b_in), _p(out, c_double), c_int64(flat.shape[0]),
        c_int32(b_in), c_int32(b_out), c_int32(pad_left), c_int(filter),
        _p(w, c_float) if w is not None else None), "ramp_filter")
    return out.reshape(rows.shape[:-1] + (b_out,))


def _geom(sino_shape, angles, axis):
    s, p, b = sino_shape
    angles = _f64(angles)
    axis = _f64(axis)
    if angles.shape != (p,) or axis.shape != (p,):
        raise ValueError("angles/axis must have shape [n_angles]")
    return s, p, b, angles, axis


def backproject(sino, angles, axis, nx, ny, pixel_size=1.0, scale=1.0):
    """sino float32 (or float64) [S,P,B] -> float64 [S,ny,nx]."""
    lib = _load()
    f64 = np.asarray(sino).dtype == np.float64
    sino = _f64(sino) if f64 else _f32(sino)
    s, p, b, angles, axis = _geom(sino.shape, angles, axis)
    img = np.empty((s, ny, nx), dtype=np.float64)
    fn = lib.oracle_backproject_f64 if f64 else lib.oracle_backproject
    _check(fn(_p(sino, c_double if f64 else c_float), c_int64(b), _p(img, c_double), c_int32(s),
              c_int32(p), c_int32(b), _p(angles, c_double), _p(axis, c_double), c_int32(nx),
              c_int32(ny), c_double(pixel_size), c_double(scale)), "backproject")
    return img


def backproject_points(sino, angles, axis, nx, ny, pts, pixel_size=1.0, scale=1.0):
    """Same definition at pixels ``pts`` = int array [n,3] of (s,i,j) -> float64 [n]."""
    lib = _load()
    sino = _f32(sino)
    s, p, b, angles, axis = _geom(sino.shape, angles, axis)
    pts = np.asarray(pts, dtype=np.int32).reshape(-1, 3)
    ps, pi, pj = _i32(pts[:, 0]), _i32(pts[:, 1]), _i32(pts[:, 2])
    out = np.empty(len(pts), dtype=np.float64)
    _check(lib.oracle_backproject_points(
        _p(sino, c_float), c_int64(b), c_int32(s), c_int32(p), c_int32(b), _p(angles, c_double),
        _p(axis, c_double), c_int32(nx), c_int32(ny), c_double(pixel_size), c_double(scale),
        c_int64(len(pts)), _p(ps, c_int32), _p(pi, c_int32), _p(pj, c_int32), _p(out, c_double)),
        "backproject_points")
    return out


def forward_project(img, angles, axis, n_bins, pixel_size=1.0, scale=1.0):
    """img float32 [S,ny,nx] -> float64 [S,P,B] (scatter form of the exact transpose)."""
    lib = _load()
    img = _f32(img)
    s, ny, nx = img.shape
    angles, axis = _f64(angles), _f64(axis)
    p = angles.shape[0]
    sino = np.empty((s, p, n_bins), dtype=np.float64)
    _check(lib.oracle_forward_project(
        _p(img, c_float), _p(sino, c_double), c_int32(s), c_int32(p), c_int32(n_bins),
        _p(angles, c_double), _p(axis, c_double), c_int32(nx), c_int32(ny), c_double(pixel_size),
        c_double(scale)), "forward_project")
    return sino


def forward_project_rows(img, angles, axis, n_bins, rows, pixel_size=1.0, scale=1.0):
    """Only rows ``rows`` = int array [n,2] of (s,p) -> float64 [n, n_bins]."""
    lib = _load()
    img = _f32(img)
    s, ny, nx = img.shape
    angles, axis = _f64(angles), _f64(axis)
    rows = np.asarray(rows, dtype=np.int32).reshape(-1, 2)
    rs, rp = _i32(rows[:, 0]), _i32(rows[:, 1])
    out = np.empty((len(rows), n_bins), dtype=np.float64)
    _check(lib.oracle_forward_project_rows(
        _p(img, c_float), c_int32(s), c_int32(angles.shape[0]), c_int32(n_bins),
        _p(angles, c_double), _p(axis, c_double), c_int32(nx), c_int32(ny), c_double(pixel_size),
        c_double(scale), c_int64(len(rows)), _p(rs, c_int32), _p(rp, c_int32), _p(out, c_double)),
        "forward_project_rows")
    return out


def fbp(sino_raw, angles, axis, nx, ny, pixel_size=1.0, filter=FILTER_RAMLAK, mode=SCAN_180,
        pts=None):
    """FILTER then BP in double.  With ``pts`` ([n,3] of (s,i,j)) only those pixels."""
    lib = _load()
    sino = _f32(sino_raw)
    s, p, b, angles, axis = _geom(sino.shape, angles, axis)
    common = [_p(sino, c_float), c_int64(b)]
    tail = [c_int32(s), c_int32(p), c_int32(b), _p(angles, c_double), _p(axis, c_double),
            c_int32(nx), c_int32(ny), c_double(pixel_size), c_int(filter), c_int(mode)]
    if pts is None:
        img = np.empty((s, ny, nx), dtype=np.float64)
        _check(lib.oracle_fbp(*common, _p(img, c_double), *tail, c_int64(-1), None, None, None,
                              None), "fbp")
        return img
    pts = np.asarray(pts, dtype=np.int32).reshape(-1, 3)
    ps, pi, pj = _i32(pts[:, 0]), _i32(pts[:, 1]), _i32(pts[:, 2])
    out = np.empty(len(pts), dtype=np.float64)
    _check(lib.oracle_fbp(*common, None, *tail, c_int64(len(pts)), _p(ps, c_int32),
                          _p(pi, c_int32), _p(pj, c_int32), _p(out, c_double)), "fbp(points)")
    return out


# ---- NEXT row N1: TV-regularised FISTA (eq. 1-3; readings R17-R20) ----------
def forward_project_f64(img, angles, axis, n_bins, pixel_size=1.0, scale=1.0):
    """img float64 [S,ny,nx] -> float64 [S,P,B]; the input is not rounded to float32."""
    lib = _load()
    img = _f64(img)
    s, ny, nx = img.shape
    angles, axis = _f64(angles), _f64(axis)
    p = angles.shape[0]
    sino = np.empty((s, p, n_bins), dtype=np.float64)
    _check(lib.oracle_forward_project_f64(
        _p(img, c_double), _p(sino, c_double), c_int32(s), c_int32(p), c_int32(n_bins),
        _p(angles, c_double), _p(axis, c_double), c_int32(nx), c_int32(ny), c_double(pixel_size),
        c_double(scale)), "forward_project_f64")
    return sino


def tv(x) -> float:
    """Isotropic total variation (eq. 2) of a stack [S,ny,nx], summed over slices."""
    lib = _load()
    lib.oracle_tv.restype = c_double
    x = _f64(x)
    s, ny, nx = x.shape
    return float(lib.oracle_tv(_p(x, c_double), c_int32(s), c_int32(ny), c_int32(nx)))


def prox_tv(z, tau, n_inner):
    """argmin_x 1/2 ||x - z||^2 + tau TV(x) per slice, n_inner dual projected-gradient steps."""
    lib = _load()
    z = _f64(z)
    s, ny, nx = z.shape
    x = np.empty_like(z)
    _check(lib.oracle_prox_tv(_p(z, c_double), _p(x, c_double), c_int32(s), c_int32(ny), c_int32(nx),
                              c_double(tau), c_int32(n_inner)), "prox_tv")
    return x


def lipschitz(angles, axis, n_bins, nx, ny, pixel_size=1.0, n_power=8) -> float:
    """1.1 x the power-iteration estimate of lambda_max(P^T P) (R17)."""
    lib = _load()
    angles, axis = _f64(angles), _f64(axis)
    out = c_double(0.0)
    _check(lib.oracle_lipschitz(c_int32(angles.shape[0]), c_int32(n_bins), _p(angles, c_double),
                                _p(axis, c_double), c_int32(nx), c_int32(ny), c_double(pixel_size),
                                c_int32(n_power), ctypes.byref(out)), "lipschitz")
    return float(out.value)


def fista_tv(data, angles, axis, nx, ny, beta, L, n_iter, n_inner=20, pixel_size=1.0):
    """data float32 [S,P,B] -> (x float64 [S,ny,nx], energy float64 [n_iter])."""
    lib = _load()
    data = _f32(data)
    s, p, b, angles, axis = _geom(data.shape, angles, axis)
    x = np.empty((s, ny, nx), dtype=np.float64)
    energy = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(lib.oracle_fista_tv(_p(data, c_float), c_int64(b), _p(x, c_double), c_int32(s), c_int32(p),
                               c_int32(b), _p(angles, c_double), _p(axis, c_double), c_int32(nx),
                               c_int32(ny), c_double(pixel_size), c_double(beta), c_double(L),
                               c_int32(n_iter), c_int32(n_inner), _p(energy, c_double)), "fista_tv")
    return x, energy[:n_iter]


def ista_tv(data, angles, axis, nx, ny, beta, L, n_iter, n_inner=20, pixel_size=1.0):
    """ISTA: fista_tv without the momentum.  -> (x float64, energy float64 [n_iter])."""
    lib = _load()
    data = _f32(data)
    s, p, b, angles, axis = _geom(data.shape, angles, axis)
    x = np.empty((s, ny, nx), dtype=np.float64)
    energy = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(lib.oracle_ista_tv(_p(data, c_float), c_int64(b), _p(x, c_double), c_int32(s), c_int32(p),
                              c_int32(b), _p(angles, c_double), _p(axis, c_double), c_int32(nx),
                              c_int32(ny), c_double(pixel_size), c_double(beta), c_double(L),
                              c_int32(n_iter), c_int32(n_inner), _p(energy, c_double)), "ista_tv")
    return x, energy[:n_iter]


FILTER_COSINE = 4


# ---- NEXT row N4: ring filter and the estimators of sec. 4 (L149-L162) ----------
def ring_filter(sino, half_width, model=None):
    """sino float32 [S,P,B] (model: same shape or None) -> float64 [S,P,B] (reading R21)."""
    lib = _load()
    sino = _f32(sino)
    s, p, b = sino.shape
    mod = None if model is None else _f32(model)
    if mod is not None and mod.shape != sino.shape:
        raise ValueError("model must have the sinogram's shape")
    out = np.empty((s, p, b), dtype=np.float64)
    _check(lib.oracle_ring_filter(_p(sino, c_float), _p(mod, c_float) if mod is not None else None,
                                  c_int64(b), _p(out, c_double), c_int32(s), c_int32(p), c_int32(b),
                                  c_int32(half_width)), "ring_filter")
    return out


def ecohe(a, b):
    """eq. 11 per slice: Cos(a - b, a) for stacks a = I(beta), b = I(0+) [S, ...] -> float64 [S]."""
    lib = _load()
    a, b = _f32(a), _f32(b)
    if a.shape != b.shape:
        raise ValueError("shapes differ")
    s = a.shape[0]
    out = np.empty(s, dtype=np.float64)
    _check(lib.oracle_ecohe(_p(a, c_float), _p(b, c_float), c_int32(s), c_int64(a[0].size), _p(out, c_double)),
           "ecohe")
    return out


def cv_distance(img, data_excl, angles_excl, axis_excl, pixel_size=1.0):
    """Cross-validation distance (L149): sum over the excluded projections of ||P x - data||^2, per slice."""
    lib = _load()
    img, data = _f32(img), _f32(data_excl)
    s, ny, nx = img.shape
    s2, e, b = data.shape
    angles, axis = _f64(angles_excl), _f64(axis_excl)
    if s2 != s or angles.shape != (e,) or axis.shape != (e,):
        raise ValueError("shape mismatch")
    out = np.empty(s, dtype=np.float64)
    _check(lib.oracle_cv_distance(_p(img, c_float), _p(data, c_float), c_int64(b), c_int32(s), c_int32(e),
                                  c_int32(b), _p(angles, c_double), _p(axis, c_double), c_int32(nx),
                                  c_int32(ny), c_double(pixel_size), _p(out, c_double)), "cv_distance")
    return out


# ---- NEXT row N3: overlapping-patch dictionary reconstruction (Alg. 1) ------
def patch_grid(ny, nx, m, st):
    na, nb = c_int32(0), c_int32(0)
    _check(_load().oracle_patch_grid(c_int32(ny), c_int32(nx), c_int32(m), c_int32(st), ctypes.byref(na),
                                     ctypes.byref(nb)), "patch_grid")
    return int(na.value), int(nb.value)


def patch_maps(ny, nx, m, st):
    """(core [ny,nx] int32 = C_j, cover [ny,nx] int32 = N_v(j))."""
    core = np.empty((ny, nx), dtype=np.int32)
    cover = np.empty((ny, nx), dtype=np.int32)
    _check(_load().oracle_patch_maps(c_int32(ny), c_int32(nx), c_int32(m), c_int32(st), _p(core, c_int32),
                                     _p(cover, c_int32)), "patch_maps")
    return core, cover


def patch_gradient(W, D, data, angles, axis, nx, ny, m, st, rho, pixel_size=1.0):
    """Algorithm 1 for one slice.  W [N,Nc] f64, D [Nc,m*m] f64, data f32 [P,B] -> (G [N,Nc], X [ny,nx], f)."""
    lib = _load()
    W, D, data = _f64(W), _f64(D), _f32(data)
    p, b = data.shape
    angles, axis = _f64(angles), _f64(axis)
    n_atoms = D.shape[0]
    G = np.empty_like(W)
    X = np.empty((ny, nx), dtype=np.float64)
    f = c_double(0.0)
    _check(lib.oracle_patch_gradient(_p(W, c_double), _p(D, c_double), _p(data, c_float), c_int64(b), c_int32(p),
                                     c_int32(b), _p(angles, c_double), _p(axis, c_double), c_int32(nx), c_int32(ny),
                                     c_double(pixel_size), c_int32(m), c_int32(st), c_int32(n_atoms), c_double(rho),
                                     _p(G, c_double), _p(X, c_double), ctypes.byref(f)), "patch_gradient")
    return G, X, float(f.value)


def soft_threshold(v, t):
    v = _f64(v)
    out = np.empty_like(v)
    _load().oracle_soft_threshold(_p(v, c_double), c_int64(v.size), c_double(t), _p(out, c_double))
    return out


def patch_lipschitz(D, angles, axis, n_bins, nx, ny, m, st, rho, pixel_size=1.0, n_power=8) -> float:
    lib = _load()
    D = _f64(D)
    angles, axis = _f64(angles), _f64(axis)
    out = c_double(0.0)
    _check(lib.oracle_patch_lipschitz(_p(D, c_double), c_int32(angles.shape[0]), c_int32(n_bins),
                                      _p(angles, c_double), _p(axis, c_double), c_int32(nx), c_int32(ny),
                                      c_double(pixel_size), c_int32(m), c_int32(st), c_int32(D.shape[0]),
                                      c_double(rho), c_int32(n_power), ctypes.byref(out)), "patch_lipschitz")
    return float(out.value)


def patch_fista(D, data, angles, axis, nx, ny, m, st, rho, beta, Lw, n_iter, pixel_size=1.0):
    """-> (W [N,Nc] f64, X [ny,nx] f64, energy [n_iter])."""
    lib = _load()
    D, data = _f64(D), _f32(data)
    p, b = data.shape
    angles, axis = _f64(angles), _f64(axis)
    na, nb = patch_grid(ny, nx, m, st)
    W = np.empty((na * nb, D.shape[0]), dtype=np.float64)
    X = np.empty((ny, nx), dtype=np.float64)
    energy = np.zeros(max(n_iter, 1), dtype=np.float64)
    _check(lib.oracle_patch_fista(_p(D, c_double), _p(data, c_float), c_int64(b), c_int32(p), c_int32(b),
                                  _p(angles, c_double), _p(axis, c_double), c_int32(nx), c_int32(ny),
                                  c_double(pixel_size), c_int32(m), c_int32(st), c_int32(D.shape[0]), c_double(rho),
                                  c_double(beta), c_double(Lw), c_int32(n_iter), _p(W, c_double), _p(X, c_double),
                                  _p(energy, c_double)), "patch_fista")
    return W, X, energy[:n_iter]
