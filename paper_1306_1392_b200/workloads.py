"""Seeded synthetic inputs shaped like the paper's synchrotron scans.

This module only *makes inputs* (phantoms, their analytic Radon transforms, noise,
scan geometry).  It holds none of the method's arithmetic (no filter, no
interpolation, no projector) and is the one module that the tests feed to both the
CUDA path and the oracle.  It imports neither of them.

The paper's own data (ESRF scans, its 2k phantom) are not
available; these inputs stand in with the paper's shapes (2k-class slices, thousands
of projections for full scans, 150-200 for reduced dose) following the recipe of
BASELINE.json `configs` / SURVEY.md sec. 8(d), restated in DESIGN.md.

Coordinates (reading R1-R3): object point (x, y) in pixel units about the
rotation axis projects onto detector coordinate  c_p + x cos(theta) + y sin(theta)
(bin centres at integers), so a line integral at bin b of projection p is taken at
signed distance  s = (b - c_p) * bin_width  with bin_width = 1.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, Optional, Sequence

import numpy as np
import torch

SEED_BASE = 0x13061392

FILTER_RAMLAK = 0
FILTER_SHEPP_LOGAN = 1
FILTER_HANN = 2
FILTER_HAMMING = 3
SCAN_180 = 0
SCAN_360 = 1
SCAN_360_HALF = 2


def _rng(cfg: int, slice_idx: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + 1000 * cfg + slice_idx))


# Device on which the sinograms are synthesised.  "cpu" (default) is what the parity tests use:
# the arrays are bit-reproducible across machines.  bench.py sets it to "cuda" so that a full
# 16-slice stack is made in seconds; the noise stream then comes from the device generator.
_DEVICE = "cpu"


def set_device(device: str) -> str:
    global _DEVICE
    prev, _DEVICE = _DEVICE, str(device)
    return prev


def _torch_gen(cfg: int, slice_idx: int) -> torch.Generator:
    g = torch.Generator(device=_DEVICE)
    g.manual_seed(SEED_BASE + 1000 * cfg + slice_idx + 500)
    return g


# ----------------------------------------------------------------------------- phantoms
def ellipse_radon(ell: np.ndarray, angles: np.ndarray, s: torch.Tensor) -> torch.Tensor:
    """Analytic Radon transform of a sum of ellipses.

    ell: [n,6] rows (x0, y0, a, b, phi, rho);  angles: [P];  s: float64 tensor [P,B] of signed
    distances from the axis.  Line integral of an ellipse of density rho:
        p(theta, s) = 2 rho a b sqrt(max(0, r^2 - (s - s0)^2)) / r^2,
        r^2 = a^2 cos^2(theta - phi) + b^2 sin^2(theta - phi),  s0 = x0 cos(theta) + y0 sin(theta)
    (a disc of radius R reduces to the chord 2 rho sqrt(R^2 - s^2)).
    """
    out = torch.zeros_like(s)
    th = torch.as_tensor(np.asarray(angles, dtype=np.float64)).to(s.device)
    for x0, y0, a, b, phi, rho in np.asarray(ell, dtype=np.float64).reshape(-1, 6):
        r2 = (a * torch.cos(th - phi)) ** 2 + (b * torch.sin(th - phi)) ** 2
        s0 = x0 * torch.cos(th) + y0 * torch.sin(th)
        d = s - s0[:, None]
        out += (2.0 * rho * a * b / r2)[:, None] * torch.sqrt(torch.clamp(r2[:, None] - d * d, min=0.0))
    return out


def polygon_radon(polys: Sequence[np.ndarray], rhos: Sequence[float], angles: np.ndarray,
                  s: torch.Tensor) -> torch.Tensor:
    """Analytic Radon transform of convex polygons (vertices counter-clockwise, [m,2]).

    The line {x cos + y sin = s} is parametrised by u along (-sin, cos); each edge is a
    half-plane that clips the interval of u; the chord is the length left."""
    out = torch.zeros_like(s)
    th = torch.as_tensor(np.asarray(angles, dtype=np.float64)).to(s.device)
    ct, st = torch.cos(th)[:, None], torch.sin(th)[:, None]
    for verts, rho in zip(polys, rhos):
        verts = np.asarray(verts, dtype=np.float64)
        lo = torch.full_like(s, -1e30)
        hi = torch.full_like(s, 1e30)
        m = len(verts)
        for e in range(m):
            (x1, y1), (x2, y2) = verts[e], verts[(e + 1) % m]
            nx_, ny_ = (y2 - y1), -(x2 - x1)            # outward normal of a CCW polygon
            off = nx_ * x1 + ny_ * y1                    # inside: n . x <= off
            # point on the line: s*(cos,sin) + u*(-sin,cos)  ->  A + u*Bc <= off
            A = s * (nx_ * ct + ny_ * st)
            Bc = (-nx_ * st + ny_ * ct).expand_as(s)
            lim = (off - A) / torch.where(Bc == 0, torch.ones_like(Bc), Bc)
            hi = torch.where(Bc > 0, torch.minimum(hi, lim), hi)
            lo = torch.where(Bc < 0, torch.maximum(lo, lim), lo)
            empty = (Bc == 0) & (A > off)
            hi = torch.where(empty, torch.full_like(hi, -1e30), hi)
        out += rho * torch.clamp(hi - lo, min=0.0)
    return out


def random_ellipses(rng, n, radius, axes=(0.05, 0.4), rho=(-1.0, 1.0), inside=True) -> np.ndarray:
    """n ellipses: centres uniform in the disc, semi-axes U(axes)*radius, angle U(0,pi), density
    U(rho); with `inside` they are rejection-sampled to lie wholly inside the disc."""
    out = []
    while len(out) < n:
        r = radius * math.sqrt(rng.uniform())
        ang = rng.uniform(0.0, 2.0 * math.pi)
        a, b = rng.uniform(axes[0], axes[1], size=2) * radius
        if inside and r + max(a, b) > radius:
            continue
        out.append((r * math.cos(ang), r * math.sin(ang), a, b, rng.uniform(0.0, math.pi),
                    rng.uniform(rho[0], rho[1])))
    return np.array(out, dtype=np.float64)


def random_convex_polygons(rng, n, radius, levels=(0.33, 0.66, 1.0)):
    polys, rhos = [], []
    while len(polys) < n:
        m = int(rng.integers(3, 8))
        r = radius * math.sqrt(rng.uniform())
        ang = rng.uniform(0.0, 2.0 * math.pi)
        size = rng.uniform(0.08, 0.35) * radius
        if r + size > radius:
            continue
        # vertices on a circle at sorted angles -> convex, counter-clockwise
        va = np.sort(rng.uniform(0.0, 2.0 * math.pi, size=m))
        if np.any(np.diff(np.concatenate([va, [va[0] + 2 * math.pi]])) > math.pi * 0.95):
            continue
        cx, cy = r * math.cos(ang), r * math.sin(ang)
        polys.append(np.stack([cx + size * np.cos(va), cy + size * np.sin(va)], axis=1))
        rhos.append(float(levels[int(rng.integers(0, len(levels)))]))
    return polys, rhos


def rasterize_ellipses(ell: np.ndarray, nx: int, ny: int, pixel_size: float = 1.0) -> np.ndarray:
    """The phantom sampled at pixel centres (ground truth for the FBP -> phantom pin)."""
    jj = (np.arange(nx) - 0.5 * (nx - 1)) * pixel_size
    ii = (np.arange(ny) - 0.5 * (ny - 1)) * pixel_size
    x, y = np.meshgrid(jj, ii)
    img = np.zeros((ny, nx), dtype=np.float64)
    for x0, y0, a, b, phi, rho in np.asarray(ell, dtype=np.float64).reshape(-1, 6):
        xr = (x - x0) * math.cos(phi) + (y - y0) * math.sin(phi)
        yr = -(x - x0) * math.sin(phi) + (y - y0) * math.cos(phi)
        img += rho * ((xr / a) ** 2 + (yr / b) ** 2 <= 1.0)
    return img


# ----------------------------------------------------------------------------- workloads
@dataclass
class Workload:
    """One synthetic scan: geometry + a slice-wise sinogram generator."""
    name: str
    cfg: int
    n_slices: int
    n_angles: int
    n_bins: int
    nx: int
    ny: int
    pixel_size: float
    angles: np.ndarray            # float64 [P], radians
    axis: np.ndarray              # float64 [P], bin coordinate of the rotation axis
    filter: int
    mode: int
    _slice_fn: Callable[["Workload", int], torch.Tensor] = field(repr=False, default=None)
    ellipses: Optional[Callable[[int], np.ndarray]] = field(repr=False, default=None)  # phantom of slice s

    def bin_offsets(self) -> torch.Tensor:
        """s[p,b] = b - c_p (float64 [P,B])."""
        b = torch.arange(self.n_bins, dtype=torch.float64, device=_DEVICE)
        return b[None, :] - torch.as_tensor(self.axis).to(_DEVICE)[:, None]

    def sinogram_slice(self, s: int) -> np.ndarray:
        return self._slice_fn(self, s).to(torch.float32).cpu().numpy()

    def sinogram_tensor(self, slices: Optional[Sequence[int]] = None) -> torch.Tensor:
        """float32 [S,P,B] torch tensor left on the synthesis device (see set_device)."""
        idx = range(self.n_slices) if slices is None else slices
        return torch.stack([self._slice_fn(self, s).to(torch.float32) for s in idx], dim=0)

    def sinogram(self, slices: Optional[Sequence[int]] = None) -> np.ndarray:
        """float32 [S,P,B] (C order) for the requested slices (default: all)."""
        idx = range(self.n_slices) if slices is None else slices
        return np.stack([self.sinogram_slice(s) for s in idx], axis=0)

    def updates(self) -> int:
        """pixel * projection * slice updates of one backprojection."""
        return self.n_slices * self.nx * self.ny * self.n_angles


def _gauss(p: torch.Tensor, rel_sigma: float, gen: torch.Generator) -> torch.Tensor:
    sigma = rel_sigma * float(p.abs().max())
    return p + sigma * torch.randn(p.shape, dtype=torch.float64, generator=gen, device=p.device)


def _poisson_log(p: torch.Tensor, photons: float, gen: torch.Generator) -> torch.Tensor:
    counts = torch.poisson(photons * torch.exp(-p), generator=gen)
    return -torch.log(torch.clamp(counts, min=1.0) / photons)


def _even_angles(n, span):
    return np.arange(n, dtype=np.float64) * (span / n)


def _sz(v, shrink, mult=1):
    return max(mult, int(round(v / shrink / mult)) * mult)


def config(cfg: int, shrink: float = 1.0, n_slices: Optional[int] = None) -> Workload:
    """The five BASELINE.json configs.  `shrink` > 1 divides every length (bins, pixels,
    projections, phantom radius) by that factor and keeps the structure; it is how the
    parity tests get cases the oracle finishes in seconds."""
    k = float(shrink)
    if cfg == 1:
        P, B, N = _sz(180, k), _sz(367, k), _sz(256, k)
        R = N / 2.0
        wl = Workload("cfg1_single_slice_256", 1, n_slices or 1, P, B, N, N, 1.0, _even_angles(P, math.pi),
                      np.full(P, (B - 1) / 2.0), FILTER_RAMLAK, SCAN_180)

        def ellipses(s):
            ell = random_ellipses(_rng(1, s), 10, R, inside=False)
            ell[:, :2] *= 0.6                       # keep most of the mass on the detector
            return ell

        def fn(w, s):
            return _gauss(ellipse_radon(ellipses(s), w.angles, w.bin_offsets()), 0.01, _torch_gen(1, s))
        wl._slice_fn = fn
        wl.ellipses = ellipses
        return wl
    if cfg == 2:
        P, B, N = _sz(2000, k), _sz(2048, k), _sz(2048, k)
        R = 1000.0 / k
        drift = _rng(2, 900).uniform(-1.5, 1.5, size=P)
        wl = Workload("cfg2_batch16_2048", 2, n_slices or 16, P, B, N, N, 1.0, _even_angles(P, math.pi),
                      (B - 1) / 2.0 + drift, FILTER_SHEPP_LOGAN, SCAN_180)

        def fn(w, s):
            ell = random_ellipses(_rng(2, s), 30, R, rho=(0.1, 1.0))
            p = ellipse_radon(ell, w.angles, w.bin_offsets())
            p = p * (2.0 / float(p.max()))
            return _poisson_log(p, 1e4, _torch_gen(2, s))
        wl._slice_fn = fn
        return wl
    if cfg == 3:
        P, B = _sz(4000, k), _sz(2048, k)
        c = round(1900.0 / k)
        N = 2 * c
        R = 1850.0 / k
        wl = Workload("cfg3_halfacq_3800", 3, n_slices or 4, P, B, N, N, 1.0, _even_angles(P, 2 * math.pi),
                      np.full(P, float(c)), FILTER_RAMLAK, SCAN_360_HALF)

        def fn(w, s):
            ell = random_ellipses(_rng(3, s), 40, R, axes=(0.03, 0.3), rho=(0.1, 1.0))
            p = ellipse_radon(ell, w.angles, w.bin_offsets())
            p = p * (2.0 / float(p.max()))
            return _gauss(p, 0.005, _torch_gen(3, s))
        wl._slice_fn = fn
        return wl
    if cfg == 4:
        P, B, N = _sz(200, k), _sz(1024, k), _sz(1024, k)
        R = 480.0 / k
        wl = Workload("cfg4_iterative_1024", 4, n_slices or 8, P, B, N, N, 1.0, _even_angles(P, math.pi),
                      np.full(P, (B - 1) / 2.0), FILTER_RAMLAK, SCAN_180)

        def fn(w, s):
            polys, rhos = random_convex_polygons(_rng(4, s), 12, R)
            p = polygon_radon(polys, rhos, w.angles, w.bin_offsets())
            p = p * (2.0 / float(p.max()))
            return _poisson_log(p, 2e3, _torch_gen(4, s))
        wl._slice_fn = fn
        return wl
    if cfg == 5:
        P, B, N = _sz(3000, k), _sz(2560, k), _sz(2560, k)
        R = 1250.0 / k
        drift = _rng(5, 900).uniform(-2.0, 2.0, size=P)
        rs = _rng(5, 901)
        spheres = []
        while len(spheres) < 15:
            r = R * math.sqrt(rs.uniform())
            ang = rs.uniform(0, 2 * math.pi)
            rad = rs.uniform(0.04, 0.25) * R
            if r + rad > R:
                continue
            spheres.append((r * math.cos(ang), r * math.sin(ang), rs.uniform(-0.5 * rad, 64.0 / k + 0.5 * rad),
                            rad, rs.uniform(0.1, 1.0)))
        wl = Workload("cfg5_throughput_stack_2560", 5, n_slices or 64, P, B, N, N, 1.0,
                      _even_angles(P, math.pi), (B - 1) / 2.0 + drift, FILTER_RAMLAK, SCAN_180)

        def fn(w, s):
            ell = [tuple(e) for e in random_ellipses(_rng(5, s), 20, R, rho=(0.1, 1.0))]
            z = s / k
            for x0, y0, z0, rad, rho in spheres:
                r2 = rad * rad - (z - z0) ** 2
                if r2 > 0:
                    ell.append((x0, y0, math.sqrt(r2), math.sqrt(r2), 0.0, rho))
            p = ellipse_radon(np.array(ell), w.angles, w.bin_offsets())
            p = p * (2.0 / float(p.max()))
            return _gauss(p, 0.01, _torch_gen(5, s))
        wl._slice_fn = fn
        return wl
    raise ValueError("cfg must be 1..5")


def custom(n_slices, n_angles, n_bins, nx, ny, pixel_size=1.0, span=math.pi, axis=None, drift=0.0,
           filter=FILTER_RAMLAK, mode=SCAN_180, n_ellipses=8, noise=0.01, seed=77, jitter_angles=0.0) -> Workload:
    """A free-form small scan for edge-case and ragged-size tests (same generator family)."""
    rng = _rng(9, seed)
    angles = _even_angles(n_angles, span)
    if jitter_angles:
        angles = angles + rng.uniform(-jitter_angles, jitter_angles, size=n_angles)
    c0 = (n_bins - 1) / 2.0 if axis is None else float(axis)
    ax = c0 + (rng.uniform(-drift, drift, size=n_angles) if drift else np.zeros(n_angles))
    R = 0.45 * min(nx, ny) * pixel_size
    wl = Workload("custom", 9, n_slices, n_angles, n_bins, nx, ny, float(pixel_size), angles, ax, filter, mode)

    def fn(w, s):
        ell = random_ellipses(_rng(9, 1000 * seed + s), n_ellipses, R, rho=(-1.0, 1.0))
        p = ellipse_radon(ell, w.angles, w.bin_offsets())
        return _gauss(p, noise, _torch_gen(9, 1000 * seed + s)) if noise else p
    wl._slice_fn = fn
    return wl


def random_image(n_slices, ny, nx, seed=0) -> np.ndarray:
    """Seeded dense float32 image stack (forward-projector and adjoint tests)."""
    return _rng(8, seed).standard_normal((n_slices, ny, nx)).astype(np.float32)


def random_sinogram(n_slices, n_angles, n_bins, seed=0) -> np.ndarray:
    return _rng(7, seed).standard_normal((n_slices, n_angles, n_bins)).astype(np.float32)


def dct_dictionary(m: int, n_atoms: int, seed: int = 0) -> np.ndarray:
    """Seeded over-complete dictionary [n_atoms, m*m] (float32, unit-norm rows) standing in for the
    learned basis of ref. [4] (fig. 5: not available).  Rows = separable 2-D cosines
    cos(pi (i + 1/2) u / q) cos(pi (j + 1/2) v / q) on an over-complete frequency grid q = ceil(sqrt(
    n_atoms)) >= m (the first row is the constant patch); a seeded permutation picks which of the q^2
    products are kept when n_atoms < q^2.  Holds none of the method's arithmetic."""
    q = int(math.ceil(math.sqrt(n_atoms)))
    q = max(q, m)
    i = np.arange(m) + 0.5
    basis = np.cos(math.pi * np.outer(np.arange(q), i) / q)          # [q, m]
    atoms = np.einsum("ui,vj->uvij", basis, basis).reshape(q * q, m * m)
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 77 + seed))
    order = np.concatenate([[0], 1 + rng.permutation(q * q - 1)])[:n_atoms]
    D = atoms[np.sort(order)]
    D = D / np.linalg.norm(D, axis=1, keepdims=True)
    return np.ascontiguousarray(D, dtype=np.float32)
