"""GPU-vs-oracle parity of the four C-ABI entry points (run on a B200 with ``-m gpu``).

Both sides get the same seeded float32 inputs from ``paper_1306_1392_b200.workloads``; the CUDA
path is called through the C ABI (ctypes binding) and compared element by element with the
double-precision oracle.  The bar is BASELINE.json's: relative L2 error <= 1e-5 and max-abs error
<= 1e-4 * max|oracle|.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

REL_L2 = 1e-5
MAX_ABS = 1e-4


@pytest.fixture(scope="module")
def lib():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; there is no CPU fallback")
    import paper_1306_1392_b200 as P
    P.binding._load()          # fail loudly if libpyhst_b200.so is missing
    yield P
    P.release_cache()


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_parity(got, want, what, rel=REL_L2, mabs=MAX_ABS):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    assert got.shape == want.shape, what
    assert np.isfinite(got).all(), what + ": non-finite output"
    num = np.linalg.norm((got - want).ravel())
    den = np.linalg.norm(want.ravel())
    peak = np.abs(want).max()
    err_max = np.abs(got - want).max()
    assert num <= rel * den + 1e-30, "%s: rel-L2 %.3e > %.1e" % (what, num / max(den, 1e-300), rel)
    assert err_max <= mabs * peak + 1e-30, "%s: max-abs %.3e > %.1e * %.3e" % (what, err_max, mabs, peak)
    return num / max(den, 1e-300)


# ------------------------------------------------------------------------------ backprojection
BP_CASES = [
    # S, P, B, nx, ny, h, axis, drift  -- ragged slice group, ragged chunk of projections, several tiles
    (1, 1, 40, 33, 21, 1.0, None, 0.0),
    (5, 37, 211, 150, 70, 1.0, None, 1.5),
    (3, 50, 97, 130, 131, 0.8, 30.2, 0.7),      # axis off centre: many pixels leave the detector
    (2, 19, 64, 200, 90, 1.3, None, 0.0),       # pixel larger than a bin: image wider than detector
    (4, 16, 300, 64, 64, 0.5, None, 2.0),       # exactly one tile and one chunk
    (9, 33, 180, 70, 129, 1.0, 179.0, 0.0),     # axis at the detector border
    (6, 70, 260, 200, 190, 1.0, None, 1.0),     # 360-degree angles: every class / row-reversal combination
    (2, 40, 64, 300, 40, 1.2, None, 0.0),       # image far wider than the detector: windows clamped on the pads
]


@pytest.mark.parametrize("variant", [1, 2, 3, 4, 6, 7])
@pytest.mark.parametrize("case", BP_CASES)
def test_backproject_matches_oracle(lib, oracle, case, variant):
    S, P, B, nx, ny, h, axis, drift = case
    wl = lib.workloads
    w = wl.custom(S, P, B, nx, ny, pixel_size=h, axis=axis, drift=drift, jitter_angles=0.01, seed=P,
                  span=2 * math.pi if P == 70 else math.pi)
    sino = wl.random_sinogram(S, P, B, seed=B)
    want = oracle.backproject(sino, w.angles, w.axis, nx, ny, pixel_size=h, scale=0.37)
    prev = lib.set_backproject_variant(variant)
    try:
        got = lib.backproject(_dev(sino), w.angles, w.axis, nx, ny, pixel_size=h, scale=0.37).cpu().numpy()
    finally:
        lib.set_backproject_variant(prev)
    assert_parity(got, want, "backproject variant %d %r" % (variant, case))


def test_backproject_config1_full(lib, oracle):
    w = lib.workloads.config(1)
    sino = lib.workloads.random_sinogram(1, w.n_angles, w.n_bins, seed=1)
    want = oracle.backproject(sino, w.angles, w.axis, w.nx, w.ny)
    got = lib.backproject(_dev(sino), w.angles, w.axis, w.nx, w.ny).cpu().numpy()
    assert_parity(got, want, "backproject cfg1")


def test_backproject_batch_independence(lib):
    """K12 on the device: a slice's result does not depend on the stack it is computed in."""
    wl = lib.workloads
    w = wl.custom(6, 40, 120, 90, 80, drift=1.0)
    sino = _dev(wl.random_sinogram(6, 40, 120, seed=5))
    full = lib.backproject(sino, w.angles, w.axis, 90, 80)
    part = lib.backproject(sino[1:6].contiguous(), w.angles, w.axis, 90, 80)   # other position in its group
    assert (full[2] == part[1]).all()
    # a stack of <= 4 slices runs the 4-slice kernel (runs of 16 pixels instead of 8: the weights are
    # stepped from other starting points), so a single slice agrees to FP32 rounding, not bit by bit
    one = lib.backproject(sino[2:3].contiguous(), w.angles, w.axis, 90, 80)
    assert float((full[2] - one[0]).abs().max()) <= 2e-5 * float(full[2].abs().max())
    prev = lib.set_backproject_variant(4)
    try:
        one8 = lib.backproject(sino[2:3].contiguous(), w.angles, w.axis, 90, 80)
    finally:
        lib.set_backproject_variant(prev)
    assert (full[2] == one8[0]).all()


@pytest.mark.parametrize("S", [4, 7, 9, 12, 20])
def test_backproject_default_kernel_choice(lib, oracle, S):
    """Automatic kernel choice: <= 4 slices the 4-slice run kernel, pairs of slice groups the 8-slice kernel, and the
    last group of an odd number (>= 3) of groups the 4-slice kernel again (no duplicate group)."""
    wl = lib.workloads
    P, B, nx, ny = 40, 210, 140, 130
    w = wl.custom(S, P, B, nx, ny, drift=1.0, jitter_angles=0.01, seed=S, span=2 * math.pi)
    sino = wl.random_sinogram(S, P, B, seed=S)
    want = oracle.backproject(sino, w.angles, w.axis, nx, ny, scale=1.3)
    got = lib.backproject(_dev(sino), w.angles, w.axis, nx, ny, scale=1.3).cpu().numpy()
    assert_parity(got, want, "backproject, default kernels, %d slices" % S)


@pytest.mark.parametrize("S", [13, 16, 18])
def test_backproject_run16_matches_oracle(lib, oracle, S):
    """pyhst_test.h variant 7: 16 slices per thread (four slice groups per block, ragged stacks read a duplicate group
    that is never stored); 360-degree angles exercise both classes and the row reversal."""
    wl = lib.workloads
    P, B, nx, ny = 45, 230, 150, 140
    w = wl.custom(S, P, B, nx, ny, drift=1.5, jitter_angles=0.01, seed=S, span=2 * math.pi)
    sino = wl.random_sinogram(S, P, B, seed=S)
    want = oracle.backproject(sino, w.angles, w.axis, nx, ny, scale=0.7)
    prev = lib.set_backproject_variant(7)
    try:
        got = lib.backproject(_dev(sino), w.angles, w.axis, nx, ny, scale=0.7).cpu().numpy()
    finally:
        lib.set_backproject_variant(prev)
    assert_parity(got, want, "backproject run16, %d slices" % S)


def test_backproject_affine_rows(lib):
    """K1 on the device: rows linear in the bin index back-project to scale * sum_p(alpha + beta t)."""
    rng = np.random.default_rng(11)
    S, P, B, nx, ny, h = 2, 23, 400, 140, 100, 1.0
    angles = np.sort(rng.uniform(0, math.pi, P))
    axis = (B - 1) / 2 + rng.uniform(-1, 1, P)
    alpha = np.round(rng.normal(size=(S, P)) * 64) / 64
    beta = np.round(rng.normal(size=(S, P)) * 64) / 1024
    sino = (alpha[..., None] + beta[..., None] * np.arange(B)).astype(np.float32)
    j = np.arange(nx) - (nx - 1) / 2
    i = np.arange(ny) - (ny - 1) / 2
    t = axis[:, None, None] + h * (j[None, None, :] * np.cos(angles)[:, None, None]
                                   + i[None, :, None] * np.sin(angles)[:, None, None])
    assert t.min() >= 0 and t.max() <= B - 1
    want = np.einsum("sp,pij->sij", alpha, np.ones_like(t)) + np.einsum("sp,pij->sij", beta, t)
    got = lib.backproject(_dev(sino), angles, axis, nx, ny, pixel_size=h).cpu().numpy()
    assert_parity(got, want, "affine rows")


# ------------------------------------------------------------------------------ forward projection
FP_CASES = [
    (1, 1, 40, 33, 21, 1.0, None, 0.0),
    (5, 45, 300, 260, 270, 1.0, None, 1.0),     # several bin segments, bands and chunks, ragged slice group
    (2, 21, 150, 100, 90, 0.72, None, 0.5),     # 4 candidate pixels per line
    (1, 9, 400, 80, 60, 2.5, None, 0.0),        # detector much longer than the image: strips off the image
    (3, 37, 211, 150, 70, 1.0, None, 1.5),
    (2, 50, 97, 130, 131, 0.8, 30.2, 0.7),
    (2, 19, 64, 200, 90, 1.3, None, 0.0),
    (2, 24, 300, 64, 64, 0.5, None, 2.0),       # pixel smaller than a bin: > 3 pixels per line in a strip
]


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("case", FP_CASES)
def test_forward_project_matches_oracle(lib, oracle, case, variant):
    S, P, B, nx, ny, h, axis, drift = case
    wl = lib.workloads
    w = wl.custom(S, P, B, nx, ny, pixel_size=h, axis=axis, drift=drift, jitter_angles=0.01, seed=P,
                  span=2 * math.pi)
    x = wl.random_image(S, ny, nx, seed=nx)
    want = oracle.forward_project(x, w.angles, w.axis, B, pixel_size=h, scale=1.7)
    prev = lib.set_forward_project_variant(variant)
    try:
        try:
            got = lib.forward_project(_dev(x), w.angles, w.axis, B, pixel_size=h, scale=1.7).cpu().numpy()
        except RuntimeError as e:
            # variant 5 forces the diagonal-line kernel, which needs >= 1 bin per pixel along a diagonal
            if variant == 5 and h < 1.0 / math.sqrt(2.0) + 0.05 and "does not cover" in str(e):
                pytest.skip("diagonal-line kernel does not cover pixel_size %g" % h)
            raise
    finally:
        lib.set_forward_project_variant(prev)
    assert_parity(got, want, "forward_project variant %d %r" % (variant, case))


def test_forward_project_axis_aligned_angles(lib, oracle):
    """theta = 0, pi/2, pi, 3pi/2 exactly: the strip degenerates onto pixel rows / columns."""
    wl = lib.workloads
    S, B, nx, ny = 2, 90, 60, 50
    angles = np.array([0.0, math.pi / 2, math.pi, 1.5 * math.pi, math.pi / 4, 3 * math.pi / 4])
    axis = np.array([44.5, 44.5, 44.0, 45.25, 44.5, 44.5])
    x = wl.random_image(S, ny, nx, seed=3)
    want = oracle.forward_project(x, angles, axis, B)
    got = lib.forward_project(_dev(x), angles, axis, B).cpu().numpy()
    assert_parity(got, want, "forward_project axis-aligned")


def _fp_variant(lib, variant, *args, **kw):
    prev = lib.set_forward_project_variant(variant)
    try:
        return lib.forward_project(*args, **kw).cpu().numpy()
    finally:
        lib.set_forward_project_variant(prev)


@pytest.mark.parametrize("S", [3, 5, 8, 13, 16, 18])
def test_forward_project_diag_slice_counts(lib, oracle, S):
    """The diagonal-line interval kernel takes 1, 2 or 4 slice groups per block (4, 8, 16 slices per thread);
    ragged stacks leave spare zero groups."""
    wl = lib.workloads
    P, B, nx, ny = 40, 140, 120, 100
    w = wl.custom(S, P, B, nx, ny, drift=1.0, jitter_angles=0.01, seed=S, span=2 * math.pi)
    x = wl.random_image(S, ny, nx, seed=S)
    want = oracle.forward_project(x, w.angles, w.axis, B)
    got = _fp_variant(lib, 5, _dev(x), w.angles, w.axis, B)
    assert lib.last_forward_project_kernel() == 5
    assert_parity(got, want, "forward_project diag, %d slices" % S)


def test_forward_project_diag_special_angles(lib, oracle):
    """Angles on and next to the image axes (left to the banded kernel below 2^-12 bins per pixel of slack),
    the diagonals (largest step, skew boundary) and both detector directions, with an integer-aligned geometry:
    odd image sizes and an integer axis put pixels exactly on interval boundaries (each must be counted once)."""
    wl = lib.workloads
    S, B, nx, ny = 4, 131, 101, 91
    eps = [0.0, 1e-6, 1e-4, 2.4e-4, 2.5e-4, 1e-3, -1e-6, -1e-4, -1e-3]
    angles = np.array([q * math.pi / 2 + e for q in range(4) for e in eps] +
                      [q * math.pi / 4 + e for q in (1, 3, 5, 7) for e in (0.0, 1e-9, -1e-9, 1e-3)] +
                      list(np.linspace(0.0, 2 * math.pi, 37, endpoint=False) + 0.0123))
    axis = np.full(angles.size, 65.0)
    x = wl.random_image(S, ny, nx, seed=5)
    want = oracle.forward_project(x, angles, axis, B)
    for variant in (0, 5):
        got = _fp_variant(lib, variant, _dev(x), angles, axis, B)
        assert_parity(got, want, "forward_project special angles, variant %d" % variant)
    # a constant image: every bin of a projection that sees the whole image carries the same mass as the oracle's
    ones = np.ones((1, ny, nx), dtype=np.float32)
    got = _fp_variant(lib, 5, _dev(ones), angles, axis, B)
    want1 = oracle.forward_project(ones, angles, axis, B)
    assert_parity(got, want1, "forward_project of ones (partition of the pixels)")
    np.testing.assert_allclose(got.sum(axis=2), want1.sum(axis=2), rtol=2e-6)
    assert (np.abs(want1.sum(axis=2) - nx * ny) < 1e-6 * nx * ny).sum() >= 40    # K2: whole image on the detector


def test_forward_project_diag_sparse_angles_and_wide_detector(lib, oracle):
    """Few projections far apart (chunks of one or two projections; windows that do not fit go to the banded
    kernel), a detector much wider than the image (blocks whose strips miss the image write zeros) and a
    pixel size above one bin."""
    wl = lib.workloads
    for (S, P, B, nx, ny, h) in [(8, 7, 700, 300, 260, 1.0), (2, 12, 900, 200, 220, 1.7), (8, 3, 64, 400, 400, 1.0)]:
        w = wl.custom(S, P, B, nx, ny, pixel_size=h, drift=2.0, jitter_angles=0.3, seed=P + S)
        x = wl.random_image(S, ny, nx, seed=P)
        want = oracle.forward_project(x, w.angles, w.axis, B, pixel_size=h)
        got = _fp_variant(lib, 5, _dev(x), w.angles, w.axis, B, pixel_size=h)
        assert_parity(got, want, "forward_project diag sparse %r" % ((S, P, B, nx, ny, h),))


def test_forward_project_kernels_agree(lib):
    """Banded, interval and diagonal-line kernels compute the same sums in different orders: FP32 rounding apart."""
    wl = lib.workloads
    S, P, B, nx, ny = 16, 96, 300, 256, 256
    w = wl.custom(S, P, B, nx, ny, drift=1.0, jitter_angles=0.002, seed=9)
    x = _dev(wl.random_image(S, ny, nx, seed=9))
    ref = _fp_variant(lib, 2, x, w.angles, w.axis, B)
    for variant in (0, 4, 5):
        got = _fp_variant(lib, variant, x, w.angles, w.axis, B)
        assert_parity(got, ref, "forward_project variant %d vs banded" % variant, rel=3e-6, mabs=3e-5)


def _fuzz_geometry(rng):
    """A random small scan: slice counts around the group sizes, random / regular / near-special angle lists, random
    pixel sizes, integer-aligned geometries (pixels exactly on bin centres and interval boundaries)."""
    S = int(rng.choice([1, 2, 4, 5, 8, 9, 12, 13, 16, 17]))
    nx, ny = int(rng.integers(20, 180)), int(rng.integers(20, 180))
    B, NP = int(rng.integers(16, 300)), int(rng.integers(1, 70))
    h = float(rng.choice([1.0, 1.0, 1.0, rng.uniform(0.72, 2.5)]))
    kind = int(rng.integers(0, 3))
    if kind == 0:
        ang = np.sort(rng.uniform(0, 2 * math.pi, NP))
    elif kind == 1:
        ang = np.arange(NP) * math.pi / NP
    else:
        base = rng.choice([0, math.pi / 4, math.pi / 2, 3 * math.pi / 4, math.pi, 1.5 * math.pi], NP)
        ang = base + rng.choice([0, 1e-9, 1e-6, 1e-4, 2.44e-4, 1e-3, -1e-7, -1e-4], NP)
    if rng.random() < 0.3:
        nx |= 1
        ny |= 1
        axis = np.full(NP, float(rng.integers(0, B)))
    else:
        axis = rng.uniform(-5, B + 5) + rng.uniform(-2, 2, NP)
    return S, NP, B, nx, ny, h, ang, axis


def test_projector_pair_fuzz(lib, oracle):
    """40 seeded random scans through the automatic kernel choices of both projectors and through the forced
    diagonal-line forward kernel (400 such cases were run once while it was written: worst rel-L2 3e-6)."""
    rng = np.random.default_rng(20241105)
    for case in range(40):
        S, NP, B, nx, ny, h, ang, axis = _fuzz_geometry(rng)
        x = rng.normal(size=(S, ny, nx)).astype(np.float32)
        want = oracle.forward_project(x, ang, axis, B, pixel_size=h)
        for variant in (0, 5):
            prev = lib.set_forward_project_variant(variant)
            try:
                got = lib.forward_project(_dev(x), ang, axis, B, pixel_size=h).cpu().numpy()
            finally:
                lib.set_forward_project_variant(prev)
            assert_parity(got, want, "fuzz case %d forward variant %d %r" % (case, variant, (S, NP, B, nx, ny, h)))
        q = rng.normal(size=(S, NP, B)).astype(np.float32)
        assert_parity(lib.backproject(_dev(q), ang, axis, nx, ny, pixel_size=h).cpu().numpy(),
                      oracle.backproject(q, ang, axis, nx, ny, pixel_size=h),
                      "fuzz case %d backproject %r" % (case, (S, NP, B, nx, ny, h)))


@pytest.mark.parametrize("B,axis", [(260, None), (120, 75.3)])
def test_adjoint_identity_on_device(lib, B, axis):
    """K3 in FP32: |<P x, y> - <x, P^T y>| <= 1e-5 ||P x|| ||y||."""
    import torch
    wl = lib.workloads
    S, P, nx, ny = 3, 61, 170, 150
    w = wl.custom(S, P, B, nx, ny, axis=axis, drift=1.0, jitter_angles=0.02)
    x = _dev(wl.random_image(S, ny, nx, seed=1))
    y = _dev(wl.random_sinogram(S, P, B, seed=2))
    Px = lib.forward_project(x, w.angles, w.axis, B)
    Pty = lib.backproject(y, w.angles, w.axis, nx, ny)
    lhs = torch.dot(Px.double().ravel(), y.double().ravel()).item()
    rhs = torch.dot(x.double().ravel(), Pty.double().ravel()).item()
    bound = 1e-5 * Px.double().norm().item() * y.double().norm().item()
    assert abs(lhs - rhs) <= bound, (lhs, rhs, bound)


def test_pitched_sinograms(lib, oracle):
    """pyhst_geom_t.sino_pitch: rows of the sinogram stack further apart than n_bins (a view of a wider stack), for the
    input of pyhst_backproject / pyhst_fbp and the output of pyhst_forward_project (every forward kernel); the gap
    between the rows is neither read nor written."""
    import torch
    wl = lib.workloads
    S, P, B, nx, ny, pitch = 6, 33, 150, 120, 110, 164
    w = wl.custom(S, P, B, nx, ny, drift=1.0, jitter_angles=0.01, seed=4, span=2 * math.pi)
    sino = wl.random_sinogram(S, P, B, seed=4)
    wide = torch.full((S, P, pitch), float("nan"), dtype=torch.float32, device="cuda")
    wide[:, :, :B] = torch.from_numpy(sino).cuda()
    view = wide[:, :, :B]
    assert not view.is_contiguous()
    assert_parity(lib.backproject(view, w.angles, w.axis, nx, ny).cpu().numpy(),
                  oracle.backproject(sino, w.angles, w.axis, nx, ny), "backproject, pitched rows")
    assert_parity(lib.fbp(view, w.angles, w.axis, nx, ny, filter=1).cpu().numpy(),
                  oracle.fbp(sino, w.angles, w.axis, nx, ny, filter=1), "fbp, pitched rows")
    x = wl.random_image(S, ny, nx, seed=4)
    want = oracle.forward_project(x, w.angles, w.axis, B)
    for variant in (0, 1, 2, 4, 5):
        out = torch.full((S, P, pitch), -7.0, dtype=torch.float32, device="cuda")
        prev = lib.set_forward_project_variant(variant)
        try:
            lib.forward_project(_dev(x), w.angles, w.axis, B, out=out[:, :, :B])
        finally:
            lib.set_forward_project_variant(prev)
        assert_parity(out[:, :, :B].cpu().numpy(), want, "forward_project variant %d, pitched rows" % variant)
        assert (out[:, :, B:] == -7.0).all().item(), "variant %d wrote between the rows" % variant


# ------------------------------------------------------------------------------ ramp filter
@pytest.mark.parametrize("f", [0, 1, 2, 3])
@pytest.mark.parametrize("b_in,b_out,pad,weights", [(367, 367, 0, False), (128, 256, 0, True),
                                                    (100, 192, 92, True), (64, 64, 0, False),
                                                    (2048, 2048, 0, False)])
def test_ramp_filter_matches_oracle(lib, oracle, f, b_in, b_out, pad, weights):
    rng = np.random.default_rng(b_in + f)
    rows = rng.normal(size=(7, b_in)).astype(np.float32)
    w = rng.uniform(0, 1, b_in).astype(np.float32) if weights else None
    want = oracle.ramp_filter(rows, n_bins_out=b_out, pad_left=pad, filter=f, col_weights=w)
    got = lib.ramp_filter(_dev(rows), n_bins_out=b_out, pad_left=pad, filter=f,
                          col_weights=None if w is None else _dev(w)).cpu().numpy()
    assert_parity(got, want, "ramp_filter")


def test_ramp_filter_zero_rows_is_a_noop(lib):
    import torch
    out = lib.ramp_filter(torch.empty((0, 64), dtype=torch.float32, device="cuda"))
    assert out.shape == (0, 64)


# ------------------------------------------------------------------------------ FBP, the five configs
def test_fbp_config1_full(lib, oracle):
    w = lib.workloads.config(1)
    sino = w.sinogram()
    want = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    got = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode).cpu().numpy()
    assert_parity(got, want, "fbp cfg1")
    # host-buffer entry point: same result through chunked copies
    got_h = lib.fbp_host(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    assert np.array_equal(got_h, got)


@pytest.mark.parametrize("cfg,shrink,n_slices", [(2, 8, 6), (3, 8, 4), (4, 4, 3), (5, 8, 9)])
def test_fbp_shrunken_configs(lib, oracle, cfg, shrink, n_slices):
    """Configs 2-5 with every length divided by `shrink` (same structure: drift, half acquisition,
    noise model), whole images compared."""
    w = lib.workloads.config(cfg, shrink=shrink, n_slices=n_slices)
    sino = w.sinogram()
    want = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    got = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode).cpu().numpy()
    assert_parity(got, want, "fbp cfg%d/%d" % (cfg, shrink))
    got_h = lib.fbp_host(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode,
                         max_slices_per_chunk=4)
    # the host pipeline works on chunks of 4 slices, which run the 4-slice backprojector (other run
    # length than the 8-slice kernel the whole stack gets): equal to FP32 rounding, and to the oracle
    assert np.abs(got_h - got).max() <= 2e-5 * np.abs(got).max()
    assert_parity(got_h, want, "fbp_host cfg%d/%d" % (cfg, shrink))


def _sample_points(rng, n, slices, ny, nx):
    pts = np.stack([rng.choice(slices, n), rng.integers(0, ny, n), rng.integers(0, nx, n)], axis=1)
    corners = [(slices[0], 0, 0), (slices[0], ny - 1, nx - 1), (slices[-1], 0, nx - 1), (slices[-1], ny - 1, 0),
               (slices[0], ny // 2, nx // 2)]
    return np.concatenate([pts, np.array(corners)], axis=0).astype(np.int32)


def test_projector_pair_config4_full(lib, oracle):
    """Config 4 (iterative): the pair P, P^T at full size on sampled rows / pixels + the K3 identity."""
    import torch
    w = lib.workloads.config(4)
    rng = np.random.default_rng(4)
    y0 = w.sinogram()
    x0 = lib.fbp(_dev(y0), w.angles, w.axis, w.nx, w.ny).contiguous()
    x0h = x0.cpu().numpy()
    Px = lib.forward_project(x0, w.angles, w.axis, w.n_bins)
    rows = np.stack([rng.integers(0, w.n_slices, 24), rng.integers(0, w.n_angles, 24)], axis=1)
    want = oracle.forward_project_rows(x0h, w.angles, w.axis, w.n_bins, rows)
    assert_parity(Px.cpu().numpy()[rows[:, 0], rows[:, 1]], want, "forward_project cfg4 rows")
    Pty = lib.backproject(_dev(y0), w.angles, w.axis, w.nx, w.ny)
    pts = _sample_points(rng, 2000, [0, w.n_slices - 1], w.ny, w.nx)
    want = oracle.backproject_points(y0, w.angles, w.axis, w.nx, w.ny, pts)
    assert_parity(Pty.cpu().numpy()[pts[:, 0], pts[:, 1], pts[:, 2]], want, "backproject cfg4 points")
    yd = _dev(y0)
    lhs = torch.dot(Px.double().ravel(), yd.double().ravel()).item()
    rhs = torch.dot(x0.double().ravel(), Pty.double().ravel()).item()
    assert abs(lhs - rhs) <= 1e-5 * Px.double().norm().item() * yd.double().norm().item()


# ------------------------------------------------------------------------------ errors
def test_invalid_arguments_are_rejected(lib):
    import torch
    wl = lib.workloads
    w = wl.custom(1, 8, 32, 16, 16)
    sino = _dev(wl.random_sinogram(1, 8, 32))
    with pytest.raises(lib.PyhstError):
        lib.backproject(sino, w.angles, w.axis, 16, 16, pixel_size=0.0)
    bad = w.angles.copy()
    bad[3] = np.nan
    with pytest.raises(lib.PyhstError):
        lib.backproject(sino, bad, w.axis, 16, 16)
    with pytest.raises(lib.PyhstError):
        lib.ramp_filter(sino.reshape(8, 32), n_bins_out=16)
    with pytest.raises(lib.PyhstError):
        lib.fbp(sino, w.angles, w.axis, 16, 16, filter=7)
    with pytest.raises(lib.PyhstError):
        lib.backproject(sino.double(), w.angles, w.axis, 16, 16)
    assert "filter" in lib.last_error() or lib.last_error() != ""
    out = torch.full((1, 16, 16), 5.0, device="cuda")
    with pytest.raises(lib.PyhstError):
        lib.backproject(sino, w.angles, w.axis, 16, 16, pixel_size=-1.0, out=out)
    assert (out == 5.0).all()          # nothing written on error


# ------------------------------------------------------------------------------ N1: TV-FISTA
# FP32 iterates drift from the double oracle as rounding accumulates through the iterations
# (SURVEY.md sec. 8(f) N1): energy within 1e-4 relative, image within 1e-3 relative L2.
FISTA_REL_ENERGY = 1e-4
FISTA_REL_L2 = 1e-3


@pytest.mark.gpu
@pytest.mark.parametrize("beta,n_iter,n_inner", [(0.0, 12, 0), (0.5, 15, 20), (3.0, 10, 7)])
def test_fista_tv_matches_oracle(lib, oracle, beta, n_iter, n_inner):
    w = lib.workloads.config(4, shrink=8, n_slices=3)          # 128^2, 25 projections x 128 bins
    data = w.sinogram()
    L_want = oracle.lipschitz(w.angles, w.axis, w.n_bins, w.nx, w.ny, n_power=8)
    want, e_want = oracle.fista_tv(data, w.angles, w.axis, w.nx, w.ny, beta, L_want, n_iter, n_inner=n_inner)
    got, e_got, L_got = lib.fista_tv(_dev(data), w.angles, w.axis, w.nx, w.ny, beta, n_iter, n_inner=n_inner,
                                     n_power=8)
    assert abs(L_got - L_want) <= 1e-5 * L_want
    np.testing.assert_allclose(e_got, e_want, rtol=FISTA_REL_ENERGY)
    assert_parity(got.cpu().numpy(), want, "fista_tv beta=%g" % beta, rel=FISTA_REL_L2, mabs=5e-3)


@pytest.mark.gpu
def test_fista_tv_ragged_shapes_and_arguments(lib, oracle):
    wl = lib.workloads
    w = wl.custom(2, 21, 75, 50, 37, pixel_size=1.0, axis=None, drift=0.5, jitter_angles=0.01, seed=5)
    data = wl.random_sinogram(2, 21, 75, seed=3)
    L = oracle.lipschitz(w.angles, w.axis, 75, 50, 37, n_power=5)
    want, e_want = oracle.fista_tv(data, w.angles, w.axis, 50, 37, 0.2, L, 6, n_inner=5)
    got, e_got, L_got = lib.fista_tv(_dev(data), w.angles, w.axis, 50, 37, 0.2, 6, n_inner=5, n_power=5)
    np.testing.assert_allclose(e_got, e_want, rtol=FISTA_REL_ENERGY)
    assert_parity(got.cpu().numpy(), want, "fista_tv ragged", rel=FISTA_REL_L2, mabs=5e-3)
    # n_iter = 0: x = 0, nothing else touched
    got0, e0, _ = lib.fista_tv(_dev(data), w.angles, w.axis, 50, 37, 0.2, 0)
    assert e0.size == 0 and float(got0.abs().max()) == 0.0
    with pytest.raises(lib.binding.PyhstError):
        lib.fista_tv(_dev(data), w.angles, w.axis, 50, 37, -1.0, 3)
    with pytest.raises(lib.binding.PyhstError):
        lib.fista_tv(_dev(data), w.angles, w.axis, 50, 37, 0.1, 3, n_power=0)


@pytest.mark.gpu
def test_fista_tv_config4_full_size(lib, oracle):
    """BASELINE.json configs[3] at full size (8 x 1024^2, 200 x 1024) in the launch configuration
    bench.py --config 4 times: the first iterations against the oracle on one slice (the oracle
    needs seconds per projector pair), the 100-iteration run via properties that hold at any size."""
    w = lib.workloads.config(4)
    data = w.sinogram()
    d_data = _dev(data)
    s0 = 3
    L_want = oracle.lipschitz(w.angles, w.axis, w.n_bins, w.nx, w.ny, n_power=8)
    want, e_want = oracle.fista_tv(data[s0:s0 + 1], w.angles, w.axis, w.nx, w.ny, 0.01, L_want, 2, n_inner=3)
    got, _, L_got = lib.fista_tv(d_data, w.angles, w.axis, w.nx, w.ny, 0.01, 2, n_inner=3, n_power=8)
    assert abs(L_got - L_want) <= 1e-5 * L_want
    assert_parity(got[s0:s0 + 1].cpu().numpy(), want, "fista_tv config 4, 2 iterations", rel=FISTA_REL_L2,
                  mabs=5e-3)
    _, e1, _ = lib.fista_tv(d_data[s0:s0 + 1].contiguous(), w.angles, w.axis, w.nx, w.ny, 0.01, 2, n_inner=3)
    np.testing.assert_allclose(e1, e_want, rtol=FISTA_REL_ENERGY)
    # 100 iterations, lambda = 0.01, 20 dual steps (the bench configuration)
    x, e, _ = lib.fista_tv(d_data, w.angles, w.axis, w.nx, w.ny, 0.01, 100, n_inner=20, n_power=8)
    x = x.cpu().numpy()
    assert np.isfinite(x).all() and np.isfinite(e).all()
    half = 0.5 * float(np.sum(data.astype(np.float64) ** 2))
    assert e[0] == pytest.approx(half, rel=1e-6)              # y0 = 0: eq. 3 = 1/2 ||data||^2
    assert e[-1] < 1e-3 * e[0] and e[-1] <= e[10] <= e[1]     # FISTA is not monotone, but it descends
    # the reconstruction explains the data: P x close to data (relative residual of the noisy scan)
    px = lib.forward_project(_dev(x), w.angles, w.axis, w.n_bins).cpu().numpy()
    rel = np.linalg.norm((px - data).ravel()) / np.linalg.norm(data.ravel())
    assert rel < 0.05
    assert 2.0 * e[-1] >= (rel * np.linalg.norm(data.ravel())) ** 2 * 0.5   # energy >= its data term (y_99 ~ x)


@pytest.mark.gpu
@pytest.mark.parametrize("f", [2, 3])
def test_fbp_windowed_ramps(lib, oracle, f):
    """N2: Hann / Hamming windows through the whole FBP (config 2 shrunk, drift, Poisson noise)."""
    w = lib.workloads.config(2, shrink=8, n_slices=5)
    sino = w.sinogram()
    want = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=f, mode=w.mode)
    got = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=f, mode=w.mode).cpu().numpy()
    assert_parity(got, want, "fbp filter %d" % f)


@pytest.mark.gpu
def test_halfacq_stitched_equals_general_path(lib, oracle):
    """N2: the folded 180-degree path of PYHST_SCAN_360_HALF against the general path (all P rows)
    and the oracle; a scan that does not pair up (odd P, drifting axis) takes the general path."""
    w = lib.workloads.config(3, shrink=8, n_slices=5)          # c = 237.5: 2c integer, P = 500
    sino = w.sinogram()
    want = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    got = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode).cpu().numpy()
    prev = lib.set_halfacq_stitch(False)
    try:
        gen = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode).cpu().numpy()
    finally:
        lib.set_halfacq_stitch(prev)
    assert_parity(got, want, "fbp half acquisition, stitched")
    assert_parity(gen, want, "fbp half acquisition, general")
    assert np.abs(got - gen).max() <= 2e-5 * np.abs(gen).max()
    assert not np.array_equal(got, gen)                         # the two paths really differ
    # unpaired scans: odd number of projections, and an axis that is not a half-integer
    for P, axis in ((101, 50.5), (100, 50.3)):
        ang = np.arange(P) * 2 * math.pi / P
        ax = np.full(P, axis)
        raw = lib.workloads.random_sinogram(2, P, 64, seed=P)
        nxy = 100
        want2 = oracle.fbp(raw, ang, ax, nxy, nxy, mode=lib.SCAN_360_HALF)
        got2 = lib.fbp(_dev(raw), ang, ax, nxy, nxy, mode=lib.SCAN_360_HALF).cpu().numpy()
        assert_parity(got2, want2, "fbp half acquisition, unpaired P=%d" % P)
    # paired, axis left of the detector centre (pad_left > 0) and integer axis
    P = 60
    ang = np.arange(P) * 2 * math.pi / P
    ax = np.full(P, 9.0)
    raw = lib.workloads.random_sinogram(3, P, 64, seed=1)
    want3 = oracle.fbp(raw, ang, ax, 110, 108, mode=lib.SCAN_360_HALF)
    got3 = lib.fbp(_dev(raw), ang, ax, 110, 108, mode=lib.SCAN_360_HALF).cpu().numpy()
    assert_parity(got3, want3, "fbp half acquisition, stitched, axis on the left")


# ------------------------------------------------------------------------------ library state
@pytest.mark.gpu
def test_calls_on_two_streams_are_serialised(lib, oracle):
    """include/pyhst.h, concurrency rule: all calls of a device share one workspace; calls on
    different streams are ordered on the device by the library (cudaStreamWaitEvent), so two
    streams that alternate between two shapes -- which regrow / reuse the same QI and FFT
    blocks -- still give the serial results."""
    import torch
    wl = lib.workloads
    wa = wl.config(2, shrink=8, n_slices=6)            # 256^2, 250 projections
    wb = wl.custom(9, 90, 300, 200, 170, drift=1.0, seed=4)
    sa, sb = _dev(wa.sinogram()), _dev(wl.random_sinogram(9, 90, 300, seed=9))
    ref_a = lib.fbp(sa, wa.angles, wa.axis, wa.nx, wa.ny, filter=wa.filter)
    ref_b = lib.fbp(sb, wb.angles, wb.axis, 200, 170)
    ref_p = lib.forward_project(ref_b, wb.angles, wb.axis, 300)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    out_a = [torch.empty_like(ref_a) for _ in range(4)]
    out_b = [torch.empty_like(ref_b) for _ in range(4)]
    out_p = [torch.empty_like(ref_p) for _ in range(4)]
    for k in range(4):                                  # no host synchronisation in between
        lib.fbp(sa, wa.angles, wa.axis, wa.nx, wa.ny, filter=wa.filter, out=out_a[k], stream=s1)
        lib.fbp(sb, wb.angles, wb.axis, 200, 170, out=out_b[k], stream=s2)
        lib.forward_project(ref_b, wb.angles, wb.axis, 300, out=out_p[k], stream=s1)
    torch.cuda.synchronize()
    for k in range(4):
        assert torch.equal(out_a[k], ref_a) and torch.equal(out_b[k], ref_b) and torch.equal(out_p[k], ref_p)
    assert_parity(ref_a.cpu().numpy(), oracle.fbp(wa.sinogram(), wa.angles, wa.axis, wa.nx, wa.ny, filter=wa.filter),
                  "fbp (serial reference of the two-stream test)")


@pytest.mark.gpu
def test_forward_projector_pads_survive_a_released_cache(lib, oracle):
    """The banded forward projector relies on zero pads around its interleaved image copy and writes
    them only once per block: after pyhst_release_cache() (or a regrown workspace) the block may come
    back at the same address holding anything, and must be zeroed again."""
    import torch
    wl = lib.workloads
    w = wl.custom(4, 40, 200, 150, 140, drift=1.0, seed=8)
    x = _dev(wl.random_image(4, 140, 150, seed=2))
    want = oracle.forward_project(x.cpu().numpy(), w.angles, w.axis, 200)
    got = lib.forward_project(x, w.angles, w.axis, 200)
    assert_parity(got.cpu().numpy(), want, "forward_project before release")
    for _ in range(3):
        lib.release_cache()
        junk = [torch.full((1 << 22,), float("nan"), device="cuda") for _ in range(8)]   # dirty the freed blocks
        del junk
        torch.cuda.empty_cache()
        got = lib.forward_project(x, w.angles, w.axis, 200)
        assert_parity(got.cpu().numpy(), want, "forward_project after release_cache")


@pytest.mark.gpu
def test_large_pixel_size_falls_back_to_the_reference_kernel(lib, oracle):
    """pixel_size ~ 6: the staged window of the tiled kernels would exceed shared memory; the
    automatic pick must take the one-thread-per-pixel kernel instead of failing."""
    wl = lib.workloads
    w = wl.custom(2, 24, 700, 90, 80, pixel_size=6.0, drift=0.5, seed=6)
    sino = wl.random_sinogram(2, 24, 700, seed=6)
    want = oracle.backproject(sino, w.angles, w.axis, 90, 80, pixel_size=6.0)
    got = lib.backproject(_dev(sino), w.angles, w.axis, 90, 80, pixel_size=6.0).cpu().numpy()
    assert_parity(got, want, "backproject pixel_size 6")
    x = wl.random_image(2, 80, 90, seed=6)
    wantp = oracle.forward_project(x, w.angles, w.axis, 700, pixel_size=6.0)
    gotp = lib.forward_project(_dev(x), w.angles, w.axis, 700, pixel_size=6.0).cpu().numpy()
    assert_parity(gotp, wantp, "forward_project pixel_size 6")


# ------------------------------------------------------------------------------ N2: cosine window
@pytest.mark.gpu
def test_cosine_window_filter_and_fbp(lib, oracle):
    rng = np.random.default_rng(44)
    rows = rng.normal(size=(5, 300)).astype(np.float32)
    want = oracle.ramp_filter(rows, n_bins_out=340, pad_left=17, filter=oracle.FILTER_COSINE)
    got = lib.ramp_filter(_dev(rows), n_bins_out=340, pad_left=17, filter=lib.FILTER_COSINE).cpu().numpy()
    assert_parity(got, want, "ramp_filter cosine")
    w = lib.workloads.config(2, shrink=8, n_slices=5)
    sino = w.sinogram()
    want = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=oracle.FILTER_COSINE, mode=w.mode)
    got = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=lib.FILTER_COSINE, mode=w.mode).cpu().numpy()
    assert_parity(got, want, "fbp cosine window")


# ------------------------------------------------------------------------------ N1: ISTA switch
@pytest.mark.gpu
def test_ista_tv_matches_oracle_and_descends(lib, oracle):
    w = lib.workloads.config(4, shrink=8, n_slices=3)
    data = w.sinogram()
    L = oracle.lipschitz(w.angles, w.axis, w.n_bins, w.nx, w.ny, n_power=8)
    want, e_want = oracle.ista_tv(data, w.angles, w.axis, w.nx, w.ny, 0.5, L, 15, n_inner=20)
    got, e_got, L_got = lib.ista_tv(_dev(data), w.angles, w.axis, w.nx, w.ny, 0.5, 15, n_inner=20, n_power=8)
    assert abs(L_got - L) <= 1e-5 * L
    np.testing.assert_allclose(e_got, e_want, rtol=FISTA_REL_ENERGY)
    assert_parity(got.cpu().numpy(), want, "ista_tv", rel=FISTA_REL_L2, mabs=5e-3)
    # the energy of eq. 3 does not increase under ISTA (inexact prox: to rounding)
    _, e_long, _ = lib.ista_tv(_dev(data), w.angles, w.axis, w.nx, w.ny, 0.5, 60, n_inner=40, n_power=8)
    assert np.all(np.diff(e_long) <= 1e-5 * e_long[0])
    # two runs are bit-identical (deterministic reductions)
    got2, e2, L2 = lib.ista_tv(_dev(data), w.angles, w.axis, w.nx, w.ny, 0.5, 15, n_inner=20, n_power=8)
    assert L2 == L_got and np.array_equal(e2, e_got) and bool((got2 == got).all())


# ------------------------------------------------------------------------------ N4
@pytest.mark.gpu
@pytest.mark.parametrize("S,P,B,r,with_model", [(1, 1, 40, 1, False), (3, 50, 211, 4, True), (2, 333, 1000, 15, False),
                                                (5, 64, 2048, 9, True)])
def test_ring_filter_matches_oracle(lib, oracle, S, P, B, r, with_model):
    rng = np.random.default_rng(S * 1000 + B)
    sino = (rng.normal(size=(S, P, B)) + 0.5 * rng.normal(size=(S, 1, B))).astype(np.float32)   # per-bin errors
    model = rng.normal(size=(S, P, B)).astype(np.float32) if with_model else None
    want = oracle.ring_filter(sino, r, model=model)
    got = lib.ring_filter(_dev(sino), r, model=None if model is None else _dev(model)).cpu().numpy()
    assert_parity(got, want, "ring_filter")
    d = _dev(sino)
    lib.ring_filter(d, r, model=None if model is None else _dev(model), out=d)                   # in place
    assert np.array_equal(d.cpu().numpy(), got)
    with pytest.raises(lib.PyhstError):
        lib.ring_filter(_dev(sino), 0)


@pytest.mark.gpu
def test_ring_filter_removes_rings_from_a_reconstruction(lib, oracle):
    """End to end: per-bin detector errors give rings in the FBP; the filter removes most of them."""
    w = lib.workloads.config(2, shrink=8, n_slices=2)
    clean = w.sinogram()
    rng = np.random.default_rng(61)
    err = np.zeros(w.n_bins, dtype=np.float32)
    err[rng.choice(w.n_bins, 12, replace=False)] = rng.choice([-0.05, 0.05], 12).astype(np.float32)
    dirty = clean + err[None, None, :]
    rec = lambda s: lib.fbp(s, w.angles, w.axis, w.nx, w.ny, filter=w.filter).cpu().numpy()
    r_clean, r_dirty = rec(_dev(clean)), rec(_dev(dirty))
    r_fixed = rec(lib.ring_filter(_dev(dirty), 3))
    e_dirty = np.linalg.norm(r_dirty - r_clean)
    e_fixed = np.linalg.norm(r_fixed - r_clean)
    assert e_fixed < 0.45 * e_dirty


@pytest.mark.gpu
def test_ecohe_and_cv_distance_match_oracle(lib, oracle):
    wl = lib.workloads
    rng = np.random.default_rng(62)
    a = rng.normal(size=(3, 201, 187)).astype(np.float32)
    b = (a + 0.3 * rng.normal(size=a.shape)).astype(np.float32)
    want = oracle.ecohe(a, b)
    got = lib.ecohe(_dev(a), _dev(b))
    np.testing.assert_allclose(got, want, rtol=1e-12, atol=1e-14)
    assert lib.ecohe(_dev(a), _dev(a)).tolist() == [0.0, 0.0, 0.0]
    assert np.array_equal(lib.ecohe(_dev(a), _dev(b)), got)                # deterministic
    # cross-validation: leave two projections out of a config-4-like scan
    w = wl.config(4, shrink=8, n_slices=2)
    data = w.sinogram()
    excl = [7, 19]
    keep = [p for p in range(w.n_angles) if p not in excl]
    x, _, _ = lib.fista_tv(_dev(np.ascontiguousarray(data[:, keep])), w.angles[keep], w.axis[keep], w.nx, w.ny,
                           0.05, 30, n_inner=10)
    d_excl = np.ascontiguousarray(data[:, excl])
    want = oracle.cv_distance(x.cpu().numpy(), d_excl, w.angles[excl], w.axis[excl])
    got = lib.cv_distance(x, _dev(d_excl), w.angles[excl], w.axis[excl])
    np.testing.assert_allclose(got, want, rtol=2e-5)
    # estimator curve: E_cohe between a weakly and a strongly regularised reconstruction is finite and in [-1, 1]
    x0, _, _ = lib.fista_tv(_dev(np.ascontiguousarray(data[:, keep])), w.angles[keep], w.axis[keep], w.nx, w.ny,
                            1e-4, 30, n_inner=10)
    e = lib.ecohe(x, x0)
    assert np.all(np.abs(e) <= 1.0) and np.all(np.isfinite(e))
    np.testing.assert_allclose(e, oracle.ecohe(x.cpu().numpy(), x0.cpu().numpy()), rtol=1e-10, atol=1e-13)


# ------------------------------------------------------------------------------ N3: overlapping patches
PATCH_REL_L2 = REL_L2    # north_star's bar also for Algorithm 1's gradient (measured <= 2.8e-6)


@pytest.mark.gpu
@pytest.mark.parametrize("ny,nx,m,st,n_atoms,rho", [(64, 64, 8, 4, 128, 0.5), (70, 93, 8, 3, 100, 1.5),
                                                    (40, 52, 4, 4, 16, 0.0), (33, 47, 6, 5, 40, 0.2)])
def test_patch_gradient_matches_oracle(lib, oracle, ny, nx, m, st, n_atoms, rho):
    """Algorithm 1 on the device against the oracle: X (eq. 7), f (eq. 8), G (eq. 9);
    ragged grids (last patch pulled back), non-overlapping patches, two slices."""
    wl = lib.workloads
    P, B = 25, int(1.5 * max(nx, ny)) | 1
    w = wl.custom(2, P, B, nx, ny, drift=0.7, jitter_angles=0.01, seed=m + st)
    data = wl.random_sinogram(2, P, B, seed=ny)
    D = wl.dct_dictionary(m, n_atoms, seed=1)
    na, nb = oracle.patch_grid(ny, nx, m, st)
    assert lib.patch_grid(ny, nx, m, st) == (na, nb)
    rng = np.random.default_rng(nx)
    W = (rng.normal(size=(2, na * nb, n_atoms)) * (rng.uniform(size=(2, na * nb, n_atoms)) < 0.2)).astype(np.float32)
    G, X, f = lib.patch_gradient(_dev(W), _dev(D), _dev(data), w.angles, w.axis, nx, ny, m, st, rho)
    f_want = 0.0
    for s in range(2):
        Gw, Xw, fw = oracle.patch_gradient(W[s].astype(np.float64), D.astype(np.float64), data[s], w.angles, w.axis,
                                           nx, ny, m, st, rho)
        assert_parity(X[s].cpu().numpy(), Xw, "patch X slice %d" % s)
        assert_parity(G[s].cpu().numpy(), Gw, "patch G slice %d" % s, rel=PATCH_REL_L2, mabs=MAX_ABS)
        f_want += fw
    assert f == pytest.approx(f_want, rel=1e-5)


@pytest.mark.gpu
def test_patch_fista_matches_oracle(lib, oracle):
    """FISTA on the coefficients (R23, R24): Lipschitz estimate, energies and iterates against the oracle
    on a reduced-projection scan (few projections + noise), 8 x 8 patches, stride 4,
    2x over-complete dictionary; then the long run descends and sparsifies."""
    wl = lib.workloads
    w = wl.config(4, shrink=16, n_slices=2)                  # 64^2, 12 projections x 64 bins
    data = w.sinogram()
    m, st, n_atoms, rho, beta = 8, 4, 128, 0.3, 0.05
    D = wl.dct_dictionary(m, n_atoms)
    Lw = oracle.patch_lipschitz(D.astype(np.float64), w.angles, w.axis, w.n_bins, w.nx, w.ny, m, st, rho, n_power=6)
    Wg, Xg, eg, Lg = lib.patch_fista(_dev(D), _dev(data), w.angles, w.axis, w.nx, w.ny, m, st, rho, beta, 12, n_power=6)
    assert abs(Lg - Lw) <= 2e-5 * Lw
    e_want = np.zeros(12)
    for s in range(2):
        Ww, Xw, ew = oracle.patch_fista(D.astype(np.float64), data[s], w.angles, w.axis, w.nx, w.ny, m, st, rho, beta,
                                        Lw, 12)
        e_want += ew
        assert_parity(Xg[s].cpu().numpy(), Xw, "patch FISTA image, slice %d" % s, rel=1e-3, mabs=5e-3)
        assert_parity(Wg[s].cpu().numpy(), Ww, "patch FISTA coefficients, slice %d" % s, rel=2e-3, mabs=1e-2)
    np.testing.assert_allclose(eg, e_want, rtol=1e-4)
    Wl, Xl, el, _ = lib.patch_fista(_dev(D), _dev(data), w.angles, w.axis, w.nx, w.ny, m, st, rho, beta, 150, n_power=6)
    assert el[-1] < 0.2 * el[0] and np.isfinite(el).all()
    frac_zero = float((Wl == 0).float().mean())
    assert frac_zero > 0.5                                   # the L1 term switches most coefficients off
    with pytest.raises(lib.PyhstError):
        lib.patch_gradient(Wl, _dev(D), _dev(data), w.angles, w.axis, w.nx, w.ny, m, 9, rho)   # stride > m


# ------------------------------------------------------------------------------ N2: fused FFT filter
@pytest.mark.gpu
@pytest.mark.parametrize("f", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("b_in,b_out,pad,weights,rows", [(367, 367, 0, False, 7), (128, 256, 0, True, 4),
                                                         (100, 192, 92, True, 9), (20, 20, 0, False, 1),
                                                         (2048, 2048, 0, False, 6), (2048, 3840, 0, True, 5),
                                                         (2560, 2560, 0, False, 3), (4096, 4096, 0, False, 2)])
def test_fused_ramp_filter_matches_oracle_and_cufft_path(lib, oracle, f, b_in, b_out, pad, weights, rows):
    """N2: the fused shared-memory FFT kernel (FFT lengths 64 .. 8192, every radix schedule 8..8 [4|2]) against
    the oracle's direct convolution and against the cuFFT path."""
    rng = np.random.default_rng(b_in + 7 * f)
    x = rng.normal(size=(rows, b_in)).astype(np.float32)
    w = rng.uniform(0, 1, b_in).astype(np.float32) if weights else None
    want = oracle.ramp_filter(x, n_bins_out=b_out, pad_left=pad, filter=f, col_weights=w)
    dw = None if w is None else _dev(w)
    prev = lib.set_filter_variant(2)
    try:
        got = lib.ramp_filter(_dev(x), n_bins_out=b_out, pad_left=pad, filter=f, col_weights=dw).cpu().numpy()
        lib.set_filter_variant(1)
        ref = lib.ramp_filter(_dev(x), n_bins_out=b_out, pad_left=pad, filter=f, col_weights=dw).cpu().numpy()
    finally:
        lib.set_filter_variant(prev)
    assert_parity(got, want, "fused ramp filter")
    assert_parity(ref, want, "cuFFT ramp filter")


@pytest.mark.gpu
def test_fbp_through_both_filter_paths(lib, oracle):
    """pyhst_fbp writes the interleaved layout straight from the filter: both filter paths, ragged slice
    group, reversed rows (360-degree angles), half acquisition (weights + extension)."""
    for cfg, shrink, n_slices in ((2, 8, 6), (3, 8, 3), (5, 8, 5)):
        w = lib.workloads.config(cfg, shrink=shrink, n_slices=n_slices)
        sino = w.sinogram()
        want = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
        for variant in (1, 2):
            prev = lib.set_filter_variant(variant)
            try:
                got = lib.fbp(_dev(sino), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode).cpu().numpy()
            finally:
                lib.set_filter_variant(prev)
            assert_parity(got, want, "fbp cfg%d, filter variant %d" % (cfg, variant))
    with pytest.raises(lib.PyhstError):
        prev = lib.set_filter_variant(2)
        try:
            lib.ramp_filter(_dev(np.zeros((2, 5000), dtype=np.float32)))        # M would be 16384
        finally:
            lib.set_filter_variant(prev)


@pytest.mark.gpu
@pytest.mark.parametrize("m,st,n_atoms", [(8, 4, 128), (8, 8, 64), (16, 9, 64), (8, 5, 256)])
def test_patch_gradient_tensor_core_gemm(lib, oracle, m, st, n_atoms):
    """The tcgen05 3xTF32 GEMM (pyhst_test.h variant 2) against the oracle and against the FP32 SIMT GEMM:
    ragged last tile of patches (N not a multiple of 128), K = 32 .. 256, N = 16 .. 256, two slices."""
    wl = lib.workloads
    ny, nx = 77, 102
    P, B = 21, 155
    w = wl.custom(2, P, B, nx, ny, drift=0.5, jitter_angles=0.01, seed=m + n_atoms)
    data = wl.random_sinogram(2, P, B, seed=n_atoms)
    D = wl.dct_dictionary(m, n_atoms, seed=2)
    na, nb = oracle.patch_grid(ny, nx, m, st)
    rng = np.random.default_rng(n_atoms)
    W = rng.normal(size=(2, na * nb, n_atoms)).astype(np.float32)
    out = {}
    for variant in (1, 2):
        prev = lib.set_patch_gemm_variant(variant)
        try:
            out[variant] = lib.patch_gradient(_dev(W), _dev(D), _dev(data), w.angles, w.axis, nx, ny, m, st, 0.8)
        finally:
            lib.set_patch_gemm_variant(prev)
    for s in range(2):
        Gw, Xw, fw = oracle.patch_gradient(W[s].astype(np.float64), D.astype(np.float64), data[s], w.angles, w.axis,
                                           nx, ny, m, st, 0.8)
        for variant in (1, 2):
            G, X, f = out[variant]
            assert_parity(X[s].cpu().numpy(), Xw, "patch X, GEMM variant %d" % variant)
            assert_parity(G[s].cpu().numpy(), Gw, "patch G, GEMM variant %d" % variant, rel=PATCH_REL_L2, mabs=MAX_ABS)
    assert not np.array_equal(out[1][0].cpu().numpy(), out[2][0].cpu().numpy())    # the two kernels really differ


# ------------------------------------------------------------------------------ workspace handling
def _dense_scan(S, n, P, B, seed):
    rng = np.random.default_rng(seed)
    angles = np.arange(P) * (math.pi / P)
    axis = (B - 1) / 2.0 + rng.uniform(-1.5, 1.5, size=P)
    x = rng.normal(size=(S, n, n)).astype(np.float32)
    return x, angles, axis


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [0, 2, 5])
def test_forward_project_smaller_stack_after_larger_one(lib, oracle, variant):
    """A stack of fewer slice groups than the one before it (the last chunk of a host pipeline) is laid out
    inside the workspace block that was zeroed for the larger stack and does not clear it again: results must
    be the same as from a freshly cleared block, bit for bit, for the sheared (diagonal-line) and the
    line-interleaved (banded) layouts, and whichever of the two the automatic choice takes."""
    n, P, B = 160, 360, 240
    big, angles, axis = _dense_scan(12, n, P, B, seed=5)
    small = _dense_scan(5, n, P, B, seed=6)[0]
    prev = lib.set_forward_project_variant(variant)
    try:
        fp = lambda x: lib.forward_project(_dev(x), angles, axis, B).cpu().numpy()
        lib.release_cache()
        ref_small = fp(small)                      # block sized and cleared for 2 slice groups
        assert_parity(ref_small, oracle.forward_project(small, angles, axis, B), "forward_project, 5 slices")
        lib.release_cache()
        ref_two = fp(small[:2])                    # one slice group (the automatic choice may differ per group count)
        lib.release_cache()
        ref_big = fp(big)                          # block sized and cleared for 3 slice groups
        assert np.array_equal(fp(small), ref_small)    # laid out as the 3-group stack, pads found zero
        assert np.array_equal(fp(big), ref_big)
        assert np.array_equal(fp(small[:2]), ref_two)
        assert np.array_equal(fp(big), ref_big)
    finally:
        lib.set_forward_project_variant(prev)


@pytest.mark.gpu
def test_forward_project_falls_back_to_banded_kernel_without_room_for_the_sheared_copies(lib, oracle):
    """Automatic kernel choice: when the block for the two sheared image copies (about 4.8x the stack) cannot be
    allocated, the call runs on the banded kernel (about 2x) instead of failing with NOMEM."""
    n, P, B = 512, 360, 512
    x, angles, axis = _dense_scan(8, n, P, B, seed=7)
    lib.release_cache()
    ref = lib.forward_project(_dev(x), angles, axis, B).cpu().numpy()
    assert lib.last_forward_project_kernel() == 5          # the diagonal-line kernel is the automatic choice here
    xd_bytes = 2 * 2 * (n + n + 7) * (n + 392) * 16         # pyhst.h: two copies, 2 slice groups
    lib.release_cache()
    prev_limit = lib.set_test_workspace_limit(xd_bytes - 1)
    try:
        got = lib.forward_project(_dev(x), angles, axis, B).cpu().numpy()
        assert lib.last_forward_project_kernel() == 2
        assert_parity(got, ref.astype(np.float64), "forward_project on the banded kernel vs the diagonal-line kernel")
        rows = [0, 89, 90, 91, 180, 359]
        want = oracle.forward_project(x[:1], angles[rows], axis[rows], B)
        assert_parity(got[:1, rows], want, "forward_project fall-back vs oracle")
        prev = lib.set_forward_project_variant(5)          # forced: no fall-back, the error is reported
        try:
            with pytest.raises(lib.PyhstError, match="refused"):
                lib.forward_project(_dev(x), angles, axis, B)
        finally:
            lib.set_forward_project_variant(prev)
    finally:
        lib.set_test_workspace_limit(prev_limit)
        lib.release_cache()
    assert np.array_equal(lib.forward_project(_dev(x), angles, axis, B).cpu().numpy(), ref)
    assert lib.last_forward_project_kernel() == 5
