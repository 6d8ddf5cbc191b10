"""GPU-vs-oracle parity at BASELINE.json's own sizes, in the launch configurations bench.py times.

north_star: "FBP and projector outputs matching the oracle within the stated tolerances on all
five configs".  Config 1 is compared whole in test_cuda_parity.py.  Here:
  * pyhst_forward_project at configs 2, 3 and 5 (default kernel, default chunking, every slice of the
    config resident): >= 64 whole detector rows per config against oracle.forward_project_rows,
    including the first / last projection and the rows on both sides of every 45-degree walk-class
    switch, first and last slice group;
  * pyhst_fbp at configs 2 and 3: the first and the last slice of the stack compared WHOLE (every
    tile of the launch), config 5 with all 64 slices resident on sampled pixels of three slices;
  * pyhst_fbp_host / pyhst_forward_project_host on the 16-slice config-2 stack in 8-slice chunks (the
    e2e configuration of bench.py: two chunks through the three-stream pipeline);
  * pyhst_fista_tv on one config-4 slice, beta = 0.01, 100 iterations x 20 dual steps, at the bar
    SURVEY.md sec. 8(f) N1 states (energy 1e-4, image rel-L2 1e-3 after 100 iterations).
Inputs are synthesised on the device (same recipe as the parity cases; bench.py does the same) and
the very float32 arrays the kernels read are copied to the host for the oracle.
"""
import math

import numpy as np
import pytest

from test_cuda_parity import FISTA_REL_ENERGY, FISTA_REL_L2, _dev, _sample_points, assert_parity, lib  # noqa: F401

pytestmark = pytest.mark.gpu


def _device_sinogram(P, w, slices=None):
    prev = P.workloads.set_device("cuda")
    try:
        return w.sinogram_tensor(slices).contiguous()
    finally:
        P.workloads.set_device(prev)


@pytest.fixture(scope="module")
def cfg2(lib, oracle):
    """Config 2 at full size: device sinogram, device FBP, and the oracle's FBP of slices 0 and 15."""
    import torch
    w = lib.workloads.config(2)
    sino = _device_sinogram(lib, w)
    img = lib.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    torch.cuda.synchronize()
    check = [0, w.n_slices - 1]
    h_sub = sino[check].cpu().numpy()
    want = oracle.fbp(h_sub, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    return w, sino, img, check, want


def test_fbp_config2_whole_slices(lib, cfg2):
    w, sino, img, check, want = cfg2
    got = img[check].cpu().numpy()
    assert_parity(got, want, "fbp cfg2, slices 0 and 15 whole")


def test_host_entry_points_config2_eight_slice_chunks(lib, oracle, cfg2):
    """The e2e configuration of bench.py: *_host with max_slices_per_chunk = 8 on 16 slices."""
    import torch
    w, sino, img, check, want = cfg2
    h_sino = torch.empty(sino.shape, dtype=torch.float32, pin_memory=True)
    h_sino.copy_(sino)
    h_img = torch.empty(img.shape, dtype=torch.float32, pin_memory=True)
    lib.fbp_host(h_sino, w.angles, w.axis, w.nx, w.ny, w.pixel_size, filter=w.filter, mode=w.mode, out=h_img,
                 max_slices_per_chunk=8)
    got = h_img.numpy()
    assert_parity(got[check], want, "fbp_host cfg2, 8-slice chunks")
    assert np.array_equal(got, img.cpu().numpy())          # same kernels, same order: bit-identical
    h_proj = torch.empty((w.n_slices, w.n_angles, w.n_bins), dtype=torch.float32, pin_memory=True)
    lib.forward_project_host(h_img, w.angles, w.axis, w.n_bins, w.pixel_size, out=h_proj, max_slices_per_chunk=8)
    rows = _fp_rows(np.random.default_rng(28), w, [0, 7, 8, 15], 32)
    sl = sorted(set(rows[:, 0].tolist()))
    sub = got[sl]
    remap = np.stack([np.searchsorted(sl, rows[:, 0]), rows[:, 1]], axis=1)
    want_rows = oracle.forward_project_rows(sub, w.angles, w.axis, w.n_bins, remap, pixel_size=w.pixel_size)
    assert_parity(h_proj.numpy()[rows[:, 0], rows[:, 1]], want_rows, "forward_project_host cfg2 rows")


def _fp_rows(rng, w, slices, n_random):
    """(s, p) rows: first / last projection, both sides of every walk-class switch (|cos| = |sin|),
    and random ones, over the given slices."""
    ang = np.asarray(w.angles)
    c, s = np.abs(np.cos(ang)), np.abs(np.sin(ang))
    cls = c >= s
    switch = np.nonzero(cls[1:] != cls[:-1])[0]
    ps = {0, len(ang) - 1}
    for k in switch:
        ps.update((int(k), int(k) + 1))
    ps = sorted(ps)
    rows = [(slices[i % len(slices)], p) for i, p in enumerate(ps)]
    rows += [(int(rng.choice(slices)), int(rng.integers(0, len(ang)))) for _ in range(n_random)]
    return np.array(rows, dtype=np.int32)


@pytest.mark.parametrize("cfg", [2, 3, 5])
def test_forward_project_full_size_rows(lib, oracle, cfg, request):
    """pyhst_forward_project in the configuration bench.py times (config 2: fp_band_kernel, 16-projection
    chunks, 2048^2), and at configs 3 (3800^2, axis 1900: most pixels project off the detector) and 5 (all
    64 slices resident), on whole detector rows."""
    import torch
    if cfg == 2:
        w, sino, img, _, _ = request.getfixturevalue("cfg2")
    else:
        w = lib.workloads.config(cfg)
        sino = _device_sinogram(lib, w)
        img = lib.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
        del sino
    proj = lib.forward_project(img, w.angles, w.axis, w.n_bins, w.pixel_size)
    torch.cuda.synchronize()
    S = w.n_slices
    slices = sorted({0, 3, S - 4, S - 1} & set(range(S)))
    rows = _fp_rows(np.random.default_rng(100 + cfg), w, slices, 64)
    assert len(rows) >= 64
    sub = img[slices].cpu().numpy()
    remap = np.stack([np.searchsorted(slices, rows[:, 0]), rows[:, 1]], axis=1)
    want = oracle.forward_project_rows(sub, w.angles, w.axis, w.n_bins, remap, pixel_size=w.pixel_size)
    got = proj[torch.as_tensor(rows[:, 0].astype(np.int64), device="cuda"),
               torch.as_tensor(rows[:, 1].astype(np.int64), device="cuda")].cpu().numpy()
    assert_parity(got, want, "forward_project cfg%d full size, %d rows" % (cfg, len(rows)))
    # every row separately as well (a single wrong row must not hide in the stack norm)
    for k in range(len(rows)):
        assert_parity(got[k], want[k], "forward_project cfg%d row (s=%d, p=%d)" % (cfg, rows[k, 0], rows[k, 1]),
                      rel=2e-5)
    del proj, img
    torch.cuda.empty_cache()


def test_fbp_config3_whole_slices(lib, oracle):
    """Config 3 (360-degree half acquisition, 4 x 3800^2): first and last slice whole.  The default
    path folds facing projections (stitched); the oracle is the general definition (R10)."""
    w = lib.workloads.config(3)
    sino = _device_sinogram(lib, w)
    img = lib.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    check = [0, w.n_slices - 1]
    want = oracle.fbp(sino[check].cpu().numpy(), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    assert_parity(img[check].cpu().numpy(), want, "fbp cfg3, slices 0 and 3 whole")


def test_fbp_config5_all_slices_resident(lib, oracle):
    """Config 5 as bench.py --config 5 launches it: all 64 slices on the device (grid.z = 8)."""
    import torch
    w = lib.workloads.config(5)
    sino = _device_sinogram(lib, w)
    img = lib.fbp(sino, w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    torch.cuda.synchronize()
    check = [0, 37, w.n_slices - 1]
    pts = _sample_points(np.random.default_rng(5), 600, list(range(len(check))), w.ny, w.nx)
    want = oracle.fbp(sino[check].cpu().numpy(), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode, pts=pts)
    sub = img[check].cpu().numpy()
    assert_parity(sub[pts[:, 0], pts[:, 1], pts[:, 2]], want, "fbp cfg5, 64 slices resident (sampled)")
    # the other 61 slices: finite, and the same slice reconstructed alone in another group position agrees
    assert bool(torch.isfinite(img).all())
    alone = lib.fbp(sino[36:41].contiguous(), w.angles, w.axis, w.nx, w.ny, filter=w.filter, mode=w.mode)
    assert float((alone[1] - img[37]).abs().max()) <= 2e-5 * float(img[37].abs().max())
    del sino, img, alone
    torch.cuda.empty_cache()


def test_fista_tv_config4_one_slice_100_iterations(lib, oracle):
    """SURVEY.md sec. 8(f) N1's bar as stated: energy rel 1e-4, image rel-L2 1e-3 after 100 iterations
    (beta = 0.01, 20 dual steps), on one full-size config-4 slice."""
    w = lib.workloads.config(4, n_slices=1)
    data = w.sinogram()
    L = oracle.lipschitz(w.angles, w.axis, w.n_bins, w.nx, w.ny, n_power=8)
    want, e_want = oracle.fista_tv(data, w.angles, w.axis, w.nx, w.ny, 0.01, L, 100, n_inner=20)
    got, e_got, L_got = lib.fista_tv(_dev(data), w.angles, w.axis, w.nx, w.ny, 0.01, 100, n_inner=20, n_power=8)
    assert abs(L_got - L) <= 1e-5 * L
    np.testing.assert_allclose(e_got, e_want, rtol=FISTA_REL_ENERGY)
    assert_parity(got.cpu().numpy(), want, "fista_tv cfg4, 100 iterations", rel=FISTA_REL_L2, mabs=5e-3)
