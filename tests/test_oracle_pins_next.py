"""Pins of the oracle functions of the NEXT rows built in round 2 -- CPU only.

N2  cosine-windowed ramp (reading R8)                                 K6c
N1  ISTA switch                                        K20, K21
N4  ring filter (L61, reading R21), E_cohe (eq. 11), cross-validation K25-K27
N3  overlapping patches (L102-L145, eq. 4-9, Algorithm 1; R22-R24)    K28-K32
Each pin fixes a function against something other than itself: closed forms typed from the
paper's formulas, numpy's FFT / dense linear algebra on matrices built entry by entry in the
tests, finite differences of eq. 8 written out in numpy, optimality conditions.
"""
import math

import numpy as np
import pytest

from test_oracle_pins import _dense_matrix
from test_oracle_pins_fista import _tiny_problem, _tv_numpy


@pytest.fixture(autouse=True)
def _one_thread(oracle):
    with oracle.threads(1):
        yield


# --------------------------------------------------------------------------- K6c: cosine window
def test_k6c_cosine_windowed_ramp(oracle):
    """R8 / N2: spectrum |w| cos(pi w), w in cycles per bin.  h_c[0] = int |w| cos(pi w) dw =
    1/pi - 2/pi^2 (integration by parts); h_c[n] from the half-bin shifts of the continuous
    band-limited ramp; even; sums to H(0) = 0."""
    h = oracle.ramp_kernel(oracle.FILTER_COSINE, np.arange(-4, 5))
    assert h[4] == pytest.approx(1 / math.pi - 2 / math.pi ** 2, rel=1e-14)
    # n = 1: (h(1/2) + h(3/2)) / 2, h(1/2) = 1/pi - 2/pi^2, h(3/2) = -1/(3 pi) - 2/(9 pi^2)
    want1 = 0.5 * ((1 / math.pi - 2 / math.pi ** 2) + (-1 / (3 * math.pi) - 2 / (9 * math.pi ** 2)))
    assert h[5] == pytest.approx(want1, rel=1e-13)
    np.testing.assert_array_equal(h, h[::-1])
    M = 4096
    lag = np.fft.fftfreq(M, 1.0 / M).astype(np.int64)
    w = np.fft.fftfreq(M)
    H = np.fft.fft(oracle.ramp_kernel(oracle.FILTER_COSINE, lag)).real
    assert np.abs(H - np.abs(w) * np.cos(math.pi * w)).max() < 3.0 / M
    assert abs(oracle.ramp_kernel(oracle.FILTER_COSINE, np.arange(-20000, 20001)).sum()) < 1e-5
    # numerical quadrature of the defining integral at a few lags
    from scipy import integrate
    for n in (0, 1, 2, 7):
        val = integrate.quad(lambda x: 2 * x * math.cos(math.pi * x) * math.cos(2 * math.pi * x * n), 0, 0.5,
                             epsabs=1e-14)[0]
        assert oracle.ramp_kernel(oracle.FILTER_COSINE, [n])[0] == pytest.approx(val, abs=1e-12)
    q = np.zeros((1, 21), dtype=np.float32)
    q[0, 8] = 1.0
    g = oracle.ramp_filter(q, n_bins_out=30, pad_left=3, filter=oracle.FILTER_COSINE)[0]
    np.testing.assert_allclose(g, oracle.ramp_kernel(oracle.FILTER_COSINE, np.arange(30) - 3 - 8), atol=1e-16)


# --------------------------------------------------------------------------- K20, K21: ISTA
def test_k20_ista_iterates_against_the_dense_matrix(oracle):
    """beta = 0: ISTA is the Landweber iteration x_{k+1} = x_k - A^T (A x_k - d) / L (no momentum)."""
    rng, angles, axis, A, P, B, n = _tiny_problem(20)
    d = rng.normal(size=(1, P, B)).astype(np.float32)
    dv = d.astype(np.float64).ravel()
    L = 1.3 * np.linalg.eigvalsh(A.T @ A)[-1]
    x = np.zeros(n * n)
    want_e = []
    for k in range(4):
        want_e.append(0.5 * np.sum((A @ x - dv) ** 2))
        x = x - A.T @ (A @ x - dv) / L
    got, e = oracle.ista_tv(d, angles, axis, n, n, 0.0, L, 4, n_inner=3)
    np.testing.assert_allclose(got.ravel(), x, rtol=0, atol=1e-12 * np.abs(x).max() * 50)
    np.testing.assert_allclose(e, want_e, rtol=1e-12)
    # FISTA differs from the third iterate on (the first two coincide: t0 = 1)
    xf2, _ = oracle.fista_tv(d, angles, axis, n, n, 0.0, L, 2)
    xi2, _ = oracle.ista_tv(d, angles, axis, n, n, 0.0, L, 2)
    np.testing.assert_array_equal(xf2, xi2)
    xf3, _ = oracle.fista_tv(d, angles, axis, n, n, 0.0, L, 3)
    assert np.abs(xf3.ravel() - oracle.ista_tv(d, angles, axis, n, n, 0.0, L, 3)[0].ravel()).max() > 1e-6


def test_k21_ista_energy_is_monotone_and_reaches_the_fista_minimum(oracle):
    """the energy of eq. 3 does not increase under ISTA (exact prox, L >= lambda_max);
    FISTA is not monotone but reaches the same minimum sooner."""
    rng, angles, axis, A, P, B, n = _tiny_problem(21, P=7, B=25, n=12)
    xs = np.zeros((n, n))
    xs[2:9, 4:10] = 1.0
    clean = A @ xs.ravel()
    d = (clean + 0.2 * rng.normal(size=clean.shape)).reshape(1, P, B).astype(np.float32)
    dv = d.astype(np.float64).ravel()
    L = oracle.lipschitz(angles, axis, B, n, n)
    beta = 0.4
    xi, ei = oracle.ista_tv(d, angles, axis, n, n, beta, L, 400, n_inner=300)
    assert np.all(np.diff(ei) <= 1e-9 * ei[0])
    # the displayed energy is eq. 3 at the iterate: recompute the last one with the dense A and numpy TV
    xi399, _ = oracle.ista_tv(d, angles, axis, n, n, beta, L, 399, n_inner=300)
    f = 0.5 * np.sum((A @ xi399.ravel() - dv) ** 2) + beta * _tv_numpy(xi399)
    assert ei[-1] == pytest.approx(f, rel=1e-10)
    xf, ef = oracle.fista_tv(d, angles, axis, n, n, beta, L, 400, n_inner=300)
    Fi = 0.5 * np.sum((A @ xi.ravel() - dv) ** 2) + beta * _tv_numpy(xi)
    Ff = 0.5 * np.sum((A @ xf.ravel() - dv) ** 2) + beta * _tv_numpy(xf)
    assert abs(Ff - Fi) <= 1e-6 * Fi                     # both have reached the minimum of eq. 3
    assert ef[40] < ei[40]                               # the accelerated scheme is ahead


# --------------------------------------------------------------------------- K25: ring filter
def test_k25_ring_filter_closed_forms(oracle):
    """R21 typed out.  A constant sinogram plus an isolated per-bin error a at b0, window 2r+1:
    mean m = c + a delta; moving average of the spike = a/(2r+1) on |b - b0| <= r; so the filter
    subtracts a (1 - 1/(2r+1)) at b0 and adds a/(2r+1) to its 2r neighbours, in every row."""
    S, P, B, r, b0, a, c = 2, 7, 40, 3, 17, 0.9, 1.25
    q = np.full((S, P, B), c, dtype=np.float32)
    q[0, :, b0] += np.float32(a)
    out = oracle.ring_filter(q, r)
    a = float(np.float32(c) + np.float32(a)) - c          # the value that was really stored
    want = np.full((P, B), c)
    want[:, b0] = c + a - a * (1 - 1.0 / (2 * r + 1))
    want[:, b0 - r:b0] += a / (2 * r + 1)
    want[:, b0 + 1:b0 + r + 1] += a / (2 * r + 1)
    np.testing.assert_allclose(out[0], want, rtol=0, atol=1e-14)
    np.testing.assert_allclose(out[1], c, rtol=0, atol=1e-14)          # slices are independent
    # clipped window at the detector edge: error at bin 0 is averaged over bins 0..r only
    q = np.zeros((1, 3, 12), dtype=np.float32)
    q[0, :, 0] = 1.0
    out = oracle.ring_filter(q, 2)[0]
    lp = np.zeros(12)
    lp[0], lp[1], lp[2] = 1 / 3, 1 / 4, 1 / 5
    np.testing.assert_allclose(out, np.tile(np.r_[1.0, np.zeros(11)] - (np.r_[1.0, np.zeros(11)] - lp), (3, 1)),
                               atol=1e-15)
    # a signal that varies with the angle but has zero angular mean is untouched; a linear trend in
    # the mean is untouched away from the edges (the moving average reproduces affine functions)
    rng = np.random.default_rng(25)
    z = rng.normal(size=(1, 8, 30))
    z -= z.mean(axis=1, keepdims=True)
    trend = (0.3 * np.arange(30) - 2.0)[None, None, :]
    q = (z + trend).astype(np.float32)
    out = oracle.ring_filter(q, 4)[0]
    np.testing.assert_allclose(out[:, 4:-4], q[0].astype(np.float64)[:, 4:-4], atol=2e-6)
    # the model (thresholded bone) is removed before the high-pass: a sharp feature
    # that the model explains is not mistaken for a ring
    bone = np.zeros((1, 5, 30), dtype=np.float32)
    bone[0, :, 12] = 3.0
    q = (np.ones((1, 5, 30)) + bone).astype(np.float32)
    np.testing.assert_allclose(oracle.ring_filter(q, 2, model=bone)[0], q[0], atol=1e-14)
    assert np.abs(oracle.ring_filter(q, 2)[0] - q[0]).max() > 1.0
    with pytest.raises(ValueError):
        oracle.ring_filter(q, 0)


# --------------------------------------------------------------------------- K26: E_cohe
def test_k26_ecohe_closed_forms(oracle):
    """eq. 11: Cos(a - b, a).  (3,4) vs (3,0): a-b = (0,4), cos = 16 / (4 * 5) = 0.8."""
    a = np.array([[3.0, 4.0], [1.0, 0.0], [2.0, 2.0], [1.0, 2.0]], dtype=np.float32)
    b = np.array([[3.0, 0.0], [1.0, 5.0], [0.0, 0.0], [2.0, 4.0]], dtype=np.float32)
    e = oracle.ecohe(a, b)
    assert e[0] == pytest.approx(0.8, abs=1e-15)
    assert e[1] == pytest.approx(0.0, abs=1e-15)          # a - b = (0,-5) is orthogonal to a
    assert e[2] == pytest.approx(1.0, abs=1e-15)          # I(0+) = 0: the difference is I(beta) itself
    assert e[3] == pytest.approx(-1.0, abs=1e-15)         # b = 2a: a - b = -a
    rng = np.random.default_rng(26)
    x, y = rng.normal(size=(1, 7, 9)).astype(np.float32), rng.normal(size=(1, 7, 9)).astype(np.float32)
    e1 = oracle.ecohe(x, y)[0]
    assert oracle.ecohe(4 * x, 4 * y)[0] == pytest.approx(e1, rel=1e-13)      # scale invariant
    assert abs(e1) <= 1.0
    assert oracle.ecohe(x, x)[0] == 0.0                   # zero difference: defined as 0


# --------------------------------------------------------------------------- K27: cross-validation
def test_k27_cv_distance_against_the_dense_matrix(oracle):
    rng, angles, axis, A, P, B, n = _tiny_problem(27, P=9, B=25, n=10)
    x = rng.normal(size=(2, n, n)).astype(np.float32)
    excl = [2, 7]
    data = rng.normal(size=(2, len(excl), B)).astype(np.float32)
    A3 = A.reshape(P, B, n * n)
    want = [sum(np.sum((A3[p] @ x[s].astype(np.float64).ravel() - data[s, e]) ** 2) for e, p in enumerate(excl))
            for s in range(2)]
    got = oracle.cv_distance(x, data, angles[excl], axis[excl])
    np.testing.assert_allclose(got, want, rtol=1e-12)
    exact = np.stack([np.stack([A3[p] @ x[s].astype(np.float64).ravel() for p in excl]) for s in range(2)])
    assert np.all(oracle.cv_distance(x, exact.astype(np.float32), angles[excl], axis[excl]) < 1e-10)


# --------------------------------------------------------------------------- K28-K32: overlapping patches
def _patch_setup(seed, ny=10, nx=12, m=4, st=2, n_atoms=20, P=8, B=21):
    rng = np.random.default_rng(seed)
    angles = np.sort(rng.uniform(0, math.pi, size=P))
    axis = (B - 1) / 2.0 + rng.uniform(-0.5, 0.5, size=P)
    A = _dense_matrix(angles, axis, nx, ny, B, 1.0)
    D = rng.normal(size=(n_atoms, m * m))
    D /= np.linalg.norm(D, axis=1, keepdims=True)
    return rng, angles, axis, A, D


def _origins(n, m, st):
    """R22 typed out: origins 0, st, 2 st, ... with the last one pulled back to n - m."""
    o = list(range(0, n - m, st)) + [n - m]
    return o


def _compose_numpy(Pm, ny, nx, m, st):
    """eq. 7 + eq. 6 typed out: every pixel takes the value of the patch with the L1-closest centre."""
    oy, ox = _origins(ny, m, st), _origins(nx, m, st)
    half = (m - 1) / 2.0
    X = np.zeros((ny, nx))
    for iy in range(ny):
        for ix in range(nx):
            best, bp = None, None
            for a, y0 in enumerate(oy):
                for b, x0 in enumerate(ox):
                    dist = abs(iy - (y0 + half)) + abs(ix - (x0 + half))
                    if best is None or dist < best - 1e-12:
                        best, bp = dist, (a, b)
            a, b = bp
            X[iy, ix] = Pm[a * len(ox) + b].reshape(m, m)[iy - oy[a], ix - ox[b]]
    return X


def _f_numpy(W, D, dv, A, ny, nx, m, st, rho):
    """eq. 8 typed out."""
    Pm = W @ D
    X = _compose_numpy(Pm, ny, nx, m, st)
    oy, ox = _origins(ny, m, st), _origins(nx, m, st)
    sim = 0.0
    for a, y0 in enumerate(oy):
        for b, x0 in enumerate(ox):
            sim += np.sum((X[y0:y0 + m, x0:x0 + m] - Pm[a * len(ox) + b].reshape(m, m)) ** 2)
    return np.sum((dv - A @ X.ravel()) ** 2) + rho * sim, X


@pytest.mark.parametrize("ny,nx,m,st", [(10, 12, 4, 2), (11, 9, 4, 3), (8, 8, 4, 4), (9, 10, 3, 1)])
def test_k28_patch_maps(oracle, ny, nx, m, st):
    """eq. 4-6: the patches cover the image, the cores partition it, each core pixel lies in its
    patch and no other patch centre is closer in the L1 norm."""
    na, nb = oracle.patch_grid(ny, nx, m, st)
    oy, ox = _origins(ny, m, st), _origins(nx, m, st)
    assert (na, nb) == (len(oy), len(ox))
    core, cover = oracle.patch_maps(ny, nx, m, st)
    ind = np.zeros((na * nb, ny, nx), dtype=int)
    for a, y0 in enumerate(oy):
        for b, x0 in enumerate(ox):
            ind[a * nb + b, y0:y0 + m, x0:x0 + m] = 1
    np.testing.assert_array_equal(cover, ind.sum(axis=0))
    assert cover.min() >= 1                                            # eq. 4
    half = (m - 1) / 2.0
    for iy in range(ny):
        for ix in range(nx):
            p = core[iy, ix]
            assert ind[p, iy, ix] == 1                                 # eq. 5: core inside the patch
            d = [abs(iy - (oy[q // nb] + half)) + abs(ix - (ox[q % nb] + half)) for q in range(na * nb)]
            assert d[p] == min(d) and p == int(np.argmin(d))           # eq. 6, smallest index among equals


def test_k29_gemm_and_composition(oracle):
    """P = W D and eq. 7 against numpy (X returned by the gradient routine)."""
    ny, nx, m, st = 10, 12, 4, 2
    rng, angles, axis, A, D = _patch_setup(29)
    na, nb = oracle.patch_grid(ny, nx, m, st)
    W = rng.normal(size=(na * nb, D.shape[0]))
    data = rng.normal(size=(len(angles), 21)).astype(np.float32)
    G, X, f = oracle.patch_gradient(W, D, data, angles, axis, nx, ny, m, st, 0.7)
    np.testing.assert_allclose(X, _compose_numpy(W @ D, ny, nx, m, st), rtol=0, atol=1e-13)
    fn, _ = _f_numpy(W, D, data.astype(np.float64).ravel(), A, ny, nx, m, st, 0.7)
    assert f == pytest.approx(fn, rel=1e-12)


@pytest.mark.parametrize("ny,nx,m,st,rho", [(10, 12, 4, 2, 0.7), (9, 9, 4, 3, 0.0), (8, 11, 3, 2, 2.5)])
def test_k30_gradient_is_the_derivative_of_eq8(oracle, ny, nx, m, st, rho):
    """Algorithm 1 / eq. 9 against central finite differences of eq. 8 written out in numpy with the
    dense projector (f is quadratic: central differences are exact up to rounding)."""
    rng, angles, axis, A, D = _patch_setup(30 + ny, ny=ny, nx=nx, m=m)
    na, nb = oracle.patch_grid(ny, nx, m, st)
    W = rng.normal(size=(na * nb, D.shape[0]))
    data = rng.normal(size=(len(angles), 21)).astype(np.float32)
    dv = data.astype(np.float64).ravel()
    G, _, _ = oracle.patch_gradient(W, D, data, angles, axis, nx, ny, m, st, rho)
    eps = 1e-3
    idx = [(int(rng.integers(0, W.shape[0])), int(rng.integers(0, W.shape[1]))) for _ in range(25)]
    idx += [(0, 0), (W.shape[0] - 1, W.shape[1] - 1), (nb - 1, 3), ((na - 1) * nb, 5)]   # corner patches
    for p, k in idx:
        Wp, Wm = W.copy(), W.copy()
        Wp[p, k] += eps
        Wm[p, k] -= eps
        fd = (_f_numpy(Wp, D, dv, A, ny, nx, m, st, rho)[0] - _f_numpy(Wm, D, dv, A, ny, nx, m, st, rho)[0]) / (2 * eps)
        assert G[p, k] == pytest.approx(fd, rel=1e-7, abs=1e-7 * np.abs(G).max())


def test_k31_soft_threshold(oracle):
    v = np.array([-3.0, -0.5, 0.0, 0.2, 0.5, 0.5000001, 7.25])
    np.testing.assert_allclose(oracle.soft_threshold(v, 0.5), [-2.5, 0.0, 0.0, 0.0, 0.0, 1e-7, 6.75], atol=1e-15)
    np.testing.assert_array_equal(oracle.soft_threshold(v, 0.0), v)


def test_k32_patch_fista(oracle):
    """First iterate by hand, the Lipschitz estimate against the dense Hessian, the energy printed,
    and the optimality conditions of min f(w) + beta ||w||_1 at convergence:
    |grad_k| <= beta where w_k = 0, grad_k = -beta sign(w_k) elsewhere."""
    ny, nx, m, st, rho, beta = 8, 8, 4, 2, 0.5, 0.3
    rng, angles, axis, A, D = _patch_setup(32, ny=ny, nx=nx, n_atoms=18, P=6, B=15)
    na, nb = oracle.patch_grid(ny, nx, m, st)
    N, Nc = na * nb, D.shape[0]
    xs = np.zeros((ny, nx))
    xs[2:6, 3:7] = 1.0
    data = (A @ xs.ravel() + 0.05 * rng.normal(size=A.shape[0])).reshape(6, 15).astype(np.float32)
    dv = data.astype(np.float64).ravel()
    # dense Hessian from the (pinned) gradient: H e_k = grad f(e_k) - grad f(0)
    zero = np.zeros((N, Nc))
    g0 = oracle.patch_gradient(zero, D, data, angles, axis, nx, ny, m, st, rho)[0].ravel()
    H = np.zeros((N * Nc, N * Nc))
    for k in range(N * Nc):
        e = np.zeros(N * Nc)
        e[k] = 1.0
        H[:, k] = oracle.patch_gradient(e.reshape(N, Nc), D, data, angles, axis, nx, ny, m, st, rho)[0].ravel() - g0
    np.testing.assert_allclose(H, H.T, atol=1e-10 * np.abs(H).max())
    lam = np.linalg.eigvalsh(0.5 * (H + H.T))[-1]
    Lw = oracle.patch_lipschitz(D, angles, axis, 15, nx, ny, m, st, rho, n_power=12)
    assert lam <= Lw <= 1.1 * lam * (1 + 1e-12)
    # first iterate: w1 = shrink(-grad f(0) / Lw, beta / Lw); energy[0] = f(0) = ||y||^2
    W1, _, e1 = oracle.patch_fista(D, data, angles, axis, nx, ny, m, st, rho, beta, Lw, 1)
    v = -g0 / Lw
    want = np.sign(v) * np.maximum(np.abs(v) - beta / Lw, 0.0)
    np.testing.assert_allclose(W1.ravel(), want, atol=1e-14)
    assert e1[0] == pytest.approx(np.sum(dv ** 2), rel=1e-13)
    # convergence: KKT of the lasso
    Wc, Xc, ec = oracle.patch_fista(D, data, angles, axis, nx, ny, m, st, rho, beta, Lw, 3000)
    g = oracle.patch_gradient(Wc, D, data, angles, axis, nx, ny, m, st, rho)[0]
    on = np.abs(Wc) > 1e-9
    assert on.sum() > 5 and (~on).sum() > 5
    assert np.abs(g[on] + beta * np.sign(Wc[on])).max() < 2e-4
    assert np.abs(g[~on]).max() <= beta * (1 + 1e-3)
    F = _f_numpy(Wc, D, dv, A, ny, nx, m, st, rho)[0] + beta * np.abs(Wc).sum()
    assert ec[-1] == pytest.approx(F, rel=1e-6) and ec[-1] < ec[0]
    np.testing.assert_allclose(Xc, _compose_numpy(Wc @ D, ny, nx, m, st), atol=1e-12)
    for k in range(10):                                   # convex: no perturbation does better
        dW = rng.normal(size=Wc.shape) * 10.0 ** rng.uniform(-4, -1)
        assert _f_numpy(Wc + dW, D, dv, A, ny, nx, m, st, rho)[0] + beta * np.abs(Wc + dW).sum() >= F - 1e-9
