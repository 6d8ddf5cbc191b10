"""Pins of the TV-FISTA oracle (NEXT row N1; eq. 1-3; readings R17-R20).

Each pin fixes an oracle function against something other than itself: closed forms of the
isotropic total variation, the exact solution of 1-D two-plateau TV denoising, optimality of the
proximal point against perturbations, a dense matrix built entry by entry in test_oracle_pins.py
(K4's routine) with numpy's symmetric eigensolver, and the O(1/k^2) FISTA bound of Beck & Teboulle.
"""
import math

import numpy as np
import pytest

from test_oracle_pins import _dense_matrix


@pytest.fixture(autouse=True)
def _one_thread(oracle):
    """The problems of this file are tiny: one OpenMP thread beats a spinning team by 20x."""
    with oracle.threads(1):
        yield


# --------------------------------------------------------------------------- K13: TV closed forms
def test_k13_tv_of_a_ramp_and_of_a_rectangle(oracle):
    ny, nx, a, b = 7, 9, 0.3, -1.1
    j, i = np.meshgrid(np.arange(nx), np.arange(ny))
    ramp = (a * j + b * i)[None].astype(np.float64)
    # interior pixels sqrt(a^2+b^2); last column only d2, last row only d1, corner nothing (R18)
    want = (ny - 1) * (nx - 1) * math.hypot(a, b) + (ny - 1) * abs(b) + (nx - 1) * abs(a)
    assert abs(oracle.tv(ramp) - want) <= 1e-12 * want
    img = np.zeros((2, 12, 15))
    img[0, 3:8, 4:11] = 1.0          # h = 5 rows, w = 7 columns, strictly inside
    img[1] = 2.5                     # constant slice: TV 0; the stack sums over slices
    # 2h + 2w unit jumps; at the pixel (i1-1, j1-1) both differences are -1: sqrt(2) instead of 2
    want = 2 * 5 + 2 * 7 - 2 + math.sqrt(2.0)
    assert abs(oracle.tv(img) - want) <= 1e-12


# --------------------------------------------------------------------------- K14: proximal step
def test_k14_prox_limits(oracle):
    rng = np.random.default_rng(14)
    z = rng.normal(size=(2, 9, 11))
    np.testing.assert_array_equal(oracle.prox_tv(z, 0.0, 50), z)        # tau = 0: identity
    np.testing.assert_array_equal(oracle.prox_tv(z, 0.3, 0), z)         # no inner step: u = z
    big = oracle.prox_tv(z, 1e3, 4000)                                   # TV dominates: the slice mean
    for s in range(2):
        np.testing.assert_allclose(big[s], z[s].mean(), rtol=0, atol=1e-6)
    # G^T p sums to zero over a slice: the mean is preserved for every tau and iteration count
    x = oracle.prox_tv(z, 0.37, 7)
    np.testing.assert_allclose(x.mean(axis=(1, 2)), z.mean(axis=(1, 2)), rtol=0, atol=1e-14)


def test_k14_prox_two_plateaus_closed_form(oracle):
    # image constant along i: d2 = 0, isotropic TV = 1-D TV along j of every row.  For a
    # non-decreasing two-plateau signal (n1 samples at a, n2 at b) the minimiser of
    # 1/2 ||x - z||^2 + tau TV(x) moves the plateaus to a + tau/n1 and b - tau/n2 (until they meet).
    n1, n2, a, b, tau = 3, 5, -0.4, 1.1, 0.6
    row = np.r_[np.full(n1, a), np.full(n2, b)]
    z = np.tile(row, (4, 1))[None]
    x = oracle.prox_tv(z, tau, 6000)
    want = np.r_[np.full(n1, a + tau / n1), np.full(n2, b - tau / n2)]
    np.testing.assert_allclose(x[0], np.tile(want, (4, 1)), rtol=0, atol=1e-7)
    # along the other axis too (transposed operand would fail one of the two)
    xt = oracle.prox_tv(np.ascontiguousarray(z.transpose(0, 2, 1)), tau, 6000)
    np.testing.assert_allclose(xt[0], np.tile(want, (4, 1)).T, rtol=0, atol=1e-7)
    # tau beyond the merge point: both plateaus at the mean
    tau_merge = (b - a) / (1.0 / n1 + 1.0 / n2)
    xm = oracle.prox_tv(z, 1.5 * tau_merge, 6000)
    np.testing.assert_allclose(xm[0], row.mean(), rtol=0, atol=1e-7)


def test_k14_prox_is_the_minimiser(oracle):
    rng = np.random.default_rng(141)
    z = rng.normal(size=(1, 10, 12)) + np.kron(rng.normal(size=(2, 3)), np.ones((5, 4)))[None]
    tau = 0.25

    def objective(x):
        return 0.5 * np.sum((x - z) ** 2) + tau * oracle.tv(x)

    x = oracle.prox_tv(z, tau, 4000)
    f0 = objective(x)
    assert f0 < objective(z) and f0 < objective(np.full_like(z, z.mean()))
    for k in range(30):                                  # strictly convex: every perturbation is worse
        d = rng.normal(size=z.shape) * 10.0 ** rng.uniform(-3, 0)
        assert objective(x + d) >= f0 - 1e-9
    # fewer inner steps are no better than many (the dual ascent converges to the same point)
    assert objective(oracle.prox_tv(z, tau, 20)) >= f0 - 1e-9


# --------------------------------------------------------------------------- K15: Lipschitz constant
@pytest.mark.parametrize("P,B,n", [(9, 21, 12), (20, 33, 16)])
def test_k15_lipschitz_bounds_the_largest_eigenvalue(oracle, P, B, n):
    rng = np.random.default_rng(15 + P)
    angles = np.sort(rng.uniform(0, math.pi, size=P))
    axis = (B - 1) / 2.0 + rng.uniform(-1.0, 1.0, size=P)
    A = _dense_matrix(angles, axis, n, n, B, 1.0)
    lam = np.linalg.eigvalsh(A.T @ A)[-1]
    L = oracle.lipschitz(angles, axis, B, n, n, n_power=8)
    assert lam <= L <= 1.1 * lam * (1 + 1e-12)           # 1.1 x an estimate from below (R17)
    assert L / 1.1 >= 0.97 * lam                          # 8 iterations from v = 1 are close


# --------------------------------------------------------------------------- K16: FISTA
def _tiny_problem(seed, P=14, B=25, n=10):
    rng = np.random.default_rng(seed)
    angles = np.sort(rng.uniform(0, math.pi, size=P))
    axis = (B - 1) / 2.0 + rng.uniform(-0.5, 0.5, size=P)
    A = _dense_matrix(angles, axis, n, n, B, 1.0)
    return rng, angles, axis, A, P, B, n


def test_k16_first_iterates_against_the_dense_matrix(oracle):
    rng, angles, axis, A, P, B, n = _tiny_problem(16)
    d = rng.normal(size=(1, P, B)).astype(np.float32)
    dv = d.astype(np.float64).ravel()
    L = 1.3 * np.linalg.eigvalsh(A.T @ A)[-1]
    # beta = 0: prox = identity.  x1 = A^T d / L (gradient sign of eq. 9, R16); t0 = 1 gives y1 = x1;
    # Beck & Teboulle's momentum with t1 = (1 + sqrt 5) / 2, t2 = (1 + sqrt(1 + 4 t1^2)) / 2
    x1 = A.T @ dv / L
    x2 = x1 - A.T @ (A @ x1 - dv) / L
    t1 = (1 + math.sqrt(5.0)) / 2
    t2 = (1 + math.sqrt(1 + 4 * t1 * t1)) / 2
    y2 = x2 + (t1 - 1) / t2 * (x2 - x1)
    x3 = y2 - A.T @ (A @ y2 - dv) / L
    for n_iter, want in ((1, x1), (2, x2), (3, x3)):
        x, e = oracle.fista_tv(d, angles, axis, n, n, 0.0, L, n_iter, n_inner=5)
        np.testing.assert_allclose(x.ravel(), want, rtol=0, atol=1e-12 * np.abs(want).max() * 50)
    # energy (eq. 3) at y_k: y0 = 0, y1 = x1, y2
    want_e = [0.5 * dv @ dv, 0.5 * np.sum((A @ x1 - dv) ** 2), 0.5 * np.sum((A @ y2 - dv) ** 2)]
    np.testing.assert_allclose(e, want_e, rtol=1e-12)


def test_k16_fista_rate_bound_and_energy(oracle):
    rng, angles, axis, A, P, B, n = _tiny_problem(161)
    xs = np.zeros((n, n))
    xs[3:7, 2:6] = 1.0
    d = (A @ xs.ravel()).reshape(1, P, B).astype(np.float32)     # consistent data, P B > n^2
    dv = d.astype(np.float64).ravel()
    xstar = np.linalg.lstsq(A, dv, rcond=None)[0]                 # F* = min 1/2 ||A x - d||^2
    fstar = 0.5 * np.sum((A @ xstar - dv) ** 2)
    L = oracle.lipschitz(angles, axis, B, n, n)
    prev = None
    for k in (5, 20, 80, 320):
        x, e = oracle.fista_tv(d, angles, axis, n, n, 0.0, L, k)
        f = 0.5 * np.sum((A @ x.ravel() - dv) ** 2)
        # F(x_k) - F* <= 2 L ||x0 - x*||^2 / (k + 1)^2   (Beck & Teboulle 2009, Thm 4.4), x0 = 0
        assert f - fstar <= 2 * L * np.sum(xstar ** 2) / (k + 1) ** 2 * (1 + 1e-9)
        assert prev is None or f <= prev
        prev = f
    assert np.abs(x.ravel() - xstar).max() < 0.2        # ill-conditioned: x converges slowly, F fast
    assert e[0] == pytest.approx(0.5 * dv @ dv, rel=1e-13)


# --------------------------------------------------------------------------- K17: the TV term acts
def test_k17_tv_term_value_and_regularisation(oracle):
    rng, angles, axis, A, P, B, n = _tiny_problem(17, P=6, B=25, n=12)   # few noisy projections
    xs = np.zeros((n, n))
    xs[2:9, 4:10] = 1.0
    clean = A @ xs.ravel()
    d = (clean + 0.3 * rng.normal(size=clean.shape)).reshape(1, P, B).astype(np.float32)
    L = oracle.lipschitz(angles, axis, B, n, n)
    x0, _ = oracle.fista_tv(d, angles, axis, n, n, 0.0, L, 300)
    x1, e1 = oracle.fista_tv(d, angles, axis, n, n, 0.8, L, 300, n_inner=40)
    assert oracle.tv(x1) < 0.5 * oracle.tv(x0)                    # beta > 0 lowers the total variation
    assert np.linalg.norm(x1.ravel() - xs.ravel()) < np.linalg.norm(x0.ravel() - xs.ravel())
    # the displayed energy converges to eq. 3 evaluated (independently, dense A) at the result
    dv = d.astype(np.float64).ravel()
    f = 0.5 * np.sum((A @ x1.ravel() - dv) ** 2) + 0.8 * oracle.tv(x1)
    assert e1[-1] == pytest.approx(f, rel=2e-3)
    assert e1[-1] < e1[0]
    # batch independence: two slices at once = each alone
    d2 = np.concatenate([d, d[:, ::-1].copy()], axis=0)
    xb, eb = oracle.fista_tv(d2, angles, axis, n, n, 0.8, L, 25, n_inner=10)
    xa, ea = oracle.fista_tv(d2[:1], angles, axis, n, n, 0.8, L, 25, n_inner=10)
    xc, ec = oracle.fista_tv(d2[1:], angles, axis, n, n, 0.8, L, 25, n_inner=10)
    np.testing.assert_array_equal(xb[0], xa[0])
    np.testing.assert_array_equal(xb[1], xc[0])
    np.testing.assert_allclose(eb, ea + ec, rtol=1e-13)


# --------------------------------------------------------------------------- K18: tau = beta / L
def _tv_numpy(x):
    """Eq. 2 with the forward differences of R18, typed out (K13 pins oracle.tv to closed forms)."""
    d1 = np.zeros_like(x)
    d2 = np.zeros_like(x)
    d1[..., :, :-1] = x[..., :, 1:] - x[..., :, :-1]
    d2[..., :-1, :] = x[..., 1:, :] - x[..., :-1, :]
    return float(np.sqrt(d1 * d1 + d2 * d2).sum())


def test_k18_prox_threshold_is_beta_over_L(oracle):
    """The minimiser of eq. 3 does not depend on the step 1/L, and x*(beta) beats
    x*(beta') on eq. 3 at beta for every other beta'.  A threshold beta (or beta L, beta / L^2 ...)
    instead of beta / L makes the fixed point the minimiser for beta L: it then moves with L, and
    the run at beta' = beta / L wins eq. 3 at beta."""
    rng, angles, axis, A, P, B, n = _tiny_problem(18, P=8, B=25, n=12)
    xs = np.zeros((n, n))
    xs[3:9, 2:7] = 1.0
    xs[5:10, 6:11] += 0.5
    clean = A @ xs.ravel()
    d = (clean + 0.2 * rng.normal(size=clean.shape)).reshape(1, P, B).astype(np.float32)
    dv = d.astype(np.float64).ravel()
    lam = np.linalg.eigvalsh(A.T @ A)[-1]
    beta = 0.5

    def F(x, b):
        return 0.5 * np.sum((A @ x.ravel() - dv) ** 2) + b * _tv_numpy(x)

    def solve(b, L):
        return oracle.fista_tv(d, angles, axis, n, n, b, L, 500, n_inner=80)[0]

    L1, L2 = 1.05 * lam, 3.0 * lam
    assert L1 > 4.0                                      # L far from 1: beta / L and beta differ
    x1, x2 = solve(beta, L1), solve(beta, L2)
    assert np.abs(x1 - x2).max() < 2e-3 * np.abs(x1).max()
    f1 = F(x1, beta)
    assert abs(F(x2, beta) - f1) < 1e-4 * f1
    for other in (beta / L1, beta * L1, beta / 3, beta * 3):
        assert F(solve(other, L1), beta) > f1 * (1 + 1e-2)
    for k in range(20):                                  # and no random perturbation does better
        assert F(x1 + rng.normal(size=x1.shape) * 10.0 ** rng.uniform(-4, -1), beta) >= f1 - 1e-9


# --------------------------------------------------------------------------- K19: isotropic coupling
def test_k19_prox_kkt_with_both_gradient_components(oracle):
    """KKT system of  min 1/2 ||x - z||^2 + tau TV(x)  with the isotropic TV of eq. 2 (PAPER.md
    L77-L78), typed out in numpy: z - x = tau G^T p with p = G x / |G x| (Euclidean norm of the
    PAIR) wherever G x != 0.  z is a tilted plane plus bumps, so both components of G x are
    non-zero at every interior pixel and p is determined everywhere by x alone.  An anisotropic
    projection (per component, or by the max norm) gives p = sign(.) instead and fails by O(1)."""
    ny, nx, tau = 14, 17, 0.05
    j, i = np.meshgrid(np.arange(nx, dtype=np.float64), np.arange(ny, dtype=np.float64))
    z = (0.7 * j - 0.45 * i + 0.35 * np.sin(0.5 * j + 0.2) * np.cos(0.4 * i))[None]
    x = oracle.prox_tv(z, tau, 20000)[0]
    d1 = np.zeros_like(x)
    d2 = np.zeros_like(x)
    d1[:, :-1] = x[:, 1:] - x[:, :-1]
    d2[:-1, :] = x[1:, :] - x[:-1, :]
    assert np.abs(d1[:-1, :-1]).min() > 0.05 and np.abs(d2[:-1, :-1]).min() > 0.05
    m = np.sqrt(d1 * d1 + d2 * d2)
    m[-1, -1] = 1.0                                      # G x = 0 there: p is multiplied by nothing
    p1, p2 = d1 / m, d2 / m
    # G^T p, adjoint of the forward differences with the zero last column / row (R18)
    gt = np.zeros_like(x)
    gt[:, :-1] -= p1[:, :-1]
    gt[:, 1:] += p1[:, :-1]
    gt[:-1, :] -= p2[:-1, :]
    gt[1:, :] += p2[:-1, :]
    np.testing.assert_allclose(z[0] - x, tau * gt, rtol=0, atol=2e-6)
    # the same test distinguishes the norms: with p = sign(d) the residual is O(tau)
    gs = np.zeros_like(x)
    s1, s2 = np.sign(d1), np.sign(d2)
    gs[:, :-1] -= s1[:, :-1]
    gs[:, 1:] += s1[:, :-1]
    gs[:-1, :] -= s2[:-1, :]
    gs[1:, :] += s2[:-1, :]
    assert np.abs(z[0] - x - tau * gs).max() > 0.2 * tau
