"""``pyhst_ring_filter_static`` against ``pyhst_ring_filter`` (run on a B200 with ``-m gpu``).

Who this entry point is for: programs in which the library is not allowed to allocate device memory --
a host application that has split the whole GPU memory into pools of its own, an acquisition loop that
cannot take the device-wide stall of cudaMalloc / cudaFree, a process that must go on correcting
sinograms after an out-of-memory condition.  The ordinary ring filter keeps its column sums in a
workspace that the library grows with cudaMalloc; the static one keeps them in a fixed 8.5 MB array
compiled into the library, so it works for ``n_slices * n_bins <= 32768`` only and every call on a
device shares (and overwrites) that one array.

What is checked: on two calls in a row with different inputs -- the second one smaller, so that it runs
over what the first left behind in the array -- the output agrees with the existing path's within the
tolerance of the other GPU tests (rel-L2 <= 1e-5, max-abs <= 1e-4 * max; the two paths run the same
kernels in the same order, so in practice they agree to the bit), and a request beyond the limit is
refused with a message instead of overrunning the array.

The file sorts last on purpose: ``pytest -x`` stops at the first failure and a failure here must not
hide the parity tests.  It needs nothing from the tests before it and passes alone in a fresh process.
"""
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


def _close(got, want, what):
    got = got.astype(np.float64)
    want = want.astype(np.float64)
    assert got.shape == want.shape and np.isfinite(got).all(), what
    num, den = np.linalg.norm((got - want).ravel()), np.linalg.norm(want.ravel())
    assert num <= REL_L2 * den + 1e-30, "%s: rel-L2 %.3e" % (what, num / max(den, 1e-300))
    assert np.abs(got - want).max() <= MAX_ABS * np.abs(want).max() + 1e-30, what


def _scan(seed, S, P, B, with_model):
    rng = np.random.default_rng(seed)
    sino = (rng.normal(size=(S, P, B)) + 0.5 * rng.normal(size=(S, 1, B))).astype(np.float32)   # per-bin errors = rings
    model = rng.normal(size=(S, P, B)).astype(np.float32) if with_model else None
    return sino, model


def test_ring_filter_static_matches_ring_filter_on_two_calls_in_a_row(lib):
    import torch
    # first call fills the whole array (16 x 2048 = the limit), the second is smaller and has a model:
    # stale contents of the first call lie under and behind everything the second one uses
    cases = [(11, 16, 96, 2048, 9, False), (12, 3, 50, 211, 4, True)]
    assert cases[0][1] * cases[0][3] == lib.binding.RING_STATIC_MAX_CELLS
    for seed, S, P, B, r, with_model in cases:
        sino, model = _scan(seed, S, P, B, with_model)
        d_model = None if model is None else _dev(model)
        want = lib.ring_filter(_dev(sino), r, model=d_model).cpu().numpy()
        out = torch.full((S, P, B), float("nan"), device="cuda", dtype=torch.float32)
        got = lib.binding.ring_filter_static(_dev(sino), r, model=d_model, out=out)
        assert got is out
        got = got.cpu().numpy()
        _close(got, want, "ring_filter_static S=%d P=%d B=%d" % (S, P, B))
        assert np.array_equal(got, want)       # same kernels, same summation order
        assert np.abs(got - sino).max() > 0    # the filter did something
    # the first case once more, in place: the array now holds the small case's leftovers
    seed, S, P, B, r, with_model = cases[0]
    sino, _ = _scan(seed, S, P, B, with_model)
    want = lib.ring_filter(_dev(sino), r).cpu().numpy()
    d = _dev(sino)
    lib.binding.ring_filter_static(d, r, out=d)
    _close(d.cpu().numpy(), want, "ring_filter_static in place")


def test_ring_filter_static_refuses_what_does_not_fit(lib):
    import torch
    S, P, B = 17, 4, 2048                      # 17 * 2048 cells > 32768
    sino = torch.zeros((S, P, B), device="cuda", dtype=torch.float32)
    out = torch.full_like(sino, 7.0)
    with pytest.raises(lib.PyhstError, match="PYHST_RING_STATIC_MAX_CELLS"):
        lib.binding.ring_filter_static(sino, 3, out=out)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())            # nothing was written
    with pytest.raises(lib.PyhstError):
        lib.binding.ring_filter_static(sino[:1], 0, out=out[:1])   # half_width < 1, as in pyhst_ring_filter
    lib.ring_filter(sino, 3, out=out)          # the allocating path takes the same stack
    torch.cuda.synchronize()
    assert bool((out == 0.0).all())
