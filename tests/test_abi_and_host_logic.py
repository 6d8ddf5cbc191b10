"""CPU-side checks (-m "not gpu"): the C-ABI library loads and exports every symbol that
include/pyhst.h declares, errors that are detectable without a device are reported, and the
multi-GPU plumbing (slice sharding, max-over-ranks, gather) works under gloo with world_size 2.
No compute call is made without a GPU.
"""
import ctypes
import math
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cuda_lib():
    from paper_1306_1392_b200 import build
    return ctypes.CDLL(build.build())


def _declared_symbols(headers=None):
    inc = os.path.join(ROOT, "include")
    names = set()
    for h in headers or sorted(f for f in os.listdir(inc) if f.endswith(".h")):
        src = open(os.path.join(inc, h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(pyhst_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_header_symbols_are_exported(cuda_lib):
    names = _declared_symbols()
    assert {"pyhst_ramp_filter", "pyhst_backproject", "pyhst_forward_project", "pyhst_fbp"} <= set(names)
    for n in names:
        assert hasattr(cuda_lib, n), "libpyhst_b200.so does not export %s" % n


def test_header_states_the_concurrency_rule_and_keeps_test_hooks_out():
    """pyhst.h promises stream-ordered calls: it must say how calls on several streams / threads /
    devices are ordered and where a call may synchronise; kernel-variant switches are test hooks."""
    text = open(os.path.join(ROOT, "include", "pyhst.h")).read()
    assert "ONE CALL IN FLIGHT PER DEVICE" in text and "cudaStreamWaitEvent" in text
    assert "FIRST call with a new shape" in text
    public = _declared_symbols(["pyhst.h"])
    assert not [n for n in public if n.startswith("pyhst_set_")]
    assert "pyhst_set_backproject_variant" in _declared_symbols(["pyhst_test.h"])


def test_binding_lists_every_header_symbol():
    from paper_1306_1392_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()


def test_library_has_sm100a_code_and_tma():
    """The shipped library carries sm_100a SASS with the TMA bulk copy (UBLKCP) in the projectors."""
    from paper_1306_1392_b200 import build
    lib = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass
    # per kernel: the product projectors stage by TMA bulk copy and synchronise through mbarriers (SYNCS); the GEMM of
    # Algorithm 1 runs on the 5th-generation tensor cores (UTCMMA = tcgen05.mma, LDTM = tcgen05.ld)
    chunks = sass.split("Function : ")
    def body(name):
        hits = [c for c in chunks if name in c.split("\n", 1)[0]]
        assert hits, name
        return "\n".join(hits)
    for name in ("bp_run8_kernel", "fp_diag_kernel"):
        k = body(name)
        assert "UBLKCP" in k and "SYNCS" in k and "FFMA" in k, name
    g = body("patch_gemm_tc_kernel")
    assert "UTCMMA" in g or "UTCHMMA" in g or "UTCQMMA" in g, "no tcgen05.mma in the tensor-core GEMM"
    assert "LDTM" in g, "no tcgen05.ld in the tensor-core GEMM"


def test_halfacq_extent_host_logic(cuda_lib, oracle):
    """Pure host function: no device needed; must agree with the oracle's reading R10."""
    cuda_lib.pyhst_halfacq_extent.argtypes = [ctypes.c_int32, ctypes.c_double,
                                              ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32)]
    for n_bins, cbar in [(2048, 1900.0), (2048, 147.0), (128, 118.0), (128, 63.5), (367, 10.25), (64, 60.0)]:
        ext, pad = ctypes.c_int32(), ctypes.c_int32()
        assert cuda_lib.pyhst_halfacq_extent(n_bins, cbar, ctypes.byref(ext), ctypes.byref(pad)) == 0
        assert (ext.value, pad.value) == oracle.halfacq_extent(n_bins, cbar)
        assert ext.value % 64 == 0 and ext.value >= 2 * max(cbar, n_bins - 1 - cbar) + 1
    assert cuda_lib.pyhst_halfacq_extent(0, 1.0, None, None) != 0


def test_argument_errors_without_device(cuda_lib):
    """Validation happens before any CUDA call: NULL pointers / bad sizes -> INVALID_ARG + message."""
    cuda_lib.pyhst_last_error.restype = ctypes.c_char_p
    cuda_lib.pyhst_ramp_filter.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32,
                                           ctypes.c_int32, ctypes.c_int32, ctypes.c_int64, ctypes.c_int,
                                           ctypes.c_void_p, ctypes.c_void_p]
    assert cuda_lib.pyhst_ramp_filter(None, None, 4, 64, 64, 0, 0, 0, None, None) == 1
    assert b"NULL" in cuda_lib.pyhst_last_error()
    assert cuda_lib.pyhst_ramp_filter(None, None, 0, 64, 64, 0, 0, 0, None, None) == 0      # empty stack: no-op
    assert cuda_lib.pyhst_ramp_filter(None, None, 0, 64, 32, 0, 0, 0, None, None) == 1      # still validated
    cuda_lib.pyhst_backproject.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_float,
                                           ctypes.c_void_p]
    assert cuda_lib.pyhst_backproject(None, None, None, 1.0, None) == 1


def test_no_cpu_fallback_without_device():
    """On a box without a GPU the product path must fail loudly, not route through the oracle."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1306_1392_b200 as P
    x = torch.zeros((1, 8, 32), dtype=torch.float32)
    with pytest.raises(P.PyhstError):
        P.backproject(x, np.zeros(8), np.full(8, 15.5), 16, 16)
    # a raw call with fake non-NULL pointers still stops at the device check (UNSUPPORTED = 2)
    lib = P.binding._load()
    ang = (ctypes.c_double * 8)(*([0.0] * 8))
    g = P.binding.Geom(1, 8, 32, 0, ang, ang, 16, 16, 1.0)
    assert lib.pyhst_backproject(ctypes.c_void_p(4096), ctypes.c_void_p(8192), ctypes.byref(g), 1.0, None) == 2
    assert "no CPU fallback" in P.last_error()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1306_1392_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "pyhst_oracle" not in text, f
    text = (open(os.path.join(ROOT, "oracle", "pyhst_oracle.c")).read()
            + open(os.path.join(ROOT, "oracle", "__init__.py")).read())
    assert not re.search(r"^\s*(import|from)\s+paper_1306_1392_b200\b", text, flags=re.M)
    assert "#include \"../paper" not in text and "pyhst.h" not in text


# ------------------------------------------------------------------ sharding (single process)
def test_slice_range_partitions_exactly():
    from paper_1306_1392_b200.sharding import slice_range
    for n in [0, 1, 5, 16, 64, 67]:
        for world in [1, 2, 3, 8]:
            spans = [slice_range(n, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        slice_range(4, 2, 2)


# ------------------------------------------------------------------ sharding under gloo, world_size 2
_WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import numpy as np, torch, torch.distributed as dist
from paper_1306_1392_b200 import sharding, workloads
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
S = 5
a, b = sharding.slice_range(S, world, rank)
w = workloads.config(1, shrink=8, n_slices=S)
local = torch.from_numpy(w.sinogram(range(a, b)))           # each rank synthesises only its slices
full = sharding.gather_slices(local, S, dist)
t = sharding.max_over_ranks(10.0 + rank, dist)
assert t == 10.0 + world - 1, t
if rank == 0:
    want = torch.from_numpy(w.sinogram())
    assert full.shape == want.shape and torch.equal(full, want)
    print("OK", flush=True)
dist.destroy_process_group()
"""


def test_gloo_world2_sharding(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % {"root": ROOT})
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29613", str(script)],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "OK" in r.stdout


def test_bench_reference_arm_runs_on_cpu():
    """bench.py --impl reference prints one JSON line with the contract's keys (tiny config 1)."""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "3", "--warmup", "2"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "ms_per_step", "higher_is_better",
              "cpu_baseline", "e2e", "config"):
        assert k in line
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    # the two arms print the same quantity on the same config
    sys.path.insert(0, ROOT)
    import bench
    from paper_1306_1392_b200 import workloads
    assert line["metric"] == bench.METRIC and line["unit"] == bench.UNIT and line["metric_version"] == bench.METRIC_VERSION
    assert line["config"] == bench._config_dict(workloads.config(1), 1)          # exactly the b200 arm's config dict
    assert (line["steps"], line["warmup"]) == (3, 2)                             # honoured (they fit --ref-seconds)
    m = line["metrics"]
    w = workloads.config(1)
    upd = m["slices_timed_per_step"] * w.nx * w.ny * w.n_angles
    assert line["value"] == pytest.approx(upd / (m["ms_backproject"] * 1e-3) / 1e9, rel=1e-9)   # BP updates / BP seconds
    assert line["ms_per_step"] == pytest.approx(m["ms_ramp_filter"] + m["ms_backproject"] + m["ms_forward_project"], rel=1e-6)
    assert line["e2e"]["value"] == line["value"] and line["cpu_baseline"]["value"] == line["value"]
    # a budget too small for the request: fewer steps are run and REPORTED, never more than asked
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "50", "--warmup", "5", "--ref-seconds", "0.5"], capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr
    short = json.loads(r.stdout.strip().splitlines()[-1])
    assert 1 <= short["steps"] < 50 and 0 <= short["warmup"] <= 5


# ------------------------------------------------------------------ diagonal-line forward projector: host tables
def _fd_plan(angles, axis, B, nx, ny, h=1.0):
    from paper_1306_1392_b200 import binding
    return binding.test_fd_plan(angles, axis, B, nx, ny, pixel_size=h)


def test_fd_plan_chunks_cover_every_projection_once(cuda_lib):
    """pyhst_test.h pyhst_test_fd_plan (host only): every projection sits in exactly one chunk of at most 16 neighbours
    of one walk class; those with fewer than 1 + 2^-12 bins per pixel along an image diagonal (an interval may then
    hold two pixels of a line) form chunks of their own."""
    P, B, n = 2000, 2048, 2048
    angles = np.arange(P) * math.pi / P
    rng = np.random.default_rng(3)
    axis = 1023.5 + rng.uniform(-1.5, 1.5, P)
    info, chunk_of, ranges = _fd_plan(angles, axis, B, n, n)
    assert info["status"] == 0
    sigma = np.abs(np.cos(angles)) + np.abs(np.sin(angles))
    near = sigma < 1.0 + 1.0 / 4096.0                                      # theta = 0 and pi / 2: two pixels per interval possible
    assert int(near.sum()) == 2 and info["left_out"] == 0 and (chunk_of >= 0).all()
    # ... they sit in chunks of their own (run by the TWO form of the kernel), after all other chunks
    near_chunks = set(chunk_of[near])
    assert not near_chunks & set(chunk_of[~near]) and min(near_chunks) > max(chunk_of[~near])
    left = np.zeros(P, dtype=bool)
    counts = np.bincount(chunk_of[~left], minlength=info["chunks"])
    assert counts.min() >= 1 and counts.max() <= info["projections_per_chunk"] == 16
    assert info["chunks"] <= 132                                          # dense list: chunks are full
    # one walk class per chunk: layout (sign of cos * sin), detector direction, skew (which of |cos|, |sin| is larger)
    cls = (np.cos(angles) * np.sin(angles) >= 0).astype(int) * 4 + (np.abs(np.sin(angles)) > np.abs(np.cos(angles))) * 2
    for c in range(info["chunks"]):
        assert len(set(cls[chunk_of == c])) == 1
    assert 64 < info["window"] <= 100 and info["zpad"] >= info["window"] + 16
    assert info["blocks"] == -(-B // (info["intervals_per_block"] - 1))
    assert ranges.min() >= 0 and ranges[:, :, 1].max() <= info["lines"] - 8


def test_fd_plan_line_ranges_contain_every_contributing_pixel(cuda_lib):
    """Brute force on a small scan: every pixel whose coordinate falls into a block's interval range lies on a stored
    line inside the range the block walks (layout 0: line = i - j + nx - 1, layout 1: line = i + j)."""
    rng = np.random.default_rng(5)
    P, B, nx, ny, h = 37, 150, 70, 50, 1.15
    angles = np.sort(rng.uniform(0, 2 * math.pi, P))
    axis = 74.0 + rng.uniform(-20, 20, P)
    info, chunk_of, ranges = _fd_plan(angles, axis, B, nx, ny, h)
    assert info["status"] == 0
    nb = info["intervals_per_block"]
    j, i = np.meshgrid(np.arange(nx), np.arange(ny))
    for p in range(P):
        c = chunk_of[p]
        if c < 0:
            continue
        a, b = h * math.cos(angles[p]), h * math.sin(angles[p])
        t = axis[p] + a * (j - (nx - 1) / 2) + b * (i - (ny - 1) / 2)
        w = (i - j + nx - 1) if a * b >= 0 else (i + j)
        for bx in range(info["blocks"]):
            mB = bx * (nb - 1) - 1
            inside = (t >= mB) & (t < mB + nb)
            if inside.any():
                lo, hi = ranges[c, bx]
                assert lo <= w[inside].min() and w[inside].max() < hi, (p, bx)


def test_fd_plan_rejects_small_pixels_and_sparse_lists_shrink_chunks(cuda_lib):
    """Pixel sizes below 1 / sqrt(2) bins leave no projection with >= 1 bin per pixel along a diagonal; a sparse angle
    list (config 4: 0.9 degrees apart) fans out and fits only a few projections into one staged window."""
    ang = np.arange(200) * math.pi / 200
    info, chunk_of, _ = _fd_plan(ang, np.full(200, 511.5), 1024, 1024, 1024, h=0.6)
    assert info["status"] != 0 and (chunk_of == -1).all()
    info, chunk_of, _ = _fd_plan(ang, np.full(200, 511.5), 1024, 1024, 1024)
    assert info["status"] == 0 and info["window"] <= 100
    per_chunk = (chunk_of >= 0).sum() / info["chunks"]
    assert 2.0 <= per_chunk <= 8.0
