#!/usr/bin/env python
"""bench.py -- throughput of the hot path on BASELINE.json's config 2, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--config C]

A *step* is one pass of the whole hot path over one synthetic batch:
pyhst_fbp (a1 ramp filter -> a2 backprojection = a4) followed by pyhst_forward_project (a3) of the
reconstructed stack.  `value` is BASELINE.json's metric, backprojection GUPS: the pixel*projection*
slice updates of the backprojection divided by the device time of the backprojection stage inside
the step (CUDA events recorded by the library on the launching stream); `metrics` carries the other
half of the metric (FBP slices/s = slices / (filter + backprojection time)), the forward projector
and the composite step; `roofline` is the backprojector's, `roofline_other` the forward projector's
and the ramp filter's.

N > 1 (torchrun, one rank per GPU): slices are independent, every rank runs the
same per-GPU stack (weak scaling, no data-path collective); time = max over ranks.

--impl reference times the oracle (oracle/, fp64 CPU) on the host cores on a bounded sample of the
same workload.  The product path never touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = ("backprojection GUPS (nominal S*nx*ny*P pixel*projection*slice updates / time of the backprojection stage; "
          "executed updates and FBP slices/s in metrics)")
# 1 (round 1): updates of the whole step / step time.  2 (round 2): backprojection updates / backprojection-stage time.
# 3: as 2, and the reference arm prints the same quantity (oracle backprojection alone); nominal counting stated.
METRIC_VERSION = 3
N_INNER_TV = 20                  # dual steps per FISTA iteration of the config-4 solve
METRIC_STEP = "projector updates/s over one hot-path step (ramp filter + backprojection + forward projection)"
UNIT = "GUPS"
FP32_LANES_PER_SM = 128          # FP32 FMA lanes per SM per clock (4 SMSP x 32)
LANE_OPS_PER_UPDATE = 2          # lerp FMA + accumulate FMA


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh), "measured"
    except OSError:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        fd, self.path = tempfile.mkstemp(suffix=".csv")
        os.close(fd)
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        with open(self.path) as fh:
            for line in fh:
                f = [x.strip() for x in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
                except ValueError:
                    continue
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        os.unlink(self.path)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), power_w_max=max(pw),
                       reasons=sorted(reasons), samples=len(sm))
        return out


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def _workload(P, args):
    w = P.workloads.config(args.config, n_slices=args.slices or None)
    return w


def _executed_bp_fraction(w):
    """Share of the nominal S*nx*ny*P backprojection updates the library executes: the stitched
    360-degree half-acquisition path (pyhst_test.h pyhst_set_halfacq_stitch) folds
    facing projections and backprojects P/2 rows when the scan pairs up (same test as csrc/api.cu)."""
    import math
    import numpy as np
    if w.mode != 2 or w.n_angles % 2:
        return 1.0
    h = w.n_angles // 2
    a, c = np.asarray(w.angles), np.asarray(w.axis)
    c2 = 2.0 * c[:h]
    ok = (np.abs(a[h:] - a[:h] - math.pi) <= 1e-10).all() and (c[h:] == c[:h]).all() and \
         (np.abs(c2 - np.rint(c2)) <= 1e-9).all()
    return 0.5 if ok else 1.0


def _config_dict(w, world, extra=None):
    d = {"workload": "BASELINE.json configs[%d] (%s): %d slices x %dx%d, %d projections x %d bins per GPU"
                     % (w.cfg - 1, w.name, w.n_slices, w.ny, w.nx, w.n_angles, w.n_bins),
         "slices_per_gpu": w.n_slices, "n_angles": w.n_angles, "n_bins": w.n_bins, "nx": w.nx, "ny": w.ny,
         "filter": ["ram-lak", "shepp-logan"][w.filter], "scan": ["180", "360", "360-half"][w.mode],
         "parallelism": "slices sharded over %d GPU(s), no collective" % world,
         "step": "pyhst_fbp (ramp filter + backprojection) then pyhst_forward_project of the result",
         "l2": "inputs larger than L2 (sinogram stack %.0f MB, image stack %.0f MB vs 126 MB L2)"
               % (w.n_slices * w.n_angles * w.n_bins * 4 / 1e6, w.n_slices * w.nx * w.ny * 4 / 1e6)}
    if extra:
        d.update(extra)
    return d


def run_b200(args):
    import torch
    import torch.distributed as dist

    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("--gpus %d needs torchrun with --nproc-per-node %d" % (args.gpus, args.gpus))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference "
                         "for the oracle baseline)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_1306_1392_b200 as P
    from paper_1306_1392_b200 import sharding

    P.binding._load()
    w = _workload(P, args)
    S, NP, B, nx, ny = w.n_slices, w.n_angles, w.n_bins, w.nx, w.ny
    # weak scaling: rank r reconstructs slices [r*S, (r+1)*S) of a world*S-slice scan
    first = sharding.slice_range(S * world, world, rank)[0]
    P.workloads.set_device("cuda")
    sino = w.sinogram_tensor(range(first, first + S)).contiguous()
    P.workloads.set_device("cpu")
    img = torch.empty((S, ny, nx), dtype=torch.float32, device="cuda")
    proj = torch.empty((S, NP, B), dtype=torch.float32, device="cuda")
    updates = S * nx * ny * NP                      # per projector call, per GPU
    updates_call = updates

    fista = w.cfg == 4 and not args.no_fista
    if fista:
        # BASELINE.json configs[3]: TV-regularised FISTA, lambda = 0.01, 100 iterations, one projector
        # pair per iteration (pyhst_fista_tv, NEXT row N1); a step = one whole reconstruction
        n_fista = 100
        updates *= n_fista
        args.no_e2e = True                          # the device-resident solver has no host entry point

    def step():
        if fista:
            P.fista_tv(sino, w.angles, w.axis, nx, ny, 0.01, n_fista, n_inner=N_INNER_TV, n_power=8,
                       pixel_size=w.pixel_size, out=img, want_energy=False)
            return
        P.fbp(sino, w.angles, w.axis, nx, ny, w.pixel_size, filter=w.filter, mode=w.mode, out=img)
        P.forward_project(img, w.angles, w.axis, B, w.pixel_size, out=proj)

    for _ in range(max(args.warmup, 1)):
        step()
    torch.cuda.synchronize()
    P.profile_read(reset=True)
    P.profile_enable(True)
    sampler = ClockSampler(local)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    ms_total = sharding.max_over_ranks(ev0.elapsed_time(ev1), dist if world > 1 else None)
    stages = P.profile_read(reset=True)
    P.profile_enable(False)
    ms_step = ms_total / args.steps

    # ---- end to end: host (pinned) buffers through the *_host entry points
    e2e = None
    if not args.no_e2e:
        h_sino = torch.empty(sino.shape, dtype=torch.float32, pin_memory=True)
        h_sino.copy_(sino)
        h_img = torch.empty((S, ny, nx), dtype=torch.float32, pin_memory=True)
        h_proj = torch.empty((S, NP, B), dtype=torch.float32, pin_memory=True)

        # chunks of the host pipeline: copies of one chunk overlap the kernels of another; 16-slice chunks (the
        # 16-slices-per-thread forward kernel) once the stack has at least two of them
        chunk = 16 if S >= 32 else 8

        def e2e_fbp():
            P.fbp_host(h_sino, w.angles, w.axis, nx, ny, w.pixel_size, filter=w.filter, mode=w.mode,
                       out=h_img, max_slices_per_chunk=chunk)

        def e2e_fp():
            P.forward_project_host(h_img, w.angles, w.axis, B, w.pixel_size, out=h_proj,
                                   max_slices_per_chunk=chunk)

        for _ in range(min(args.warmup, 2) or 1):
            e2e_fbp()
            e2e_fp()
        n_e2e = max(1, min(args.steps, 5))
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t_fbp = t_fp = 0.0
        for _ in range(n_e2e):                      # the *_host calls synchronise before returning
            t0 = time.perf_counter()
            e2e_fbp()
            t1 = time.perf_counter()
            e2e_fp()
            t_fbp += t1 - t0
            t_fp += time.perf_counter() - t1
        torch.cuda.synchronize()
        mx = lambda v: sharding.max_over_ranks(v, dist if world > 1 else None)
        ms_fbp_h, ms_fp_h = mx(t_fbp * 1e3) / n_e2e, mx(t_fp * 1e3) / n_e2e
        ms_e2e = ms_fbp_h + ms_fp_h
        e2e = {"value": updates * world / (ms_fbp_h * 1e-3) / 1e9, "unit": UNIT,
               "what": "backprojection updates / wall time of pyhst_fbp_host (ramp filter + backprojection with the "
                       "H2D copy of the raw sinograms and the D2H copy of the slices inside the timed region)",
               "fbp_slices_per_s": S * world / (ms_fbp_h * 1e-3),
               "forward_projection_gups": updates * world / (ms_fp_h * 1e-3) / 1e9,
               "step_gups": 2 * updates * world / (ms_e2e * 1e-3) / 1e9,
               "ms_fbp_host": ms_fbp_h, "ms_forward_project_host": ms_fp_h, "ms_per_step": ms_e2e,
               "steps": n_e2e,
               "h2d_bytes_per_step": int(h_sino.numel() * 4 + h_img.numel() * 4),
               "d2h_bytes_per_step": int(h_img.numel() * 4 + h_proj.numel() * 4),
               "api": "pyhst_fbp_host + pyhst_forward_project_host (pinned host buffers, %d-slice chunks, "
                      "copies overlapped with kernels)" % chunk}
        P.profile_read(reset=True)
        del h_sino, h_img, h_proj

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks, peaks_kind = _peaks()
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    f_max = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    peak_tflops = n_sm * FP32_LANES_PER_SM * 2 * f_max / 1e12   # FP32 FMA issue peak at max clock

    bp_exec = _executed_bp_fraction(w)

    def kernel_roofline(stage, name, executed=1.0, calls_per_step=1):
        # one "launch" of the roofline = one call of the stage (all S*nx*ny*P updates); the run8
        # backprojector covers it with two kernel launches (class A, then class B projections)
        ms, launches, _ = stages[stage]
        if launches == 0:
            return None
        kernels_per_call = max(1, round(launches / (args.steps * calls_per_step)))
        launches = args.steps * calls_per_step
        avg_ms = ms / launches
        upd = updates_call * executed
        ach = upd * LANE_OPS_PER_UPDATE * 2 / (avg_ms * 1e-3) / 1e12
        r = {"kernel": name, "bound": "alu", "achieved": ach, "peak": peak_tflops, "unit": "TFLOP/s",
             "frac": ach / peak_tflops, "traffic": None, "avg_ms": avg_ms, "launches": launches,
             "kernels_per_launch": kernels_per_call,
             "updates_per_launch": upd, "nominal_updates_per_launch": updates_call,
             "flop_per_update": 2 * LANE_OPS_PER_UPDATE,
             "gups": upd / (avg_ms * 1e-3) / 1e9,
             "peak_note": "%d SMs x 128 FP32 lanes x 2 flop x %.0f MHz (sm_max_mhz, %s peaks file); "
                          "algorithmic work = 2 FMA per (pixel, projection, slice)"
                          % (n_sm, f_max / 1e6, peaks_kind)}
        if clocks.get("sm_mhz"):
            r["frac_at_sampled_clock"] = r["frac"] * (f_max / 1e6) / clocks["sm_mhz"]
        tr = _traffic().get("config%d" % w.cfg, {}).get(stage) if not args.slices else None
        if tr is not None:
            # a stored number (one ncu --set full capture, not this run): only valid for the kernel it was taken on
            captured = str(_traffic().get("_kernels", {}).get(stage, ""))
            if captured and captured in name:
                r["traffic"] = tr
                r["traffic_source"] = _traffic_source()
            else:
                r["traffic_source"] = "none: the stored capture is of '%s', this run used '%s'" % (captured, name)
        return r

    calls = n_fista if fista else 1
    r_bp = kernel_roofline("backproject", "bp_run8_kernel<0> + bp_run8_kernel<1>", executed=bp_exec, calls_per_step=calls)
    fp_names = {1: "fp_gather_kernel", 2: "fp_band_kernel", 3: "fp_ivl_kernel", 4: "fp_ivl_kernel (8 slices)",
                5: "fp_diag_kernel"}
    r_fp = kernel_roofline("forward_project", fp_names.get(P.last_forward_project_kernel(), "forward projector"),
                           calls_per_step=calls)
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    ms_bp = stages["backproject"][0] / args.steps
    ms_fp = (stages["forward_project"][0] + stages["transpose"][0]) / args.steps
    ms_filter = stages["ramp_filter"][0] / args.steps
    ms_tv = stages["tv_solver"][0] / args.steps
    others = []
    if ms_filter > 0 and not fista:
        # a1 is HBM-bound: algorithmic bytes = one read of the raw row + one write of the filtered row
        fbytes = 4.0 * S * NP * (B + (B if w.mode != 2 else P.halfacq_extent(B, float(w.axis.mean()))[0]))
        others.append({"kernel": "ramp filter (a1)", "bound": "hbm", "achieved": fbytes / (ms_filter * 1e-3) / 1e9,
                       "peak": hbm, "unit": "GB/s", "frac": fbytes / (ms_filter * 1e-3) / 1e9 / hbm,
                       "traffic": _traffic().get("config%d" % w.cfg, {}).get("ramp_filter") if not args.slices else None,
                       "traffic_source": _traffic_source(),
                       "avg_ms": ms_filter, "bytes_per_launch": fbytes,
                       "peak_note": "hbm_gbs of MEASURED_PEAKS.json (%s); algorithmic bytes = 4 (B_in + B_out) per row" % peaks_kind})
    if fista and ms_tv > 0:
        # N1: the dual steps dominate the solver's own kernels; algorithmic bytes of ONE dual step =
        # read z, p1, p2 + write p1', p2' = 5 image stacks
        dbytes = 5.0 * 4.0 * S * nx * ny
        n_dual = n_fista * N_INNER_TV
        others.append({"kernel": "ftv_dual_fused_kernel (+ residual / step / finish kernels of pyhst_fista_tv)",
                       "bound": "hbm", "achieved": dbytes * n_dual / (ms_tv * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                       "frac": dbytes * n_dual / (ms_tv * 1e-3) / 1e9 / hbm, "traffic": None,
                       "avg_ms": ms_tv / n_dual, "launches": n_dual, "bytes_per_launch": dbytes,
                       "note": "one 'launch' = one dual step of 168 MB algorithmic traffic at config 4; the fused kernel "
                               "runs 5 steps per kernel launch out of shared memory, so the fraction can exceed 1",
                       "peak_note": "hbm_gbs of MEASURED_PEAKS.json (%s)" % peaks_kind})
    own = sum(v[1] for v in stages.values())
    bp_gups = updates_call * calls * world / (ms_bp * 1e-3) / 1e9 if ms_bp else None
    if fista:
        roofs = sorted([x for x in (r_bp, r_fp) if x], key=lambda r: -r["avg_ms"] * r["launches"])
        metric, value = METRIC_STEP + " -- pyhst_fista_tv solve", 2 * updates * world / (ms_step * 1e-3) / 1e9
    else:
        roofs = [x for x in (r_bp, r_fp) if x]       # the stated metric is the backprojector's: it leads
        metric, value = METRIC, bp_gups
    line = {
        "metric": metric, "metric_version": METRIC_VERSION, "value": value, "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "impl": "b200",
        "config": _config_dict(w, world, {"step": "pyhst_fista_tv: 100 FISTA iterations (lambda 0.01, 20 dual "
                                          "steps each), one forward/back projector pair per iteration; "
                                          "updates counted for the 200 projector calls only"} if fista else None),
        "metrics": {"backprojection_gups": bp_gups,
                    "backprojection_gups_executed": bp_gups * bp_exec if bp_gups else None,
                    "backprojection_executed_fraction": bp_exec,
                    "forward_projection_gups": updates * world / (ms_fp * 1e-3) / 1e9 if ms_fp else None,
                    "fbp_slices_per_s": S * world / ((ms_filter + ms_bp) * 1e-3) if (ms_bp and not fista) else None,
                    "step_gups": 2 * updates * world / (ms_step * 1e-3) / 1e9,
                    "ms_ramp_filter": ms_filter, "ms_backproject": ms_bp, "ms_forward_project": ms_fp,
                    "ms_tv_solver_kernels": ms_tv,
                    "note": "per-stage device ms of rank 0 (CUDA events recorded by the library on the launching "
                            "stream, inside the timed region); backprojection_gups counts the nominal S*nx*ny*P "
                            "updates, _executed what the kernel really does (the stitched half-acquisition path "
                            "backprojects P/2 folded rows)"},
        "clocks": clocks, "e2e": e2e,
        "gpu_launches": own, "gpu_launches_per_step": own / args.steps,
        "library_launches": {"cufft_execs": sum(v[2] for v in stages.values())},
        "roofline": roofs[0] if roofs else None, "roofline_other": roofs[1:] + others,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(P.workloads, args)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _traffic():
    """dram bytes per launch from the committed ncu --set full capture (profiles/traffic.json)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            return json.load(fh)
    except (OSError, ValueError):
        return {}


def _traffic_source():
    t = _traffic()
    return "stored: %s; captured at commit %s on %s" % (t.get("_source", "profiles/traffic.json"), t.get("_head", "?"),
                                                       t.get("_date", "?"))


def _oracle_sample(wl_mod, args):
    """One bounded sample of the workload for the oracle: the first `cpu_slices` slices (default 1) at
    full size -- all projections, bins and pixels, so every inner loop has the workload's own length."""
    w = wl_mod.config(args.config, n_slices=max(1, args.cpu_slices))
    sino = w.sinogram()
    return w, sino


def _time_oracle_step(oracle, w, sino):
    """One hot-path step in the oracle, as it stands, stage by stage: ramp filter (direct convolution, fp64),
    backprojection of the filtered rows (scale pi / P), forward projection of the float32-rounded result.
    oracle.fbp is exactly filter then backprojection (pin K12); the half-acquisition mode has no separate
    stages in the oracle and is timed as one FBP.  Returns (total, filter, backprojection, forward) seconds."""
    import math
    import numpy as np
    t0 = time.perf_counter()
    if w.mode != 2:
        q = oracle.ramp_filter(sino, filter=w.filter)
        t1 = time.perf_counter()
        scale = (math.pi if w.mode == 0 else 2.0 * math.pi) / w.n_angles
        img = oracle.backproject(q, w.angles, w.axis, w.nx, w.ny, pixel_size=w.pixel_size, scale=scale)
    else:
        t1 = t0
        img = oracle.fbp(sino, w.angles, w.axis, w.nx, w.ny, pixel_size=w.pixel_size, filter=w.filter, mode=w.mode)
    t2 = time.perf_counter()
    oracle.forward_project(img.astype(np.float32), w.angles, w.axis, w.n_bins, pixel_size=w.pixel_size)
    t3 = time.perf_counter()
    return t3 - t0, t1 - t0, t2 - t1, t3 - t2


def cpu_baseline(wl_mod, args):
    import oracle
    oracle.build()
    w, sino = _oracle_sample(wl_mod, args)
    sec, sec_filter, sec_bp, sec_fp = _time_oracle_step(oracle, w, sino)
    upd = w.n_slices * w.nx * w.ny * w.n_angles
    # value = the metric's own quantity (backprojection updates / time of the oracle's backprojection); the oracle's
    # filter is the direct O(B^2) convolution (its definition, not an FFT), so the stages are listed one by one
    return {"value": upd / sec_bp / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "seconds": sec, "seconds_ramp_filter": sec_filter, "seconds_backproject": sec_bp,
            "seconds_forward_project": sec_fp, "step_gups": 2 * upd / sec / 1e9,
            "projector_pair_gups": 2 * upd / max(sec_bp + sec_fp, 1e-9) / 1e9,
            "sample": "%d of the config's slices at full size (%dx%d, %d projections x %d bins): oracle ramp filter "
                      "(direct O(B^2) convolution), backprojection and forward projection (fp64, OpenMP), one pass; "
                      "value = updates / backprojection seconds%s"
                      % (w.n_slices, w.ny, w.nx, w.n_angles, w.n_bins,
                         " (half acquisition: filter included, the oracle has one FBP routine for it)" if w.mode == 2 else "")}


def run_reference(args):
    """The oracle as it stands on the host cores, printing the SAME quantity as the b200 arm: backprojection updates
    per second of the backprojection stage.  config / metric / unit are the b200 arm's; each step is a bounded sample
    of that workload (cpu_baseline.sample says which).  --steps / --warmup are honoured as long as the run stays
    within --ref-seconds (default 200 s; estimated from the first step), else fewer steps are run and reported."""
    rank, world = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1)
    if rank != 0:
        return
    from paper_1306_1392_b200 import workloads as wl_mod
    import oracle
    oracle.build()
    w, sino = _oracle_sample(wl_mod, args)
    full = wl_mod.config(args.config, n_slices=args.slices or None)
    first = _time_oracle_step(oracle, w, sino)           # warm-up step 1 (or, with --warmup 0, timed step 1)
    fit = max(1, int(args.ref_seconds / max(first[0], 1e-9)))
    warmup = min(args.warmup, max(0, fit - 1))
    steps = max(1, min(args.steps, fit - warmup))
    runs = [first] if warmup == 0 else []
    for _ in range(max(0, warmup - 1)):
        _time_oracle_step(oracle, w, sino)
    while len(runs) < steps:
        runs.append(_time_oracle_step(oracle, w, sino))
    sec, sec_filter, sec_bp, sec_fp = [sum(r[k] for r in runs) / len(runs) for k in range(4)]
    upd = w.n_slices * w.nx * w.ny * w.n_angles
    val = upd / sec_bp / 1e9
    sample = ("each step = %d of %d slices of the config at full size: oracle ramp filter, backprojection, forward "
              "projection; value = that sample's backprojection updates / its backprojection seconds"
              % (w.n_slices, full.n_slices))
    line = {"impl": "reference", "metric": METRIC, "metric_version": METRIC_VERSION, "value": val, "unit": UNIT,
            "n_gpus": args.gpus, "steps": steps, "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _config_dict(full, 1),
            "reference": "oracle/ (fp64 CPU, OpenMP) on the host cores; " + sample,
            "metrics": {"backprojection_gups": val, "step_gups": 2 * upd / sec / 1e9,
                        "projector_pair_gups": 2 * upd / max(sec_bp + sec_fp, 1e-9) / 1e9,
                        "ms_ramp_filter": sec_filter * 1e3, "ms_backproject": sec_bp * 1e3,
                        "ms_forward_project": sec_fp * 1e3, "slices_timed_per_step": w.n_slices},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_extra(args):
    """Timings of the NEXT-row entry points that are not part of the hot-path step (profiles/r02_ncu_kernels.md
    sec. 5, 6): `--extra patch` = pyhst_patch_gradient on a config-4-sized problem (8 x 1024^2, 200 x 1024, 8 x 8 patches
    at stride 4, 128 atoms) with both GEMM kernels; `--extra estimators` = pyhst_ring_filter / pyhst_ecohe on
    config-2-sized operands.  One JSON line; CUDA events, `--steps` timed calls after `--warmup`."""
    import torch
    import paper_1306_1392_b200 as P
    wl = P.workloads

    def timeit(f):
        for _ in range(max(args.warmup, 1)):
            f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    out = {"extra": args.extra, "steps": args.steps, "warmup": args.warmup, "data": "synthetic"}
    if args.extra == "patch":
        w = wl.config(4)
        S, n, m, st, n_atoms = w.n_slices, w.nx, 8, 4, 128
        wl.set_device("cuda")
        data = w.sinogram_tensor(range(S)).contiguous()
        wl.set_device("cpu")
        D = torch.from_numpy(wl.dct_dictionary(m, n_atoms, seed=1)).cuda()
        na, nb = P.patch_grid(n, n, m, st)
        torch.manual_seed(0)
        W = (torch.randn((S, na * nb, n_atoms), device="cuda") * 0.01).contiguous()
        out["workload"] = "pyhst_patch_gradient: %d slices of %dx%d, %d x %d sinograms, %d patches of %dx%d per slice, %d atoms" \
                          % (S, n, n, w.n_angles, w.n_bins, na * nb, m, m, n_atoms)
        for variant, name in ((1, "ms_fp32_simt_gemm"), (2, "ms_tcgen05_3xtf32_gemm")):
            prev = P.set_patch_gemm_variant(variant)
            try:
                out[name] = timeit(lambda: P.patch_gradient(W, D, data, w.angles, w.axis, n, n, m, st, 0.8, want_f=False))
            finally:
                P.set_patch_gemm_variant(prev)
    else:
        S, NP, B, n = 16, 2000, 2048, 2048
        sino = torch.rand((S, NP, B), device="cuda")
        res = torch.empty_like(sino)
        a, b = torch.rand((S, n, n), device="cuda"), torch.rand((S, n, n), device="cuda")
        out["workload"] = "config-2-sized operands: %d x %d x %d sinogram stack, two %d x %dx%d image stacks" % (S, NP, B, S, n, n)
        t = timeit(lambda: P.ring_filter(sino, 8, out=res))
        out["ring_filter"] = {"ms": t, "gb_per_s": 3 * sino.numel() * 4 / t / 1e6, "bytes_counted": "3 x stack (mean pass, subtract pass in + out)"}
        t = timeit(lambda: P.ecohe(a, b))
        out["ecohe"] = {"ms": t, "gb_per_s": 2 * a.numel() * 4 / t / 1e6, "bytes_counted": "2 x stack; time includes the D2H of the results"}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number 1..5 (default 2)")
    ap.add_argument("--slices", type=int, default=0, help="override slices per GPU")
    ap.add_argument("--cpu-slices", type=int, default=1, help="slices in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-fista", action="store_true",
                    help="config 4: time FBP + forward projection instead of the 100-iteration TV-FISTA")
    ap.add_argument("--extra", default="", choices=["", "patch", "estimators"],
                    help="time pyhst_patch_gradient / the estimators instead of the hot-path step (see run_extra)")
    ap.add_argument("--ref-seconds", type=float, default=200.0,
                    help="--impl reference: time budget within which --steps / --warmup are honoured")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        sys.stderr.write("note: fewer than 3 warm-up steps; the number is not a valid bench value\n")
    if args.extra:
        run_extra(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
