#!/usr/bin/env python
"""bench.py -- throughput of the multi-view Richardson-Lucy hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

A *step* is one iteration of efficient-OSEM (eq. 109-112 with the compound kernels of eq. 105):
every view blurs psi, forms the quotient, back-projects it and updates psi (V view-updates,
8 kernel launches each).  The workload is BASELINE.json configs[3] (512x512x256, 7 views, PSFs
21x21x45: the volume north_star quotes its target on), seeded and synthetic (mvd_synth).  Metric: Gvoxel-view
updates/s = Nx*Ny*Nz*V*K / t / 1e9 on un-padded voxels, inputs resident in HBM, CUDA events on
the launching stream, max over ranks.  The path does not shard (OSEM is a strict sequence of
global FFTs): --gpus N runs N independent replicas, no collective on
the data path.

One JSON line on stdout (rank 0).  Extra objects: `roofline` (dominant kernel class, algorithmic
bytes / live CUDA-event time), `kernels` (every class), `cpu_baseline` (the fp64 oracle timed on
this box's host cores on a bounded sample), `e2e` (whole job through the public API from pinned
host buffers: H2D of the views, mvd_create, all iterations, D2H of the estimate).

`sustained`: the same step replayed back to back for >= 3 s (the board reaches its power cap), with its
own clock summary.  --impl reference times the oracle itself (rank 0 only): one view-update of
efficient-OSEM per step on the SAME workload (config 4 at full size: about 2 s per step on 16 cores).

Other workloads, each still one JSON line:
    --config 5                    BASELINE configs[4] whole (1024x1024x512, 6 views)
    --config 5 --blocked 256      the same volume as 256^3 blocks + halo r (mvd_deconvolve_blocked, 5 iterations)
    --config 5 --psf-sweep        one record per PSF box 9^3 ... 31x31x63 in "sweep"
    --mode view-parallel          combined efficient variant, views dealt over the ranks, one all-reduce(PRODUCT)
                                  per iteration; scaling "strong"
    --mode block-replicas         config 5 blocks dealt over the ranks (the paper's 2-GPU mode, L225); "strong"
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gvoxel-view updates/s per iteration (fp32)"
UNIT = "Gvv/s"
FALLBACK_HBM_GBS = 6650.0     # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
NOMINAL_HBM_GBS = 8000.0      # north_star's "roughly 8 TB/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------
# clocks: NVML sampling thread (falls back to nothing if NVML is unavailable)
# ------------------------------------------------------------------------------------------
REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
           0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
           0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}


class ClockSampler:
    def __init__(self, index, period=0.02):
        self.samples = []          # (t, sm_mhz, reasons_mask, power_w)
        self.period = period
        self.stop_flag = threading.Event()
        self.ok = False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                import torch
                uuid = "GPU-" + str(torch.cuda.get_device_properties(index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            log("[bench] NVML unavailable: %r" % (e,))
        self.th = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                try:
                    pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                except Exception:
                    pw = float("nan")
                self.samples.append((time.perf_counter(), float(mhz), int(mask), pw))
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.ok:
            self.th.start()

    def stop(self):
        self.stop_flag.set()
        if self.ok:
            self.th.join(timeout=2)

    def summary(self, t0, t1):
        inside = [s for s in self.samples if t0 <= s[0] <= t1]
        window = "timed region"
        if not inside:
            inside = self.samples[-3:]
            window = "nearest samples (timed region shorter than the sampling period)"
        if not inside:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0, "window": "none"}
        mask = 0
        for s in inside:
            mask |= s[2]
        reasons = [name for bit, name in REASONS.items() if mask & bit and name != "gpu_idle"]
        return {"sm_mhz": float(np.median([s[1] for s in inside])), "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(inside), "window": window,
                "power_w_max": float(np.nanmax([s[3] for s in inside]))}


# ------------------------------------------------------------------------------------------
# algorithmic bytes per launch of every kernel class
# ------------------------------------------------------------------------------------------
def algorithmic_bytes(dims, fft_dims):
    nx, ny, nz = dims
    mx, my, mz = fft_dims            # mx = complex half-row length
    row = 8 * mx                     # bytes of one complex work-buffer row
    n = nx * ny * nz
    return {
        "y_fwd": row * ny * nz + row * my * nz,
        "y_inv": row * my * nz + row * ny * nz,
        "z_conv": 2 * row * my * nz + row * my * mz,
        "x_quot": 2 * row * ny * nz + 4 * n,
        "x_update": 2 * row * ny * nz + 8 * n,
        "x_accum": 2 * row * ny * nz + 12 * n,
        "x_load": row * ny * nz + 4 * n,
    }


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel_class, k):
    """(dram bytes per launch of the class, source string) from the newest committed `ncu --set full`
    capture (profiles/r*_traffic.csv; its first line is a comment naming the commit it was taken at),
    or (None, None)."""
    import glob
    for p in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv")), reverse=True):
        try:
            lines = open(p).read().splitlines()
            stamp = lines[0].lstrip("# ").strip() if lines and lines[0].startswith("#") else "build not recorded"
            for line in lines:
                if line.startswith("#") or line.startswith("config"):
                    continue
                cfg, cls, val = line.split(",")
                if int(cfg) == k and cls == kernel_class:
                    return int(val), "%s (%s)" % (os.path.relpath(p, ROOT), stamp)
        except Exception:
            continue
    return None, None


# ------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------
def load_problem(k, rank, world, dist):
    """rank 0 draws the problem; with several ranks it is handed over through /tmp."""
    import mvd_synth
    if world == 1:
        return mvd_synth.make_problem(k)
    tmp = os.path.join(tempfile.gettempdir(), "mvd_bench_cfg%d_%s" % (k, os.environ.get("MASTER_PORT", "0")))
    if rank == 0:
        p = mvd_synth.make_problem(k)
        os.makedirs(tmp, exist_ok=True)
        for v, (a, b) in enumerate(zip(p.views, p.psfs)):
            np.save(os.path.join(tmp, "view%d.npy" % v), a)
            np.save(os.path.join(tmp, "psf%d.npy" % v), b)
        dist.barrier()
        return p
    dist.barrier()
    nv = len(mvd_synth.CONFIGS[k]["angles"])
    views = [np.load(os.path.join(tmp, "view%d.npy" % v)) for v in range(nv)]
    psfs = [np.load(os.path.join(tmp, "psf%d.npy" % v)) for v in range(nv)]
    rec = mvd_synth.CONFIGS[k]
    return mvd_synth.Problem(k, rec["dims"], rec["psf"], None, psfs, views, rec["iterations"], rec["variants"])


def max_over_ranks(values, world, dist, device):
    """Element-wise maximum of a list of floats over all ranks (the slowest replica sets the time)."""
    if world == 1:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def replica_throughput(world, units_per_replica_step, steps, ms):
    """Whole-job value of `world` independent replicas: all units of all ranks over the slowest rank's time."""
    return world * units_per_replica_step * steps / (ms * 1e-3) / 1e9


def cpu_baseline(prob, budget_s=12.0):
    """The oracle as it stands, on this box's host cores: whole view-updates of efficient-OSEM on
    the full volume until `budget_s` seconds are spent (at least one)."""
    from oracle import mvd_oracle as O
    cores = len(os.sched_getaffinity(0))
    o = O.Oracle(prob.views, prob.psfs, "osem")
    n = 0
    t0 = time.perf_counter()
    while n < prob.n_views:
        o.view_update(n)                                          # one line of eq. 109-112, as Oracle.iterate runs it
        n += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    nvox = float(np.prod(prob.dims))
    return {"value": nvox * n / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "first %d of %d view-updates of one efficient-OSEM iteration on the full %dx%dx%d volume "
                      "(fp64, scipy.fft with %d workers), %.1f s" % (n, prob.n_views, *prob.dims, cores, dt)}


SWEEP_BOXES = ((9, 9, 9), (13, 13, 27), (17, 17, 35), (21, 21, 45), (25, 25, 51), (31, 31, 63))   # BASELINE configs[4]


def sweep_psfs(k, box):
    """PSFs of config k's recipe on another box: sigma_xy = r_x / 4, sigma_z = r_z / 3.5."""
    import mvd_synth
    rec = mvd_synth.CONFIGS[k]
    sxy, sz = max((box[0] - 1) / 2 / 4.0, 0.5), max((box[2] - 1) / 2 / 3.5, 0.5)
    return [mvd_synth.gaussian_psf(box, sxy, sz, a) for a in rec["angles"]]


def other_configs(k_main, stream, peak, barrier, sampler, warmup):
    """The other BASELINE workloads, device-resident, for the `configs` array of the default line: configs 1-3
    (L2-resident: the DRAM fraction says little there, the Gvv/s is the figure), and config 5 whole when the GPU has
    the memory free.  One record each: graph replay, `warmup` warm-up iterations, then timed iterations under CUDA events
    on the library's stream.  The algorithmic bytes are SURVEY 8(d)'s formula with the build's FFT lengths."""
    import torch
    import mvd_synth
    import paper_1308_0730_b200 as mvd
    out = []
    for k in (1, 2, 3, 5):
        if k == k_main:
            continue
        rec = mvd_synth.CONFIGS[k]
        nvox, V = int(np.prod(rec["dims"])), len(rec["angles"])
        if k == 5:
            free = torch.cuda.mem_get_info()[0]
            if free < 60e9:
                out.append({"config": k, "skipped": "%.0f GB of HBM free, 60 GB wanted" % (free / 1e9)})
                continue
        t = time.perf_counter()
        prob = mvd_synth.make_problem(k)
        draw_s = time.perf_counter() - t
        dv = [torch.from_numpy(v).cuda() for v in prob.views]
        d = mvd.Deconvolver(dv, prob.psfs, variant="osem", stream=stream, use_graph=True)
        steps = 5 if k == 5 else 30
        for _ in range(max(3, warmup)):
            d.iterate(1)
        launches0 = d.launch_count
        ms, t0, t1 = time_steps(d, stream, steps, barrier)
        per = ms / steps
        alg = algorithmic_bytes(prob.dims, d.fft_dims)
        step_bytes = V * (2 * alg["y_fwd"] + 2 * alg["y_inv"] + 2 * alg["z_conv"] + alg["x_quot"] + alg["x_update"])
        gbs = step_bytes / (per * 1e-3) / 1e9
        out.append({"config": k, "workload": "%dx%dx%d, %d views, PSF %dx%dx%d, efficient-OSEM" % (*prob.dims, V, *prob.psf_dims),
                    "fft_dims": list(d.fft_dims), "steps": steps, "ms_per_step": per, "value": nvox * V / (per * 1e-3) / 1e9,
                    "unit": UNIT, "gpu_launches": d.launch_count - launches0,
                    "algorithmic_bytes_per_vv": step_bytes / (nvox * V), "achieved_gbs": gbs, "frac_of_measured": gbs / peak,
                    "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS,
                    "l2": ("work buffer %.0f MB: L2-resident, DRAM fraction not meaningful" if k < 4 else
                           "work buffer %.0f MB: streams from HBM") % (8 * np.prod(d.fft_dims[:2]) * prob.dims[2] / 1e6),
                    "workspace_gb": d.workspace_bytes / 1e9, "sm_mhz": sampler.summary(t0, t1)["sm_mhz"],
                    "draw_s": draw_s})
        log("[bench] config %d: %.3f ms per iteration" % (k, per))
        d.close()
        del d, dv, prob
        torch.cuda.empty_cache()
    return out


def time_steps(d, stream, steps, barrier):
    """CUDA-event time (ms) of `steps` calls of d.iterate(1) on the library's stream, plus the wall-clock window."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    e0.record(stream)
    for _ in range(steps):
        d.iterate(1)
    e1.record(stream)
    barrier()
    return e0.elapsed_time(e1), t0, time.perf_counter()


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1308_0730_b200 as mvd

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU path; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    mvd.load_library()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    k = args.config
    if args.mode == "block-replicas" or args.blocked or args.psf_sweep:
        k = args.config = 5 if args.config == 4 else args.config      # these are config-5 workloads (BASELINE configs[4])
    t = time.perf_counter()
    prob = load_problem(k, rank, world, dist)
    log("[bench] rank %d: config %d drawn in %.1f s" % (rank, k, time.perf_counter() - t))
    V, dims = prob.n_views, prob.dims
    nvox = float(np.prod(dims))

    host_views = [torch.from_numpy(v).pin_memory() for v in prob.views] if not (args.blocked or args.psf_sweep or args.mode != "replicas") \
        else [torch.from_numpy(v) for v in prob.views]
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dev_views = [h.to("cuda", non_blocking=True) for h in host_views]
    stream.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    peak, peak_src = hbm_peak()
    base = {"metric": METRIC, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "vs_baseline": None, "dtype": "f32", "data": "synthetic"}
    wl = "BASELINE configs[%d]: %dx%dx%d, %d views, PSF %dx%dx%d" % (k - 1, *dims, V, *prob.psf_dims)

    def emit(line):
        sampler.stop()
        if rank == 0:
            print(json.dumps(line), flush=True)
        if world > 1:
            dist.destroy_process_group()

    # ============================ view-parallel combined variant ============================
    if args.mode == "view-parallel":
        # eq. 104 + eq. 44 with the views dealt round-robin over the ranks: per iteration each
        # rank's partial product, ONE all-reduce(PRODUCT) of N floats over NCCL, the same root update everywhere
        if V < world:
            raise SystemExit("bench.py: view-parallel needs at least one view per rank (%d views, %d ranks)" % (V, world))
        mine = mvd.split_views(V, world, rank)
        d = mvd.ViewParallelDeconvolver([dev_views[v] for v in mine], prob.psfs, variant="efficient", rank=rank,
                                        world=world, group=None, stream=stream)
        for v in range(V):
            if v not in mine:
                dev_views[v] = None
        torch.cuda.empty_cache()
        for _ in range(args.warmup):
            d.iterate(1)
        launches0 = d.d.launch_count
        ms, t0, t1 = time_steps(d, stream, args.steps, barrier)
        launches = d.d.launch_count - launches0
        ms = max_over_ranks([ms], world, dist, "cuda")[0]
        stats = d.get_stats()
        if not np.isfinite(stats["flux"]):
            raise SystemExit("bench.py: non-finite estimate")
        line = dict(base, value=nvox * V * args.steps / (ms * 1e-3) / 1e9, ms_per_step=ms / args.steps, scaling="strong",
                    config={"workload": wl + ", combined efficient variant (MVD_EFFICIENT), one step = one iteration",
                            "fft_dims": list(d.d.fft_dims), "voxel_views_per_step": nvox * V,
                            "parallelism": "view-parallel x%d: views %s on rank 0; one all-reduce(PRODUCT) of %.0f MB per "
                                           "iteration" % (world, mine, nvox * 4 / 1e6),
                            "l2": "inputs larger than L2", "cuda_graph": False},
                    clocks=sampler.summary(t0, t1), gpu_launches=launches, e2e=None, roofline=None, flux=stats["flux"])
        d.close()
        return emit(line)

    # ============================ block-wise processing (config 5) ============================
    if (args.blocked and not args.psf_sweep) or args.mode == "block-replicas":
        # R13 / PAPER.md L943, L225: 256^3 blocks + halo r, every block an independent problem; with several ranks
        # the blocks are dealt round-robin (the paper's two-GPU mode) and no rank talks to another
        B = args.blocked or 256
        iters = prob.iterations
        kw = dict(block_rank=rank, block_world=world) if args.mode == "block-replicas" else {}
        reps = []
        for rep in range(1 + max(1, args.repeats)):                    # first pass = warm-up (allocator, attributes)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            t0 = time.perf_counter()
            e0.record(stream)
            out, launches = mvd.deconvolve_blocked(dev_views, prob.psfs, (B, B, B), iters, variant="osem", stream=stream, **kw)
            e1.record(stream)
            barrier()
            t1 = time.perf_counter()
            if rep:
                reps.append(e0.elapsed_time(e1))
            if not bool(torch.isfinite(out[::37, ::41, ::43]).all()):
                raise SystemExit("bench.py: non-finite estimate")
            del out
        ms = max_over_ranks([float(np.median(reps))], world, dist, "cuda")[0]
        nblocks = int(np.prod([-(-n // B) for n in dims]))
        replicas = args.mode != "block-replicas"
        units = nvox * V * iters * (world if replicas else 1)
        line = dict(base, steps=iters, warmup=1, value=units / (ms * 1e-3) / 1e9, ms_per_step=ms / iters,
                    scaling="weak" if replicas else "strong",
                    config={"workload": wl + ", efficient-OSEM as %d blocks of %d^3 + halo r (mvd_deconvolve_blocked: gather, "
                                             "per-shape contexts and precompute, %d iterations per block, paste); value counts "
                                             "the useful (un-padded, un-haloed) voxels" % (nblocks, B, iters),
                            "parallelism": ("replicas x%d" % world) if replicas else "blocks dealt round-robin over %d ranks, no collective" % world,
                            "l2": "inputs larger than L2", "cuda_graph": False, "ms_total": ms, "repeats": len(reps)},
                    clocks=sampler.summary(t0, t1), gpu_launches=launches, e2e=None, roofline=None)
        return emit(line)

    # ============================ PSF-size sweep (config 5, whole volume) ============================
    if args.psf_sweep:
        # the PSF size drives the padding (and the block overhead).  The views are those of the config-5
        # draw (timing does not depend on the values); only the PSF box handed to the library changes
        sweep = []
        for box in SWEEP_BOXES:
            psfs = sweep_psfs(k, box)
            if args.blocked:
                # the same sweep in block-wise mode, where the PSF half-size sets the halo and so the overhead (L240)
                B, iters, reps = args.blocked, prob.iterations, []
                for rep in range(1 + max(1, args.repeats)):            # first pass = warm-up
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    barrier()
                    e0.record(stream)
                    out, _ = mvd.deconvolve_blocked(dev_views, psfs, (B, B, B), iters, variant="osem", stream=stream)
                    e1.record(stream)
                    barrier()
                    if rep:
                        reps.append(e0.elapsed_time(e1))
                    del out
                halo = [(b - 1) // 2 for b in box]
                ext = float(np.prod([B + 2 * h for h in halo])) / B ** 3
                med = float(np.median(reps))
                sweep.append({"psf_box": list(box), "block": B, "halo": halo, "iterations": iters, "ms_total": med,
                              "ms_total_min_max": [min(reps), max(reps)],
                              "ms_per_step": med / iters, "value": nvox * V * iters / (med * 1e-3) / 1e9,
                              "extended_over_central_voxels_interior_block": ext})
                log("[bench] blocked sweep %s: %.1f ms" % (box, med))
                continue
            d = mvd.Deconvolver(dev_views, psfs, variant="osem", stream=stream, use_graph=True)
            for _ in range(args.warmup):
                d.iterate(1)
            ms, t0, t1 = time_steps(d, stream, args.steps, barrier)
            alg = algorithmic_bytes(dims, d.fft_dims)
            step_bytes = V * (2 * alg["y_fwd"] + 2 * alg["y_inv"] + 2 * alg["z_conv"] + alg["x_quot"] + alg["x_update"])
            per = ms / args.steps
            sweep.append({"psf_box": list(box), "fft_dims": list(d.fft_dims), "ms_per_step": per,
                          "value": nvox * V / (per * 1e-3) / 1e9, "algorithmic_bytes_per_vv": step_bytes / (nvox * V),
                          "achieved_gbs": step_bytes / (per * 1e-3) / 1e9,
                          "frac_of_measured": step_bytes / (per * 1e-3) / 1e9 / peak,
                          "frac_of_nominal_8TBs": step_bytes / (per * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
                          "workspace_gb": d.workspace_bytes / 1e9, "sm_mhz": sampler.summary(t0, t1)["sm_mhz"]})
            log("[bench] sweep %s: %.2f ms" % (box, per))
            d.close()
            del d
            torch.cuda.empty_cache()
        ref = [r for r in sweep if tuple(r["psf_box"]) == tuple(prob.psf_dims)] or sweep[-1:]
        line = dict(base, value=ref[0]["value"], ms_per_step=ref[0]["ms_per_step"], scaling="weak",
                    config={"workload": wl + " swept over PSF boxes 9^3 ... 31x31x63, efficient-OSEM, %s; `value` is the "
                                             "%dx%dx%d record" % (("as %d^3 blocks + halo r" % args.blocked) if args.blocked else "whole volume",
                                                                  *ref[0]["psf_box"]), "cuda_graph": not args.blocked,
                            "l2": "inputs larger than L2", "parallelism": "single GPU"},
                    clocks=sampler.summary(0, time.perf_counter()), gpu_launches=None, e2e=None, roofline=None, sweep=sweep,
                    peak_source=peak_src)
        return emit(line)

    # ============================ the headline workload: replicas of efficient-OSEM ============================
    use_graph = not args.no_graph
    t = time.perf_counter()
    d = mvd.Deconvolver(dev_views, prob.psfs, variant="osem", stream=stream, use_graph=use_graph)
    create_ms = (time.perf_counter() - t) * 1e3
    fft_dims = d.fft_dims
    workspace_gb = d.workspace_bytes / 1e9

    # ---- device-resident timing: W warm-up steps, then exactly K steps ---------------------------
    # The timed region replays each iteration as one CUDA graph (the library's use_graph option):
    # the same 8V kernel launches, without the host launch gaps.
    for _ in range(args.warmup):
        d.iterate(1)
    launches0 = d.launch_count
    ms, t0, t1 = time_steps(d, stream, args.steps, barrier)
    launches = d.launch_count - launches0
    clocks = sampler.summary(t0, t1)
    stats = d.get_stats()
    if not np.isfinite(stats["flux"]):
        raise SystemExit("bench.py: non-finite estimate")

    # ---- sustained: the same step back to back for >= sustained_s seconds (power cap reached) ----
    sustained = None
    if args.sustained_s > 0:
        n = max(args.steps, int(np.ceil(args.sustained_s * 1e3 / (ms / args.steps))))
        ms_s, s0, s1 = time_steps(d, stream, n, barrier)
        ms_s = max_over_ranks([ms_s], world, dist, "cuda")[0]
        sustained = {"steps": n, "seconds": ms_s * 1e-3, "ms_per_step": ms_s / n,
                     "value": replica_throughput(world, nvox * V, n, ms_s), "unit": UNIT, "clocks": sampler.summary(s0, s1)}

    # ---- the same K steps as plain launches with a CUDA-event pair around every launch: the
    #      per-kernel durations behind `kernels` and `roofline` (a graph cannot carry those events) --
    if use_graph:
        d.close()
        d = mvd.Deconvolver(dev_views, prob.psfs, variant="osem", stream=stream, use_graph=False)
        for _ in range(args.warmup):
            d.iterate(1)
    d.profile(True)
    ms_plain, _, _ = time_steps(d, stream, args.steps, barrier)
    classes = d.profile_read()
    d.profile(False)

    ms, ms_plain = max_over_ranks([ms, ms_plain], world, dist, "cuda")
    value = replica_throughput(world, nvox * V, args.steps, ms)

    # ---- roofline of the dominant kernel class --------------------------------------------------
    alg = algorithmic_bytes(dims, fft_dims)
    kernels = {}
    for name, (tms, n) in classes.items():
        if n:
            per = tms / n
            kernels[name] = {"launches": n, "avg_ms": per, "share": tms / ms_plain,
                             "algorithmic_bytes": alg[name], "achieved_gbs": alg[name] / (per * 1e-3) / 1e9}
    step_bytes = sum(alg[name] * kk["launches"] for name, kk in kernels.items()) / max(args.steps, 1)
    roofline = None
    if kernels:
        top = max(kernels, key=lambda n: kernels[n]["share"])
        a = kernels[top]["achieved_gbs"]
        traffic, traffic_src = ncu_traffic(top, k)
        roofline = {"bound": "hbm", "kernel": top, "achieved": a, "peak": peak, "unit": "GB/s", "frac": a / peak,
                    "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": alg[top],
                    "step": {"algorithmic_bytes": step_bytes,
                             "achieved": step_bytes / (ms / args.steps * 1e-3) / 1e9,
                             "frac_of_measured": step_bytes / (ms / args.steps * 1e-3) / 1e9 / peak,
                             "frac_of_nominal_8TBs": step_bytes / (ms / args.steps * 1e-3) / 1e9 / NOMINAL_HBM_GBS}}
        if sustained:
            sustained["achieved_gbs"] = step_bytes / (sustained["ms_per_step"] * 1e-3) / 1e9
            sustained["frac_of_measured"] = sustained["achieved_gbs"] / peak
            sustained["frac_of_nominal_8TBs"] = sustained["achieved_gbs"] / NOMINAL_HBM_GBS

    # ---- end to end from pinned host buffers, through the public API -----------------------------
    e2e = None
    e2e_timelapse = None
    if args.e2e_jobs > 0:
        iters = prob.iterations
        out_host = torch.empty(prob.views[0].shape, dtype=torch.float32).pin_memory()
        h2d = sum(h.numel() * 4 for h in host_views)
        d2h = out_host.numel() * 4
        d.close()
        del d, dev_views
        torch.cuda.empty_cache()

        copy_stream = torch.cuda.Stream()

        def job():
            # the views are copied on their own stream; mvd_create waits for them (views_ready) only
            # where it first reads them, so the copy overlaps the PSF precompute
            with torch.cuda.stream(copy_stream):
                dv = [h.to("cuda", non_blocking=True) for h in host_views]
                ready = torch.cuda.Event()
                ready.record(copy_stream)
            dd = mvd.Deconvolver(dv, prob.psfs, variant="osem", stream=stream, use_graph=use_graph,
                                 views_ready=ready)
            dd.iterate(iters)
            dd.get_estimate_host(out_host.numpy())
            dd.close()

        job()                                          # warm-up job (allocator, page-ins)
        barrier()
        tw0 = time.perf_counter()
        for _ in range(args.e2e_jobs):
            job()
        barrier()
        dt = time.perf_counter() - tw0
        dt = max_over_ranks([dt], world, dist, "cuda")[0]
        cold = {"value": world * nvox * V * iters * args.e2e_jobs / dt / 1e9, "unit": UNIT,
                "step": "one whole cold job: H2D of the %d views from pinned host memory, mvd_create (PSF precompute, "
                        "spectra; overlaps the H2D), %d iterations, D2H of the estimate; wall clock between "
                        "synchronisations" % (V, iters),
                "jobs": args.e2e_jobs, "ms_per_job": dt / args.e2e_jobs * 1e3}

        # ---- time-lapse stream (series of time-points with the same PSFs): two contexts created
        #      once, each with its own device view buffers; per time-point: H2D of its views into the buffers,
        #      mvd_restart, all iterations, D2H of the estimate.  The next time-point's H2D and the previous one's D2H
        #      overlap the current one's iterations; the contexts (PSF precompute) are paid once per series ----
        T = max(4, 3 * args.e2e_jobs)
        ctxs, outs = [], []
        for i in range(2):
            st = torch.cuda.Stream()
            with torch.cuda.stream(copy_stream):
                bufs = [h.to("cuda", non_blocking=True) for h in host_views]
                ready = torch.cuda.Event()
                ready.record(copy_stream)
            dd = mvd.Deconvolver(bufs, prob.psfs, variant="osem", stream=st, use_graph=use_graph, views_ready=ready)
            dd.iterate(1)                              # graph capture, first-use costs
            ctxs.append((dd, bufs))
            outs.append(torch.empty(prob.views[0].shape, dtype=torch.float32).pin_memory())
        barrier()                                      # the first-use iterations have read the view buffers

        def stream_series(n):
            pending, done = None, None
            for i in range(n):
                dd, bufs = ctxs[i % 2]
                if done is not None:                   # one time-point's kernels at a time: the other context's stream
                    dd.stream.wait_event(done)         # starts when the previous time-point's iterations have finished
                with torch.cuda.stream(copy_stream):
                    for b, h in zip(bufs, host_views):
                        b.copy_(h, non_blocking=True)
                    ready = torch.cuda.Event()
                    ready.record(copy_stream)
                dd.restart(ready)
                dd.iterate(iters)
                done = torch.cuda.Event()
                done.record(dd.stream)
                if pending is not None:                # blocks until time-point i-1 is done and copied out
                    pending[0].get_estimate_host(pending[1].numpy())
                pending = (dd, outs[i % 2])
            pending[0].get_estimate_host(pending[1].numpy())

        stream_series(2)                               # warm-up
        barrier()
        tw0 = time.perf_counter()
        stream_series(T)
        barrier()
        dts = max_over_ranks([time.perf_counter() - tw0], world, dist, "cuda")[0]
        for dd, _ in ctxs:
            dd.close()
        # `e2e` is the cold job (what one call of the public API costs, mvd_create included), as in round 1; the
        # time-lapse stream is reported beside it under its own key so that the two are never compared as one series
        e2e = dict(cold, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h)
        e2e_timelapse = {"value": world * nvox * V * iters * T / dts / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "step": "one time-point of a time-lapse series (same PSFs, PAPER.md L64/L242): H2D of its %d views from pinned "
                       "host memory into a context's view buffers, mvd_restart, %d iterations, D2H of the estimate into pinned "
                       "host memory; %d time-points through two contexts so that copies overlap the other context's "
                       "iterations; mvd_create is paid once per series and is outside the timed region (`e2e` is the "
                       "single job that includes it); wall clock between synchronisations" % (V, iters, T),
               "time_points": T, "ms_per_time_point": dts / T * 1e3}

    configs = None
    if world == 1 and k == 4 and not args.no_configs:
        configs = other_configs(k, stream, peak, barrier, sampler, args.warmup)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(prob)

    line = dict(base, value=value, ms_per_step=ms / args.steps, scaling="weak",
                config={"workload": wl + ", efficient-OSEM (MVD_OSEM + compound kernels), one step = one iteration",
                        "fft_dims": list(fft_dims), "voxel_views_per_step": nvox * V,
                        "parallelism": "replicas x%d (no data-path collective)" % world,
                        "l2": "inputs larger than L2 (one view-update streams %.1f GB)" % (step_bytes / V / 1e9 if kernels else 0.0),
                        "cuda_graph": bool(use_graph)},
                clocks=clocks, gpu_launches=launches, e2e=e2e, e2e_timelapse=e2e_timelapse, roofline=roofline, kernels=kernels, sustained=sustained,
                cpu_baseline=cpu, configs=configs, create_ms=create_ms, ms_per_step_plain_launches_with_events=ms_plain / args.steps,
                workspace_gb=workspace_gb, flux=stats["flux"])
    emit(line)


# ------------------------------------------------------------------------------------------
# reference arm: the oracle, on the host
# ------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    import mvd_synth
    from oracle import mvd_oracle as O

    k = args.config
    prob = mvd_synth.make_problem(k)                     # the SAME workload as our arm, at full size
    dims = prob.dims
    cores = len(os.sched_getaffinity(0))
    o = O.Oracle(prob.views, prob.psfs, "osem")
    V = prob.n_views
    nvox = float(np.prod(dims))

    for i in range(args.warmup):
        o.view_update(i % V)
    t0 = time.perf_counter()
    for i in range(args.steps):
        o.view_update((args.warmup + i) % V)
    dt = time.perf_counter() - t0
    value = nvox * args.steps / dt / 1e9
    sample = ("BASELINE configs[%d]: %dx%dx%d, %d views, PSF %dx%dx%d, efficient-OSEM; the oracle as it stands (fp64 "
              "numpy/scipy.fft, %d workers); each step is ONE view-update (1/%d of an iteration, views in index order) of "
              "the full volume" % (k - 1, *dims, V, *prob.psf_dims, cores, V))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": sample, "voxel_views_per_step": nvox},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE config number 1..5 (default 4, the target volume)")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "view-parallel", "block-replicas"],
                    help="what --gpus N ranks do (DESIGN.md section 10); default: N independent replicas of the OSEM workload")
    ap.add_argument("--blocked", type=int, default=0, metavar="B", help="config 5 as B^3 blocks + halo (mvd_deconvolve_blocked)")
    ap.add_argument("--psf-sweep", action="store_true", help="config 5 whole, one record per PSF box 9^3 ... 31x31x63")
    ap.add_argument("--repeats", type=int, default=3, help="timed repeats of the blocked job (median)")
    ap.add_argument("--sustained-s", type=float, default=3.0, help="seconds of back-to-back steps for the `sustained` leg (0 = skip)")
    ap.add_argument("--no-graph", action="store_true", help="time plain launches instead of one CUDA graph per iteration")
    ap.add_argument("--e2e-jobs", type=int, default=2)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-configs", action="store_true", help="skip the `configs` array (configs 1-3 and 5 beside the default config 4)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
