#!/usr/bin/env python
"""bench.py -- times the TOI hot path (steps a1..a7 of DESIGN.md: plane fit, rotation, weighting,
gridding, inverse FFT, correction + crop) on BASELINE.json configs[1]: one MeerKAT-shaped snapshot
(2016 baselines x 4096 channels x 4 pols, 2048^2 image, uniform weighting), seeded synthetic data.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 2]

Prints ONE JSON line (rank 0).  `value` = visibilities (baseline-channel samples) gridded per second
over all ranks with inputs resident in HBM; `e2e` = the same through the C ABI with pinned HOST
buffers (H2D of every input and D2H of the image inside the timed region); `roofline` = the
gridding kernel (+ the sparse clear of its grid) against the measured HBM copy rate;
`roofline_natural` / `stages_ms_natural` = the same workload under the paper's own natural weighting;
`workloads` = BASELINE.json configs[3] and configs[4] (natural); `stream` = configs[2], 1500 snapshots
through toi_image_stream from a pinned pool of distinct snapshots; `cpu_baseline` = the fp64 oracle on
the host cores.  --impl reference times the oracle itself (the only "reference" this paper-only task has).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

METRIC = "visibilities gridded per second, whole snapshot hot path (ms/snapshot in ms_per_step)"
UNIT = "vis/s"
PAPER_MS_PER_SNAPSHOT_H100 = 120.0   # PAPER.md:456, end to end incl. FITS writing: context only
STAGE_KEYS = ["ms_planefit", "ms_weight", "ms_grid", "ms_fft", "ms_crop", "ms_total", "ms_clear", "ms_clear_density"]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=2, choices=[1, 2, 4, 5],
                    help="BASELINE.json config id (2 = configs[1], the metric's workload)")
    ap.add_argument("--weighting", default=None, choices=[None, "natural", "uniform"])
    ap.add_argument("--gridder", default="sliding", choices=["sliding", "atomic"])
    ap.add_argument("--stream-snapshots", type=int, default=1500,
                    help="length of the streamed (configs[2]) run reported under `stream`; 0 = skip")
    ap.add_argument("--stream-pool", type=int, default=16,
                    help="distinct pinned snapshots the streamed run cycles through")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra-workloads", action="store_true",
                    help="skip the natural-weighting arm and configs[3] / configs[4]")
    ap.add_argument("--cpu-snapshots", type=int, default=2)
    return ap.parse_args()


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    return rank, local, world


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if (t0 is None or t >= t0 - 0.2) and (t1 is None or t <= t1 + 0.2)]
        rows = rows or [r for _, r in self.rows]
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                smax.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload(args):
    from paper_2512_06254_b200 import synth
    wl = synth.CONFIGS[args.workload]
    weighting = args.weighting or wl.weighting
    return wl, weighting


def algorithmic_bytes(wl, weighting):
    """what the method must move, per snapshot, given the MS layout."""
    S = wl.n_baselines * wl.n_chan
    G = 2 * wl.image_size
    per_sample = wl.n_pol * (8 + 4 + 1)                       # vis c64 + weight f32 + flag u8, per pol
    grid = G * G * 8
    out = {"samples": S, "input": S * per_sample, "grid": grid,
           "gridding": S * per_sample + grid,                  # every input byte once + grid written once
           "density": S * wl.n_pol * (4 + 1) + G * G * 4 if weighting == "uniform" else 0,
           # rows r+w, then r+w of the N of G = 2N columns the crop reads (pruned transform)
           "fft_min": 3 * grid, "crop": wl.image_size ** 2 * (8 + 4)}
    return out


def config_dict(wl, weighting, args, world):
    in_mb = wl.n_baselines * wl.n_chan * wl.n_pol * 13 / 1e6
    return {"workload": "BASELINE.json configs[%d] %s: %d baselines x %d channels x %d pols, %dx%d image, "
                        "G=%d, W=7, %s weighting, seeded synthetic (synth.py)" %
                        (wl.config_id - 1, wl.name, wl.n_baselines, wl.n_chan, wl.n_pol, wl.image_size,
                         wl.image_size, 2 * wl.image_size, weighting),
            "samples_per_snapshot": wl.n_baselines * wl.n_chan,
            "input_bytes_per_snapshot": wl.n_baselines * wl.n_chan * wl.n_pol * 13 + wl.n_baselines * 24,
            "gridder": args.gridder,
            "l2": "inputs (%.0f MB) + grid and FFT workspace (2 x %.0f MB) streamed every step: far larger than "
                  "the 126 MB L2; no flush needed" % (in_mb, (2 * wl.image_size) ** 2 * 8 / 1e6),
            "parallelism": "snapshots sharded over %d GPU(s), no collective" % world}


def oracle_snapshot_seconds(snap_np, wl, weighting, repeats, threads=None):
    """The oracle as it stands (Tier G, fp64, OpenMP) on one snapshot, `repeats` times -> seconds each,
    plus its own per-stage wall clock of the last call."""
    import oracle
    wt = oracle.UNIFORM if weighting == "uniform" else oracle.NATURAL
    all_cores = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    times, info = [], None
    try:
        for _ in range(repeats):
            t0 = time.perf_counter()
            rc, _, info, _ = oracle.image_gridded(snap_np["uvw_m"], snap_np["vis"], snap_np["weights"], snap_np["flags"],
                                                  snap_np["chan_freq_hz"], wl.image_size, wl.cell_size_deg,
                                                  weighting=wt, pol_a=0, pol_b=wl.n_pol - 1)
            times.append(time.perf_counter() - t0)
            assert rc == 0
        stages = {k: 1e3 * v for k, v in oracle.last_stage_seconds().items()}
        cores = oracle.num_threads()
    finally:
        if threads:
            oracle.set_num_threads(all_cores)
    return times, int(info["n_gridded"]), cores, stages


def make_inputs(wl, device, snapshot=0):
    from paper_2512_06254_b200 import synth
    return synth.make_snapshot(wl, snapshot, device=device)


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; rank 0 only."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    wl, weighting = workload(args)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    snap = make_inputs(wl, dev)
    snap_np = {k: (v.cpu().numpy() if v is not None else None) for k, v in snap.items()}
    del snap
    steps = max(1, min(args.steps, 20))
    warm = max(0, min(args.warmup, 1))
    oracle_snapshot_seconds(snap_np, wl, weighting, max(1, warm))
    times, n_gridded, cores, stages = oracle_snapshot_seconds(snap_np, wl, weighting, steps)
    ms = 1e3 * sum(times) / len(times)
    S = wl.n_baselines * wl.n_chan
    value = S / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": max(1, warm), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(wl, weighting, args, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "stages_ms": stages,
                             "sample": "%d full snapshot(s) of the workload, one per step" % steps},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def time_stages(toi, plan, snap, stream, reps):
    """Per-stage durations (CUDA events inside the library, on `stream`; every call synchronises)."""
    acc = {k: [] for k in STAGE_KEYS}
    info = None
    # warm-up of the timed path itself: a call with `info` launches the sparse clear as a kernel of its own,
    # which the untimed steps before never did (lazy module loading put 50-80 us into its first launch)
    for _ in range(2):
        toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream, want_info=True)
    for _ in range(reps):
        _, info, _ = toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                            stream=stream, want_info=True)
        for k in STAGE_KEYS:
            acc[k].append(getattr(info, k))
    return ({k: sum(v) / len(v) for k, v in acc.items()}, {k: min(v) for k, v in acc.items()}, int(info.n_gridded))


def time_3d(toi, plan, snap, stream, reps=3):
    """Near-coplanar 3-D mode (NEXT-2): N_slab x K Chebyshev-moment passes, parameters chosen from the
    snapshot (Eqs. 25-27); the call synchronises once, so its own CUDA-event time is reported."""
    toi.toi_image_snapshot_3d(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
    t3d, i3 = [], None
    for _ in range(reps):
        _, i3, _ = toi.toi_image_snapshot_3d(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
        t3d.append(i3["ms_total"])
    return {"ms": sum(t3d) / len(t3d), "ms_min": min(t3d), "n_slab": i3["n_slab"], "K": i3["K"], "passes": i3["n_passes"],
            "phi_max": i3["phi_max"], "expansion_error": i3["expansion_error"]}


def roofline_of(wl, weighting, stages, stages_min, peak, peak_src, kernel):
    """Gridding against the HBM roofline: algorithmic bytes (every input byte once + the grid once) over
    the gridding kernel + the sparse clear of its grid, both timed in situ with CUDA events.  Under
    uniform weighting the density map's clear is a launch of its own in the timed calls
    (ms_clear_density): it belongs to the density pass, whose algorithmic bytes hold that map's zero
    fill, and is charged there (density_gbs)."""
    ab = algorithmic_bytes(wl, weighting)
    grid_ms = stages["ms_grid"] + stages["ms_clear"]
    achieved = ab["gridding"] / (grid_ms * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": kernel + " + k_clear_tiles (sparse clear of the gridding grid)",
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "frac_of_8tbs_nominal": achieved / 8000.0, "peak_source": peak_src,
            "algorithmic_bytes": ab["gridding"], "ms": grid_ms, "ms_kernel": stages["ms_grid"],
            "ms_clear": stages["ms_clear"], "ms_kernel_min": stages_min["ms_grid"],
            "vis_per_s": ab["samples"] / (grid_ms * 1e-3)}


def run_side_workload(toi, wl, weighting, local, gridder, stream, steps, with_3d):
    """One more (workload, weighting) pair, device-resident: whole-step time + stages.  Rank 0 only."""
    snap = make_inputs(wl, "cuda")
    freq = snap["chan_freq_hz"].cpu()
    wt = toi.TOI_WEIGHT_UNIFORM if weighting == "uniform" else toi.TOI_WEIGHT_NATURAL
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, freq, wl.image_size, wl.cell_size_deg, weighting=wt,
                               pol_a=0, pol_b=wl.n_pol - 1, input_location=toi.TOI_MEM_DEVICE, device=local,
                               gridder=gridder, enable_3d=with_3d)
    try:
        def step():
            toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
        for _ in range(3):
            step()
        toi.toi_plan_sync(plan)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            step()
        e1.record(stream)
        torch.cuda.synchronize()
        ms_step = e0.elapsed_time(e1) / steps
        stages, stages_min, n_gridded = time_stages(toi, plan, snap, stream, max(5, min(steps, 20)))
        m3 = time_3d(toi, plan, snap, stream) if with_3d else None
    finally:
        toi.toi_plan_destroy(plan)
        del snap
        torch.cuda.empty_cache()
    return ms_step, stages, stages_min, n_gridded, m3


def run_ours(args):
    from paper_2512_06254_b200 import binding as toi
    from paper_2512_06254_b200 import shard
    rank, local, world = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: libtoi has no CPU fallback"
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    toi.load()
    wl, weighting = workload(args)
    wt = toi.TOI_WEIGHT_UNIFORM if weighting == "uniform" else toi.TOI_WEIGHT_NATURAL
    gridder = {"sliding": toi.TOI_GRIDDER_SLIDING, "atomic": toi.TOI_GRIDDER_ATOMIC}[args.gridder]
    S = wl.n_baselines * wl.n_chan
    N = wl.image_size
    snap = make_inputs(wl, "cuda")            # seeded generator, on the device; every rank the same shape
    freq = snap["chan_freq_hz"].cpu()
    stream = torch.cuda.Stream()

    # ---------------- device-resident arm: `value` ----------------
    with_3d = args.gridder != "atomic"
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, freq, N, wl.cell_size_deg, weighting=wt,
                               pol_a=0, pol_b=wl.n_pol - 1, input_location=toi.TOI_MEM_DEVICE, device=local,
                               gridder=gridder, enable_3d=with_3d)

    def step():
        toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)

    for _ in range(max(3, args.warmup)):
        step()
    toi.toi_plan_sync(plan)
    launches_per_step = toi.toi_last_launch_count(plan)
    sampler = ClockSampler(local)
    sampler.start()
    # the sampler needs ~0.3 s to come up; the GPU keeps working meanwhile (more untimed warm-up steps): a
    # timed region of a few ms that starts on a GPU that has just idled measures its clock ramp, not the path
    t_busy = time.time() + 0.3
    while time.time() < t_busy:
        for _ in range(50):
            step()
        torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    shard.barrier()
    torch.cuda.synchronize()
    t_wall0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    shard.barrier()
    t_wall1 = time.time()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop(t_wall0, t_wall1)
    ms_total, units = shard.reduce_timing(ms_total, float(S) * args.steps, device="cuda")
    ms_step = ms_total / args.steps
    value = units / (ms_total * 1e-3)

    stages, stages_min, n_gridded = time_stages(toi, plan, snap, stream, max(5, min(args.steps, 20)))
    # ---------------- NEXT rows, timed on their own (not part of `value`): re-projection of the
    # image just made with the snapshot's own V, and the difference of two ring images ----------------
    ptr_a, _, _ = toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
    ptr_b, _, _ = toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
    out_img = torch.empty((N, N), dtype=torch.float32, device="cuda")
    extra = {}
    for name, fn in (("ms_reproject", lambda: toi.toi_reproject(plan, ptr_b, out_img, stream=stream)),
                     ("ms_difference", lambda: toi.toi_difference(plan, ptr_b, ptr_a, out_img, stream=stream))):
        for _ in range(3):
            fn()
        best, tot, reps = 1e9, 0.0, 10
        for _ in range(reps):
            x0, x1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            x0.record(stream)
            fn()
            x1.record(stream)
            torch.cuda.synchronize()
            t = x0.elapsed_time(x1)
            best, tot = min(best, t), tot + t
        extra[name] = tot / reps
        extra[name + "_min"] = best
    del out_img
    if with_3d:
        extra["mode_3d"] = time_3d(toi, plan, snap, stream)
    toi.toi_plan_destroy(plan)
    return dict(rank=rank, local=local, world=world, wl=wl, weighting=weighting, wt=wt, gridder=gridder, S=S, N=N,
                snap=snap, freq=freq, stream=stream, ms_step=ms_step, value=value, clocks=clocks, stages=stages,
                stages_min=stages_min, n_gridded=n_gridded, launches_per_step=launches_per_step, extra=extra)


def pinned_h2d_peak_gbs(n_bytes=1 << 30, repeats=5):
    """This box's pinned host->device copy rate: the PCIe roofline of the e2e / streamed numbers."""
    h = torch.empty(n_bytes, dtype=torch.uint8).pin_memory()
    d = torch.empty(n_bytes, dtype=torch.uint8, device="cuda")
    best = 0.0
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        d.copy_(h, non_blocking=True)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, n_bytes / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    del h, d
    return best


def run_e2e(r, args):
    """Same metric through the C ABI with HOST (pinned) buffers: every step copies its inputs H2D and
    reads the image back D2H inside the timed region."""
    from paper_2512_06254_b200 import binding as toi
    from paper_2512_06254_b200 import shard
    from paper_2512_06254_b200 import synth
    wl, snap, stream, N = r["wl"], r["snap"], r["stream"], r["N"]
    host = {k: (snap[k].cpu().pin_memory() if snap[k] is not None else None)
            for k in ("uvw_m", "vis", "weights", "flags")}
    h2d = sum(t.numel() * t.element_size() for t in host.values() if t is not None)
    d2h = N * N * 4
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, r["freq"], N, wl.cell_size_deg, weighting=r["wt"],
                               pol_a=0, pol_b=wl.n_pol - 1, input_location=toi.TOI_MEM_HOST, device=r["local"],
                               gridder=r["gridder"])
    out = torch.empty((N, N), dtype=torch.float32).pin_memory()

    def step():
        ptr, _, _ = toi.toi_image_snapshot(plan, host["uvw_m"], host["vis"], host["weights"], host["flags"],
                                           stream=stream)
        toi.toi_copy_image_to_host(plan, ptr, N, out=out)

    steps = max(3, min(args.steps, 20))
    for _ in range(3):
        step()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    shard.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    shard.barrier()
    ms = max(e0.elapsed_time(e1), wall_ms)          # the D2H is synchronous: wall clock bounds it
    ms, units = shard.reduce_timing(ms, float(r["S"]) * steps, device="cuda")
    e2e = {"value": units / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / steps, "steps": steps,
           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "h2d_gbs_per_gpu": h2d * steps / (ms * 1e-3) / 1e9}

    # streamed run, BASELINE.json configs[2]: `--stream-snapshots` (1500) consecutive toi_image_stream
    # snapshots fed from a pinned pool of `--stream-pool` DISTINCT snapshots of the run (evenly spaced
    # indices: hour angle advancing, pulsar on and off), generated on the GPU by the seeded generator
    # and copied into pinned host memory before the timed region; pinned ring -> copy stream ->
    # compute stream, events only.  1500 x 429.5 MB cannot be held, so the stream cycles through the pool.
    stream_res = None
    if args.stream_snapshots > 0 and r["rank"] == 0 and wl.config_id == 2:
        w3 = synth.CONFIG3
        n_pool = max(1, min(args.stream_pool, args.stream_snapshots))
        idxs = sorted({int(round(k * (w3.n_snapshots - 1) / max(1, n_pool - 1))) for k in range(n_pool)})
        pool = []
        t_gen = time.perf_counter()
        for i in idxs:
            d = make_inputs(w3, "cuda", snapshot=i)
            pool.append({k: (d[k].cpu().pin_memory() if d[k] is not None else None)
                         for k in ("uvw_m", "vis", "weights", "flags")})
            del d
        torch.cuda.empty_cache()
        t_gen = time.perf_counter() - t_gen

        def fill(idx, slot):
            h = pool[idx % len(pool)]
            slot.uvw_m = h["uvw_m"].data_ptr()
            slot.vis = h["vis"].data_ptr()
            slot.weights = h["weights"].data_ptr() if h["weights"] is not None else None
            slot.flags = h["flags"].data_ptr() if h["flags"] is not None else None
            return 0
        toi.toi_image_stream(plan, 4, fill)                     # warm-up
        st = toi.toi_image_stream(plan, args.stream_snapshots, fill)
        n_done = max(1, int(st["n_done"]))
        stream_res = {"workload": "BASELINE.json configs[2] meerkat_stream: config 2's layout, %d snapshots 2 s apart, "
                                  "on/off 5 mJy pulsar, uniform weighting" % w3.n_snapshots,
                      "snapshots": int(st["n_done"]), "ms_per_snapshot": st["gpu_ms"] / n_done,
                      "seconds_total_gpu_events": st["gpu_ms"] * 1e-3, "seconds_total_wall": st["wall_s"],
                      "wall_ms_per_snapshot": 1e3 * st["wall_s"] / n_done,
                      "h2d_gbs": st["h2d_bytes"] / (st["gpu_ms"] * 1e-3) / 1e9,
                      "h2d_ms_mean": st["h2d_ms_sum"] / n_done,
                      "compute_ms_mean": st["compute_ms_sum"] / n_done,
                      "pool": {"distinct_snapshots": len(pool), "snapshot_indices": idxs,
                               "pinned_bytes": len(pool) * h2d, "generate_s": t_gen},
                      "source": "pinned pool of distinct seeded snapshots, cycled (DESIGN.md section 4); images stay on the GPU"}
        # the same stream with the output side on: re-projection of every image (interpolate stage)
        # and its D2H through the pinned ring to a host sink (copy_cpu stage)
        seen = []
        n_out = max(4, min(args.stream_snapshots, 300))
        toi.toi_stream_set_output(plan, product=toi.TOI_OUT_REPROJECT_EXACT,
                                  host_sink=lambda idx, image: seen.append(idx), image_size=N)
        toi.toi_image_stream(plan, 4, fill)
        del seen[:]
        st = toi.toi_image_stream(plan, n_out, fill)
        stream_res["with_output"] = {
            "snapshots": int(st["n_done"]), "images_on_host": len(seen),
            "ms_per_snapshot": st["gpu_ms"] / max(1, st["n_done"]),
            "wall_ms_per_snapshot": 1e3 * st["wall_s"] / max(1, st["n_done"]),
            "h2d_gbs": st["h2d_bytes"] / (st["gpu_ms"] * 1e-3) / 1e9,
            "d2h_bytes_per_snapshot": st["d2h_bytes"] / max(1, st["n_done"]),
            "d2h_ms_mean": st["d2h_ms_sum"] / max(1, st["n_done"]),
            "what": "re-projected (exact) image of every snapshot delivered to a host callback"}
        toi.toi_stream_set_output(plan)
        del pool
    toi.toi_plan_destroy(plan)
    return e2e, stream_res


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel: read off the
# `ncu --set full` capture named in `source` (a recorded measurement of the same command line, taken
# on `date`; this run cannot observe DRAM counters itself).  The sparse clear is a separate launch,
# and most of the reductions stay in the 126 MB L2 until the FFT reads them, hence the small write figure.
NCU_TRAFFIC = {
    ("2", "uniform", "sliding"): {"bytes": 471379456 + 6023680, "source": "profiles/r2_k_grid_pair8_c2_uniform_full.txt",
                                  "date": "round 2, commit 88344db (the kernel this run times)"},
    ("2", "natural", "sliding"): {"bytes": 459376640 + 5765376, "source": "profiles/r2_k_grid_pair8_c2_natural_full.txt",
                                  "date": "round 2, commit 88344db (the kernel this run times)"},
    ("4", "natural", "sliding"): {"bytes": 4022963000 + 106629376, "source": "profiles/r2_k_grid_pair8_c4_natural_full.txt",
                                  "date": "round 2, commit 88344db (the kernel this run times)"},
    ("2", "uniform", "atomic"): {"bytes": 454289920 + 15841024, "source": "profiles/r2_k_grid_atomic_c2_uniform_full.txt",
                                 "date": "round 2, commit d446d56"},
}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    from paper_2512_06254_b200 import binding as toi
    from paper_2512_06254_b200 import synth
    r = run_ours(args)
    pcie_before = pinned_h2d_peak_gbs() if r["rank"] == 0 else 0.0
    e2e, stream_res = run_e2e(r, args)
    rank, world, wl, weighting = r["rank"], r["world"], r["wl"], r["weighting"]
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()
        return
    ab = algorithmic_bytes(wl, weighting)
    peak, peak_src = measured_peaks()
    kernel = {"sliding": "k_grid_pair8", "atomic": "k_grid_atomic"}[args.gridder]
    roofline = roofline_of(wl, weighting, r["stages"], r["stages_min"], peak, peak_src, kernel)
    tr = NCU_TRAFFIC.get((str(args.workload), weighting, args.gridder))
    roofline["traffic"] = None if tr is None else tr["bytes"]
    roofline["traffic_source"] = None if tr is None else "%s, %s" % (tr["source"], tr["date"])
    stages = {k: round(v, 5) for k, v in r["stages"].items()}
    if weighting == "uniform" and r["stages"]["ms_weight"] > 0:
        stages["density_gbs"] = ab["density"] / ((r["stages"]["ms_weight"] + r["stages"]["ms_clear_density"]) * 1e-3) / 1e9
    stages["fft_gbs_min_traffic"] = ab["fft_min"] / (r["stages"]["ms_fft"] * 1e-3) / 1e9
    stages["crop_gbs"] = ab["crop"] / (r["stages"]["ms_crop"] * 1e-3) / 1e9
    # NEXT rows, timed alone: N^2 x (4 read + 4 written) resp. (8 read + 4 written)
    n2 = float(r["N"]) ** 2
    stages["ms_reproject"] = round(r["extra"]["ms_reproject"], 5)
    stages["reproject_gbs"] = n2 * 8 / (r["extra"]["ms_reproject_min"] * 1e-3) / 1e9
    stages["ms_difference"] = round(r["extra"]["ms_difference"], 5)
    stages["difference_gbs"] = n2 * 12 / (r["extra"]["ms_difference_min"] * 1e-3) / 1e9
    stages["mode_3d"] = r["extra"].get("mode_3d")
    # the pinned-copy rate of a fresh 1 GiB buffer varies by 2-4 % from allocation to allocation (where
    # the pinned pages land): measured before and after the e2e / streamed runs, the better one is the roofline
    pcie = max(pcie_before, pinned_h2d_peak_gbs())
    e2e["pcie_peak_gbs_measured"] = pcie
    e2e["pcie_frac"] = e2e["h2d_gbs_per_gpu"] / pcie
    if stream_res is not None:
        stream_res["pcie_frac"] = stream_res["h2d_gbs"] / pcie

    # ---------------- the paper's own weighting on the same workload, and the other configs ----------------
    line_extra = {}
    if not args.no_extra_workloads and args.workload == 2:
        other = "natural" if weighting == "uniform" else "uniform"
        ms_o, st_o, stmin_o, ng_o, _ = run_side_workload(toi, wl, other, r["local"], r["gridder"], r["stream"],
                                                         args.steps, False)
        line_extra["ms_per_step_" + other] = ms_o
        line_extra["stages_ms_" + other] = {k: round(v, 5) for k, v in st_o.items()}
        rf = roofline_of(wl, other, st_o, stmin_o, peak, peak_src, kernel)
        tro = NCU_TRAFFIC.get((str(args.workload), other, args.gridder))
        rf["traffic"] = None if tro is None else tro["bytes"]
        rf["traffic_source"] = None if tro is None else "%s, %s" % (tro["source"], tro["date"])
        line_extra["roofline_" + other] = rf
        wls = []
        for cid in (4, 5):
            w = synth.CONFIGS[cid]
            ms_w, st_w, stmin_w, ng_w, m3 = run_side_workload(toi, w, "natural", r["local"], r["gridder"], r["stream"],
                                                              max(5, min(args.steps, 10)), cid == 5 and args.gridder != "atomic")
            rw = roofline_of(w, "natural", st_w, stmin_w, peak, peak_src, kernel)
            entry = {"workload": config_dict(w, "natural", args, 1)["workload"], "ms_per_step": ms_w,
                     "value": w.n_baselines * w.n_chan / (ms_w * 1e-3), "unit": UNIT,
                     "stages_ms": {k: round(v, 5) for k, v in st_w.items()}, "n_gridded": ng_w,
                     "ms_grid": st_w["ms_grid"], "ms_clear": st_w["ms_clear"], "frac": rw["frac"],
                     "frac_of_8tbs_nominal": rw["frac_of_8tbs_nominal"], "achieved_gbs": rw["achieved"],
                     "algorithmic_bytes": rw["algorithmic_bytes"]}
            if m3 is not None:
                entry["mode_3d"] = m3
            wls.append(entry)
        line_extra["workloads"] = wls

    cpu = None
    if not args.no_cpu_baseline:
        snap_np = {k: (v.cpu().numpy() if v is not None else None) for k, v in r["snap"].items()}
        times, _, cores, st_all = oracle_snapshot_seconds(snap_np, wl, weighting, max(1, args.cpu_snapshots))
        sec = sum(times) / len(times)
        t1, _, _, st_one = oracle_snapshot_seconds(snap_np, wl, weighting, 1, threads=1)
        cpu = {"value": r["S"] / sec, "unit": UNIT, "cores": cores, "kind": "oracle", "ms_per_snapshot": sec * 1e3,
               "stages_ms": {k: round(v, 2) for k, v in st_all.items()},
               "one_thread": {"ms_per_snapshot": t1[0] * 1e3, "value": r["S"] / t1[0],
                              "stages_ms": {k: round(v, 2) for k, v in st_one.items()}},
               "sample": "%d full snapshot(s) of the same workload on all cores + 1 on one thread "
                         "(fp64 Tier G oracle, OpenMP; its own per-stage wall clock)" % len(times)}
    line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": r["ms_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config_dict(wl, weighting, args, world),
            "e2e": e2e, "gpu_launches": r["launches_per_step"] * args.steps, "clocks": r["clocks"],
            "roofline": roofline, "cpu_baseline": cpu, "stages_ms": stages, "stream": stream_res,
            "n_gridded_per_snapshot": r["n_gridded"],
            "context": {"paper_ms_per_snapshot_h100_end_to_end": PAPER_MS_PER_SNAPSHOT_H100,
                        "note": "PAPER.md:456, 1770 bl x 1024 ch incl. FITS writing; not the target"}}
    line.update(line_extra)
    print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
