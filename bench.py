#!/usr/bin/env python
"""bench.py -- times the TOI hot path (steps a1..a7 of DESIGN.md: plane fit, rotation, weighting,
gridding, inverse FFT, correction + crop) on BASELINE.json configs[1]: one MeerKAT-shaped snapshot
(2016 baselines x 4096 channels x 4 pols, 2048^2 image, uniform weighting), seeded synthetic data.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 2]

Prints ONE JSON line (rank 0).  `value` = visibilities (baseline-channel samples) gridded per second
over all ranks with inputs resident in HBM; `e2e` = the same through the C ABI with pinned HOST
buffers (H2D of every input and D2H of the image inside the timed region); `roofline` = the
gridding kernel against the measured HBM copy rate; `cpu_baseline` = the fp64 oracle on the host
cores.  --impl reference times the oracle itself (the only "reference" this paper-only task has).
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


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=2, choices=[1, 2, 4, 5],
                    help="BASELINE.json config id (2 = configs[1], the metric's workload)")
    ap.add_argument("--weighting", default=None, choices=[None, "natural", "uniform"])
    ap.add_argument("--gridder", default="sliding", choices=["sliding", "pair7", "sliding7", "atomic"])
    ap.add_argument("--stream-snapshots", type=int, default=60,
                    help="length of the streamed (config-3-shaped) run reported under `stream`; 0 = skip")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-snapshots", type=int, default=3)
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
    return {"workload": "BASELINE.json configs[%d] %s: %d baselines x %d channels x %d pols, %dx%d image, "
                        "G=%d, W=7, %s weighting, seeded synthetic (synth.py)" %
                        (wl.config_id - 1, wl.name, wl.n_baselines, wl.n_chan, wl.n_pol, wl.image_size,
                         wl.image_size, 2 * wl.image_size, weighting),
            "samples_per_snapshot": wl.n_baselines * wl.n_chan,
            "input_bytes_per_snapshot": wl.n_baselines * wl.n_chan * wl.n_pol * 13 + wl.n_baselines * 24,
            "gridder": args.gridder,
            "l2": "inputs (%.0f MB) larger than the 126 MB L2; no flush needed" %
                  (wl.n_baselines * wl.n_chan * wl.n_pol * 13 / 1e6),
            "parallelism": "snapshots sharded over %d GPU(s), no collective" % world}


def oracle_snapshot_seconds(snap_np, wl, weighting, repeats):
    """The oracle as it stands (Tier G, fp64, OpenMP) on one snapshot, `repeats` times -> seconds each."""
    import oracle
    wt = oracle.UNIFORM if weighting == "uniform" else oracle.NATURAL
    times = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        rc, _, info, _ = oracle.image_gridded(snap_np["uvw_m"], snap_np["vis"], snap_np["weights"], snap_np["flags"],
                                              snap_np["chan_freq_hz"], wl.image_size, wl.cell_size_deg,
                                              weighting=wt, pol_a=0, pol_b=wl.n_pol - 1)
        times.append(time.perf_counter() - t0)
        assert rc == 0
    return times, int(info["n_gridded"]), oracle.num_threads()


def make_inputs(wl, device):
    from paper_2512_06254_b200 import synth
    return synth.make_snapshot(wl, 0, device=device)


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
    times, n_gridded, cores = oracle_snapshot_seconds(snap_np, wl, weighting, steps)
    ms = 1e3 * sum(times) / len(times)
    S = wl.n_baselines * wl.n_chan
    value = S / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": max(1, warm), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(wl, weighting, args, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": "%d full snapshot(s) of the workload, one per step" % steps},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


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
    gridder = {"sliding": toi.TOI_GRIDDER_SLIDING, "pair7": toi.TOI_GRIDDER_PAIR7, "sliding7": toi.TOI_GRIDDER_SLIDING7,
               "atomic": toi.TOI_GRIDDER_ATOMIC}[args.gridder]
    S = wl.n_baselines * wl.n_chan
    N = wl.image_size
    snap = make_inputs(wl, "cuda")            # seeded generator, on the device; every rank the same shape
    freq = snap["chan_freq_hz"].cpu()
    stream = torch.cuda.Stream()

    # ---------------- device-resident arm: `value` ----------------
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, freq, N, wl.cell_size_deg, weighting=wt,
                               pol_a=0, pol_b=wl.n_pol - 1, input_location=toi.TOI_MEM_DEVICE, device=local,
                               gridder=gridder)

    def step():
        toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)

    for _ in range(max(3, args.warmup)):
        step()
    toi.toi_plan_sync(plan)
    launches_per_step = toi.toi_last_launch_count(plan)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
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

    # ---------------- per-stage durations (CUDA events inside the library, on `stream`) ----------------
    stage_keys = ["ms_planefit", "ms_weight", "ms_grid", "ms_fft", "ms_crop", "ms_total", "ms_zero"]
    acc = {k: [] for k in stage_keys}
    info = None
    for _ in range(max(5, min(args.steps, 20))):
        _, info, _ = toi.toi_image_snapshot(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                            stream=stream, want_info=True)
        for k in stage_keys:
            acc[k].append(getattr(info, k))
    stages = {k: sum(v) / len(v) for k, v in acc.items()}
    stages_min = {k: min(v) for k, v in acc.items()}
    n_gridded = int(info.n_gridded)
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
    # near-coplanar 3-D mode (NEXT-2): N_slab x K Chebyshev-moment passes, parameters chosen from the
    # snapshot (Eqs. 25-27); the call synchronises once, so its own CUDA-event time is reported
    toi.toi_image_snapshot_3d(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
    t3d = []
    for _ in range(3):
        _, i3, _ = toi.toi_image_snapshot_3d(plan, snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"], stream=stream)
        t3d.append(i3["ms_total"])
    extra["mode_3d"] = {"ms": sum(t3d) / len(t3d), "n_slab": i3["n_slab"], "K": i3["K"], "passes": i3["n_passes"],
                        "phi_max": i3["phi_max"], "expansion_error": i3["expansion_error"]}
    toi.toi_plan_destroy(plan)
    # the grid's zero fill alone (same size, same API call the library uses), best of 5
    zbuf = torch.empty(4 * N * N * 2, dtype=torch.float32, device="cuda")   # G x G complex64
    zero_alone_ms = 1e9
    for _ in range(6):
        z0, z1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        z0.record(stream)
        with torch.cuda.stream(stream):
            zbuf.zero_()
        z1.record(stream)
        torch.cuda.synchronize()
        zero_alone_ms = min(zero_alone_ms, z0.elapsed_time(z1))
    del zbuf
    return dict(rank=rank, local=local, world=world, wl=wl, weighting=weighting, wt=wt, gridder=gridder, S=S, N=N,
                snap=snap, freq=freq, stream=stream, ms_step=ms_step, value=value, clocks=clocks, stages=stages,
                stages_min=stages_min, n_gridded=n_gridded, launches_per_step=launches_per_step,
                zero_alone_ms=zero_alone_ms, extra=extra)


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

    # streamed run (config-3-shaped): pinned replay pool -> copy stream -> compute stream, events only
    stream_res = None
    if args.stream_snapshots > 0 and r["rank"] == 0:
        def fill(idx, slot):
            slot.uvw_m = host["uvw_m"].data_ptr()
            slot.vis = host["vis"].data_ptr()
            slot.weights = host["weights"].data_ptr() if host["weights"] is not None else None
            slot.flags = host["flags"].data_ptr() if host["flags"] is not None else None
            return 0
        toi.toi_image_stream(plan, 4, fill)                     # warm-up
        st = toi.toi_image_stream(plan, args.stream_snapshots, fill)
        stream_res = {"snapshots": int(st["n_done"]), "ms_per_snapshot": st["gpu_ms"] / max(1, st["n_done"]),
                      "wall_ms_per_snapshot": 1e3 * st["wall_s"] / max(1, st["n_done"]),
                      "h2d_gbs": st["h2d_bytes"] / (st["gpu_ms"] * 1e-3) / 1e9,
                      "h2d_ms_mean": st["h2d_ms_sum"] / max(1, st["n_done"]),
                      "compute_ms_mean": st["compute_ms_sum"] / max(1, st["n_done"]),
                      "source": "replay pool of 1 pinned snapshot (DESIGN.md section 4); images stay on the GPU"}
        # the same stream with the output side on: re-projection of every image (interpolate stage)
        # and its D2H through the pinned ring to a host sink (copy_cpu stage)
        seen = []
        toi.toi_stream_set_output(plan, product=toi.TOI_OUT_REPROJECT_EXACT,
                                  host_sink=lambda idx, image: seen.append(idx), image_size=N)
        toi.toi_image_stream(plan, 4, fill)
        del seen[:]
        st = toi.toi_image_stream(plan, args.stream_snapshots, fill)
        stream_res["with_output"] = {
            "snapshots": int(st["n_done"]), "images_on_host": len(seen),
            "ms_per_snapshot": st["gpu_ms"] / max(1, st["n_done"]),
            "wall_ms_per_snapshot": 1e3 * st["wall_s"] / max(1, st["n_done"]),
            "h2d_gbs": st["h2d_bytes"] / (st["gpu_ms"] * 1e-3) / 1e9,
            "d2h_bytes_per_snapshot": st["d2h_bytes"] / max(1, st["n_done"]),
            "d2h_ms_mean": st["d2h_ms_sum"] / max(1, st["n_done"]),
            "what": "re-projected (exact) image of every snapshot delivered to a host callback"}
        toi.toi_stream_set_output(plan)
    toi.toi_plan_destroy(plan)
    return e2e, stream_res


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
# `ncu --set full` captures summarised under profiles/ (a recorded measurement of the same command,
# not something this run can observe).  The 134 MB grid zero fill is a separate cudaMemsetAsync and
# most of the reductions stay in the 126 MB L2 until the FFT reads them, hence the small write figure.
NCU_TRAFFIC = {
    ("2", "uniform", "sliding"): {"bytes": 471329280 + 5403136, "source": "profiles/r1_k_grid_pair8_full.txt"},
    ("2", "natural", "sliding"): {"bytes": 459540992 + 5927424, "source": "profiles/r1_k_grid_pair8_natural_full.txt"},
    ("2", "uniform", "pair7"): {"bytes": 473425920 + 5772032, "source": "profiles/r1_k_grid_pair_full.txt"},
    ("2", "uniform", "sliding7"): {"bytes": 461792768 + 6813696, "source": "profiles/r1_k_grid_sliding_full.txt"},
}


def ncu_traffic(args, weighting):
    t = NCU_TRAFFIC.get((str(args.workload), weighting, args.gridder))
    return None if t is None else t["bytes"]


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    r = run_ours(args)
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
    # gridding kernel (CUDA events on its stream, while the side stream zero-fills the next
    # snapshot's buffers under it) + the zero fill of one grid timed alone with CUDA events: the fill
    # overlaps the kernels of the previous snapshot, so its in-situ duration (ms_zero) is not a cost
    zero_alone_ms = r["zero_alone_ms"]
    grid_ms = r["stages"]["ms_grid"] + zero_alone_ms
    achieved = ab["gridding"] / (grid_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "%s (+ grid zero fill on the side stream)" % {"sliding": "k_grid_pair8", "pair7": "k_grid_pair", "sliding7": "k_grid_sliding", "atomic": "k_grid_atomic"}[args.gridder], "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "frac_of_8tbs_nominal": achieved / 8000.0,
                "peak_source": peak_src, "traffic": ncu_traffic(args, weighting),
                "algorithmic_bytes": ab["gridding"], "ms": grid_ms, "ms_kernel": r["stages"]["ms_grid"],
                "ms_zero_fill_alone": zero_alone_ms, "ms_zero_fill_in_situ": r["stages"]["ms_zero"], "ms_min": r["stages_min"]["ms_grid"],
                "vis_per_s": r["S"] / (grid_ms * 1e-3)}
    stages = {k: round(v, 5) for k, v in r["stages"].items()}
    if weighting == "uniform" and r["stages"]["ms_weight"] > 0:
        stages["density_gbs"] = ab["density"] / ((r["stages"]["ms_weight"] + 0.5 * zero_alone_ms) * 1e-3) / 1e9
    stages["fft_gbs_min_traffic"] = ab["fft_min"] / (r["stages"]["ms_fft"] * 1e-3) / 1e9
    stages["crop_gbs"] = ab["crop"] / (r["stages"]["ms_crop"] * 1e-3) / 1e9
    # NEXT rows, timed alone: N^2 x (4 read + 4 written) resp. (8 read + 4 written)
    n2 = float(r["N"]) ** 2
    stages["ms_reproject"] = round(r["extra"]["ms_reproject"], 5)
    stages["reproject_gbs"] = n2 * 8 / (r["extra"]["ms_reproject_min"] * 1e-3) / 1e9
    stages["ms_difference"] = round(r["extra"]["ms_difference"], 5)
    stages["difference_gbs"] = n2 * 12 / (r["extra"]["ms_difference_min"] * 1e-3) / 1e9
    stages["mode_3d"] = r["extra"]["mode_3d"]
    pcie = pinned_h2d_peak_gbs()
    e2e["pcie_peak_gbs_measured"] = pcie
    e2e["pcie_frac"] = e2e["h2d_gbs_per_gpu"] / pcie
    if stream_res is not None:
        stream_res["pcie_frac"] = stream_res["h2d_gbs"] / pcie
        stream_res["extrapolated_s_for_1500_snapshots"] = 1.5 * stream_res["ms_per_snapshot"]
    cpu = None
    if not args.no_cpu_baseline:
        snap_np = {k: (v.cpu().numpy() if v is not None else None) for k, v in r["snap"].items()}
        times, _, cores = oracle_snapshot_seconds(snap_np, wl, weighting, max(1, args.cpu_snapshots))
        sec = sum(times) / len(times)
        cpu = {"value": r["S"] / sec, "unit": UNIT, "cores": cores, "kind": "oracle", "ms_per_snapshot": sec * 1e3,
               "sample": "%d full snapshot(s) of the same workload (fp64 Tier G oracle, OpenMP)" % len(times)}
    line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": r["ms_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config_dict(wl, weighting, args, world),
            "e2e": e2e, "gpu_launches": r["launches_per_step"] * args.steps, "clocks": r["clocks"],
            "roofline": roofline, "cpu_baseline": cpu, "stages_ms": stages, "stream": stream_res,
            "n_gridded_per_snapshot": r["n_gridded"],
            "context": {"paper_ms_per_snapshot_h100_end_to_end": PAPER_MS_PER_SNAPSHOT_H100,
                        "note": "PAPER.md:456, 1770 bl x 1024 ch incl. FITS writing; not the target"}}
    print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
