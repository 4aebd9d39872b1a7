#!/usr/bin/env python
"""bench.py -- throughput of the Dykstra projection hot path on B200 (one JSON line on stdout).

A "step" = one smre_project call = the whole hot path over one
synthetic workload.  Default workload = BASELINE.json configs[1]: 512x512, sides 1-8 (204
families), standard Dykstra, 200 sweeps.  Metric: Dykstra sweeps/s (window-projections/s is
reported beside it).  N > 1: replicas only -- every rank projects its own
image, no collective on the data path; value = sweeps of all ranks / max-over-ranks time.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--schedule auto|graph|conveyor]
  python bench.py --impl reference ...      # times the fp64 CPU oracle (rank 0 only)
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import smre_inputs as si  # noqa: E402

METRIC = "dykstra_sweeps_per_s"
UNIT = "sweeps/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


def profile_metric(workload_name, key):
    """A per-launch number taken from the committed ncu summaries (profiles/r02_measured.txt, written from the
    captures named there): DRAM traffic of the C1 kernel, thread-instructions of the ICD kernels.  None if absent."""
    p = os.path.join(ROOT, "profiles", "r02_measured.txt")
    try:
        d = json.load(open(p))
        return d.get(workload_name, {}).get(key), "profiles/r02_measured.txt (" + d.get("_source", "?") + ")"
    except (OSError, ValueError):
        return None, None


def cpu_info():
    """Host description printed beside the oracle timing."""
    model = "?"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    try:
        gcc = subprocess.run(["gcc", "--version"], capture_output=True, text=True).stdout.splitlines()[0]
    except (OSError, IndexError):
        gcc = "?"
    from oracle import smre_oracle
    return {"cpu_model": model, "nproc": os.cpu_count(), "compiler": gcc, "cflags": " ".join(smre_oracle.CFLAGS)}


def workload_numbers(w):
    """Per-step unit counts and algorithmic HBM bytes."""
    B, H, W = w.batch, w.H, w.W
    if w.variant == "standard":
        F = si.std_family_count(w.sides)
        wins = si.std_windows_per_sweep(H, W, w.sides) * B
        # q_f read + q_f write per pixel per family per sweep (x stays on chip / in L2),
        # + zeroing q once per call + x in / x out
        bytes_step = w.n_sweeps * F * B * H * W * 8 + F * B * H * W * 4 + 2 * B * H * W * 4
        passes = F
    else:
        K = int(np.floor(np.log2(max(w.sides))))
        wins = si.icd_windows_per_cycle(H, W, K) * B
        bytes_step = (K + 1) * B * H * W * 8
        passes = len(si.icd_level_passes(K))
    return {"families": passes, "windows_per_sweep": wins, "bytes_per_step": bytes_step}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def time_oracle(w, budget_sweeps):
    """The oracle as it stands, single thread, on a bounded sample of the workload."""
    from oracle import smre_oracle
    smre_oracle.build()
    y = w.y if w.y.ndim == 2 else w.y[0]
    t0 = time.perf_counter()
    smre_oracle.project(y, w.sides, w.c, budget_sweeps, w.variant)
    dt = time.perf_counter() - t0
    frames = "frame 0 of %d, " % w.batch if w.y.ndim == 3 else ""
    return budget_sweeps / dt, dt, \
        f"{frames}first {budget_sweeps} of {w.n_sweeps} sweeps of {w.name} ({w.H}x{w.W}), gcc -O2, 1 thread"


def run_reference(args, w, rank):
    if rank != 0:
        return
    nums = workload_numbers(w)
    sample_sweeps = max(1, min(w.n_sweeps, args.ref_sweeps))
    times = []
    for i in range(args.warmup + args.steps):
        v, dt, sample = time_oracle(w, sample_sweeps)
        if i >= args.warmup:
            times.append(dt)
    dt = float(np.mean(times))
    value = sample_sweeps / dt / w.batch          # whole job: all frames
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "note": w.note, "variant": w.variant, "n_sweeps": w.n_sweeps,
                   "step": f"bounded sample: {sample}"},
        "window_projections_per_s": value * nums["windows_per_sweep"],
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, **cpu_info()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_gpu(args, w, rank, world):
    import torch

    import paper_1503_03492_b200 as smre

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and this library has no CPU path")
    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    sched = {"auto": smre.SMRE_SCHED_AUTO, "graph": smre.SMRE_SCHED_GRAPH,
             "persistent": smre.SMRE_SCHED_PERSISTENT, "conveyor": smre.SMRE_SCHED_PERSISTENT,
             "strips": smre.SMRE_SCHED_STRIPS}[args.schedule]
    # N > 1: a stack of frames is split by frame (no collective; outputs stay on their rank), a single image is
    # replicated
    from paper_1503_03492_b200.replicas import shard_workload
    y_part, first_frame, frames_in_job, scaling = shard_workload(w.y, rank, world)
    frames_total = w.batch
    w.y = y_part
    nums = workload_numbers(w)
    sol = smre.Solver(w.H, w.W, w.sides, w.c, w.variant, w.batch, sched)
    stream = torch.cuda.Stream()
    y = torch.from_numpy(np.ascontiguousarray(w.y)).cuda()
    out = torch.empty_like(y)
    y_pin = torch.from_numpy(np.ascontiguousarray(w.y)).pin_memory()
    out_pin = torch.empty_like(y_pin).pin_memory()
    # Between timed iterations nothing useful survives in L2 for the standard variant: its q planes
    # (F*B*H*W*4 bytes, 204 MiB for C1) exceed the 126 MB L2 and are re-zeroed every call; for the
    # incomplete variant a >L2 scratch buffer is rewritten between steps.
    flush = None
    if w.variant != "standard" or sol.info[2] < 160 * 2 ** 20:
        flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    done = torch.zeros(max(w.batch, 1), dtype=torch.int32, device="cuda")

    def step_device():
        if args.tol is not None:
            smre.smre_project_tol(sol.handle, y.data_ptr(), out.data_ptr(), w.n_sweeps, args.tol, done.data_ptr(),
                                  stream.cuda_stream)
        else:
            smre.smre_project(sol.handle, y.data_ptr(), out.data_ptr(), w.n_sweeps, stream.cuda_stream)

    def step_host():
        smre.smre_project_host(sol.handle, y_pin.data_ptr(), out_pin.data_ptr(), w.n_sweeps, stream.cuda_stream)

    def timed(step_fn, n_warm, n_steps, sample_clocks):
        """Returns (wall seconds bracketing exactly n_steps, summed CUDA-event seconds of the steps)."""
        with torch.cuda.stream(stream):
            for _ in range(n_warm):
                if flush is not None:
                    flush.fill_(1)
                step_fn()
            barrier()
            sampler = ClockSampler(local) if sample_clocks else None
            if sampler:
                sampler.start()
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                   for _ in range(n_steps)]
            barrier()
            t0 = time.perf_counter()
            for a, b in evs:
                if flush is not None:
                    flush.fill_(1)
                a.record(stream)
                step_fn()
                b.record(stream)
            barrier()
            wall = time.perf_counter() - t0
            clocks = sampler.stop() if sampler else None
        dev = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
        return wall, dev, clocks

    wall, dev, clocks = timed(step_device, args.warmup, args.steps, rank == 0)
    launch = sol.last_launch
    wall_e, dev_e, _ = timed(step_host, max(1, args.warmup // 2), args.steps, False)

    from paper_1503_03492_b200.replicas import max_over_ranks as _max_over_ranks

    def max_over_ranks(v):
        return _max_over_ranks(v, dist, "cuda")

    dev, dev_e, wall_e = max_over_ranks(dev), max_over_ranks(dev_e), max_over_ranks(wall_e)
    # whole job: replicas multiply the work, frame shards split it (the metric counts sweeps of the job's call)
    sweeps_per_call = w.n_sweeps
    if args.tol is not None:                  # what the stop rule actually ran (the slowest frame / tile)
        torch.cuda.synchronize()
        sweeps_per_call = int(done.cpu().numpy()[:max(w.batch, 1) if w.variant == "standard" else 1].max())
    sweeps_total = sweeps_per_call * args.steps * (world if scaling == "weak" else 1)
    value = sweeps_total / dev
    e2e_value = sweeps_total / wall_e          # host-call wall time: the call blocks until the D2H copy is done

    if rank == 0:
        peak, peak_src, _ = measured_peaks()
        per_launch_s = dev / args.steps                       # persistent: one kernel = one step
        kernel = {smre.SMRE_SCHED_PERSISTENT: "conveyor_kernel", smre.SMRE_SCHED_STRIPS: "strips_kernel"}.get(
            launch[0], "family_pass_kernel")
        if w.variant != "standard":
            kernel = "icd_shift_kernel"
        achieved = nums["bytes_per_step"] / per_launch_s / 1e9
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": None, "peak_source": peak_src, "kernel": kernel,
                    "algorithmic_bytes_per_step": nums["bytes_per_step"],
                    "note": "achieved = dense-model bytes of one whole step (all launches of the step) / "
                            "CUDA-event time of the step; see DESIGN.md sec. 7"}
        if w.variant == "standard" and launch[0] == smre.SMRE_SCHED_STRIPS and w.n_sweeps == 200 and args.tol is None:
            # dram__bytes_read.sum + dram__bytes_write.sum of this launch, from the committed ncu --set full capture of
            # the same command; the kernel skips stores that would not change memory, so the dense-model fraction
            # (frac) and the fraction of the bytes actually moved (achieved_dram_frac) are both given
            t, src = profile_metric(w.name, "dram_bytes_per_launch")
            roofline["traffic"] = t
            roofline["traffic_source"] = src
            if t:
                roofline["achieved_dram_frac"] = t / per_launch_s / 1e9 / peak
        if w.variant != "standard":
            # ICD keeps q in registers: it is bound by instruction issue, not by HBM.  Numerator:
            # thread-instructions the shift kernels EXECUTE per call (ncu smsp__thread_inst_executed.sum of the
            # committed capture of this workload), not a model; peak = 148 SMs x 128 lanes x sm_max_mhz.
            _, _, sm_max = measured_peaks()
            lane_instr, src = profile_metric(w.name, "thread_inst_per_call")
            peak_alu = 148 * 128 * sm_max * 1e6
            roofline = {"bound": "alu", "achieved": (lane_instr / per_launch_s / 1e12) if lane_instr else None,
                        "peak": peak_alu / 1e12, "unit": "T lane-instr/s",
                        "frac": (lane_instr / per_launch_s / peak_alu) if lane_instr else None, "traffic": None,
                        "kernel": kernel, "hbm_frac": achieved / peak, "thread_inst_per_call": lane_instr,
                        "thread_inst_source": src,
                        "note": "executed thread-instructions per call (ncu) / time; peak = 148 SMs x 128 lanes x "
                                "sm_max_mhz; hbm_frac is reported so that nobody reads ICD as a bandwidth result"}
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            sample_sweeps = max(1, min(w.n_sweeps, args.ref_sweeps))
            v, dt, sample = time_oracle(w, sample_sweeps)
            cpu = {"value": v / w.batch, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                   "seconds": dt, **cpu_info()}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev / args.steps * 1e3, "higher_is_better": True,
            "scaling": scaling, "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "note": w.note, "variant": w.variant, "n_sweeps": w.n_sweeps,
                       "H": w.H, "W": w.W, "batch": frames_total, "frames_per_rank": w.batch,
                       "families": nums["families"],
                       "windows_per_sweep": nums["windows_per_sweep"],
                       "schedule": ("icd_shifts" if w.variant != "standard" else {1: "graph", 2: "conveyor", 3: "strips"}.get(launch[0], str(launch[0]))),
                       "tiles": [launch[2], launch[3]],
                       "l2": ("q planes (204 MiB for C1, > 126 MB L2) are rewritten by every step: nothing of a step survives "
                              "in L2 for the next one") if flush is None else "256 MiB flush between steps",
                       "parallelism": ("1 GPU" if world == 1 else
                                       "frames sharded over ranks, no collective" if scaling == "strong" else "replicas only")},
            "window_projections_per_s": value * nums["windows_per_sweep"] * (world if scaling == "strong" else 1),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(y_pin.numel() * 4),
                    "d2h_bytes_per_step": int(out_pin.numel() * 4), "ms_per_step": wall_e / args.steps * 1e3},
            "gpu_launches": int(launch[1]) * args.steps,
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
            "wall_ms_per_step": wall / args.steps * 1e3,
        }
        if args.tol is not None:
            dn = done.cpu().numpy()
            line["roofline"] = None           # the byte / instruction models above assume a fixed count
            line["config"]["stop_rule"] = {"tol": args.tol, "max_sweeps": w.n_sweeps,
                                           "iterations_done": [int(v) for v in (dn[:w.batch] if w.variant == "standard" else dn[:1])],
                                           "note": "smre_project_tol: Alg. 2 / Listing 3 stop rule decided on the device; value "
                                                   "counts the iterations of the slowest frame / tile; ms_per_step is the "
                                                   "time to convergence; e2e is the fixed-count host call and does not apply"}
        print(json.dumps(line), flush=True)
    sol.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_admm(args, w):
    """--admm N: N iterations of the ADMM around the projection (smre_admm, NEXT-2) on the config's image (first frame
    of a stack), App. B parameters, delta = 0 so that exactly N iterations run.  One GPU."""
    import torch
    import paper_1503_03492_b200 as smre
    torch.cuda.set_device(0)
    img = np.ascontiguousarray(w.y if w.y.ndim == 2 else w.y[0]).astype(np.float32)
    n_sweeps = args.n_sweeps or 20
    gamma = 8.0
    sol = smre.Solver(w.H, w.W, w.sides, w.c, w.variant, 1)
    I = torch.from_numpy(img).cuda()
    for _ in range(max(1, args.warmup)):
        smre.admm(sol, I, args.sigma, gamma=gamma, delta=0.0, max_iter=min(args.admm, 5), n_sweeps=n_sweeps)
    sampler = ClockSampler(0)
    sampler.start()
    torch.cuda.synchronize()
    evs = []
    t0 = time.perf_counter()
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        x, eps, it = smre.admm(sol, I, args.sigma, gamma=gamma, delta=0.0, max_iter=args.admm, n_sweeps=n_sweeps)
        b.record()
        evs.append((a, b))
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    clocks = sampler.stop()
    dev = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    iters = args.admm * args.steps
    # the projection alone, same handle and sweep count
    out = torch.empty_like(I)
    sol.project(I, n_sweeps, out=out)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(20):
        sol.project(I, n_sweeps, out=out)
    b.record()
    torch.cuda.synchronize()
    proj_ms = a.elapsed_time(b) / 20
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import smre_oracle
        t1 = time.perf_counter()
        smre_oracle.admm(img, w.sides, w.c.astype(np.float64), 0 if w.variant == "standard" else 1, n_sweeps, args.sigma,
                         6.192, 1.8, 1.2, 0.12, 1.0, gamma, 0.0, 2)
        dt = time.perf_counter() - t1
        cpu = {"value": 2 / dt, "unit": "iterations/s", "cores": 1, "kind": "oracle", "sample": "2 iterations of the same call",
               "seconds": dt, **cpu_info()}
    launches_per_iter = 6 + int(sol.last_launch[1])
    print(json.dumps({
        "metric": "admm_iterations_per_s", "value": iters / dev, "unit": "iterations/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dev / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name + "_admm", "variant": w.variant, "H": w.H, "W": w.W, "iterations_per_call": args.admm,
                   "n_sweeps_per_projection": n_sweeps, "sigma_psf": args.sigma, "gamma": gamma,
                   "parameters": "App. B: rho1 6.192, rho2 1.8, alpha1 1.2, alpha2 0.12, regularization 1",
                   "note": "smre_admm (NEXT-2): host-synchronous call, delta = 0"},
        "ms_per_iteration": dev / iters * 1e3, "projection_ms": proj_ms,
        "projection_share": proj_ms / (dev / iters * 1e3),
        "e2e": {"value": iters / wall, "unit": "iterations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 8,
                "note": "image resident; the call reads back the stop flag every 8 iterations"},
        "gpu_launches": launches_per_iter * iters, "clocks": clocks, "roofline": None, "cpu_baseline": cpu,
    }), flush=True)
    sol.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1)")
    ap.add_argument("--n-sweeps", type=int, default=None, help="override the config's sweep count (debug)")
    ap.add_argument("--schedule", default="auto", choices=["auto", "graph", "persistent", "conveyor", "strips"])
    ap.add_argument("--ref-sweeps", type=int, default=200, help="oracle sample size in sweeps (~12 s on C1)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--admm", type=int, default=None, help="time N iterations of smre_admm on the config's image instead")
    ap.add_argument("--sigma", type=float, default=1.5, help="PSF standard deviation of --admm")
    ap.add_argument("--tol", type=float, default=None,
                    help="run smre_project_tol with this tolerance (n_sweeps = max) and report the iterations done")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    w = si.config(args.config, args.n_sweeps)
    if args.impl == "reference":
        run_reference(args, w, rank)
        return
    if args.admm is not None:
        if rank == 0:
            run_admm(args, w)
        return
    run_gpu(args, w, rank, world)


if __name__ == "__main__":
    main()
