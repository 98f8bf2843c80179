#!/usr/bin/env python
"""bench.py -- QTAM forward+inverse throughput on B200 through the C ABI (libqtam.so).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--batch B] [--impl reference]

A step is one pass of the whole hot path over one batch of synthetic strain: forward (long R2C,
window gather + baseband shift + short IFFT per row), [row-median threshold for cfg5], inverse
(per-row FFT, overlap reduction, 1/P, long C2R).  Default workload: BASELINE.json configs[2]
("cfg3": 256 x 4 s at 4096 Hz, complex64, forward+inverse), the first configuration that exercises
the forward+inverse metric; see DESIGN.md "Measurement".  One JSON line is printed by rank 0.

Timing: W >= 3 warm-up steps, then K steps each bracketed by CUDA events on the launch stream with an
L2 flush (a 512 MB device memset) before every step, outside the event brackets; barrier +
torch.cuda.synchronize() on both sides; max over ranks.  Multi-GPU: the batch shards over ranks with
no data-path collective (weak scaling: every rank gets its own `batch` segments).
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2603_29785_b200 import dist_utils, inputs  # noqa: E402

METRIC = "QTAM fwd+inv input samples/s"
UNIT = "samples/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="cfg3", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--batch", type=int, default=0, help="segments per GPU (default: the configuration's)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--overlap", type=float, default=1.0, help="clamp_overlap (R7); 1.0 = paper literal")
    ap.add_argument("--e2e-chunks", type=int, default=2, help="chunks of the batch pipelined over H2D | kernels | D2H")
    ap.add_argument("--no-largest-batch", action="store_true",
                    help="skip the extra pass at a batch of 8 segments per SM (SURVEY.md 8(d) 'largest batch')")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def measured_traffic(workload, batch, kernel):
    """dram__bytes_read + dram__bytes_write of one launch from the committed ncu --set full capture
    (profiles/r1_dram_traffic.csv, see the .md beside it); None when no capture matches this run."""
    path = os.path.join(ROOT, "profiles", "r1_dram_traffic.csv")
    try:
        with open(path) as f:
            for line in f.read().splitlines()[1:]:
                w, b, k, v = line.split(",")
                if w == workload and int(b) == batch and k == kernel:
                    return float(v)
    except Exception:
        pass
    return None


def compulsory_bytes_per_segment(cfg, ctot):
    """forward r*N + c*C_tot, inverse c*C_tot + r*N; threshold fused -> 0 extra, as a
    separate in-place pass 2*c*C_tot (what this build does today)."""
    r = 8 if cfg["dtype"] == "f64" else 4
    c = 2 * r
    n = cfg["N"]
    total = 0
    if "forward" in cfg["calls"]:
        total += r * n + c * ctot
    if "inverse" in cfg["calls"]:
        total += c * ctot + r * n
    return total


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons of one GPU with NVML while the timed region runs"""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, nm in names.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.005)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


# --------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on the host cores
# --------------------------------------------------------------------------------------------------
def oracle_step_fn(cfg, name, overlap, nseg):
    from oracle.qtam_ref import RefPlan, set_threads, threads
    # torchrun exports OMP_NUM_THREADS=1 for every rank; the baseline is "the oracle on the box's host cores"
    set_threads(len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
    plan = RefPlan(fs, N, Q, fmin, fmax, rows, clamp_overlap=overlap)
    x = inputs.make_batch(name, batch=nseg).astype(np.float64)

    def step():
        Y = plan.forward(x, engine=1)
        if "threshold" in cfg["calls"]:
            Y = plan.threshold(Y, 3.0)
        if "inverse" in cfg["calls"]:
            plan.inverse(Y, engine=1)

    return step, threads()


def time_oracle(cfg, name, overlap, budget_s=25.0, max_seg=None):
    """times the oracle's FFT-engine path on a bounded sample sized for about `budget_s` of work"""
    probe = 4
    step, cores = oracle_step_fn(cfg, name, overlap, probe)
    t0 = time.perf_counter(); step(); t1 = time.perf_counter() - t0
    nseg = int(max(probe, min(max_seg or 10 ** 9, probe * budget_s / max(t1, 1e-3))))
    nseg = min(nseg, 4096)
    step, cores = oracle_step_fn(cfg, name, overlap, nseg)
    t0 = time.perf_counter(); step(); dt = time.perf_counter() - t0
    return nseg * cfg["N"] / dt, cores, nseg, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = inputs.CONFIGS[args.workload]
    # each step a bounded sample of the workload: a few seconds of CPU work
    probe_step, cores = oracle_step_fn(cfg, args.workload, args.overlap, 4)
    t0 = time.perf_counter(); probe_step(); t1 = time.perf_counter() - t0
    total_steps = args.steps + args.warmup
    per_step_budget = max(0.5, min(4.0, 150.0 / max(total_steps, 1)))
    nseg = int(max(1, min(cfg["batch"], 4 * per_step_budget / max(t1, 1e-3))))
    step, cores = oracle_step_fn(cfg, args.workload, args.overlap, nseg)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    value = nseg * cfg["N"] / dt
    sample = f"{nseg} of {cfg['batch']} segments per step, oracle FFT engine (fp64), OpenMP"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args, cfg, nseg, None),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def workload_config(args, cfg, batch, plan):
    c = {
        "workload": f"{args.workload}: {batch} x {cfg['N']} samples at {cfg['fs']:g} Hz, "
                    f"Q-planes {cfg['Q']}, {cfg['rows']} rows each over {cfg['fmin']:g}-{cfg['fmax']:g} Hz, "
                    f"calls {'+'.join(cfg['calls'])}",
        "baseline_config_index": cfg["idx"] - 1,
        "batch_per_gpu": batch, "N": cfg["N"], "fs": cfg["fs"], "clamp_overlap": args.overlap,
        "l2_policy": "512 MB device memset before every timed step (outside the event brackets)",
    }
    if plan is not None:
        c["coeffs_per_segment"] = plan.ctot
        c["rows"] = plan.n_rows
    return c


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2603_29785_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the QTAM path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = inputs.CONFIGS[args.workload]
    batch = args.batch or cfg["batch"]
    dtype = cfg["dtype"]
    fs, N, Q, fmin, fmax, rows = inputs.plan_args(args.workload)
    plan = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype=dtype, max_batch=batch, clamp_overlap=args.overlap)
    rdt = torch.float64 if dtype == "f64" else torch.float32
    cdt = torch.complex128 if dtype == "f64" else torch.complex64

    # each rank gets its own segments (weak scaling, no collective on the data path)
    first, _ = dist_utils.shard_segments(rank, world, batch)
    x_np = inputs.make_batch(args.workload, batch=batch, first_segment=first)
    x_pin = torch.from_numpy(x_np).pin_memory()
    d_x = x_pin.to(dev)
    d_coef = torch.empty((batch, plan.ctot), dtype=cdt, device=dev)
    d_out = torch.empty((batch, N), dtype=rdt, device=dev)
    out_pin = torch.empty((batch, N), dtype=rdt).pin_memory()
    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)
    calls = cfg["calls"]
    launches = [0]

    def step():
        if "threshold" in calls:
            plan.forward_threshold(d_x, 3.0, out=d_coef)     # forward + row-median threshold, one call
        else:
            plan.forward(d_x, out=d_coef)
        launches[0] += plan.last_launch_count()
        if "inverse" in calls:
            plan.inverse(d_coef, out=d_out)
            launches[0] += plan.last_launch_count()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps, profile):
        plan.profile_enable(profile, max_launches=max(64, 64 * nsteps))
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
        launches[0] = 0
        barrier()
        for s, e in ev:
            flush.zero_()
            s.record()
            step()
            e.record()
        barrier()
        ms = sum(s.elapsed_time(e) for s, e in ev)
        stats = plan.profile_read() if profile else []
        plan.profile_enable(False)
        return ms, stats, launches[0]

    W = max(args.warmup, 3)
    for _ in range(W):
        step()
    torch.cuda.synchronize()

    # ---- the timed region: exactly K steps, each bracketed by CUDA events on the launch stream (-> value),
    # then the same K steps again with the library's launch profile on (two more events around every kernel
    # launch: about 8 % of a cfg3 step) for the per-kernel durations of the roofline line.  Clocks are
    # sampled across both passes.
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    ms_plain, _, n_launch = timed(args.steps, False)
    ms_total, stats, _ = timed(args.steps, True)
    clocks = sampler.stop()

    # context: the same step captured once into a CUDA graph and replayed (the calls neither allocate nor
    # synchronise), timed the same way
    ms_graph = None
    if world == 1:
        try:
            cg = torch.cuda.CUDAGraph()
            with torch.cuda.graph(cg):
                step()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            torch.cuda.synchronize()
            for s0, s1 in ev:
                flush.zero_()
                s0.record(); cg.replay(); s1.record()
            torch.cuda.synchronize()
            ms_graph = sum(a.elapsed_time(b) for a, b in ev) / args.steps
        except Exception as exc:      # reported, never fatal: the eager numbers above are the result
            ms_graph = f"capture failed: {exc}"

    # ---- end to end through the public API with host buffers (pinned), copies inside the timing.
    # The batch goes through in `--e2e-chunks` chunks on three streams (H2D | forward[+threshold]+inverse |
    # D2H), so that the PCIe copies of one chunk overlap the kernels of another; every step still copies
    # all of its inputs in and all of its results out.
    coef_pin = None
    if "inverse" not in calls:
        coef_pin = torch.empty((batch, plan.ctot), dtype=cdt).pin_memory()
    nch = max(1, min(args.e2e_chunks, batch))
    bounds = [(c * batch // nch, (c + 1) * batch // nch) for c in range(nch)]
    s_in, s_cmp, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    ev_in = [torch.cuda.Event() for _ in bounds]
    ev_cmp = [torch.cuda.Event() for _ in bounds]
    ev_out = [torch.cuda.Event() for _ in bounds]
    primed = [False]

    def e2e_step():
        for c, (lo, hi) in enumerate(bounds):
            with torch.cuda.stream(s_in):
                if primed[0]:
                    s_in.wait_event(ev_cmp[c])          # the previous step's kernels have read d_x[lo:hi]
                d_x[lo:hi].copy_(x_pin[lo:hi], non_blocking=True)
                ev_in[c].record(s_in)
            with torch.cuda.stream(s_cmp):
                s_cmp.wait_event(ev_in[c])
                if primed[0]:
                    s_cmp.wait_event(ev_out[c])         # the previous step's D2H has read the result buffer
                if "threshold" in calls:
                    plan.forward_threshold(d_x[lo:hi], 3.0, out=d_coef[lo:hi])
                else:
                    plan.forward(d_x[lo:hi], out=d_coef[lo:hi])
                launches[0] += plan.last_launch_count()
                if "inverse" in calls:
                    plan.inverse(d_coef[lo:hi], out=d_out[lo:hi])
                ev_cmp[c].record(s_cmp)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_cmp[c])
                if "inverse" in calls:
                    out_pin[lo:hi].copy_(d_out[lo:hi], non_blocking=True)
                else:
                    coef_pin[lo:hi].copy_(d_coef[lo:hi], non_blocking=True)
                ev_out[c].record(s_out)
        primed[0] = True

    def fork():
        cur = torch.cuda.current_stream()
        for s_ in (s_in, s_cmp, s_out):
            s_.wait_stream(cur)

    def join():
        cur = torch.cuda.current_stream()
        for s_ in (s_in, s_cmp, s_out):
            cur.wait_stream(s_)

    fork()
    for _ in range(3):
        e2e_step()
    join()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(3, min(args.steps, 50))
    e0.record()
    fork()
    for _ in range(n_e2e):
        e2e_step()
    join()
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1) / n_e2e
    # what came back over PCIe is what the device-resident path computes (kernels are deterministic)
    step()
    torch.cuda.synchronize()
    e2e_ok = bool(torch.equal(out_pin, d_out.cpu())) if "inverse" in calls else bool(torch.equal(coef_pin, d_coef.cpu()))
    h2d = x_pin.numel() * x_pin.element_size()
    d2h = (out_pin.numel() * out_pin.element_size()) if "inverse" in calls else (coef_pin.numel() * coef_pin.element_size())

    # ---- max over ranks
    ms_total, ms_plain, ms_e2e = dist_utils.max_over_ranks([ms_total, ms_plain, ms_e2e], device=dev)
    ms_step = ms_plain / args.steps
    units = world * batch * N
    value = dist_utils.aggregate_throughput(world, batch, N, ms_step)

    # ---- round-trip error against Pi_C x (verification outside the timed region; torch.fft is
    # used here only to build the projection, never on the product path)
    rt_err = None
    if "inverse" in calls and "threshold" not in calls:
        _, cover = plan.frame(-1)
        cov = torch.from_numpy(cover).to(dev)
        X = torch.fft.rfft(d_x.double(), dim=-1)
        proj = torch.fft.irfft(torch.where(cov[None, :], X, torch.zeros_like(X)), n=N, dim=-1)
        step()
        err = (d_out.double() - proj).norm(dim=-1) / proj.norm(dim=-1)
        rt_err = float(err.max().item())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, from the launch profile of the timed region
    peak, peak_src = measured_peaks()
    roof = None
    kernels = []
    if stats:
        tot_ms = sum(s["ms"] for s in stats)
        for s in sorted(stats, key=lambda s: -s["ms"]):
            avg_ms = s["ms"] / s["launches"]
            gbs = s["algo_bytes"] / s["launches"] / (avg_ms * 1e-3) / 1e9
            kernels.append({"name": s["name"], "launches_per_step": s["launches"] / args.steps,
                            "avg_ms": avg_ms, "share": s["ms"] / tot_ms, "algo_gbs": gbs,
                            "algo_bytes": s["algo_bytes"] / s["launches"]})
        top = kernels[0]
        roof = {"bound": "hbm", "kernel": top["name"], "achieved": top["algo_gbs"], "peak": peak,
                "unit": "GB/s", "frac": top["algo_gbs"] / peak,
                "traffic": measured_traffic(args.workload, batch, top["name"]),
                "algo_bytes_per_launch": top["algo_bytes"],
                "peak_source": peak_src, "avg_launch_ms": top["avg_ms"], "share_of_step": top["share"]}
    comp = compulsory_bytes_per_segment(cfg, plan.ctot) * batch
    path_gbs = comp / (ms_step * 1e-3) / 1e9

    # ---- the same step at a batch that fills every SM several times over ("largest batch")
    largest = None
    if world == 1 and not args.batch and not args.no_largest_batch and cfg["N"] <= 32768:
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        big = 8 * sms
        x_big = torch.from_numpy(inputs.make_batch(args.workload, batch=min(big, 2 * batch))).to(dev)
        x_big = x_big.repeat((big + x_big.shape[0] - 1) // x_big.shape[0], 1)[:big].contiguous()
        plan_b = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype=dtype, max_batch=big, clamp_overlap=args.overlap)
        c_big = torch.empty((big, plan_b.ctot), dtype=cdt, device=dev)
        o_big = torch.empty((big, N), dtype=rdt, device=dev)

        def step_big():
            if "threshold" in calls:
                plan_b.forward_threshold(x_big, 3.0, out=c_big)
            else:
                plan_b.forward(x_big, out=c_big)
            if "inverse" in calls:
                plan_b.inverse(c_big, out=o_big)

        for _ in range(3):
            step_big()
        torch.cuda.synchronize()
        nb = 10
        plan_b.profile_enable(True, max_launches=64 * nb)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nb)]
        for s0, e0_ in evs:
            flush.zero_()
            s0.record(); step_big(); e0_.record()
        torch.cuda.synchronize()
        ms_b = sum(a.elapsed_time(b) for a, b in evs) / nb
        st_b = plan_b.profile_read()
        plan_b.profile_enable(False)
        comp_b = compulsory_bytes_per_segment(cfg, plan_b.ctot) * big
        largest = {"batch": big, "ms_per_step": ms_b, "value": big * N / (ms_b * 1e-3), "unit": UNIT,
                   "path_gbs": comp_b / (ms_b * 1e-3) / 1e9, "path_frac_of_peak": comp_b / (ms_b * 1e-3) / 1e9 / peak,
                   "kernels": [{"name": k["name"], "avg_ms": k["ms"] / k["launches"],
                                "algo_gbs": k["algo_bytes"] / k["ms"] / 1e6,
                                "frac_of_peak": k["algo_bytes"] / k["ms"] / 1e6 / peak}
                               for k in sorted(st_b, key=lambda k: -k["ms"])]}
        plan_b.close()
        del x_big, c_big, o_big

    # ---- cuFFT (through torch.fft) on the same shapes, side by side as a reference only (north_star): the
    # long real transforms and one batched complex transform per length bucket -- cuFFT does the FFTs alone,
    # without the gather / window / shift, the overlap sum or 1/P, and writes one row per (plane, row)
    cufft = None
    if world == 1:
        def ev_time(fn, reps=10):
            fn(); torch.cuda.synchronize()
            tot = 0.0
            for _ in range(reps):
                flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record(); torch.cuda.synchronize()
                tot += a.elapsed_time(b)
            return tot / reps
        try:
            spec_t = torch.fft.rfft(d_x, dim=-1)
            cufft = {"rfft_ms": ev_time(lambda: torch.fft.rfft(d_x, dim=-1)),
                     "irfft_ms": ev_time(lambda: torch.fft.irfft(spec_t, n=N, dim=-1)), "buckets": []}
            hist = {}
            for r_ in plan.rows:
                hist[int(r_.M)] = hist.get(int(r_.M), 0) + 1
            tot_c2c = 0.0
            for M_, cnt in sorted(hist.items()):
                if batch * cnt * M_ * 8 > (6 << 30):
                    continue
                buf = torch.randn(batch * cnt, M_, dtype=cdt, device=dev)
                t_ = ev_time(lambda: torch.fft.ifft(buf, dim=-1))
                cufft["buckets"].append({"M": M_, "rows": cnt, "c2c_ms": t_})
                tot_c2c += t_
                del buf
            cufft["c2c_all_buckets_ms"] = tot_c2c
            cufft["note"] = "FFTs only, out of place, one launch per length; context, not the target"
            del spec_t
        except Exception as exc:
            cufft = {"unavailable": str(exc)}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, cores, nseg, dt = time_oracle(cfg, args.workload, args.overlap)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{nseg} segments of the same workload, one pass ({dt:.1f} s), oracle FFT engine fp64"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": W, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if dtype == "f32" else "f64", "data": "synthetic",
        "config": workload_config(args, cfg, batch, plan),
        "clocks": clocks,
        "e2e": {"value": units / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e, "chunks": nch,
                "equals_device_resident_result": e2e_ok},
        "gpu_launches": n_launch,
        "roofline": roof,
        "path": {"compulsory_bytes_per_step": comp, "achieved_gbs": path_gbs, "frac_of_peak": path_gbs / peak,
                 "frac_of_8tbs": path_gbs / 8000.0, "ms_per_step_with_launch_profile": ms_total / args.steps, "ms_per_step_cuda_graph": ms_graph},
        "kernels": kernels,
        "round_trip_err": rt_err,
        "largest_batch": largest,
        "cufft_side_by_side": cufft,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
