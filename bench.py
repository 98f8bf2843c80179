#!/usr/bin/env python
"""bench.py -- QTAM forward+inverse throughput on B200 through the C ABI (libqtam.so).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--batch B] [--impl reference]

A step is one pass of the whole hot path over one batch of synthetic strain: forward (long R2C,
window gather + baseband shift + short IFFT per row), [row-median threshold for cfg5], inverse
(per-row FFT, overlap reduction, 1/P, long C2R).  Default workload: BASELINE.json configs[3]
("cfg4": 16 x 64 s at 16384 Hz, N = 2^20, complex64, forward+inverse), the largest single-GPU
configuration (2.93 GB of compulsory traffic per step); the same run also times configs 2, 3, 5 and the
fp64 variant of 5, each at its own batch and at a larger one.  See DESIGN.md "Measurement".  Rank 0 prints ONE
compact JSON line (under 2 KB: the contract's keys, roofline, e2e, cpu_baseline) as the last line of stdout;
the per-kernel tables and the records of the other configurations go to gpurun_out/bench_detail.json
(`--detail`), whose path the line carries.

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
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="cfg4", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--batch", type=int, default=0, help="segments per GPU (default: the configuration's)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--overlap", type=float, default=1.0, help="clamp_overlap (R7); 1.0 = paper literal")
    ap.add_argument("--e2e-chunks", type=int, default=2, help="chunks of the batch pipelined over H2D | kernels | D2H")
    ap.add_argument("--no-largest-batch", action="store_true",
                    help="skip the extra passes at a batch scaled up until throughput saturates (SURVEY.md 8(d))")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the records of the other BASELINE configurations (`configs` in the JSON line)")
    ap.add_argument("--dtype", default="", choices=["", "f32", "f64"], help="override the configuration's dtype")
    ap.add_argument("--time-layout-calls", type=int, default=0, metavar="B",
                    help="also time qtam_forward_length / qtam_resample / qtam_inverse_length at the paper's image shape "
                         "(62 x 669 minimal, 62 x 12289 standard, PAPER.md:343) on B segments; goes to the detail file")
    ap.add_argument("--detail", default=os.path.join("gpurun_out", "bench_detail.json"),
                    help="where the per-kernel tables and the records of the other configurations go")
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


def csrc_hash():
    """sha256 (first 16 hex digits) over the kernel sources: a DRAM-traffic capture is only valid for the
    sources it was taken from"""
    import hashlib
    d = os.path.join(ROOT, "paper_2603_29785_b200", "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".hpp", ".cpp")):
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def measured_traffic(workload, batch, kernel):
    """(dram__bytes_read + dram__bytes_write of one launch, source) from the committed ncu --set full captures
    profiles/r*_dram_traffic.csv (see the .md beside each), newest round first.  A row counts only if it was
    captured from the very kernel sources of this run (csrc hash) at this workload and batch: (None, why)
    otherwise -- ncu cannot run inside a timed bench, so the number can only come from a capture, never from
    this process."""
    import glob
    want = csrc_hash()
    seen = False
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_dram_traffic.csv")), reverse=True):
        try:
            with open(path) as f:
                for line in f.read().splitlines()[1:]:
                    w, b, k, v, sha = line.split(",")[:5]
                    if w == workload and int(b) == batch and k == kernel:
                        seen = True
                        if sha == want:
                            return float(v), f"profiles/{os.path.basename(path)} (ncu --set full, csrc {sha})"
        except Exception:
            pass
    return None, ("capture is from other kernel sources (csrc hash mismatch)" if seen
                  else "no ncu capture for this workload / batch / kernel")


def compulsory_bytes_per_segment(cfg, ctot):
    """forward r*N + c*C_tot, inverse c*C_tot + r*N; the threshold moves no compulsory bytes
    (float plans run it in the forward's epilogue; as a separate in-place pass it is design traffic)."""
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


HEADLINE_LIMIT = 2048      # bytes: the driver keeps a bounded tail of stdout and parses the last line


def headline_json(line):
    """the ONE line rank 0 prints last: the contract's keys, the roofline of the top kernel, cpu_baseline and
    e2e, compact separators, floats rounded to 6 significant digits.  Per-kernel tables, the other configurations
    and the largest-batch records go to the detail file (write_detail), never into this line: round 2's line grew
    to 23 KB and the driver could not parse it.  Raises if the line would not fit HEADLINE_LIMIT."""
    def rnd(v):
        if isinstance(v, float):
            return float(f"{v:.6g}")
        if isinstance(v, dict):
            return {k: rnd(x) for k, x in v.items()}
        if isinstance(v, (list, tuple)):
            return [rnd(x) for x in v]
        return v
    text = json.dumps(rnd(line), separators=(",", ":"))
    if len(text) >= HEADLINE_LIMIT:
        raise ValueError(f"bench.py headline is {len(text)} bytes (limit {HEADLINE_LIMIT}): move keys to the detail file")
    return text


def write_detail(path, detail):
    """per-kernel tables, largest-batch and other-configuration records as indented JSON; returns the path
    written relative to the repo root (or why it was not written: the headline never depends on it)"""
    try:
        full = path if os.path.isabs(path) else os.path.join(ROOT, path)
        os.makedirs(os.path.dirname(full), exist_ok=True)
        with open(full, "w") as f:
            json.dump(detail, f, indent=1)
        return os.path.relpath(full, ROOT)
    except Exception as exc:
        return f"not written: {exc}"


def time_layout_calls(torch, binding, dev, nseg, flush):
    """the paper's output-length calls (include/qtam.h says they are direct sums, a layout converter and
    not a step of the hot path) at the paper's own shape: ms per call on `nseg` segments, CUDA events, L2 flushed"""
    fs, N, Q, fmin, fmax, rows = inputs.plan_args("paper6s")
    out = {"segments": nseg, "N": N}
    x = torch.from_numpy(inputs.make_batch("paper6s", batch=min(nseg, 8))).to(dev).repeat((nseg + 7) // 8, 1)[:nseg].contiguous()

    def ev(fn, reps=3):
        fn(); torch.cuda.synchronize()
        tot = 0.0
        for _ in range(reps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            tot += a.elapsed_time(b)
        return tot / reps
    for mode in ("minimal", "standard"):
        g = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype="f32", max_batch=nseg, out_length=mode)
        n = g.output_length()
        img = g.forward_length(x)
        rec = {"rows": g.n_rows, "n": n, "forward_length_ms": ev(lambda: g.forward_length(x)),
               "inverse_length_ms": ev(lambda: g.inverse_length(img))}
        if mode == "minimal":
            rec["resample_to_standard_ms"] = ev(lambda: g.resample(img, to_standard=True))
        rec["image_bytes"] = img.numel() * img.element_size()
        out[mode] = rec
        del img
        g.close()
    return out


def workload_config(args, cfg, batch, plan):
    c = {
        "workload": f"{args.workload}: {batch} x {cfg['N']} samples at {cfg['fs']:g} Hz, "
                    f"Q-planes {cfg['Q']}, {cfg['rows']} rows each over {cfg['fmin']:g}-{cfg['fmax']:g} Hz, "
                    f"calls {', '.join(cfg['calls'])}",
        "baseline_config_index": cfg["idx"] - 1,
        "batch_per_gpu": batch, "N": cfg["N"], "fs": cfg["fs"], "clamp_overlap": args.overlap,
        "l2_policy": "512 MB device memset before every timed step (outside the event brackets)",
    }
    return c


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------
LARGEST = {"cfg2": 592, "cfg3": 1184, "cfg4": 48, "cfg5": 4096}   # batches at which throughput has saturated


class Workload:
    """one configuration at one batch on this rank: plan, device buffers, the step, timing helpers"""

    def __init__(self, torch, binding, dev, name, dtype, batch, overlap, first_segment=0, x_np=None):
        self.torch, self.name, self.dtype, self.batch, self.dev = torch, name, dtype, batch, dev
        self.cfg = dict(inputs.CONFIGS[name], dtype=dtype)
        fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
        self.N = N
        self.plan = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype=dtype, max_batch=batch, clamp_overlap=overlap)
        self.rdt = torch.float64 if dtype == "f64" else torch.float32
        self.cdt = torch.complex128 if dtype == "f64" else torch.complex64
        if x_np is None:
            x_np = inputs.make_batch(name, batch=batch, first_segment=first_segment, dtype=dtype)
        elif x_np.shape[0] < batch:       # a larger batch re-uses the generated segments (the path is data-oblivious)
            x_np = np.tile(x_np, ((batch + x_np.shape[0] - 1) // x_np.shape[0], 1))[:batch]
        self.x_np = np.ascontiguousarray(x_np[:batch])
        self.d_x = torch.from_numpy(self.x_np).to(dev)
        self.d_coef = torch.empty((batch, self.plan.ctot), dtype=self.cdt, device=dev)
        self.d_out = torch.empty((batch, N), dtype=self.rdt, device=dev)
        self.calls = self.cfg["calls"]
        self.launches = 0

    def step(self, lo=0, hi=None):
        p, hi = self.plan, self.batch if hi is None else hi
        if "threshold" in self.calls:
            p.forward_threshold(self.d_x[lo:hi], 3.0, out=self.d_coef[lo:hi])   # forward + row-median threshold
        else:
            p.forward(self.d_x[lo:hi], out=self.d_coef[lo:hi])
        self.launches += p.last_launch_count()
        if "inverse" in self.calls:
            p.inverse(self.d_coef[lo:hi], out=self.d_out[lo:hi])
            self.launches += p.last_launch_count()

    def timed(self, nsteps, profile, flush, barrier):
        """nsteps steps, each bracketed by CUDA events on the launch stream with an L2 flush before it (outside
        the brackets); returns (sum of ms, per-kernel stats, launches)"""
        torch = self.torch
        self.plan.profile_enable(profile, max_launches=max(64, 64 * nsteps))
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
        self.launches = 0
        barrier()
        for s, e in ev:
            flush.zero_()
            s.record()
            self.step()
            e.record()
        barrier()
        ms = sum(s.elapsed_time(e) for s, e in ev)
        stats = self.plan.profile_read() if profile else []
        self.plan.profile_enable(False)
        return ms, stats, self.launches

    def compulsory_bytes(self):
        return compulsory_bytes_per_segment(self.cfg, self.plan.ctot) * self.batch

    def round_trip_err(self):
        """worst segment of |inverse(forward(x)) - Pi_C x| / |Pi_C x| (verification outside the timed region;
        torch.fft only builds the projection, it is never on the product path)"""
        torch = self.torch
        if "inverse" not in self.calls or "threshold" in self.calls:
            return None
        _, cover = self.plan.frame(-1)
        cov = torch.from_numpy(cover).to(self.dev)
        self.step()
        worst = 0.0
        for b0 in range(0, self.batch, 64):
            xs = self.d_x[b0:b0 + 64].double()
            X = torch.fft.rfft(xs, dim=-1)
            proj = torch.fft.irfft(torch.where(cov[None, :], X, torch.zeros_like(X)), n=self.N, dim=-1)
            err = (self.d_out[b0:b0 + 64].double() - proj).norm(dim=-1) / proj.norm(dim=-1)
            worst = max(worst, float(err.max().item()))
        return worst

    def close(self):
        self.plan.close()
        del self.d_x, self.d_coef, self.d_out


def kernel_table(stats, nsteps, peak):
    """per kernel: launches per step, average launch duration, share of the summed kernel time, compulsory
    (algo) and design bytes per launch and the rates they imply"""
    out = []
    tot_ms = sum(s["ms"] for s in stats) or 1.0
    for s in sorted(stats, key=lambda s: -s["ms"]):
        avg_ms = s["ms"] / s["launches"]
        algo, design = s["algo_bytes"] / s["launches"], s["design_bytes"] / s["launches"]
        out.append({"name": s["name"], "launches_per_step": s["launches"] / nsteps, "avg_ms": avg_ms,
                    "share": s["ms"] / tot_ms, "algo_bytes": algo, "design_bytes": design,
                    "algo_gbs": algo / (avg_ms * 1e-3) / 1e9, "frac_of_peak": algo / (avg_ms * 1e-3) / 1e9 / peak,
                    "design_gbs": design / (avg_ms * 1e-3) / 1e9})
    return out


def record(w, nsteps, warmup, flush, barrier, peak):
    """ms per step, samples/s, fraction of the HBM roofline on compulsory bytes and the per-kernel table"""
    for _ in range(max(3, warmup)):
        w.step()
    w.torch.cuda.synchronize()
    ms_plain, _, n_launch = w.timed(nsteps, False, flush, barrier)
    ms_prof, stats, _ = w.timed(nsteps, True, flush, barrier)
    ms = ms_plain / nsteps
    comp = w.compulsory_bytes()
    gbs = comp / (ms * 1e-3) / 1e9
    return {"batch": w.batch, "dtype": w.dtype, "steps": nsteps, "ms_per_step": ms,
            "value": w.batch * w.N / (ms * 1e-3), "unit": UNIT, "compulsory_bytes_per_step": comp,
            "path_gbs": gbs, "path_frac_of_peak": gbs / peak, "gpu_launches_per_step": n_launch / nsteps,
            "ms_per_step_with_launch_profile": ms_prof / nsteps, "kernels": kernel_table(stats, nsteps, peak)}


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
    dtype = args.dtype or cfg["dtype"]
    N = cfg["N"]
    peak, peak_src = measured_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # each rank gets its own segments (weak scaling, no collective on the data path)
    first, _ = dist_utils.shard_segments(rank, world, batch)
    w = Workload(torch, binding, dev, args.workload, dtype, batch, args.overlap, first_segment=first)
    plan, calls = w.plan, w.calls
    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)

    W = max(args.warmup, 3)
    for _ in range(W):
        w.step()
    torch.cuda.synchronize()

    # ---- the timed region: exactly K steps, each bracketed by CUDA events on the launch stream (-> value),
    # then the same K steps again with the library's launch profile on (two more events around every kernel
    # launch) for the per-kernel durations of the roofline line.  Clocks are sampled across both passes.
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    ms_plain, _, n_launch = w.timed(args.steps, False, flush, barrier)
    ms_total, stats, _ = w.timed(args.steps, True, flush, barrier)
    clocks = sampler.stop()

    # context: the same step captured once into a CUDA graph and replayed (the calls neither allocate nor
    # synchronise), timed the same way
    ms_graph = None
    if world == 1:
        try:
            cg = torch.cuda.CUDAGraph()
            with torch.cuda.graph(cg):
                w.step()
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
    x_pin = torch.from_numpy(w.x_np).pin_memory()
    d_x, d_coef, d_out = w.d_x, w.d_coef, w.d_out
    out_pin = torch.empty((batch, N), dtype=w.rdt).pin_memory()
    coef_pin = None
    if "inverse" not in calls:
        coef_pin = torch.empty((batch, plan.ctot), dtype=w.cdt).pin_memory()
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
                w.step(lo, hi)
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
    w.step()
    torch.cuda.synchronize()
    e2e_ok = bool(torch.equal(out_pin, d_out.cpu())) if "inverse" in calls else bool(torch.equal(coef_pin, d_coef.cpu()))
    h2d = x_pin.numel() * x_pin.element_size()
    d2h = (out_pin.numel() * out_pin.element_size()) if "inverse" in calls else (coef_pin.numel() * coef_pin.element_size())
    del x_pin, out_pin, coef_pin

    # ---- max over ranks
    ms_total, ms_plain, ms_e2e = dist_utils.max_over_ranks([ms_total, ms_plain, ms_e2e], device=dev)
    ms_step = ms_plain / args.steps
    units = world * batch * N
    value = dist_utils.aggregate_throughput(world, batch, N, ms_step)
    rt_err = w.round_trip_err()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, from the launch profile of the timed region: COMPULSORY bytes of
    # that launch (samples in / coefficients / samples out) over its CUDA-event duration
    kernels = kernel_table(stats, args.steps, peak)
    roof = None
    if kernels:
        top = kernels[0]
        traffic, traffic_src = measured_traffic(args.workload, batch, top["name"])
        roof = {"bound": "hbm", "kernel": top["name"], "achieved": top["algo_gbs"], "peak": peak,
                "unit": "GB/s", "frac": top["algo_gbs"] / peak, "traffic": traffic, "traffic_source": traffic_src,
                "algo_bytes_per_launch": top["algo_bytes"], "design_bytes_per_launch": top["design_bytes"],
                "peak_source": peak_src, "avg_launch_ms": top["avg_ms"], "share_of_step": top["share"]}
    comp = w.compulsory_bytes()
    path_gbs = comp / (ms_step * 1e-3) / 1e9

    # ---- the same step at a batch that has saturated the throughput ("largest batch"), and the
    # other BASELINE configurations at their own batch and at their largest one (fewer steps each)
    n_side = max(5, min(args.steps, 20))
    largest, others = None, {}
    x_main = w.x_np
    if world == 1 and not args.batch and not args.no_largest_batch:
        big = LARGEST[args.workload] if args.workload in LARGEST else None
        if big and big > batch:
            w.close()
            wb = Workload(torch, binding, dev, args.workload, dtype, big, args.overlap, x_np=x_main)
            largest = record(wb, n_side, 3, flush, barrier, peak)
            largest["round_trip_err"] = wb.round_trip_err()
            wb.close()
            del wb
            w = None
    if world == 1 and not args.batch and not args.no_other_configs:
        if w is not None:
            w.close()
            w = None
        for name, dt in (("cfg2", "f32"), ("cfg3", "f32"), ("cfg5", "f32"), ("cfg5", "f64"), ("cfg4", "f32"), ("cfg1", "f64"),
                         ("paper6s", "f32")):
            if name == args.workload and dt == dtype:
                continue
            key = name if dt == inputs.CONFIGS[name]["dtype"] else f"{name}_{dt}"
            try:
                wo = Workload(torch, binding, dev, name, dt, inputs.CONFIGS[name]["batch"], args.overlap)
                rec = record(wo, n_side, 3, flush, barrier, peak)
                rec["round_trip_err"] = wo.round_trip_err()
                xo = wo.x_np
                wo.close()
                big = LARGEST.get(name)
                if big and not args.no_largest_batch:
                    if dt == "f64":
                        big //= 2
                    wb = Workload(torch, binding, dev, name, dt, big, args.overlap, x_np=xo)
                    rec["largest_batch"] = record(wb, max(5, n_side // 2), 3, flush, barrier, peak)
                    rec["largest_batch"]["round_trip_err"] = wb.round_trip_err()
                    wb.close()
                others[key] = rec
            except Exception as exc:          # one configuration failing must not lose the headline
                others[key] = {"error": str(exc)}
            torch.cuda.empty_cache()

    # ---- cuFFT (through torch.fft) on the same shapes, side by side as a reference only (north_star): the
    # long real transforms alone, without the gather / window / shift, the overlap sum or 1/P
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
            xs = torch.from_numpy(x_main).to(dev)
            spec_t = torch.fft.rfft(xs, dim=-1)
            cufft = {"rfft_ms": ev_time(lambda: torch.fft.rfft(xs, dim=-1)),
                     "irfft_ms": ev_time(lambda: torch.fft.irfft(spec_t, n=N, dim=-1)),
                     "note": "the long real FFTs only, out of place; context, not the target"}
            del spec_t, xs
        except Exception as exc:
            cufft = {"unavailable": str(exc)}

    layout = None
    if world == 1 and args.time_layout_calls > 0:
        try:
            layout = time_layout_calls(torch, binding, dev, args.time_layout_calls, flush)
        except Exception as exc:
            layout = {"error": str(exc)}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, cores, nseg, dt = time_oracle(cfg, args.workload, args.overlap)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{nseg} segments of the same workload, one pass ({dt:.1f} s), oracle FFT engine fp64"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": W, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": dtype, "data": "synthetic",
        "config": workload_config(args, cfg, batch, plan),
        "clocks": clocks,
        "e2e": {"value": units / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e, "chunks": nch,
                "equals_device_resident_result": e2e_ok},
        "gpu_launches": n_launch,
        "roofline": roof,
        "path": {"compulsory_bytes_per_step": comp, "achieved_gbs": path_gbs, "frac_of_peak": path_gbs / peak,
                 "ms_per_step_cuda_graph": ms_graph},
        "round_trip_err": rt_err,
        "cpu_baseline": cpu,
        "csrc_hash": csrc_hash(),
    }
    detail = {
        "headline": line,
        "path": {"frac_of_8tbs": path_gbs / 8000.0, "ms_per_step_with_launch_profile": ms_total / args.steps,
                 "coeffs_per_segment": plan.ctot, "rows": plan.n_rows},
        "kernels": kernels, "largest_batch": largest, "configs": others, "cufft_side_by_side": cufft,
        "layout_calls_at_the_papers_shape": layout,
    }
    line["detail"] = write_detail(args.detail, detail)
    try:
        text = headline_json(line)
    except ValueError:            # never lose the headline to its own size: fall back to the contract's keys alone
        keep = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "clocks", "e2e", "gpu_launches", "cpu_baseline", "csrc_hash", "detail")
        small = {k: line[k] for k in keep}
        small["config"] = {"workload": args.workload, "baseline_config_index": cfg["idx"] - 1, "batch_per_gpu": batch}
        small["roofline"] = {k: roof[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic")} if roof else None
        text = headline_json(small)
    sys.stdout.flush()
    print(text, flush=True)
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
