#!/usr/bin/env python
"""bench.py -- deconvolved Mvoxel/s of the plane-wise multi-view RL hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--path auto|direct|fft]
    python bench.py --impl reference ...      # the fp64 CPU oracle, as it stands, on the host cores

One "step" = one pass of the whole hot path (a0..a5: ingest, T iterations x V views of blur, ratio,
back-projection, update) over one synthetic stack shaped like a BASELINE.json config.  BASELINE.json's
`metric` names no config, so the headline line is the LARGEST single-GPU workload, config 4 (2 views x
2048 planes of 2048x800 uint16, 41x41 PSFs, 10 iterations: 13.4 GB in, 13.4 GB out), and the same JSON
line carries `per_config`: value, e2e, roofline (every kernel class) and clocks of configs 1-5.

  value      device-resident throughput: inputs already in HBM, CUDA events on the launching stream
             around K calls of mvd_deconvolve_planes, max over ranks.
  e2e        the same metric through mvd_deconvolve_host: pinned HOST buffers in, pinned HOST buffer
             out, H2D and D2H inside the timed region (3-stream pipeline).
  roofline   the dominant kernel class: algorithmic bytes (FFT engine) or flops (direct engine) per
             launch / its mean launch duration from CUDA events recorded by the library around every
             launch on the launching stream (extra profiled steps right after the timed ones).
  cpu_baseline  the oracle on a bounded sample of the same workload on this box's host cores.
Multi-GPU: planes are independent, so ranks take disjoint plane ranges of a world x N plane job with no
collective in the data path ("weak" scaling); NCCL is used only for the barrier and the max-over-ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "deconvolved Mvoxel/s (planes*pixels*views*iters/s)"
UNIT = "Mvoxel/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-5) of the headline line")
    ap.add_argument("--per-config", default="1,2,3,4,5", help="configs reported in `per_config` (N = 1 only; '' = none)")
    ap.add_argument("--per-config-steps", type=int, default=5, help="timed steps of the per_config entries")
    ap.add_argument("--planes", type=int, default=0, help="override the number of planes (0 = the config's)")
    ap.add_argument("--shape", default="", help="WxH: the config's views, PSFs and iteration count on planes of another size "
                                                "(measurement of other shapes; the headline stays the config's own)")
    ap.add_argument("--path", default="auto", choices=["auto", "direct", "fft"])
    ap.add_argument("--chunk", type=int, default=0, help="mvd_set_chunk_planes (0 = library default)")
    ap.add_argument("--batch", type=int, default=0, help="mvd_set_batch_planes (0 = library default)")
    ap.add_argument("--streams", type=int, default=0, help="mvd_set_resident_streams (0 = library default)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-planes", type=int, default=0, help="planes in the oracle sample (0 = 2 per core, <= 32)")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------
# inputs
# ---------------------------------------------------------------------------------------------
def make_stack(cfg, n_canonical=64):
    """uint16 [V][N][H][W]: the first planes are the canonical seeded planes of the config (the ones the
    parity tests check), the rest repeat them cyclically with fresh seeded Poisson-like jitter so that the
    whole stack has the recipe's distribution without minutes of host-side generation."""
    from paper_1503_07998_b200 import synth
    psfs = synth.config_psfs(cfg.cid)
    n0 = min(cfg.N, n_canonical)
    base = synth.views(cfg, range(n0), psfs)
    if n0 == cfg.N:
        return psfs, base
    out = np.empty((cfg.V, cfg.N, cfg.H, cfg.W), dtype=np.uint16)
    out[:, :n0] = base
    rng = np.random.default_rng([synth.SEED, cfg.cid, 31337])
    for p0 in range(n0, cfg.N, n0):
        n = min(n0, cfg.N - p0)
        shift = (int(rng.integers(0, cfg.H)), int(rng.integers(0, cfg.W)))
        out[:, p0:p0 + n] = np.roll(base[:, :n], shift, axis=(2, 3))
    return psfs, out


# ---------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock, power and throttle reasons sampled every ~10 ms through NVML (nvidia-ml-py) while the
    timed region runs; falls back to `nvidia-smi -lms 100` when NVML cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.rows, self.proc, self.index, self.stop_flag, self.thread = [], None, index, False, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.nv = pynvml
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nv = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _poll(self):
        nv = self.nv
        bits = [getattr(nv, n, 0) for n in ("nvmlClocksEventReasonHwSlowdown", "nvmlClocksEventReasonHwThermalSlowdown",
                                            "nvmlClocksEventReasonSwThermalSlowdown", "nvmlClocksEventReasonSwPowerCap")]
        legacy = [getattr(nv, n, 0) for n in ("nvmlClocksThrottleReasonHwSlowdown", "nvmlClocksThrottleReasonHwThermalSlowdown",
                                              "nvmlClocksThrottleReasonSwThermalSlowdown", "nvmlClocksThrottleReasonSwPowerCap")]
        bits = [b or l for b, l in zip(bits, legacy)]
        try:
            mx = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
        except Exception:
            mx = 0
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                try:
                    why = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    why = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.rows.append((time.time(), [str(sm), str(mx), f"{pw:.2f}"] +
                                  ["Active" if (why & b) else "Not Active" for b in bits]))
            except Exception:
                pass
            time.sleep(0.01)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self):
        self.stop_flag = True
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self, t0, t1, t_load0=None):
        """Samples inside the timed region; a region too short for three samples also takes the
        warm-up steps right before it (the same kernels under the same load)."""
        rows = [r for t, r in self.rows if t0 - 0.005 <= t <= t1 + 0.005 and len(r) >= 7]
        if len(rows) < 3 and t_load0 is not None:
            rows = [r for t, r in self.rows if t_load0 <= t <= t1 + 0.15 and len(r) >= 7]
        rows = rows or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = [float(r[0]) for r in rows if r[0].replace(".", "").isdigit()]
        reasons = [n for k, n in enumerate(self.NAMES) if any(r[3 + k].lower().startswith("active") for r in rows)]
        pw = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": float(rows[0][1]),
                "power_w_max": max(pw) if pw else None, "samples": len(rows), "reasons": reasons,
                "source": "nvml" if getattr(self, "nv", None) else "nvidia-smi"}


# ---------------------------------------------------------------------------------------------
# the oracle as CPU baseline / reference arm
# ---------------------------------------------------------------------------------------------
def oracle_sample(cfg, psfs, views, n_planes, steps=1, warmup=0):
    """Mvoxel/s of oracle/mvd_oracle on the first n_planes planes (one plane per thread)."""
    from oracle import mvd_oracle
    cores = mvd_oracle.n_cores()
    sub = np.ascontiguousarray(views[:, :n_planes])
    for _ in range(warmup):
        mvd_oracle.deconvolve(sub, psfs, cfg.T, cfg.eps, n_threads=cores)
    t0 = time.perf_counter()
    for _ in range(steps):
        mvd_oracle.deconvolve(sub, psfs, cfg.T, cfg.eps, n_threads=cores)
    dt = (time.perf_counter() - t0) / steps
    units = n_planes * cfg.W * cfg.H * cfg.V * cfg.T
    return units / dt / 1e6, dt, min(cores, n_planes), cores


def cpu_baseline(cfg, psfs, views, n_forced=0, target_s=15.0):
    """The oracle as it stands on a bounded sample of this workload: one plane per core and one RL
    iteration as a pilot, then as many planes (all T iterations) -- or, when a single plane's T
    iterations alone exceed the budget, as many iterations of one plane per core -- as fit ~target_s."""
    import dataclasses
    from oracle import mvd_oracle
    cores = mvd_oracle.n_cores()
    N, T = cfg.N, cfg.T
    n0 = max(1, min(N, cores))
    if n_forced:
        val, dt, used, cores = oracle_sample(cfg, psfs, views, min(n_forced, N))
        n, Ts = min(n_forced, N), T
    else:
        _, t1, _, _ = oracle_sample(dataclasses.replace(cfg, T=1), psfs, views, n0)       # pilot
        if t1 * T <= target_s:
            n, Ts = int(min(N, n0 * max(1, int(target_s / (t1 * T))))), T
        else:
            n, Ts = n0, max(1, int(target_s / t1))
        val, dt, used, cores = oracle_sample(dataclasses.replace(cfg, T=Ts), psfs, views, n)
    return {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "seconds": round(dt, 2),
            "sample": f"first {n} of {N} planes, {Ts} of {T} iterations, one plane per thread"}


def config_record(cfg, world=1):
    """The workload-defining part of the JSON line's `config`, shared by both arms (the reference arm runs a
    bounded sample of the SAME workload; the sample is described under `cpu_baseline.sample`)."""
    in_b = cfg.V * cfg.N * cfg.H * cfg.W * 2
    out_b = cfg.N * cfg.H * cfg.W * 4
    return {"workload": cfg.name, "planes_per_gpu": cfg.N, "plane": f"{cfg.W}x{cfg.H}", "views": cfg.V,
            "psf": cfg.K, "iterations": cfg.T,
            "l2": ("inputs+outputs per step (%.0f MB) exceed the 126 MB L2; no flush" % ((in_b + out_b) / 1e6))
                  if in_b + out_b > 126e6 else
                  ("inputs+outputs per step (%.2f MB) fit the 126 MB L2; a 256 MB buffer is written between "
                   "timed steps (flush)" % ((in_b + out_b) / 1e6)),
            "parallelism": f"planes sharded over {world} GPU(s), no collective"}


def run_reference(args, cfg):
    """--impl reference: the oracle as it stands on the host cores, on the headline arm's config.  Each step is a
    bounded sample of that workload (the first n planes, Ts of its T iterations, one plane per thread) sized
    by a one-iteration pilot so that the whole --steps K --warmup W run ends within a few minutes; the
    metric counts exactly the voxel-view-iterations the sample did."""
    import dataclasses
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import mvd_oracle
    from paper_1503_07998_b200 import synth
    cores = mvd_oracle.n_cores()
    steps, warm = max(1, args.steps), max(0, args.warmup)
    n = args.cpu_planes or max(1, min(cfg.N, cores))
    psfs = synth.config_psfs(cfg.cid)
    views = synth.views(cfg, range(n), psfs)
    _, t1, _, _ = oracle_sample(dataclasses.replace(cfg, T=1), psfs, views, n)            # pilot
    per_step = 150.0 / (steps + warm)
    Ts = int(max(1, min(cfg.T, per_step // max(t1, 1e-9))))   # one iteration of one plane per thread is the smallest sample
    sub = dataclasses.replace(cfg, T=Ts)
    val, dt, used, cores = oracle_sample(sub, psfs, views, n, steps=steps, warmup=warm)
    sample = (f"per step: first {n} of {cfg.N} planes, {Ts} of {cfg.T} iterations, one plane per thread "
              f"({n * cfg.W * cfg.H * cfg.V * Ts} voxel-view-iterations)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_record(cfg, max(1, args.gpus)),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------------
# ours
# ---------------------------------------------------------------------------------------------
def algorithmic_work(cls, cfg, n_planes, K):
    """(amount per launch, unit) of one launch of kernel class `cls` over n_planes planes."""
    vox = n_planes * cfg.W * cfg.H
    table = {
        "init_mean": (vox * (2 * cfg.V + 4), "B"),
        "direct_blur_ratio": (vox * 2.0 * K * K, "flop"),          # K^2 FMA per voxel
        "direct_backproject_update": (vox * 2.0 * K * K, "flop"),
        "sep_blur_ratio": (vox * 2.0 * 2 * K, "flop"),             # separable PSF: K FMA per voxel and pass, two passes
        "sep_backproject_update": (vox * 2.0 * 2 * K, "flop"),
        "fft_rows_first": (vox * (2 * cfg.V + 4 + 4), "B"),        # phi_v u16 in, psi + row spectrum out
        "fft_cols_otf": (vox * 8, "B"),                            # spectrum in + out (OTF is L2-resident)
        "fft_rows_ratio": (vox * 10, "B"),                         # spectrum in, phi u16 in, spectrum out
        "fft_rows_update": (vox * 16, "B"),                        # spectrum in, psi in+out, spectrum out
        "small_resident": (vox * (2 * cfg.V + 4), "B"),            # whole RL run on chip: views in, psi out
    }
    return table.get(cls, (0, "B"))


def passes_per_step(cls, cfg):
    """Launches of class `cls` that one plane goes through in one step."""
    return {"init_mean": 1, "fft_rows_first": 1, "small_resident": 1,
            "fft_cols_otf": 2 * cfg.T * cfg.V}.get(cls, cfg.T * cfg.V)


def load_traffic_table():
    """profiles/ncu_traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum per launch of each kernel class
    from the committed `ncu --set full` captures (one row per config and class, with its source file)."""
    import csv
    table = {}
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for row in csv.DictReader(r for r in f if not r.startswith("#")):
                table[(int(row["config"]), row["kernel_class"])] = (
                    float(row["dram_bytes_per_launch"]), float(row["planes_per_launch"]), row["source"])
    except OSError:
        pass
    return table


def make_roofline(prof, prof_steps, cfg, N, K, path_name, peaks, traffic_table, fp32_peak):
    """`roofline` of the dominant kernel class plus the same figures for every class (`per_class`)."""
    fp32_tf, fp32_mhz = fp32_peak
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (of fallback)"
    total_ms = sum(v[0] for v in prof.values()) or 1.0
    per_class = {}
    for cls, (ms, n) in prof.items():
        if not n or cls == "setup":
            continue
        launches_per_step = max(n // prof_steps, 1)
        planes = N * passes_per_step(cls, cfg) / launches_per_step          # mean planes per launch
        work, wunit = algorithmic_work(cls, cfg, planes, K)
        avg_s = ms * 1e-3 / n
        rec = {"ms_per_step": round(ms / prof_steps, 4), "launches_per_step": launches_per_step,
               "avg_launch_us": avg_s * 1e6, "planes_per_launch": planes, "share_of_step": ms / total_ms}
        if wunit == "flop":
            rec.update(bound="alu", achieved=work / avg_s / 1e12, peak=fp32_tf, unit="TFLOP/s",
                       algorithmic_flop_per_launch=work)
        else:
            rec.update(bound="hbm", achieved=work / avg_s / 1e9, peak=hbm, unit="GB/s",
                       algorithmic_bytes_per_launch=work)
        rec["frac"] = rec["achieved"] / rec["peak"] if rec["peak"] else None
        t = traffic_table.get((cfg.cid, cls)) if path_name == "fft" else None
        rec["traffic"] = t[0] * planes / t[1] if t else None
        if t:
            rec["traffic_source"] = f"{t[2]} (ncu --set full; bytes per launch of {t[1]:g} planes, scaled to {planes:g})"
            rec["frac_of_traffic"] = rec["traffic"] / avg_s / 1e9 / hbm
        per_class[cls] = rec
    top = max(per_class, key=lambda k: per_class[k]["share_of_step"])
    roof = dict(per_class[top])
    roof["kernel"] = top
    roof["peak_source"] = hbm_src if roof["bound"] == "hbm" else (
        f"measured FFMA micro-kernel in this run at {fp32_mhz:.0f} MHz (nominal 148 SM x 128 lanes x 2 x 1.965 GHz = 74.4)")
    roof["launches_profiled"] = prof[top][1]
    roof["per_class"] = {k: {kk: vv for kk, vv in v.items() if kk != "traffic_source"} for k, v in per_class.items()}
    return roof


def run_config(cfg, args, steps, warmup, world, local, peaks, traffic_table, fp32_peak, do_e2e=True):
    """One config on this rank's GPU: device-resident value, e2e through the host pipeline, per-class
    roofline, clocks.  Returns a dict (times are this rank's; the caller reduces over ranks)."""
    import torch
    from paper_1503_07998_b200 import binding, shard
    psfs, views = make_stack(cfg)
    V, N, H, W, K, T = cfg.V, cfg.N, cfg.H, cfg.W, cfg.K, cfg.T
    units = cfg.units
    path = {"auto": None, "direct": binding.PATH_DIRECT, "fft": binding.PATH_FFT}[args.path]
    host_in = torch.from_numpy(views.view(np.int16)).pin_memory()
    host_out = torch.empty((N, H, W), dtype=torch.float32).pin_memory()
    h2d_bytes = int(views.nbytes)
    if world > 1:
        views = None            # N ranks on one host: keep only the pinned copy (the oracle sample runs at N = 1 only)
    dev_in = host_in.cuda()
    dev_out = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
    stream = torch.cuda.Stream()
    small = h2d_bytes + N * H * W * 4 <= 126e6              # fits L2: flush between timed steps
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if small else None

    def barrier():
        import torch.distributed as dist
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    m = binding.Mvd(W, H, V, psfs, K, T, cfg.eps, path)
    if args.chunk:
        m.set_chunk_planes(args.chunk)
    if args.batch:
        m.set_batch_planes(args.batch)
    if args.streams:
        m.set_resident_streams(args.streams)
    m.reserve(N)
    path_name = binding.PATH_NAMES[m.path]

    # ---- device-resident: warm-up, then exactly `steps` timed steps ---------------------------
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    t_load0 = time.time()
    for _ in range(max(warmup, 3)):
        m.deconvolve_planes(dev_in, dev_out, N, stream)
    barrier()
    m.launch_count_reset()
    t_wall0 = time.time()
    if small:
        # steps are timed one by one (CUDA events on the launching stream) with an L2 flush in between
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for e0, e1 in evs:
            with torch.cuda.stream(stream):
                flush.fill_(1)
            e0.record(stream)
            m.deconvolve_planes(dev_in, dev_out, N, stream)
            e1.record(stream)
        barrier()
        ms = sum(e0.elapsed_time(e1) for e0, e1 in evs)
    else:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            m.deconvolve_planes(dev_in, dev_out, N, stream)
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
    t_wall1 = time.time()
    launches = m.launch_count()
    clocks = sampler.summary(t_wall0, t_wall1, t_load0)
    ms_max = shard.max_over_ranks(ms, device="cuda")          # device time of the slowest rank
    value = shard.job_throughput(units * steps, ms_max * 1e-3, world) / 1e6

    # ---- launch-bound stacks: the same call captured once into a CUDA graph and replayed (mvd_reserve makes the call
    # capturable: it only enqueues) -- reported beside `value`, which stays the eager call a user makes ----------
    graph = None
    if small:
        try:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                m.deconvolve_planes(dev_in, dev_out, N, stream)
            for _ in range(3):
                g.replay()
            torch.cuda.synchronize()
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for e0, e1 in evs:
                flush.fill_(1)
                e0.record()
                g.replay()
                e1.record()
            torch.cuda.synchronize()
            gms = sum(e0.elapsed_time(e1) for e0, e1 in evs)
            graph = {"value": units * steps / (gms * 1e-3) / 1e6, "unit": UNIT, "ms_per_step": gms / steps,
                     "what": "mvd_deconvolve_planes captured into one CUDA graph, replayed"}
            del g
        except Exception as exc:   # capture is a convenience measurement, never the headline
            graph = {"error": str(exc)[:200]}

    # ---- per-kernel durations (CUDA events inside the library, launching stream) ------------
    m.profile_enable(True)
    prof_steps = 2
    for _ in range(prof_steps):
        m.deconvolve_planes(dev_in, dev_out, N, stream)
    prof = m.profile_read()
    m.profile_enable(False)
    torch.cuda.synchronize()
    roof = make_roofline(prof, prof_steps, cfg, N, K, path_name, peaks, traffic_table, fp32_peak)

    # ---- end to end: pinned host -> host through mvd_deconvolve_host -------------------------
    e2e = None
    if do_e2e:
        m.deconvolve_planes(dev_in, dev_out, N, stream)      # the profiled steps ran single-stream: same bits, but redo
        for _ in range(max(1, min(warmup, 2))):
            m.deconvolve_host(host_in, host_out, N)
        barrier()
        # sub-millisecond steps: enough of them to time by wall clock; steps of a few milliseconds: at least 20
        e2e_steps = max(steps, 50) if small else (max(steps, 20) if ms_max / steps < 50.0 else steps)
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            m.deconvolve_host(host_in, host_out, N)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, device="cuda")
        e2e = {"value": shard.job_throughput(units * e2e_steps, dt, world) / 1e6, "unit": UNIT,
               "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": int(host_out.numel() * 4),
               "ms_per_step": dt * 1e3 / e2e_steps, "steps": e2e_steps}
        e2e["ratio_to_device_resident"] = e2e["value"] / value
        # context: what the PCIe link alone allows -- the step's input copied host -> device and its output device -> host
        # at the same time on two streams, nothing else running (an upper bound for any host-to-host figure)
        s_up, s_dn = torch.cuda.Stream(), torch.cuda.Stream()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        s_up.wait_event(ev[0]); s_dn.wait_event(ev[0])
        with torch.cuda.stream(s_up):
            dev_in.copy_(host_in, non_blocking=True)
        with torch.cuda.stream(s_dn):
            host_out.copy_(dev_out, non_blocking=True)
        torch.cuda.current_stream().wait_stream(s_up); torch.cuda.current_stream().wait_stream(s_dn)
        ev[1].record()
        torch.cuda.synchronize()
        link_ms = ev[0].elapsed_time(ev[1])
        e2e["pcie_copies_alone_ms"] = link_ms
        e2e["pcie_bound_value"] = units / (link_ms * 1e-3) / 1e6
        e2e["ratio_to_min_of_resident_and_pcie_bound"] = e2e["value"] / min(value, e2e["pcie_bound_value"])
        same = True
        for p0 in range(0, N, 256):                          # compare in slices: no second 13 GB host copy
            same = same and bool(torch.equal(host_out[p0:p0 + 256], dev_out[p0:p0 + 256].cpu()))
        e2e["bit_identical_to_device_resident"] = same
    sampler.stop()
    m.destroy()
    rec = {"value": value, "ms_per_step": ms_max / steps, "steps": steps, "e2e": e2e, "roofline": roof,
           "clocks": clocks, "gpu_launches": launches, "path": path_name, "graph_replay": graph,
           "whole_step_algorithmic_GBps": (42.0 if path_name == "fft" else 22.0) * units / (ms_max / steps * 1e-3) / 1e9}
    return rec, psfs, views


def main():
    args = parse()
    from paper_1503_07998_b200 import synth
    cfg = synth.config(args.config)
    if args.planes:
        cfg = cfg.with_planes(args.planes)
    if args.shape:
        import dataclasses
        w, h = (int(x) for x in args.shape.lower().split("x"))
        cfg = dataclasses.replace(cfg, W=w, H=h, name=f"{cfg.name} on {w}x{h} planes")
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    from paper_1503_07998_b200 import binding, build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libmvd has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        if local == 0:
            build.build()              # one rank per node compiles; the others wait for the .so
        dist.barrier()
    build.build()

    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except OSError:
        peaks = {}
    traffic_table = {} if args.shape else load_traffic_table()      # the ncu captures belong to the configs' own shapes
    fp32_peak = binding.measure_fp32_peak()

    main_rec, psfs, views = run_config(cfg, args, args.steps, args.warmup, world, local, peaks, traffic_table,
                                       fp32_peak, do_e2e=not args.no_e2e)

    # ---- the oracle beside it (rank 0, N = 1 only): a bounded sample of about 10-30 s of CPU work ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(cfg, psfs, views, args.cpu_planes)
    del psfs, views

    # ---- every config, shorter (N = 1 only): value, e2e, per-class roofline, clocks ---------------
    per_config = None
    if world == 1 and args.per_config and not args.planes and not args.shape:
        per_config = []
        for cid in [int(c) for c in args.per_config.split(",") if c]:
            if cid == cfg.cid:
                rec = dict(main_rec)
            else:
                c2 = synth.config(cid)
                rec, _, _ = run_config(c2, args, max(1, args.per_config_steps), 3, world, local, peaks,
                                       traffic_table, fp32_peak, do_e2e=not args.no_e2e)
            rec = {"config": cid, **config_record(synth.config(cid), world), **rec}
            per_config.append(rec)

    # ---- the direct engine (FP32-bound; the fallback for shapes the FFT engine does not take), driver-measured on
    # config 2's shape with 128 planes: value and the FFMA-pipe roofline of its two kernels ----------------------
    direct = None
    if world == 1 and args.per_config and not args.planes and not args.shape and args.path == "auto":
        import copy
        a2 = copy.copy(args)
        a2.path = "direct"
        c2 = synth.config(2).with_planes(128)
        rec, _, _ = run_config(c2, a2, max(1, args.per_config_steps), 3, world, local, peaks, traffic_table,
                               fp32_peak, do_e2e=False)
        direct = {"config": 2, **config_record(c2, world), **rec}

    if rank == 0:
        conf = config_record(cfg, world)
        conf["path"] = main_rec["path"]
        print(json.dumps({
            "metric": METRIC, "value": main_rec["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": main_rec["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": conf, "clocks": main_rec["clocks"], "e2e": main_rec["e2e"],
            "gpu_launches": main_rec["gpu_launches"], "roofline": main_rec["roofline"], "cpu_baseline": cpu,
            "whole_step_algorithmic_GBps": main_rec["whole_step_algorithmic_GBps"],
            "fp32_peak_measured_tflops": fp32_peak[0], "per_config": per_config, "direct_engine": direct,
            "context": "paper Table 1 (other hardware, FFT implementation, whole workflow): 1128 Mvoxel/s "
                       "at 2048^3 on a GTX Titan Black; plane-wise speedups up to 25x / 75x over 3D "
                       "deconvolution with / without GPU (PAPER.md:31, :164-175)"}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
