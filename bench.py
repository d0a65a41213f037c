#!/usr/bin/env python
"""bench.py -- deconvolved Mvoxel/s of the plane-wise multi-view RL hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--path auto|direct|fft]
    python bench.py --impl reference ...      # the fp64 CPU oracle, as it stands, on the host cores

One "step" = one pass of the whole hot path (a0..a5: ingest, T iterations x V views of blur, ratio,
back-projection, update) over one synthetic stack shaped like BASELINE.json's config (default:
configs[1] = "config 2", 2 views x 512 planes of 512x256 uint16, 21x21 PSFs, 10 iterations).

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
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); 2 = configs[1]")
    ap.add_argument("--planes", type=int, default=0, help="override the number of planes (0 = the config's)")
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


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import mvd_oracle
    from paper_1503_07998_b200 import synth
    cores = mvd_oracle.n_cores()
    n = args.cpu_planes or max(1, min(cfg.N, cores))
    psfs = synth.config_psfs(cfg.cid)
    views = synth.views(cfg, range(n), psfs)
    steps, warm = max(1, args.steps), min(args.warmup, 1)
    val, dt, used, cores = oracle_sample(cfg, psfs, views, n, steps=steps, warmup=warm)
    sample = f"first {n} planes of the {cfg.N}-plane stack per step, one plane per thread"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "planes_per_step": n},
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
        "fft_rows_first": (vox * (2 * cfg.V + 4 + 4), "B"),        # phi_v u16 in, psi + row spectrum out
        "fft_cols_otf": (vox * 8, "B"),                            # spectrum in + out (OTF is L2-resident)
        "fft_rows_ratio": (vox * 10, "B"),                         # spectrum in, phi u16 in, spectrum out
        "fft_rows_update": (vox * 16, "B"),                        # spectrum in, psi in+out, spectrum out
    }
    return table.get(cls, (0, "B"))


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture
# (profiles/r1_final_launches.md), keyed by (config id, planes per launch, kernel class)
NCU_TRAFFIC = {
    (2, 512, "fft_cols_otf"): 485.4e6,
    (2, 512, "fft_rows_ratio"): 635.2e6,
    (2, 512, "fft_rows_update"): 1032.5e6,
}


def main():
    args = parse()
    from paper_1503_07998_b200 import synth
    cfg = synth.config(args.config)
    if args.planes:
        cfg = cfg.with_planes(args.planes)
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    from paper_1503_07998_b200 import binding, build, shard

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
    psfs, views = make_stack(cfg)
    V, N, H, W, K, T = cfg.V, cfg.N, cfg.H, cfg.W, cfg.K, cfg.T
    units = cfg.units                                     # voxel-view-iterations per step per rank
    path = {"auto": None, "direct": binding.PATH_DIRECT, "fft": binding.PATH_FFT}[args.path]

    host_in = torch.from_numpy(views.view(np.int16)).pin_memory()
    host_out = torch.empty((N, H, W), dtype=torch.float32).pin_memory()
    dev_in = host_in.cuda()
    dev_out = torch.empty((N, H, W), dtype=torch.float32, device="cuda")
    stream = torch.cuda.Stream()

    def barrier():
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
    path_name = binding.PATH_NAMES[m.path]

    # ---- device-resident: warm-up, then exactly K timed steps -------------------------------
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    t_load0 = time.time()
    for _ in range(max(args.warmup, 3)):
        m.deconvolve_planes(dev_in, dev_out, N, stream)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m.launch_count_reset()
    barrier()
    t_wall0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        m.deconvolve_planes(dev_in, dev_out, N, stream)
    e1.record(stream)
    barrier()
    t_wall1 = time.time()
    launches = m.launch_count()
    ms = e0.elapsed_time(e1)
    clocks = sampler.summary(t_wall0, t_wall1, t_load0)
    ms_max = shard.max_over_ranks(ms, device="cuda")          # device time of the slowest rank
    value = shard.job_throughput(units * args.steps, ms_max * 1e-3, world) / 1e6

    # ---- per-kernel durations (CUDA events inside the library, launching stream) ------------
    m.profile_enable(True)
    prof_steps = 2
    for _ in range(prof_steps):
        m.deconvolve_planes(dev_in, dev_out, N, stream)
    prof = m.profile_read()
    m.profile_enable(False)
    torch.cuda.synchronize()
    total_prof_ms = sum(v[0] for v in prof.values()) or 1.0
    top = max(prof, key=lambda k: prof[k][0])
    top_ms, top_n = prof[top]
    passes = {"init_mean": 1, "fft_rows_first": 1, "fft_cols_otf": 2 * T * V}.get(top, T * V)   # per plane per step
    launches_per_step = max(top_n // prof_steps, 1)
    chunk_planes = N * passes / launches_per_step                      # mean planes per launch
    work, wunit = algorithmic_work(top, cfg, chunk_planes, K)
    avg_s = top_ms * 1e-3 / max(top_n, 1)
    fp32_tf, fp32_mhz = binding.measure_fp32_peak()
    if wunit == "flop":
        achieved = work / avg_s / 1e12
        roof = {"bound": "alu", "achieved": achieved, "peak": fp32_tf, "unit": "TFLOP/s",
                "frac": achieved / fp32_tf, "traffic": None,
                "peak_source": f"measured FFMA micro-kernel in this run at {fp32_mhz:.0f} MHz "
                               f"(nominal 148 SM x 128 lanes x 2 x 1.965 GHz = 74.4)"}
    else:
        achieved = work / avg_s / 1e9
        peak = float(peaks.get("hbm_gbs", 6650.0))
        roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None, "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)"
                if "hbm_gbs" in peaks else "fallback 6650 GB/s (of fallback)"}
    roof["traffic"] = NCU_TRAFFIC.get((cfg.cid, int(round(chunk_planes)), top)) if path_name == "fft" else None
    roof["algorithmic_bytes_per_launch" if wunit == "B" else "algorithmic_flop_per_launch"] = work
    roof["traffic_source"] = "profiles/r1_final_launches.md (ncu --set full, bytes per launch)" if roof["traffic"] else None
    roof.update({"kernel": top, "launches_profiled": top_n, "avg_launch_us": avg_s * 1e6,
                 "share_of_step": top_ms / total_prof_ms, "planes_per_launch": chunk_planes,
                 "per_class_ms_per_step": {k: round(v[0] / prof_steps, 4) for k, v in prof.items() if v[1]}})

    # ---- end to end: pinned host -> host through mvd_deconvolve_host -------------------------
    e2e = None
    if not args.no_e2e:
        for _ in range(max(1, min(args.warmup, 2))):
            m.deconvolve_host(host_in, host_out, N)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            m.deconvolve_host(host_in, host_out, N)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, device="cuda")
        e2e = {"value": shard.job_throughput(units * args.steps, dt, world) / 1e6, "unit": UNIT,
               "h2d_bytes_per_step": int(views.nbytes), "d2h_bytes_per_step": int(host_out.numel() * 4),
               "ms_per_step": dt * 1e3 / args.steps, "ratio_to_device_resident": None}
        e2e["ratio_to_device_resident"] = e2e["value"] / value
        same = bool(torch.equal(host_out, dev_out.cpu()))
        e2e["bit_identical_to_device_resident"] = same
    sampler.stop()

    # ---- the oracle beside it (rank 0, N = 1 only): a bounded sample of about 10-30 s of CPU work ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(cfg, psfs, views, args.cpu_planes)
    m.destroy()

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "planes_per_gpu": N, "path": path_name,
                       "l2": "inputs+outputs per step (%.0f MB) exceed the 126 MB L2; no flush" %
                             ((views.nbytes + N * H * W * 4) / 1e6),
                       "parallelism": f"planes sharded over {world} GPU(s), no collective"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "cpu_baseline": cpu,
            "fp32_peak_measured_tflops": fp32_tf,
            "context": "paper Table 1 (other hardware, FFT implementation, whole workflow): 1128 Mvoxel/s "
                       "at 2048^3 on a GTX Titan Black; plane-wise speedups up to 25x / 75x over 3D "
                       "deconvolution with / without GPU (PAPER.md:31, :164-175)"}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
