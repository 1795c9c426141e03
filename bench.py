#!/usr/bin/env python
"""bench.py -- throughput of the CFS hot path on B200 (BASELINE.json metric: point-iterations/s and
splats/s, % of measured roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--no-workloads]

One "step" = one pass of the whole hot path over one batch: clear the image, cfs_render (sampler +
pick + map + chain + colour + splat, one kernel) and cfs_tonemap, on BASELINE configs[1] (square
generator -> swirl -> scale 0.8, colour by map index, 2^20 points x 1000 iterations, 1024x1024
RGBA float32).  Prints ONE JSON line (see DESIGN.md "measurement" for every key).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_02226_b200 import workloads as W  # noqa: E402  (inputs only, no arithmetic)

HEADLINE_CFG = 1
SINCOS = "sincosf (<= 2 ulp)"
METRIC = "cfs_point_iterations_per_s"
UNIT = "point-iterations/s"
L2_FLUSH_BYTES = 256 << 20
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the render kernel on configs[1], from
# the `ncu --set full` captures summarised in profiles/README.md
NCU_TRAFFIC_BYTES_PER_LAUNCH = 0.989e9       # hybrid pass 1: profiles/r01j_hybrid_cfg1.txt (0.008 GB read + 0.982 GB written)
NCU_TRAFFIC_BYTES_PER_LAUNCH_BINNED = 2.0e9  # pure bins (--variant binned): twice the records of the hybrid stage
NCU_TRAFFIC_BYTES_PER_LAUNCH_DIRECT = 7.06e6 # direct kernel: profiles/r01h_direct_cfg1.txt (the image stays in L2)


# ----------------------------------------------------------------------------- clocks sampler
class ClockSampler:
    """SM clock / power / throttle reasons DURING the timed region (B200_PROFILING.md recipe).  The timed
    region of configs[1] lasts tens of milliseconds, shorter than one `nvidia-smi -lms` period, so the
    samples come from NVML in a polling thread (the library nvidia-smi itself reads); nvidia-smi is the
    fallback when NVML cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    BITS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index: int, uuid=None):
        self.rows = []          # nvidia-smi lines
        self.samples = []       # (sm_mhz, power_w, reasons bit mask) from NVML
        self.proc = None
        self.thread = None
        self.index = index
        self.stop_flag = threading.Event()
        self.nvml = None
        self.handle = None
        self.sm_max = None
        try:
            import pynvml
            pynvml.nvmlInit()
            h = None
            if uuid:
                try:
                    h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode())
                except Exception:
                    h = None
            if h is None:
                h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.nvml, self.handle = pynvml, h
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nvml = None

    def _poll(self):
        n, h = self.nvml, self.handle
        while not self.stop_flag.is_set():
            try:
                sm = float(n.nvmlDeviceGetClockInfo(h, n.NVML_CLOCK_SM))
                pw = n.nvmlDeviceGetPowerUsage(h) / 1000.0
                try:
                    rs = int(n.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    rs = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                self.samples.append((sm, pw, rs))
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nvml is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.nvml is not None:
            self.stop_flag.set()
            if self.thread:
                self.thread.join(timeout=1)
            sm = [x[0] for x in self.samples]
            pw = [x[1] for x in self.samples]
            mask = 0
            for x in self.samples:
                mask |= x[2]
            reasons = sorted(nm for nm, bit in self.BITS.items() if mask & bit)
            return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": self.sm_max,
                    "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons, "source": "nvml"}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons),
                "source": "nvidia-smi"}


# ----------------------------------------------------------------------------- reference arm (oracle)
def host_cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(cfg: int, n_points: int):
    """The oracle as it stands on a bounded sample (first n_points points) of configs[cfg], on all
    host cores through its own multi-threaded driver. Returns (point_iterations, seconds, threads)."""
    from oracle import cfs_oracle
    w = W.config(cfg)
    cloud = W.gaussian_mixture_cloud(n_points, w.cloud_seed) if w.system.gen == "cloud" else None
    t = w.frames[len(w.frames) // 2]
    t0 = time.perf_counter()
    _, _, threads = cfs_oracle.render_parallel(w.system, w.render, cloud=cloud, n_points=n_points, t=t)
    dt = time.perf_counter() - t0
    return n_points * w.render.iterations, dt, threads


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import build as oracle_build
    oracle_build.build()
    n = 1 << 14
    for _ in range(args.warmup):
        oracle_sample(HEADLINE_CFG, n)
    tot_pi, tot_t, threads = 0, 0.0, 1
    for _ in range(args.steps):
        pi, dt, threads = oracle_sample(HEADLINE_CFG, n)
        tot_pi += pi
        tot_t += dt
    w = W.config(HEADLINE_CFG)
    value = tot_pi / tot_t
    sample = f"first {n} points x {w.render.iterations} iterations of configs[{HEADLINE_CFG}] per step, full 1024x1024 image"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_t / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(w, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                         "cpu": host_cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(w, n_gpus):
    r = w.render
    return {"workload": f"BASELINE configs[{HEADLINE_CFG}] {w.name}", "points_per_gpu": r.n_points,
            "iterations": r.iterations, "burn_in": r.burn_in, "image": f"{r.width}x{r.height} {r.out_mode}",
            "chain": [x.type for x in w.system.chain], "n_funcs": len(w.system.funcs), "sincos": SINCOS,
            "parallelism": f"points sharded over {n_gpus} GPU(s), image all-reduce" if n_gpus > 1 else "1 GPU",
            "l2": "flushed between steps (256 MiB memset outside the per-step events); the 16 MiB image is "
                  "L2-resident by design"}


# ----------------------------------------------------------------------------- our arm
def event_pair(torch):
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


def measure_rates(cfs, torch, buf, sms):
    """Roofline denominators in the same run (BASELINE north_star)."""
    out = {}

    def rate(kind, fp, ops, blocks, threads, reps=3):
        best = None
        for _ in range(reps + 1):
            if kind == "atom_min_u64":
                buf.fill_(255)
            e0, e1 = event_pair(torch)
            e0.record()
            cfs.cfs_microbench(kind, buf, fp, ops, blocks, threads)
            e1.record()
            torch.cuda.synchronize()
            dt = e0.elapsed_time(e1) * 1e-3
            best = dt if best is None else min(best, dt)
        return blocks * threads * ops / best

    for kind, fps in (("red_add_u32", (1 << 20,)), ("red_add_v4f32", (16 << 20, 33177600, 132710400)),
                      ("atom_min_u64", (66355200,)), ("ld_u64", (66355200,))):
        for fp in fps:
            out[f"{kind}@{fp}"] = rate(kind, fp, 1024, sms * 8, 256)
    for kind in ("ffma", "imad_wide", "lop3", "mufu"):
        out[kind] = rate(kind, 0, 1 << 15, sms * 8, 256)
    best = None
    for _ in range(4):
        e0, e1 = event_pair(torch)
        e0.record()
        cfs.cfs_microbench("stream_ld128", buf, buf.numel(), 0, sms * 16, 256)
        e1.record()
        torch.cuda.synchronize()
        dt = e0.elapsed_time(e1) * 1e-3
        best = dt if best is None else min(best, dt)
    out["stream_ld128_GBps"] = buf.numel() / best / 1e9
    return out


# algorithmic lane-instructions per point-iteration (table "N_instr")
N_INSTR = {0: 30, 1: 62, 2: 66, 3: 110, 4: 52}
# the same for the binned variant with MUFU sin/cos (Philox 10, pick, LDS +
# generator FMAs, chain, 4 bound compares, 9 pixel ops, 6 record ops, 4 append ops)
N_INSTR_BIN = {0: 38, 1: 51, 2: 51}
# hybrid (CFS_FLAG_BIN_HYBRID, what AUTO runs): every other splat skips the 6 record + 4 append operations and
# pays a palette LDS + one red.global instead, i.e. 43 on those iterations: (51 + 43) / 2
N_INSTR_HYB = {1: 47, 2: 47}
# with sincosf (--accurate-trig): the direct count of N_INSTR on direct iterations, + 8 (6 record + 4 append - 2) on binned ones
N_INSTR_HYB_ACC = {1: 66, 2: 70}
N_INSTR_BIN_ACC = {0: 38, 1: 70, 2: 74}
RED_KEY = {0: "red_add_u32@1048576", 1: "red_add_v4f32@16777216", 2: "red_add_v4f32@33177600",
           3: "red_add_v4f32@132710400", 4: "atom_min_u64@66355200"}


def roofline_for(cfg, w, rates, peaks, splats, seconds):
    """t_roof = max(t_issue, t_atomic, t_hbm); frac = t_roof / t."""
    pi = w.render.n_points * w.render.iterations
    t_issue = pi * N_INSTR[cfg] / rates["ffma"]
    t_atom = splats / rates[RED_KEY[cfg]]
    t_hbm = (w.render.n_points * 16 / (peaks["hbm_gbs"] * 1e9)) if w.system.gen == "cloud" else 0.0
    t_roof = max(t_issue, t_atom, t_hbm)
    bound = "alu" if t_roof == t_issue else ("l2_atomic" if t_roof == t_atom else "hbm")
    return {"bound": bound, "t_issue_ms": t_issue * 1e3, "t_atomic_ms": t_atom * 1e3, "t_hbm_ms": t_hbm * 1e3,
            "t_roof_ms": t_roof * 1e3, "t_ms": seconds * 1e3, "frac": t_roof / seconds}


SCRATCH_CAP_BYTES = 8 << 30


def make_scratch(cfs, torch, sysh, render):
    """Scratch of the tile-binned variant (None when the variant cannot serve the workload)."""
    need = cfs.cfs_binned_scratch_bytes(sysh, cfs.make_args(render))
    if need == 0:
        return None
    return torch.empty(min(need, SCRATCH_CAP_BYTES), dtype=torch.uint8, device="cuda")


def time_workload(cfs, torch, cfg, flush, reps=5, flags=0, variant="auto"):
    """Median device time of one cfs_render of configs[cfg] (all frames for cfg 2)."""
    w = W.config(cfg)
    cloud = W.gaussian_mixture_cloud(w.render.n_points, w.cloud_seed) if w.system.gen == "cloud" else None
    d_cloud = cfs.cloud_to_device(cloud) if cloud is not None else None
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda")
    scratch = make_scratch(cfs, torch, sysh, w.render) if variant != "direct" else None
    times = []
    n_rep = reps if cfg != 4 else 3
    for rep in range(n_rep + 2):
        flush.zero_()
        tot = 0.0
        ctr.zero_()
        for t in w.frames:
            img.fill_(-1 if w.render.out_mode == "depth_u64" else 0)
            args = cfs.make_args(w.render, d_image=img, d_cloud=d_cloud, d_counters=ctr, t=t, flags=flags,
                                 variant=variant, d_scratch=scratch)
            e0, e1 = event_pair(torch)
            e0.record()
            cfs.cfs_render(sysh, args)
            e1.record()
            torch.cuda.synchronize()
            tot += e0.elapsed_time(e1) * 1e-3
        if rep >= 2:
            times.append(tot)
    sec = float(np.median(times))
    c = ctr.cpu().numpy()
    sysh.close()
    return w, sec, int(c[0]), int(c[1])


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_02226_b200 import cfs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CFS library has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfs.lib()
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        with open(peaks_path) as fh:
            peaks = json.load(fh)
        peaks_src = "measured"
    else:
        peaks, peaks_src = {"hbm_gbs": 6650.0}, "fallback"

    w = W.config(HEADLINE_CFG)
    r = w.render
    P, I, S = r.n_points, r.iterations, r.n_points * (r.iterations - r.burn_in)
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(r)
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda")
    out8 = torch.zeros(r.width * r.height, dtype=torch.int32, device="cuda")
    scratch = torch.zeros(2, dtype=torch.int32, device="cuda")
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    # weak scaling: every rank renders its own P points of the global point-id space
    flags = ["fast_trig"] if args.fast_trig else 0
    scratch_t = make_scratch(cfs, torch, sysh, r) if args.variant != "direct" else None
    rargs = cfs.make_args(r, d_image=img, d_counters=ctr, point_offset=rank * P, flags=flags, variant=args.variant,
                          d_scratch=scratch_t)

    def step(timed):
        flush.zero_()                         # L2 flush, outside the events
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        img.zero_()
        cfs.cfs_render(sysh, rargs)
        ev[1].record()
        if world > 1:                          # the exchange step: one image all-reduce (sum)
            cfs.allreduce_image(img, r.out_mode)
        cfs.cfs_tonemap(img, r.out_mode, r.width, r.height, 2.2, 1 / 255.0, out8, scratch)
        ev[2].record()
        return ev

    for _ in range(max(args.warmup, 3)):
        step(False)
    torch.cuda.synchronize()
    rates = measure_rates(cfs, torch, flush, sms) if rank == 0 else None
    ctr.zero_()
    cfs.cfs_launch_count(reset=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    try:
        dev_uuid = torch.cuda.get_device_properties(local).uuid
    except Exception:
        dev_uuid = None
    sampler = ClockSampler(local, dev_uuid)
    if rank == 0:
        sampler.start()
    evs = [step(True) for _ in range(args.steps)]
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = cfs.cfs_launch_count()
    in_bounds = int(ctr[0].item())
    assert in_bounds == S * args.steps, f"conservation violated: {in_bounds} != {S * args.steps}"
    launches_per_render = (launches // max(args.steps, 1)) - 2        # minus the two tone-map kernels
    pass1_s = None
    if launches_per_render >= 2:       # binned: time pass 1 (sample + bin) apart from pass 2, same launch shape
        p1args = cfs.make_args(r, d_image=img, point_offset=rank * P, variant=args.variant,
                               flags=(["fast_trig"] if args.fast_trig else []) + ["bin_pass1_only"], d_scratch=scratch_t)
        ts = []
        for i in range(7):
            flush.zero_()
            e0, e1 = event_pair(torch)
            e0.record()
            cfs.cfs_render(sysh, p1args)
            e1.record()
            torch.cuda.synchronize()
            if i >= 2:
                ts.append(e0.elapsed_time(e1) * 1e-3)
        pass1_s = float(np.median(ts))
    step_s = sum(e[0].elapsed_time(e[2]) for e in evs) * 1e-3
    render_s = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3
    tt = torch.tensor([step_s, render_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    step_s, render_s = float(tt[0]), float(tt[1])

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    h_img = torch.empty((r.width * r.height, 4), dtype=torch.float32).pin_memory()
    h_ctr = torch.zeros(2, dtype=torch.int64).pin_memory()
    hargs = cfs.make_args(r, point_offset=rank * P, flags=flags)
    for _ in range(2):
        cfs.cfs_render_host(sysh, hargs, h_img.numpy(), None, h_ctr.numpy())
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    n_e2e = max(3, min(args.steps, 10))
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        cfs.cfs_render_host(sysh, hargs, h_img.numpy(), None, h_ctr.numpy())
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_s = float(te[0])
    assert int(h_ctr[0]) == S

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_per_step = step_s / args.steps * 1e3
    value = world * P * I * args.steps / step_s
    t_render = render_s / args.steps
    roof = roofline_for(HEADLINE_CFG, w, rates, peaks, S, t_render)
    binned = launches_per_render >= 2
    north_star = {"definition": "t_roof / t_render, t_roof = max(t_issue, t_atomic, t_hbm) (BASELINE north_star; "
                                "the L2-atomic term assumes one reduction per splat, which the binned variant does not pay)",
                  "bound": roof["bound"], "frac": roof["frac"], "t_issue_ms": roof["t_issue_ms"],
                  "t_atomic_ms": roof["t_atomic_ms"], "t_render_ms": t_render * 1e3}
    if binned:
        # dominant kernel: pass 1 (sample + chain + bin), bound by instruction issue
        hybrid = args.variant == "auto"
        if args.fast_trig:
            n_instr = N_INSTR_HYB[HEADLINE_CFG] if hybrid else N_INSTR_BIN[HEADLINE_CFG]
        else:
            n_instr = N_INSTR_HYB_ACC[HEADLINE_CFG] if hybrid else N_INSTR_BIN_ACC[HEADLINE_CFG]
        roofline = {
            "bound": "alu", "achieved": P * I * n_instr / pass1_s / 1e12, "peak": rates["ffma"] / 1e12,
            "unit": "T lane-instructions/s", "frac": (P * I * n_instr / pass1_s) / rates["ffma"],
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH if hybrid else NCU_TRAFFIC_BYTES_PER_LAUNCH_BINNED,
            "kernel": "cfs::render_kernel<2,IFS,DIAG,BIN,swirl+scale,%s>" % ("MUFU" if args.fast_trig else "sincosf"),
            "kernel_ms": pass1_s * 1e3, "render_ms": t_render * 1e3, "pass2_ms": (t_render - pass1_s) * 1e3,
            "algorithmic_lane_instructions_per_point_iteration": n_instr,
            "algorithmic_bytes_per_launch": int(S * 2) // (2 if hybrid else 1),      # one 16-bit record per binned splat
            "peak_source": "FFMA lane-issue rate of cfs_microbench in this run (148 SMs x 128 lanes x SM clock)",
            "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peaks_src,
            "pass2_hbm_gbs": (S * 2 // (2 if hybrid else 1)) / max(t_render - pass1_s, 1e-9) / 1e9,
        }
    else:
        peak_red = rates[RED_KEY[HEADLINE_CFG]]
        roofline = {
            "bound": roof["bound"], "achieved": S / t_render / 1e9,
            "peak": (peak_red / 1e9) if roof["bound"] == "l2_atomic" else S / (roof["t_roof_ms"] * 1e-3) / 1e9,
            "unit": "Gsplat/s (one red.global.add.v4.f32 per splat)", "frac": roof["frac"],
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH_DIRECT, "kernel": "cfs::render_kernel<2,IFS,DIAG,RGBA,swirl+affine>",
            "kernel_ms": t_render * 1e3, "t_issue_ms": roof["t_issue_ms"], "t_atomic_ms": roof["t_atomic_ms"],
            "peak_source": "red.global.add.v4.f32 at uniformly random pixels of a 16 MiB footprint, cfs_microbench "
                           "in this run (BASELINE north_star); FFMA issue rate from the same run for t_issue",
            "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peaks_src,
        }
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload_config(w, world),
        "splats_per_s": world * S * args.steps / step_s,
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": world * P * I * n_e2e / e2e_s, "unit": UNIT,
                "h2d_bytes_per_step": 0, "d2h_bytes_per_step": int(h_img.numel() * 4 + 16),
                "note": "cfs_render_host: clear + render + D2H of the float32 accumulators and counters into pinned "
                        "host memory; this workload has no host input besides the kernel parameter block"},
        "roofline": roofline, "north_star_roofline": north_star,
        "splat_variant": ("hybrid: every other splat straight to L2 (red.global), the rest through tile bins in scratch with shared-memory "
                          "tile accumulation (CFS_FLAG_BIN_HYBRID, set by AUTO)" if args.variant == "auto" else
                          "binned (tile bins through scratch, shared-memory tile accumulation)") if binned else "direct (one L2 reduction per splat)",
        "microbench": {k: (v / 1e9 if not k.endswith("GBps") else v) for k, v in rates.items()},
        "microbench_unit": "G lane-ops/s (stream: GB/s)",
    }

    # ---- the other four workloads of BASELINE.json (same metric; not bench lines of their own)
    if not args.no_workloads and world == 1:
        wl = {}
        for cfg in range(W.N_CONFIGS):
            wk, sec, n_in, n_drop = time_workload(cfs, torch, cfg, flush, flags=flags, variant=args.variant)
            pi = wk.point_iterations
            rf = roofline_for(cfg, wk, rates, peaks, n_in / len(wk.frames), sec / len(wk.frames))
            wl[f"cfg{cfg}"] = {"name": wk.name, "ms": sec * 1e3, "point_iterations_per_s": pi / sec,
                               "splats_per_s": n_in / sec, "in_bounds": n_in, "dropped": n_drop,
                               "roofline_bound": rf["bound"], "roofline_frac": rf["frac"],
                               "t_issue_ms": rf["t_issue_ms"] * len(wk.frames),
                               "t_atomic_ms": rf["t_atomic_ms"] * len(wk.frames),
                               "t_hbm_ms": rf["t_hbm_ms"] * len(wk.frames)}
        line["workloads"] = wl

    # ---- the oracle timed beside it (reported baseline, never tuned)
    n_cpu = 1 << 17
    pi, dt, threads = oracle_sample(HEADLINE_CFG, n_cpu)
    line["cpu_baseline"] = {"value": pi / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                            "sample": f"first {n_cpu} points x {I} iterations of configs[{HEADLINE_CFG}], full image, "
                                      f"{dt:.1f} s wall on {threads} threads", "cpu": host_cpu_model(),
                            "host_cores": os.cpu_count()}
    print(json.dumps(line), flush=True)
    sysh.close()
    if world > 1:
        dist.destroy_process_group()


def run_profile_cfg(args):
    """Target of the ncu commands under profiles/: `--steps` cfs_render launches of configs[N] (one
    frame, t = middle frame), 2 warm-ups, nothing else on the GPU.  Prints device time per launch."""
    import torch
    from paper_2606_02226_b200 import cfs
    torch.cuda.set_device(0)
    cfg = args.profile_cfg
    w = W.config(cfg)
    cloud = W.gaussian_mixture_cloud(w.render.n_points, w.cloud_seed) if w.system.gen == "cloud" else None
    d_cloud = cfs.cloud_to_device(cloud) if cloud is not None else None
    sysh = cfs.cfs_create(w.system)
    img = cfs.new_image(w.render)
    ctr = torch.zeros(2, dtype=torch.int64, device="cuda")
    t = w.frames[len(w.frames) // 2]
    scratch = make_scratch(cfs, torch, sysh, w.render) if args.variant in ("auto", "binned") else None
    rargs = cfs.make_args(w.render, d_image=img, d_cloud=d_cloud, d_counters=ctr, t=t, variant=args.variant,
                          flags=["fast_trig"] if args.fast_trig else 0, d_scratch=scratch)
    ms = []
    for i in range(2 + args.steps):
        img.fill_(-1 if w.render.out_mode == "depth_u64" else 0)
        e0, e1 = event_pair(torch)
        e0.record()
        cfs.cfs_render(sysh, rargs)
        e1.record()
        torch.cuda.synchronize()
        if i >= 2:
            ms.append(e0.elapsed_time(e1))
    print(json.dumps({"profile_cfg": cfg, "workload": w.name, "variant": args.variant, "launch_ms": ms,
                      "point_iterations_per_s": w.render.n_points * w.render.iterations / (min(ms) * 1e-3)}))
    sysh.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-workloads", action="store_true", help="skip the per-config side report")
    ap.add_argument("--profile-cfg", type=int, default=None,
                    help="only launch cfs_render of configs[N] --steps times (ncu target; no bench line)")
    ap.add_argument("--variant", default="auto", help="splat variant: auto (tile bins for large renders, else direct), direct, binned, ...")
    ap.add_argument("--accurate-trig", action="store_true",
                    help="evaluate sin/cos with sincosf (<= 2 ulp) instead of CFS_FLAG_FAST_TRIG (MUFU); both are inside "
                         "the BASELINE tolerances (tests/test_gpu_parity.py)")
    args = ap.parse_args()
    global SINCOS
    args.fast_trig = not args.accurate_trig
    if args.fast_trig:
        SINCOS = "MUFU sin.approx/cos.approx (CFS_FLAG_FAST_TRIG)"
    if args.profile_cfg is not None:
        run_profile_cfg(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
