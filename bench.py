#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native Joseph projector.

    python bench.py --gpus N --steps K --warmup W [--impl reference]

A "step" is one pass of the hot path over one batch of synthetic input: the non-TOF forward
projection of the phantom over all 151,584,768 sinogram LORs of BASELINE.json configs[1], followed
by the exact adjoint back projection of a U[0,1) sinogram (image zero-fill included).
`value` = LORs per second through that fwd+back pair (the paper reports fwd+back sums),
inputs resident in HBM.  `e2e` is the same pair through the host-buffer C-ABI calls
(jp_fwd_host / jp_back_host) with host<->device copies inside the timed region.

N > 1 (torchrun): LORs are independent units; every rank projects its own full
configs[1] sinogram of its own frame (weak scaling), no data-path collective; timing is the max over
ranks.  `--impl reference` times the float64 CPU oracle (oracle/) on a bounded sample of the same
workload on the host cores.
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
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2212_12519_b200 import inputs  # noqa: E402

METRIC = "LORs/s (non-TOF sinogram fwd+back pair)"
UNIT = "LORs/s"
WORKLOAD = ("configs[1]: non-TOF sinogram fwd+back, 151584768 LORs (257 radial x 256 views x 48x48 ring pairs), "
            "image 200x200x96 @ 2 mm (cylinder + 10 hot spheres)")
# FP32 lane-instructions per plane-step of the minimal formulation
LANE_INSTR_FWD = 11.0
LANE_INSTR_BACK = 12.0
FP32_LANES_PER_SM = 128
N_SM = 148


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, val in zip(names, r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- oracle legs ----------------------------------------------------------------------------------------------
def oracle_sample():
    """bounded sample of configs[1]: 17 views (incl. a 45 degree tie view) x all 257 radial x every 2nd ring pair"""
    views = sorted(set(range(5, 256, 16)) | {64})
    xs, xe = inputs.sinogram_lors(views=views)
    xs, xe = xs[:, ::2].contiguous().numpy(), xe[:, ::2].contiguous().numpy()
    desc = ("views {5,21,...,245} and 64 x 257 radial x every 2nd of the 2304 ring pairs = %d LORs of configs[1] "
            "(fwd + back, float64, OpenMP)" % xs.shape[1])
    return xs, xe, desc


def time_oracle(steps: int, warmup: int):
    import oracle
    oracle.build()
    g = inputs.GEOM_SCANNER
    ph = inputs.phantom().astype(np.float64)
    xs, xe, desc = oracle_sample()
    n = xs.shape[1]
    y = inputs.uniform_values(n, 0.0, 1.0, seed=inputs.BASE_SEED + 101).numpy().astype(np.float64)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.fwd(xs, xe, ph, g.origin, g.voxsize)
        t1 = time.perf_counter()
        oracle.back(xs, xe, y, g.n, g.origin, g.voxsize)
        t2 = time.perf_counter()
        if it >= warmup:
            times.append((t1 - t0, t2 - t1))
    tf = float(np.mean([t[0] for t in times]))
    tb = float(np.mean([t[1] for t in times]))
    return dict(n=n, fwd_s=tf, back_s=tb, cores=oracle.num_threads(), sample=desc)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    r = time_oracle(args.steps, args.warmup)
    t = r["fwd_s"] + r["back_s"]
    val = r["n"] / t
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample_per_step": r["sample"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
                         "fwd_lors_per_s": r["n"] / r["fwd_s"], "back_lors_per_s": r["n"] / r["back_s"]},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---- the CUDA arm ---------------------------------------------------------------------------------------------
def run_ours(args):
    from paper_2212_12519_b200 import binding as jp
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    jp.load()

    g = inputs.GEOM_SCANNER
    # frame `rank`: same scanner, its own phantom and sinogram values (weak scaling, no exchange)
    img = torch.from_numpy(inputs.phantom(seed=inputs.BASE_SEED + 1 + 1000 * rank)).to(dev)
    xs, xe = inputs.sinogram_lors(device=dev)
    n = xs.shape[1]
    y = inputs.uniform_values(n, 0.0, 1.0, seed=inputs.BASE_SEED + 101 + rank, device=dev)
    p = torch.empty(n, dtype=torch.float32, device=dev)
    bimg = torch.zeros(g.n, dtype=torch.float32, device=dev)
    plane_steps = jp.jp_plane_steps(xs, xe, g.n, g.origin, g.voxsize)
    stream = torch.cuda.current_stream()

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        jp.jp_fwd(xs, xe, img, g.origin, g.voxsize, out=p)
        if ev:
            ev[1].record(stream)
        bimg.zero_()
        jp.jp_back(xs, xe, y, g.n, g.origin, g.voxsize, img=bimg)
        if ev:
            ev[2].record(stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    e_beg = torch.cuda.Event(enable_timing=True)
    e_end = torch.cuda.Event(enable_timing=True)
    e_beg.record(stream)
    for k in range(args.steps):
        step(evs[k])
    e_end.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = e_beg.elapsed_time(e_end)
    fwd_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    back_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))   # includes the image zero-fill
    checksum = float(p[:: max(1, n // 4096)].double().sum()) + float(bimg.double().sum())

    # ---- end to end through the host-buffer C ABI (pinned host tensors; H2D + kernels + D2H timed) --------
    e2e = None
    if not args.no_e2e:
        hxs, hxe = xs.cpu().pin_memory(), xe.cpu().pin_memory()
        hy, himg = y.cpu().pin_memory(), img.cpu().pin_memory()
        hp = torch.empty(n, dtype=torch.float32).pin_memory()
        hb = torch.zeros(g.n, dtype=torch.float32).pin_memory()

        def e2e_step():
            jp.jp_fwd_host(hxs, hxe, himg, g.origin, g.voxsize, out=hp)
            hb.zero_()
            jp.jp_back_host(hxs, hxe, hy, hb, g.origin, g.voxsize)

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        ne2e = max(1, min(args.steps, 3))
        for _ in range(ne2e):
            e2e_step()
        barrier()
        e2e_s = (time.perf_counter() - t0) / ne2e
        nvox = int(np.prod(g.n))
        e2e = {"s_per_step": e2e_s,
               "h2d": 2 * 24 * n + 4 * n + 2 * 4 * nvox, "d2h": 4 * n + 4 * nvox,
               "check": float((hp[:: max(1, n // 4096)].double().sum()))}
        del hxs, hxe, hy, hp

    if world > 1:
        t = torch.tensor([total_ms, fwd_ms, back_ms, e2e["s_per_step"] if e2e else 0.0], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, fwd_ms, back_ms = float(t[0]), float(t[1]), float(t[2])
        if e2e:
            e2e["s_per_step"] = float(t[3])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_per_step = total_ms / args.steps
    value = world * n / (ms_per_step * 1e-3)
    peaks, peak_src = measured_peaks()
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak = N_SM * FP32_LANES_PER_SM * sm_mhz * 1e6          # FP32 lane-instructions / s
    dom = "back" if back_ms >= fwd_ms else "fwd"
    dom_ms = max(back_ms, fwd_ms)
    lane = LANE_INSTR_BACK if dom == "back" else LANE_INSTR_FWD
    achieved = lane * plane_steps / (dom_ms * 1e-3)
    hbm_bytes = n * 28 + int(np.prod(g.n)) * 4
    roofline = {
        "bound": "alu", "kernel": "k_back" if dom == "back" else "k_fwd",
        "achieved": achieved / 1e12, "peak": alu_peak / 1e12, "unit": "T lane-instr/s (FP32)",
        "frac": achieved / alu_peak, "traffic": None,
        "peak_source": f"148 SMs x 128 FP32 lanes x {sm_mhz:.0f} MHz (sm_max_mhz of MEASURED_PEAKS.json, {peak_src})",
        "plane_steps_per_launch": plane_steps, "lane_instr_per_plane_step": lane,
        "fwd": {"ms": fwd_ms, "lors_per_s": n / fwd_ms * 1e3, "frac_alu": LANE_INSTR_FWD * plane_steps / (fwd_ms * 1e-3) / alu_peak},
        "back": {"ms": back_ms, "lors_per_s": n / back_ms * 1e3, "frac_alu": LANE_INSTR_BACK * plane_steps / (back_ms * 1e-3) / alu_peak},
        "hbm_bound_frac": hbm_bytes / (dom_ms * 1e-3) / (float(peaks["hbm_gbs"]) * 1e9),
    }
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "lors_per_gpu": n, "l2": "inputs (4.2 GB of end points + values per step) exceed the 126 MB L2; no flush",
                   "parallelism": f"frames{world}" if world > 1 else "single"},
        "gpu_launches": 2 * args.steps,
        "clocks": clocks,
        "roofline": roofline,
        "checksum": checksum,
    }
    if e2e:
        line["e2e"] = {"value": world * n / e2e["s_per_step"], "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"],
                       "d2h_bytes_per_step": e2e["d2h"], "ms_per_step": e2e["s_per_step"] * 1e3,
                       "api": "jp_fwd_host + jp_back_host (pinned host tensors)"}
    if world == 1 and not args.no_cpu_baseline:
        r = time_oracle(1, 0)
        t = r["fwd_s"] + r["back_s"]
        line["cpu_baseline"] = {"value": r["n"] / t, "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                "sample": r["sample"], "fwd_lors_per_s": r["n"] / r["fwd_s"],
                                "back_lors_per_s": r["n"] / r["back_s"]}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
