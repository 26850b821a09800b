#!/usr/bin/env python
"""bench.py -- benchmark of the B200-native Joseph projector.

    python bench.py --gpus N --steps K --warmup W [--config {0,1,2,3,4,5}] [--check] [--impl reference]

A "step" is one pass of the hot path over one batch of synthetic input.  The default workload is
BASELINE.json configs[1] (the configuration the headline LORs/s is quoted on): the non-TOF forward
projection of the phantom over all 151,584,768 sinogram LORs followed by the exact adjoint back projection
of a U[0,1) sinogram (image zero-fill included).  `value` = LORs per second through that fwd+back pair
(the paper reports fwd+back sums), inputs resident in HBM.  `e2e` is the same pair through the
host-buffer C-ABI calls (jp_fwd_host / jp_back_host) with host<->device copies inside the timed region.
The default run also times configs[2], [3] and [4] briefly and reports them under "other_configs"
(BASELINE.json metric: LORs/s fwd, back and TOF-LM events/s, each with its roofline fraction);
`--config C` makes configs[C] the timed workload of the line instead (used for the ncu captures in profiles/);
`--check` adds `parity` to the line: the float64 oracle run on the FULL config (outside the timed region; configs[4]:
40 M events x 20 subsets x 3 iterations, about ten minutes on 16 cores) against the CUDA results of the same inputs,
with the oracle's wall time per direction (`oracle_full`).  configs[0] (50,000 LORs, 4e5 plane-steps) is launch-bound.

N > 1 (torchrun): LORs are independent units; every rank projects its own full frame (weak
scaling), no data-path collective; timing is the max over ranks.  `--impl reference` times the float64 CPU
oracle (oracle/) on a bounded sample of the same workload on the host cores.
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

G = inputs.GEOM_SCANNER
NVOX = int(np.prod(G.n))
TOFP = inputs.TofParams()
TOF_ARGS = (TOFP.tofbin_width, TOFP.sigma_tof, TOFP.n_sigmas, TOFP.n_tofbins)

# FP32 lane-instructions per plane-step of the minimal formulation
LANE = {"fwd": 11.0, "back": 12.0, "lm": 40.0, "sino": 112.0}
FP32_LANES_PER_SM = 128
N_SM = 148
# ncu figures of the dominant kernels (dram bytes per launch, issue-slot / l1tex / L2 utilisation), read from the text
# summary of the one `ncu --set full` capture per config committed under profiles/ (the file names its commands and
# the commit it was taken at); a number measured under the profiler is never a bench value -- these only explain it
NCU_CSV = os.path.join(ROOT, "profiles", "r03_kernel_metrics.csv")


def ncu_metrics():
    out = {}
    if not os.path.exists(NCU_CSV):
        return out
    import csv
    with open(NCU_CSV) as fh:
        for r in csv.DictReader(fh):
            out[(int(r["config"]), r["direction"])] = r
    return out


def ncu_note(c, direction):
    r = ncu_metrics().get((c, direction))
    if not r:
        return None
    f = lambda k: float(r[k]) if r.get(k) not in (None, "") else None
    dur = (f("duration_ms") or 0.0) * 1e-3
    rate = lambda k: (f(k) / dur) if (dur > 0 and f(k) is not None) else None
    atomics = {   # north_star (d) "atomic throughput": counts per launch (profiles/r03_kernel_metrics.md) over ncu's duration
        "shared_atomic_warp_instr_per_s": rate("shared_atom_inst"), "global_red_warp_instr_per_s": rate("red_inst"),
        "global_red_sectors_per_s": rate("red_sectors"),
        "global_red_GBps_at_l2": (rate("red_sectors") * 32 / 1e9) if rate("red_sectors") is not None else None,
        "shared_wavefronts_per_s": rate("shared_wavefronts"),
        "shared_bank_conflict_share": (f("shared_bank_conflicts") / f("shared_wavefronts")) if f("shared_wavefronts") else None}
    return {"source": "profiles/r03_kernel_metrics.csv (ncu --set full, commit %s)" % r.get("commit", "?"), "kernel": r["kernel"],
            "atomics": atomics,
            "duration_ms": f("duration_ms"), "dram_bytes_per_launch": (f("dram_read_bytes") or 0) + (f("dram_write_bytes") or 0),
            "issue_slots_busy_pct": f("issue_pct"), "l1tex_throughput_pct": f("l1tex_pct"), "l2_throughput_pct": f("lts_pct"),
            "fma_pipe_pct": f("fma_pipe_pct"), "l1_hit_pct": f("l1_hit_pct"), "l2_hit_pct": f("l2_hit_pct"),
            "warp_instr_per_plane_step": f("warp_instr_per_step")}


SPEC = {
    0: dict(metric="LORs/s (non-TOF fwd+back pair, small case)", unit="LORs/s",
            workload="configs[0]: non-TOF fwd+back, 50000 random chords of a cylinder (r 150 mm, |z| < 40 mm), image "
                     "32x32x16 @ 4 mm U[0,1); LAUNCH-BOUND (4.06e5 plane-steps: microseconds of work per call), a "
                     "roofline fraction is not meaningful for it",
            l2="inputs (1.4 MB) fit in L2: a 256 MB buffer is overwritten between timed steps (L2 flush, outside the "
               "per-direction events)"),
    1: dict(metric="LORs/s (non-TOF sinogram fwd+back pair)", unit="LORs/s",
            workload="configs[1]: non-TOF sinogram fwd+back, 151584768 LORs (257 radial x 256 views x 48x48 ring "
                     "pairs), image 200x200x96 @ 2 mm (cylinder + 10 hot spheres)",
            l2="inputs (4.2 GB of end points + values per step) exceed the 126 MB L2; no flush"),
    2: dict(metric="LORs/s (TOF sinogram fwd+back pair, 29 TOF bins per LOR)", unit="LORs/s",
            workload="configs[2]: TOF sinogram fwd+back, one OSEM subset = 16 views x 257 radial x 2304 ring pairs "
                     "= 9474048 LORs x 29 TOF bins of 17 mm, sigma 13.6 mm, 3 sigma; same scanner and phantom",
            l2="inputs (227 MB of end points + 1.1 GB of TOF sinogram per direction) exceed the 126 MB L2; no flush"),
    3: dict(metric="events/s (TOF listmode fwd+back pair)", unit="events/s",
            workload="configs[3]: TOF listmode fwd+back, 40000000 events sampled from the phantom (crystal-snapped "
                     "end points, int16 TOF bin), sorted once by the listmode plan; results in caller order",
            l2="inputs (1.04 GB of sorted events + 0.32 GB of per-event values per step) exceed the 126 MB L2; no flush"),
    5: dict(metric="LORs/s (TOF sinogram OSEM with mult / contam, one full iteration of 16 subsets)", unit="LORs/s",
            workload="SURVEY 8(f) row 3: TOF sinogram OSEM on the full configs[1] sinogram x 29 TOF bins (151584768 LORs, "
                     "17.6 GB emission + 17.6 GB contamination sinograms resident in HBM), 16 subsets of 16 views (the "
                     "configs[2] subset structure), multiplicative factors per LOR; one step = one full iteration",
            l2="every iteration streams 3.6 GB of end points and 35 GB of sinograms; no flush"),
    4: dict(metric="events/s (TOF listmode OSEM, one full iteration of 20 subsets)", unit="events/s",
            workload="configs[4]: listmode OSEM on the configs[3] events, 20 subsets, sens = non-TOF A^T 1 over all "
                     "configs[1] LORs; one step = one full iteration (20 x (fwd, ratio, back, update))",
            l2="every iteration streams all 1.04 GB of sorted events; no flush"),
}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """SM clock / throttle reasons sampled while the timed region runs: NVML (nvidia_ml_py) every 5 ms; if NVML cannot be
    used, `nvidia-smi -lms` (which delivers a sample every ~60 ms at best)"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []       # nvidia-smi rows
        self.samples = []    # NVML: (sm_mhz, reasons bit mask)
        self.proc = None
        self.nvml = None
        self.stop_flag = False
        self.max_mhz = None

    def _nvml_handle(self):
        import pynvml
        pynvml.nvmlInit()
        try:
            uuid = str(torch.cuda.get_device_properties(self.index).uuid)
            if not uuid.startswith("GPU-"):
                uuid = "GPU-" + uuid
            h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
        except Exception:
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            ids = [v for v in vis.split(",") if v.strip() != ""]
            phys = int(ids[self.index]) if ids and all(v.strip().isdigit() for v in ids) else self.index
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
        return pynvml, h

    def _poll(self, pynvml, h):
        get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self.stop_flag:
            try:
                self.samples.append((float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)), int(get_reasons(h))))
            except Exception:
                break
            time.sleep(0.005)

    def start(self):
        try:
            pynvml, h = self._nvml_handle()
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
            self.thread = threading.Thread(target=self._poll, args=(pynvml, h), daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.nvml is not None:
            self.stop_flag = True
            self.thread.join(timeout=2)
            p = self.nvml
            bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
            reasons = sorted(n for n, b in bits.items() if any(m & b for _, m in self.samples))
            sm = [c for c, _ in self.samples]
            return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": self.max_mhz, "samples": len(sm),
                    "reasons": reasons, "source": "NVML, 5 ms"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
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
                "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi -lms"}


# ---- oracle legs (cpu_baseline and --impl reference): the float64 oracle on a bounded sample ------------------
def time_oracle(config: int, steps: int, warmup: int):
    """(units in the sample, mean fwd s, mean back s, cores, description); for config 4 fwd_s = whole iteration"""
    import oracle
    oracle.build()
    ph = inputs.phantom().astype(np.float64)
    if config == 0:
        c0 = inputs.config0()
        g0 = c0["geom"]
        xs, xe, n = c0["xstart"], c0["xend"], c0["xstart"].shape[1]
        desc = "the whole of configs[0]: %d LORs (fwd + back, float64, OpenMP)" % n
        i0, y0 = c0["img"].astype(np.float64), c0["y"].astype(np.float64)
        f = lambda: oracle.fwd(xs, xe, i0, g0.origin, g0.voxsize)
        b = lambda: oracle.back(xs, xe, y0, g0.n, g0.origin, g0.voxsize)
    elif config == 1:
        # 17 views (incl. a 45 degree tie view) x all 257 radial x every 2nd ring pair
        views = sorted(set(range(5, 256, 16)) | {64})
        xs, xe = inputs.sinogram_lors(views=views)
        xs, xe = xs[:, ::2].contiguous().numpy(), xe[:, ::2].contiguous().numpy()
        n = xs.shape[1]
        desc = ("views {5,21,...,245} and 64 x 257 radial x every 2nd of the 2304 ring pairs = %d LORs of configs[1] "
                "(fwd + back, float64, OpenMP)" % n)
        y = inputs.uniform_values(n, 0.0, 1.0, seed=inputs.BASE_SEED + 101).numpy().astype(np.float64)
        f = lambda: oracle.fwd(xs, xe, ph, G.origin, G.voxsize)
        b = lambda: oracle.back(xs, xe, y, G.n, G.origin, G.voxsize)
    elif config == 5:
        xs, xe = inputs.sinogram_lors(views=inputs.SUBSET_VIEWS)
        xs, xe = xs[:, ::24].contiguous().numpy(), xe[:, ::24].contiguous().numpy()
        n = xs.shape[1]
        desc = ("one OSEM subset update (fwd, ratio, back, image update) with mult and contam on every 24th LOR of one "
                "16-view subset = %d LORs x 29 TOF bins (float64, numpy + OpenMP projectors)" % n)
        rng = np.random.default_rng(5)
        y5, m5, c5 = rng.random((n, 29)), rng.uniform(0.2, 1.0, n), np.full((n, 29), 0.05)
        s5 = np.ones((1,) + tuple(G.n))
        f = lambda: oracle.sino_osem_tof(xs, xe, [0, n], y5, m5, c5, s5, np.ones(G.n), G.origin, G.voxsize, *TOF_ARGS,
                                         n_iter=1)
        b = lambda: None
    elif config == 2:
        xs, xe = inputs.sinogram_lors(views=inputs.SUBSET_VIEWS)
        xs, xe = xs[:, ::24].contiguous().numpy(), xe[:, ::24].contiguous().numpy()
        n = xs.shape[1]
        desc = ("every 24th LOR of the configs[2] subset = %d LORs x 29 TOF bins (fwd + back, float64, OpenMP)" % n)
        y = inputs.uniform_values((n, 29), 0.0, 1.0, seed=inputs.BASE_SEED + 102).numpy().astype(np.float64)
        f = lambda: oracle.fwd_tof_sino(xs, xe, ph, G.origin, G.voxsize, *TOF_ARGS)
        b = lambda: oracle.back_tof_sino(xs, xe, y, G.n, G.origin, G.voxsize, *TOF_ARGS)
    else:
        n = 1_000_000
        xs, xe, tb = inputs.listmode_events(n, img=inputs.phantom(), chunk=2_000_000)
        xs, xe, tb = xs.numpy(), xe.numpy(), tb.numpy()
        if config == 3:
            desc = "1000000 events of the configs[3] model (CPU-seeded) (fwd + back, float64, OpenMP)"
            y = inputs.uniform_values(n, 0.5, 2.0, seed=inputs.BASE_SEED + 103).numpy().astype(np.float64)
            f = lambda: oracle.fwd_tof_lm(xs, xe, tb, ph, G.origin, G.voxsize, *TOF_ARGS[:3])
            b = lambda: oracle.back_tof_lm(xs, xe, tb, y, G.n, G.origin, G.voxsize, *TOF_ARGS[:3])
        else:
            desc = ("one OSEM iteration (20 subsets) on 1000000 events of the configs[3] model, sens = ones "
                    "(float64, OpenMP)")
            sens = np.ones(G.n)
            f = lambda: oracle.lm_osem(xs, xe, tb, sens, np.ones(G.n, dtype=np.float32), G.origin, G.voxsize,
                                       *TOF_ARGS[:3], n_subsets=20, n_iter=1)
            b = lambda: None
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        f()
        t1 = time.perf_counter()
        b()
        t2 = time.perf_counter()
        if it >= warmup:
            times.append((t1 - t0, t2 - t1))
    tf = float(np.mean([t[0] for t in times]))
    tb_ = float(np.mean([t[1] for t in times]))
    return dict(n=n, fwd_s=tf, back_s=tb_, cores=oracle.num_threads(), sample=desc)


def cpu_baseline_dict(config: int, r: dict):
    t = r["fwd_s"] + r["back_s"]
    d = {"value": r["n"] / t, "unit": SPEC[config]["unit"], "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
         "sample_kind": "bounded sample of the workload, one run (the full config is timed under --check: parity.oracle_full)"}
    if config < 4:
        d["fwd_per_s"] = r["n"] / r["fwd_s"]
        d["back_per_s"] = r["n"] / r["back_s"]
    return d


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = args.config
    r = time_oracle(c, args.steps, args.warmup)
    t = r["fwd_s"] + r["back_s"]
    val = r["n"] / t
    line = {
        "impl": "reference", "metric": SPEC[c]["metric"], "value": val, "unit": SPEC[c]["unit"], "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": SPEC[c]["workload"], "sample_per_step": r["sample"]},
        "cpu_baseline": cpu_baseline_dict(c, r),
        "e2e": {"value": val, "unit": SPEC[c]["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---- the CUDA arm: one Workload per BASELINE.json config -------------------------------------------------------
class Workload:
    """set-up (untimed) of configs[c] on `dev`; step(ev) enqueues one pass on the current stream and records
    the events ev[0] (start), ev[1] (forward done), ev[2] (back done) when given."""

    def __init__(self, c: int, jp, dev, rank: int):
        self.c, self.jp, self.dev = c, jp, dev
        self.stream = torch.cuda.current_stream()
        self.tof = jp.make_tof(*TOF_ARGS)
        self.img = torch.from_numpy(inputs.phantom(seed=inputs.BASE_SEED + 1 + 1000 * rank)).to(dev)
        self.bimg = torch.zeros(G.n, dtype=torch.float32, device=dev)
        self.plan = None
        self.splan = None
        self.plan_s = None
        self.g = G
        self.flush = None
        if c == 0:
            c0 = inputs.config0()
            self.g = c0["geom"]
            self.xs, self.xe = torch.from_numpy(c0["xstart"]).to(dev), torch.from_numpy(c0["xend"]).to(dev)
            self.img = torch.from_numpy(c0["img"]).to(dev)
            self.y = torch.from_numpy(c0["y"]).to(dev)
            self.n = self.xs.shape[1]
            self.p = torch.empty(self.n, dtype=torch.float32, device=dev)
            self.bimg = torch.zeros(self.g.n, dtype=torch.float32, device=dev)
            self.plane_steps = jp.jp_plane_steps(self.xs, self.xe, self.g.n, self.g.origin, self.g.voxsize)
            self.kinds = ("fwd", "back")
            self.launches = 2
            self.hbm_bytes = self.n * 28 + int(np.prod(self.g.n)) * 4
            self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
        elif c == 5:
            nsub = 16
            order = [m + nsub * k for m in range(nsub) for k in range(inputs.N_VIEWS // nsub)]   # subset-major views
            self.xs, self.xe = inputs.sinogram_lors(views=order, device=dev)
            self.n = self.xs.shape[1]
            per = self.n // nsub
            self.off = [m * per for m in range(nsub + 1)]
            nb = TOFP.n_tofbins
            self.y = inputs.uniform_values((self.n, nb), 0.0, 1.0, seed=inputs.BASE_SEED + 105 + rank, device=dev)
            self.contam = torch.full((self.n, nb), 0.05, dtype=torch.float32, device=dev)
            self.mult = inputs.uniform_values(self.n, 0.2, 1.0, seed=inputs.BASE_SEED + 205 + rank, device=dev)
            self.ws = torch.empty(jp.jp_sino_osem_tof_workspace_bytes(self.off, self.n, self.tof), dtype=torch.uint8,
                                  device=dev)
            self.make_sino_plan()
            if self.splan is not None:
                self.sens = jp.jp_sino_sens_tof_planned(self.splan, self.off, self.mult, G.n, G.origin, G.voxsize, self.tof)
            else:
                self.sens = jp.jp_sino_sens_tof(self.xs, self.xe, self.off, self.mult, G.n, G.origin, G.voxsize, self.tof)
            self.x = torch.ones(G.n, dtype=torch.float32, device=dev)
            self.plane_steps = jp.jp_plane_steps(self.xs, self.xe, G.n, G.origin, G.voxsize)
            self.kinds = ("sino", "sino")
            self.launches = nsub * 3     # per subset: weight table, fused forward + ratio + back kernel, image update
            self.hbm_bytes = self.n * (24 + 4 + 2 * 4 * nb) // 2   # x 2 in the roofline dict: end points, mult, y + contam once per iteration
        elif c in (1, 2):
            self.xs, self.xe = inputs.sinogram_lors(views=None if c == 1 else inputs.SUBSET_VIEWS, device=dev)
            self.n = self.xs.shape[1]
            shape = self.n if c == 1 else (self.n, TOFP.n_tofbins)
            self.y = inputs.uniform_values(shape, 0.0, 1.0, seed=inputs.BASE_SEED + 100 + c + rank, device=dev)
            self.p = torch.empty(shape, dtype=torch.float32, device=dev)
            self.plane_steps = jp.jp_plane_steps(self.xs, self.xe, G.n, G.origin, G.voxsize)
            self.kinds = ("fwd", "back") if c == 1 else ("sino", "sino")
            self.launches = 2 if c == 1 else 8   # unplanned: c1 one tile kernel per direction; c2: pad/unpad, 2 tables, kernel
            self.make_sino_plan()
            if self.splan is not None:
                self.launches = 4   # per direction: c1 the track table + the whole-track kernel; c2 the weight table + the tile kernel
            self.hbm_bytes = (self.n * 28 + NVOX * 4) if c == 1 else (self.n * (24 + 4 * TOFP.n_tofbins) + NVOX * 4)
        else:
            nev = int(os.environ.get("JP_BENCH_EVENTS", "40000000"))
            self.xs, self.xe, self.tb = inputs.listmode_events(nev, seed=inputs.BASE_SEED + 3 + rank, device=dev,
                                                               img=inputs.phantom())
            self.n = self.xs.shape[1]
            self.plane_steps = jp.jp_plane_steps_tof_lm(self.xs, self.xe, self.tb, G.n, G.origin, G.voxsize, self.tof)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            self.plan = jp.LmPlan(self.xs, self.xe, self.tb, G.n, G.origin, G.voxsize, self.tof,
                                  n_subsets=1 if c == 3 else 20)   # configs[3] has no subsets: one sorted list
            torch.cuda.synchronize()
            self.plan_s = time.perf_counter() - t0
            self.kinds = ("lm", "lm")
            self.hbm_bytes = self.n * 30 + NVOX * 4
            if c == 3:
                self.y = inputs.uniform_values(self.n, 0.5, 2.0, seed=inputs.BASE_SEED + 103 + rank, device=dev)
                self.p = torch.empty(self.n, dtype=torch.float32, device=dev)
                # per direction: the edge table, and per principal axis (x, y) the bin-weight table + the line-tile kernel
                self.launches = 2 * (1 + 2 * 2)
            else:
                self.sens = torch.ones(G.n, dtype=torch.float32, device=dev)   # replaced by A^T 1 in setup_sens()
                self.x = torch.ones(G.n, dtype=torch.float32, device=dev)
                # per subset: brick forward, float-atomic adjoint per axis (x, y), update; + two tables per call
                self.launches = 4 * 20 + 2

    def make_sino_plan(self):
        """sinogram plan of the workload's LOR list (set-up, timed separately: `plan_s`); JP_BENCH_UNPLANNED=1 in the
        environment times the unplanned per-LOR kernels instead (A/B measurements)"""
        self.splan = None
        if os.environ.get("JP_BENCH_UNPLANNED", "0") == "1":
            return
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        self.splan = self.jp.SinoPlan(self.xs, self.xe)
        torch.cuda.synchronize()
        self.plan_s = time.perf_counter() - t0

    def setup_sens(self):
        """configs[4]: sens = non-TOF back projection of ones over all configs[1] LORs (one-time, untimed)"""
        sx, se = inputs.sinogram_lors(device=self.dev)
        self.sens.zero_()
        self.jp.jp_back(sx, se, torch.ones(sx.shape[1], device=self.dev), G.n, G.origin, G.voxsize, img=self.sens)
        torch.cuda.synchronize()

    def step(self, ev=None):
        jp, c, s = self.jp, self.c, self.stream
        if self.flush is not None:
            self.flush.zero_()
        if ev:
            ev[0].record(s)
        if c == 0:
            jp.jp_fwd(self.xs, self.xe, self.img, self.g.origin, self.g.voxsize, out=self.p)
        elif c == 1:
            if self.splan is not None:
                jp.jp_fwd_planned(self.splan, self.img, G.origin, G.voxsize, out=self.p)
            else:
                jp.jp_fwd(self.xs, self.xe, self.img, G.origin, G.voxsize, out=self.p)
        elif c == 2:
            if self.splan is not None:
                jp.jp_fwd_tof_sino_planned(self.splan, self.img, G.origin, G.voxsize, self.tof, out=self.p)
            else:
                jp.jp_fwd_tof_sino(self.xs, self.xe, self.img, G.origin, G.voxsize, self.tof, out=self.p)
        elif c == 3:
            jp.jp_fwd_tof_lm_planned(self.plan, self.img, out=self.p)
        elif c == 5:
            if self.splan is not None:
                jp.jp_sino_osem_tof_planned(self.splan, self.off, self.y, self.mult, self.contam, self.sens, self.x,
                                            G.origin, G.voxsize, self.tof, n_iter=1, workspace=self.ws)
            else:
                jp.jp_sino_osem_tof(self.xs, self.xe, self.off, self.y, self.mult, self.contam, self.sens, self.x,
                                    G.origin, G.voxsize, self.tof, n_iter=1, workspace=self.ws)
        else:
            jp.jp_lm_osem_planned(self.plan, self.sens, self.x, n_iter=1)
        if ev:
            ev[1].record(s)
        if c < 4:
            self.bimg.zero_()
        if c == 0:
            jp.jp_back(self.xs, self.xe, self.y, self.g.n, self.g.origin, self.g.voxsize, img=self.bimg)
        elif c == 1:
            if self.splan is not None:
                jp.jp_back_planned(self.splan, self.y, G.n, G.origin, G.voxsize, img=self.bimg)
            else:
                jp.jp_back(self.xs, self.xe, self.y, G.n, G.origin, G.voxsize, img=self.bimg)
        elif c == 2:
            if self.splan is not None:
                jp.jp_back_tof_sino_planned(self.splan, self.y, G.n, G.origin, G.voxsize, self.tof, img=self.bimg)
            else:
                jp.jp_back_tof_sino(self.xs, self.xe, self.y, G.n, G.origin, G.voxsize, self.tof, img=self.bimg)
        elif c == 3:
            jp.jp_back_tof_lm_planned(self.plan, self.y, img=self.bimg)
        if ev:
            ev[2].record(s)

    def time_nontof_listmode(self, reps=3):
        """NON-TOF fwd / back over the configs[3] events, unsorted (jp_fwd /
        jp_back on the acquisition order) and through the plan (sorted, line tiles); ms per call"""
        jp, s = self.jp, self.stream
        out = {}
        y = self.y
        p = torch.empty(self.n, dtype=torch.float32, device=self.dev)
        calls = {
            "unsorted": (lambda: jp.jp_fwd(self.xs, self.xe, self.img, G.origin, G.voxsize, out=p),
                         lambda: jp.jp_back(self.xs, self.xe, y, G.n, G.origin, G.voxsize, img=self.bimg)),
            "planned": (lambda: jp.jp_fwd_lm_planned(self.plan, self.img, out=p),
                        lambda: jp.jp_back_lm_planned(self.plan, y, img=self.bimg)),
        }
        for name, (f, b) in calls.items():
            f(); self.bimg.zero_(); b()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ev[0].record(s)
            for _ in range(reps):
                f()
            ev[1].record(s)
            for _ in range(reps):
                self.bimg.zero_()
                b()
            ev[2].record(s)
            torch.cuda.synchronize()
            fm, bm = ev[0].elapsed_time(ev[1]) / reps, ev[1].elapsed_time(ev[2]) / reps
            out[name] = {"fwd_ms": fm, "back_ms": bm, "fwd_events_per_s": self.n / fm * 1e3,
                         "back_events_per_s": self.n / bm * 1e3}
        out["plane_steps"] = self.jp.jp_plane_steps(self.xs, self.xe, G.n, G.origin, G.voxsize)
        return out

    def time_plan_order_io(self, reps=5):
        """configs[3] with the per-event arrays in PLAN order (jp_*_tof_lm_planned_sorted): no gather /
        scatter through the permutation; ms per call"""
        jp, s = self.jp, self.stream
        ys = jp.jp_lm_plan_permute(self.plan, self.y, True)
        ps = torch.empty(self.n, dtype=torch.float32, device=self.dev)
        f = lambda: jp.jp_fwd_tof_lm_planned_sorted(self.plan, self.img, out=ps)
        b = lambda: jp.jp_back_tof_lm_planned_sorted(self.plan, ys, img=self.bimg)
        f(); self.bimg.zero_(); b()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record(s)
        for _ in range(reps):
            f()
        ev[1].record(s)
        for _ in range(reps):
            self.bimg.zero_()
            b()
        ev[2].record(s)
        torch.cuda.synchronize()
        fm, bm = ev[0].elapsed_time(ev[1]) / reps, ev[1].elapsed_time(ev[2]) / reps
        return {"fwd_ms": fm, "back_ms": bm, "fwd_events_per_s": self.n / fm * 1e3, "back_events_per_s": self.n / bm * 1e3}

    def time_nonaligned_tracks(self, reps=5):
        """tracks whose length is not a multiple of the 768-LOR tile: the 36-ring sub-scanner of every 4th view of
        configs[1] (36 x 36 = 1296 ring pairs per track, 21.3 M LORs); ms per call and plane-steps per second"""
        jp, s = self.jp, self.stream
        xs, xe = inputs.sinogram_lors(views=range(0, inputs.N_VIEWS, 4), device=self.dev)
        idx = torch.arange(xs.shape[1], device=self.dev)
        keep = ((idx // 48) % 48 < 36) & (idx % 48 < 36)
        xs, xe = xs[:, keep].contiguous(), xe[:, keep].contiguous()
        n = xs.shape[1]
        y = inputs.uniform_values(n, 0.0, 1.0, seed=inputs.BASE_SEED + 136, device=self.dev)
        p = torch.empty(n, dtype=torch.float32, device=self.dev)
        steps = jp.jp_plane_steps(xs, xe, G.n, G.origin, G.voxsize)
        plan = jp.SinoPlan(xs, xe)
        out = {"lors": n, "track_length": plan.track_length, "plane_steps": steps}
        calls = {"planned": (lambda: jp.jp_fwd_planned(plan, self.img, G.origin, G.voxsize, out=p),
                             lambda: jp.jp_back_planned(plan, y, G.n, G.origin, G.voxsize, img=self.bimg)),
                 "unplanned": (lambda: jp.jp_fwd(xs, xe, self.img, G.origin, G.voxsize, out=p),
                               lambda: jp.jp_back(xs, xe, y, G.n, G.origin, G.voxsize, img=self.bimg))}
        for name, (f, b) in calls.items():
            f(); self.bimg.zero_(); b()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ev[0].record(s)
            for _ in range(reps):
                f()
            ev[1].record(s)
            for _ in range(reps):
                self.bimg.zero_()
                b()
            ev[2].record(s)
            torch.cuda.synchronize()
            fm, bm = ev[0].elapsed_time(ev[1]) / reps, ev[1].elapsed_time(ev[2]) / reps
            out[name] = {"fwd_ms": fm, "back_ms": bm, "fwd_plane_steps_per_s": steps / fm * 1e3,
                         "back_plane_steps_per_s": steps / bm * 1e3}
        plan.destroy()
        return out

    def time_osem_paths(self, iters=3):
        """A/B of the kernels behind one OSEM iteration (jp_lm_plan_set_path): 2 = quad image both ways (round 1),
        3 = image bricks forward + float atomics back (what the plan chooses, the timed configuration); ms per iteration"""
        out = {}
        for path, name in ((2, "quad_both_ways"), (3, "bricks_forward_float_adjoint")):
            self.plan.set_path(path)
            self.x.fill_(1.0)
            self.jp.jp_lm_osem_planned(self.plan, self.sens, self.x, n_iter=1)
            ts = []
            for _ in range(iters):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(self.stream)
                self.jp.jp_lm_osem_planned(self.plan, self.sens, self.x, n_iter=1)
                e1.record(self.stream)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            out[name] = {"ms_per_iteration": float(np.median(ts)), "min_ms": float(min(ts))}
        self.plan.set_path(0)
        return out

    def time_osem_with_resolution_model(self, iters=2):
        """the same OSEM iteration with the 4.5 mm FWHM image-based resolution model
         in every subset (2 x 20 Gaussian smoothings per iteration); seconds per iteration"""
        sig = 4.5 / 2.3548200450309493
        self.jp.jp_lm_osem_planned_res(self.plan, self.sens, self.x, n_iter=1, res_sigma_mm=sig)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.stream)
        self.jp.jp_lm_osem_planned_res(self.plan, self.sens, self.x, n_iter=iters, res_sigma_mm=sig)
        e1.record(self.stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / iters

    def checksum(self):
        if self.c >= 4:
            return float(self.x.double().sum())
        p = self.p.reshape(-1)
        return float(p[:: max(1, p.numel() // 4096)].double().sum()) + float(self.bimg.double().sum())

    # ---- end to end with HOST buffers: H2D of the step's inputs, the calls, D2H of the results, all timed ------
    def e2e_setup(self):
        """host-side copies of the step's inputs in pinned memory + the hybrid handle (jp_hybrid over this rank's GPU)"""
        jp, c = self.jp, self.c
        pin = lambda t: t.cpu().pin_memory()
        nvox = int(np.prod(self.g.n))
        self.hyb = jp.Hybrid([self.dev.index if self.dev.index is not None else 0]) if c < 4 else None
        if c in (0, 1):
            self.h = dict(xs=pin(self.xs), xe=pin(self.xe), y=pin(self.y), img=pin(self.img),
                          p=torch.empty(self.n, dtype=torch.float32).pin_memory(),
                          b=torch.zeros(self.g.n, dtype=torch.float32).pin_memory())
            self.e2e_api = "jp_hybrid_set_lors + jp_hybrid_fwd + jp_hybrid_back (pinned host tensors; the LOR list is uploaded once per step)"
            self.h2d, self.d2h = 24 * self.n + 4 * self.n + 4 * nvox, 4 * self.n + 4 * nvox
        elif c == 2:
            self.h = dict(xs=pin(self.xs), xe=pin(self.xe), y=pin(self.y), img=pin(self.img),
                          p=torch.empty_like(self.p, device="cpu").pin_memory(),
                          b=torch.zeros(G.n, dtype=torch.float32).pin_memory())
            self.e2e_api = "jp_hybrid_set_lors + jp_hybrid_fwd_tof_sino + jp_hybrid_back_tof_sino (pinned host tensors)"
            self.h2d = 24 * self.n + 4 * self.y.numel() + 4 * NVOX
            self.d2h = 4 * self.p.numel() + 4 * NVOX
        elif c == 3:
            self.h = dict(xs=pin(self.xs), xe=pin(self.xe), tb=pin(self.tb), y=pin(self.y), img=pin(self.img),
                          p=torch.empty(self.n, dtype=torch.float32).pin_memory(),
                          b=torch.zeros(G.n, dtype=torch.float32).pin_memory())
            self.e2e_api = ("jp_hybrid_set_lors (events + TOF bins, builds the listmode plan) + jp_hybrid_fwd_tof_lm + "
                            "jp_hybrid_back_tof_lm (pinned host tensors)")
            self.h2d = 26 * self.n + 4 * self.n + 4 * NVOX
            self.d2h = 4 * self.n + 4 * NVOX
        else:
            self.h = dict(xs=pin(self.xs), xe=pin(self.xe), tb=pin(self.tb), sens=pin(self.sens),
                          x=torch.ones(G.n, dtype=torch.float32).pin_memory(),
                          xo=torch.empty(G.n, dtype=torch.float32).pin_memory())
            self.e2e_api = ("pinned host -> device copies of the events and sens, jp_lm_plan_create, "
                            "jp_lm_osem_planned (1 iteration), image device -> pinned host")
            self.h2d = 26 * self.n + 2 * 4 * NVOX
            self.d2h = 4 * NVOX

    def e2e_step(self):
        jp, c, h, g = self.jp, self.c, self.h, self.g
        if c < 4:
            hy = self.hyb
            h["b"].zero_()
            if c in (0, 1):
                hy.set_lors(h["xs"], h["xe"])
                hy.fwd(h["img"], g.origin, g.voxsize, out=h["p"])
                hy.back(h["y"], h["b"], g.origin, g.voxsize)
            elif c == 2:
                hy.set_lors(h["xs"], h["xe"])
                hy.fwd_tof_sino(h["img"], g.origin, g.voxsize, self.tof, out=h["p"])
                hy.back_tof_sino(h["y"], h["b"], g.origin, g.voxsize, self.tof)
            else:
                hy.set_lors(h["xs"], h["xe"], h["tb"], g.n, g.origin, g.voxsize, self.tof)
                hy.fwd_tof_lm(h["img"], out=h["p"])
                hy.back_tof_lm(h["y"], h["b"])
            return
        self.xs.copy_(h["xs"], non_blocking=True)
        self.xe.copy_(h["xe"], non_blocking=True)
        self.tb.copy_(h["tb"], non_blocking=True)
        plan = self.jp.LmPlan(self.xs, self.xe, self.tb, G.n, G.origin, G.voxsize, self.tof, n_subsets=20)
        old, self.plan = self.plan, plan
        self.sens.copy_(h["sens"], non_blocking=True)
        self.x.copy_(h["x"], non_blocking=True)
        self.step()
        torch.cuda.synchronize()
        self.plan = old
        plan.destroy()
        h["xo"].copy_(self.x, non_blocking=True)
        torch.cuda.synchronize()

    def e2e_check(self):
        """the e2e results must be the step's results (a copy that silently failed would leave the buffers untouched)"""
        if self.c >= 4:
            return True
        p, b = self.h["p"].to(self.dev).reshape(-1), self.h["b"].to(self.dev)
        self.step()
        torch.cuda.synchronize()
        ok_p = float((p - self.p.reshape(-1)).abs().max()) <= 2e-5 * float(self.p.abs().max())
        ok_b = float((b - self.bimg).abs().max()) <= 1e-4 * float(self.bimg.abs().max())
        return bool(ok_p and ok_b)


def check_parity(w: Workload):
    """parity of the workload's CUDA results against the oracle run on the whole config on the host cores:
    forward rel-L2 and max-abs / max|oracle| over ALL outputs, back projection max-abs / max|oracle| over ALL voxels
    with the DENSE input, the GPU adjoint gap, and the oracle's wall time per direction (`oracle_full`)"""
    import oracle
    oracle.build()
    jp, c, g = w.jp, w.c, w.g
    tol = {"fwd_rel_l2": 1e-5, "max_abs_rel": 1e-4, "adjoint_gap": 1e-4, "osem_rel_l2": 1e-4, "osem_max_abs_rel": 1e-3}
    out = {"oracle_cores": oracle.num_threads(), "tolerances": tol}
    f64 = lambda t: t.detach().cpu().numpy().astype(np.float64)

    def cmp_fwd(got, ref):
        d = got - ref
        return float(np.linalg.norm(d) / np.linalg.norm(ref)), float(np.abs(d).max() / np.abs(ref).max())

    if c in (0, 1, 2, 3):
        w.step()
        torch.cuda.synchronize()
        xs, xe = w.xs.cpu().numpy(), w.xe.cpu().numpy()
        img64 = f64(w.img)
        t0 = time.perf_counter()
        if c in (0, 1):
            ref = oracle.fwd(xs, xe, img64, g.origin, g.voxsize)
        elif c == 2:
            ref = oracle.fwd_tof_sino(xs, xe, img64, g.origin, g.voxsize, *TOF_ARGS)
        else:
            tb = w.tb.cpu().numpy()
            ref = oracle.fwd_tof_lm(xs, xe, tb, img64, g.origin, g.voxsize, *TOF_ARGS[:3])
        t1 = time.perf_counter()
        rel, mx = cmp_fwd(f64(w.p).reshape(ref.shape), ref)
        del ref
        y64 = f64(w.y)
        t2 = time.perf_counter()
        if c in (0, 1):
            bref = oracle.back(xs, xe, y64, g.n, g.origin, g.voxsize)
        elif c == 2:
            bref = oracle.back_tof_sino(xs, xe, y64, g.n, g.origin, g.voxsize, *TOF_ARGS)
        else:
            bref = oracle.back_tof_lm(xs, xe, tb, y64, g.n, g.origin, g.voxsize, *TOF_ARGS[:3])
        t3 = time.perf_counter()
        bmx = float(np.abs(f64(w.bimg) - bref).max() / np.abs(bref).max())
        a = float((w.p.double().reshape(-1) * w.y.double().reshape(-1)).sum())
        b = float((w.img.double() * w.bimg.double()).sum())
        out.update({"fwd_rel_l2": rel, "fwd_max_abs_rel": mx, "back_max_abs_rel": bmx, "adjoint_gap": abs(a - b) / abs(a),
                    "units_checked": int(w.n), "back_input": "dense",
                    "oracle_full": {"fwd_s": t1 - t0, "back_s": t3 - t2, "units": int(w.n),
                                    "fwd_per_s": w.n / (t1 - t0), "back_per_s": w.n / (t3 - t2)}})
        out["pass"] = bool(rel <= tol["fwd_rel_l2"] and mx <= tol["max_abs_rel"] and bmx <= tol["max_abs_rel"]
                           and out["adjoint_gap"] <= tol["adjoint_gap"])
    elif c == 4:
        n_iter = 3
        x = torch.ones(G.n, dtype=torch.float32, device=w.dev)
        jp.jp_lm_osem_planned(w.plan, w.sens, x, n_iter=n_iter)
        torch.cuda.synchronize()
        xs, xe, tb = w.xs.cpu().numpy(), w.xe.cpu().numpy(), w.tb.cpu().numpy()
        t0 = time.perf_counter()
        ref = oracle.lm_osem(xs, xe, tb, f64(w.sens), np.ones(G.n, dtype=np.float32), G.origin, G.voxsize,
                             *TOF_ARGS[:3], n_subsets=20, n_iter=n_iter)
        t1 = time.perf_counter()
        got = f64(x)
        rel = float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
        mx = float(np.abs(got - ref).max() / np.abs(ref).max())
        out.update({"osem_rel_l2": rel, "osem_max_abs_rel": mx, "events": int(w.n), "n_subsets": 20, "n_iter": n_iter,
                    "image_max": float(ref.max()), "image_sum": float(ref.sum()), "finite": bool(np.isfinite(got).all()),
                    "oracle_full": {"s_per_iteration": (t1 - t0) / n_iter, "events": int(w.n)}})
        out["pass"] = bool(rel <= tol["osem_rel_l2"] and mx <= tol["osem_max_abs_rel"] and out["finite"])
        # the same reconstruction through the other kernel paths of the plan (jp_lm_plan_set_path), against the same oracle image
        out["paths"] = {}
        for path, name in ((2, "quad_both_ways"),):
            w.plan.set_path(path)
            xp = torch.ones(G.n, dtype=torch.float32, device=w.dev)
            jp.jp_lm_osem_planned(w.plan, w.sens, xp, n_iter=n_iter)
            gp = f64(xp)
            out["paths"][name] = {"osem_rel_l2": float(np.linalg.norm(gp - ref) / np.linalg.norm(ref)),
                                  "osem_max_abs_rel": float(np.abs(gp - ref).max() / np.abs(ref).max())}
        w.plan.set_path(0)
    else:
        out["skipped"] = "the 40 GB sinogram OSEM workload is checked per subset in tests/test_gpu_fullsize.py"
    return out


def measure(w: Workload, steps: int, warmup: int, barrier, sampler=None):
    """warm-up, then `steps` timed steps between CUDA events on the launching stream"""
    for _ in range(warmup):
        w.step()
    barrier()
    if sampler:
        sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    e_beg, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e_beg.record(w.stream)
    for k in range(steps):
        w.step(evs[k])
    e_end.record(w.stream)
    barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = e_beg.elapsed_time(e_end)
    f = [e[0].elapsed_time(e[1]) for e in evs]
    b = [e[1].elapsed_time(e[2]) for e in evs]                         # includes the image zero-fill
    if w.flush is not None:   # the L2 flush between steps is not part of a step
        total_ms = float(np.sum(f) + np.sum(b))
    w.step_ms = {"fwd": f, "back": b}
    return total_ms, float(np.mean(f)), float(np.mean(b)), clocks


def spread(ms):
    """median / min / max of the per-step CUDA-event times (median and min of the repetitions)"""
    a = np.asarray(ms, dtype=np.float64)
    return {"median_ms": float(np.median(a)), "min_ms": float(a.min()), "max_ms": float(a.max()), "n": int(a.size)}


def roofline_dict(w: Workload, fwd_ms: float, back_ms: float):
    peaks, peak_src = measured_peaks()
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak = N_SM * FP32_LANES_PER_SM * sm_mhz * 1e6          # FP32 lane-instructions / s
    kf, kb = w.kinds
    planned = getattr(w, "splan", None) is not None
    names = {0: ("k_fwd_tile (per-LOR path: random chords are not tracks)", "k_back_tile (per-LOR path)"),
             1: ("k_fwd_track<104, 9>", "k_back_track<104, 9>") if planned else ("k_fwd_tile<104, list>", "k_back_tile<104, list>"),
             2: ("k_tof_sino_tile<6,fwd>", "k_tof_sino_tile<6,back>") if planned else ("k_tof_sino_win<6,fwd>", "k_tof_sino_win<6,back>"),
             3: ("k_fwd_tof_lm_tile", "k_back_tof_lm_tile"),
             4: ("k_brick_fwd (forward sums on TMA-loaded image bricks) + k_back_tof_lm_quad<ratio> (float atomics)", ""),
             5: ("k_tof_sino_tile<6,osem> (forward + ratio + back per track slice)" if planned else
                 "k_tof_sino_osem<6> (forward + ratio + back per LOR block)", "")}[w.c]
    src = (f"148 SMs x 128 FP32 lanes x {sm_mhz:.0f} MHz (sm_max_mhz of MEASURED_PEAKS.json, {peak_src})")
    if w.c in (4, 5):
        lane = 2 * LANE["lm" if w.c == 4 else "sino"]
        achieved = lane * w.plane_steps / (fwd_ms * 1e-3)
        return {"bound": "alu", "kernel": names[0], "achieved": achieved / 1e12, "peak": alu_peak / 1e12,
                "unit": "T lane-instr/s (FP32)", "frac": achieved / alu_peak,
                "traffic": (ncu_note(w.c, "iter") or {}).get("dram_bytes_per_launch"), "ncu": {"iter": ncu_note(w.c, "iter")},
                "peak_source": src,
                "plane_steps_per_iteration": w.plane_steps, "lane_instr_per_plane_step": lane,
                "hbm_bound_frac": 2 * w.hbm_bytes / (fwd_ms * 1e-3) / (float(peaks["hbm_gbs"]) * 1e9)}
    dom = "back" if back_ms >= fwd_ms else "fwd"
    dom_ms = max(back_ms, fwd_ms)
    lane = LANE[kb] if dom == "back" else LANE[kf]
    achieved = lane * w.plane_steps / (dom_ms * 1e-3)
    per = lambda ms, k: {"ms": ms, "per_s": w.n / ms * 1e3, "frac_alu": LANE[k] * w.plane_steps / (ms * 1e-3) / alu_peak}
    return {"bound": "alu", "kernel": names[1] if dom == "back" else names[0], "achieved": achieved / 1e12,
            "peak": alu_peak / 1e12, "unit": "T lane-instr/s (FP32)", "frac": achieved / alu_peak,
            "traffic": (ncu_note(w.c, dom) or {}).get("dram_bytes_per_launch"),
            "ncu": {"fwd": ncu_note(w.c, "fwd"), "back": ncu_note(w.c, "back")},
            "algorithmic_bytes_per_launch": w.hbm_bytes,
            "peak_source": src, "plane_steps_per_launch": w.plane_steps, "lane_instr_per_plane_step": lane,
            "fwd": per(fwd_ms, kf), "back": per(back_ms, kb),
            # the same work counted in flops against 2 flop x lane peak (a tighter roof for the non-TOF
            # pair: 16 / 14 flop per plane-step forward / back; the headline `frac` counts instruction slots)
            **({"flop_based": {"peak_tflops": 2 * alu_peak / 1e12,
                               "fwd_frac": 16.0 * w.plane_steps / (fwd_ms * 1e-3) / (2 * alu_peak),
                               "back_frac": 14.0 * w.plane_steps / (back_ms * 1e-3) / (2 * alu_peak)}} if w.c == 1 else {}),
            "hbm_bound_frac": w.hbm_bytes / (dom_ms * 1e-3) / (float(peaks["hbm_gbs"]) * 1e9)}


def run_sharded_osem(jp, dev, rank, world, barrier, steps, warmup):
    """configs[4] with the 40 M events SHARDED over the ranks (multi_gpu.shard_events: contiguous shards
    that start at a multiple of n_subsets), a listmode plan per rank, and per OSEM subset ONE all-reduce(sum) of the
    15.36 MB image over NCCL (multi_gpu.lm_osem_sharded); the sensitivity image is a sharded non-TOF back projection of
    ones over the configs[1] views of the rank + one all-reduce.  Strong scaling: the total work is fixed.
    Returns (ms per iteration on this rank, dict)."""
    from paper_2212_12519_b200 import multi_gpu
    tof = jp.make_tof(*TOF_ARGS)
    nev = int(os.environ.get("JP_BENCH_EVENTS", "40000000"))
    n_subsets = 20
    xs, xe, tb = inputs.listmode_events(nev, seed=inputs.BASE_SEED + 3, device=dev, img=inputs.phantom())   # same list on every rank
    lo, hi = multi_gpu.shard_events(nev, rank, world, n_subsets)
    xs, xe, tb = xs[:, lo:hi].contiguous(), xe[:, lo:hi].contiguous(), tb[lo:hi].contiguous()
    plan = jp.LmPlan(xs, xe, tb, G.n, G.origin, G.voxsize, tof, n_subsets=n_subsets)
    views = range(rank * inputs.N_VIEWS // world, (rank + 1) * inputs.N_VIEWS // world)
    sx, se = inputs.sinogram_lors(views=views, device=dev)
    sens = torch.empty(G.n, dtype=torch.float32, device=dev)
    multi_gpu.back_sharded(multi_gpu.CudaOps(jp, lors=(sx, se), geom=G), torch.ones(sx.shape[1], device=dev), sens)
    del sx, se
    ops = multi_gpu.CudaOps(jp, plan=plan)
    x = torch.ones(G.n, dtype=torch.float32, device=dev)
    for _ in range(max(warmup, 1)):
        multi_gpu.lm_osem_sharded(ops, sens, x, n_subsets, 1)
    barrier()
    st = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(steps):
        multi_gpu.lm_osem_sharded(ops, sens, x, n_subsets, 1)
    e1.record(st)
    barrier()
    ms = e0.elapsed_time(e1) / steps
    info = {"events": nev, "events_on_rank0": hi - lo if rank == 0 else None, "n_subsets": n_subsets,
            "collective": "all_reduce(sum) of the %d-voxel float32 image per OSEM subset (%d per iteration) over %s"
                          % (NVOX, n_subsets, "NCCL" if world > 1 else "one rank (no exchange)"),
            "image_sum": float(x.double().sum()), "finite": bool(torch.isfinite(x).all())}
    plan.destroy()
    return ms, info


def measure_fp32_rate(jp, dev):
    """FFMA lane-instructions per second of jp_fma_burn (148 x 8 CTAs of 256 threads, 8 independent chains per thread),
    best of 5 after a warm-up, CUDA events on the current stream"""
    import ctypes
    from paper_2212_12519_b200 import build as jp_build
    mb = ctypes.CDLL(jp_build.MICROBENCH_LIB)            # bench-only library (csrc/bench/jp_microbench.cu), not the product ABI
    mb.jp_fma_burn.restype = ctypes.c_int
    mb.jp_fma_burn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
    scratch = torch.zeros(4, dtype=torch.float32, device=dev)
    blocks, iters = N_SM * 8, 20000
    n = blocks * 256 * 16 * iters
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert mb.jp_fma_burn(scratch.data_ptr(), blocks, iters, st) == 0
    best = 0.0
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        assert mb.jp_fma_burn(scratch.data_ptr(), blocks, iters, st) == 0
        e1.record()
        torch.cuda.synchronize()
        best = max(best, n / (e0.elapsed_time(e1) * 1e-3))
    return best


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

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    c = args.config
    if c == 4 and (world > 1 or args.sharded):
        # the 40 M events of ONE reconstruction sharded over the ranks, one all-reduce of the image per subset
        ms, info = run_sharded_osem(jp, dev, rank, world, barrier, args.steps, args.warmup)
        if world > 1:
            t = torch.tensor([ms], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t[0])
        if rank == 0:
            line = {"metric": SPEC[4]["metric"], "value": info["events"] / (ms * 1e-3), "unit": SPEC[4]["unit"],
                    "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                    "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                    "config": {"workload": SPEC[4]["workload"] + "; events sharded over the ranks (SURVEY.md 8(e))",
                               "parallelism": f"event shards x{world}", "l2": SPEC[4]["l2"]},
                    # per subset: 2 tables, brick forward, adjoint per axis, quad merge, update
                    "gpu_launches": 8 * 20 * args.steps, "s_per_iteration": ms * 1e-3, "sharded": info}
            print(json.dumps(line), flush=True)
        if world > 1:
            dist.destroy_process_group()
        return
    w = Workload(c, jp, dev, rank)
    if c == 4:
        w.setup_sens()
    total_ms, fwd_ms, back_ms, clocks = measure(w, args.steps, args.warmup, barrier,
                                                ClockSampler(local) if rank == 0 else None)
    checksum = w.checksum()

    e2e_s = None
    if not args.no_e2e and c != 5:   # configs 5 keeps 40 GB of sinograms resident by design: no host leg
        w.e2e_setup()
        w.e2e_step()
        barrier()
        t0 = time.perf_counter()
        ne2e = max(1, min(args.steps, 10))
        for _ in range(ne2e):
            w.e2e_step()
        barrier()
        e2e_s = (time.perf_counter() - t0) / ne2e
        e2e_ok = w.e2e_check()
        w.h = None
        if getattr(w, "hyb", None) is not None:
            w.hyb.destroy()

    sharded = None
    if world > 1 and c == 1 and not args.no_other:
        # the path's one exchange step on this node: configs[4] with the events sharded over the ranks (NCCL all-reduce)
        w_keep = w
        ms_sh, sharded = run_sharded_osem(jp, dev, rank, world, barrier, 3, 1)
        w = w_keep
    if world > 1:
        t = torch.tensor([total_ms, fwd_ms, back_ms, e2e_s or 0.0, ms_sh if sharded else 0.0], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, fwd_ms, back_ms = float(t[0]), float(t[1]), float(t[2])
        if e2e_s is not None:
            e2e_s = float(t[3])
        if sharded:
            sharded["ms_per_iteration"] = float(t[4])
            sharded["events_per_s"] = sharded["events"] / (float(t[4]) * 1e-3)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_per_step = total_ms / args.steps
    line = {
        "metric": SPEC[c]["metric"], "value": world * w.n / (ms_per_step * 1e-3), "unit": SPEC[c]["unit"],
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": SPEC[c]["workload"], "units_per_gpu": w.n, "l2": SPEC[c]["l2"],
                   "parallelism": f"frames{world}" if world > 1 else "single"},
        "gpu_launches": w.launches * args.steps,
        "clocks": clocks,
        "roofline": roofline_dict(w, fwd_ms, back_ms),
        "timing": ({"fwd": spread(w.step_ms["fwd"]), "back": spread(w.step_ms["back"])} if c < 4 else
                   {"iteration": spread(w.step_ms["fwd"])}),
        "checksum": checksum,
    }
    if c in (2, 5):
        line["roofline"]["note"] = ("SURVEY.md 8(d) charges 112 FP32 lane-instructions per plane-step (the per-LOR minimal formulation: "
                                    "~7 erf evaluations per step).  The track-tile kernels evaluate the TOF weights once per "
                                    "(group of LORs of equal length, plane) and execute far fewer instructions per step, so `frac` can "
                                    "exceed 1: it is kept for continuity; the kernels' real limiter is the shared-memory pipe -- see "
                                    "roofline.ncu (issue slots, l1tex) and hbm_bound_frac")
    if c in (3, 4):
        line["roofline"]["note"] = ("SURVEY.md 8(d) charges 40 FP32 lane-instructions per plane-step (two 10-instruction erf "
                                    "evaluations); the kernels use table look-ups (fewer instructions), so `frac` overstates the FP32 "
                                    "pipe use: see roofline.ncu (issue slots, l1tex)")
    if c == 0:
        line["roofline"]["note"] = ("launch-bound: 4.06e5 plane-steps are microseconds of work per call; the fraction "
                                    "is reported as SURVEY.md 8(d) asks, it says nothing about the kernels")
    if w.plan_s is not None:
        line["config"]["plan_s"] = w.plan_s
    # A/B switches read from the environment change what is timed: the line says so (the driver sets neither)
    overrides = {k: os.environ[k] for k in ("JP_BENCH_EVENTS", "JP_BENCH_UNPLANNED") if k in os.environ}
    if overrides:
        line["config"]["env_overrides"] = overrides
        line["config"]["workload"] += " [NOT the stated config: environment overrides " + json.dumps(overrides) + "]"
    if sharded:
        line["sharded_osem"] = sharded
    if world == 1:
        rate = measure_fp32_rate(jp, dev)
        line["roofline"]["fp32_ffma_measured"] = {"value": rate / 1e12, "unit": "T lane-instr/s (FP32 FFMA, libjp_microbench.so)",
                                                  "frac_of_nominal_peak": rate / (line["roofline"]["peak"] * 1e12)}
    if c == 1 and world == 1 and not args.no_other:
        line["nonaligned_tracks_36_rings"] = w.time_nonaligned_tracks()
    if c == 3:
        line["nontof_listmode"] = w.time_nontof_listmode()
        line["plan_order_io"] = w.time_plan_order_io()
    if c >= 4:
        line["s_per_iteration"] = ms_per_step * 1e-3
    if c == 4:
        line["s_per_iteration_with_resolution_model"] = w.time_osem_with_resolution_model()
        line["osem_paths"] = w.time_osem_paths()
    if e2e_s is not None:
        line["e2e"] = {"value": world * w.n / e2e_s, "unit": SPEC[c]["unit"], "h2d_bytes_per_step": w.h2d,
                       "d2h_bytes_per_step": w.d2h, "ms_per_step": e2e_s * 1e3, "api": w.e2e_api,
                       "results_match_device_step": e2e_ok}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_dict(c, time_oracle(c, 1, 0))
    if args.check and world == 1:
        line["parity"] = check_parity(w)
    # ---- the other configs, briefly (single GPU, default workload only) -----------------------------------
    if world == 1 and c == 1 and not args.no_other:
        del w
        torch.cuda.empty_cache()
        other = {}
        for oc in (2, 3, 4, 5):
            ow = Workload(oc, jp, dev, rank)
            if oc == 4:
                ow.setup_sens()
            nb = 6
            t_ms, f_ms, b_ms, _ = measure(ow, nb, 3, barrier)
            r = roofline_dict(ow, f_ms, b_ms)
            d = {"units": ow.n, "ms_per_step": t_ms / nb, "per_s": ow.n / (t_ms / nb * 1e-3), "unit": SPEC[oc]["unit"],
                 "plane_steps": ow.plane_steps, "frac_alu": r["frac"]}
            if oc == 5:
                d["s_per_iteration"] = t_ms / nb * 1e-3
            elif oc == 4:
                d["s_per_iteration"] = t_ms / nb * 1e-3
                d["s_per_iteration_with_resolution_model"] = ow.time_osem_with_resolution_model()
                d["osem_paths"] = ow.time_osem_paths()
            else:
                d["fwd"], d["back"] = r["fwd"], r["back"]
            if oc == 3:
                d["nontof_listmode"] = ow.time_nontof_listmode()
                d["plan_order_io"] = ow.time_plan_order_io()
            if ow.plan_s is not None:
                d["plan_s"] = ow.plan_s
            other[f"configs[{oc}]" if oc < 5 else "sino_osem_8f3"] = d
            del ow
            torch.cuda.empty_cache()
        line["other_configs"] = other
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4, 5])
    ap.add_argument("--check", action="store_true",
                    help="run the float64 oracle on the FULL config (outside the timed region) and add `parity` to the line")
    ap.add_argument("--sharded", action="store_true",
                    help="--config 4: run the sharded OSEM driver (multi_gpu.lm_osem_sharded) even on one GPU")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the brief configs[2..4] runs of the default line")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
