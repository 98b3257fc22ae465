#!/usr/bin/env python
"""bench.py -- MSUPS and fraction of the HBM roofline of the fused D3Q15 site update.

Contract (one JSON line on stdout, printed by rank 0):
  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload bigtree|tree|aneurysm|cube|pipe]
                  [--scheme aa|two_lattice] [--store f64|f32] [--order morton|raster|tiled]
                  [--lattice d3q15|d3q19] [--inner S] [--impl ours|reference]

* metric/unit: BASELINE.json's metric -- fluid site updates per second, in MSUPS
  (= fluid sites x LB time steps / seconds / 1e6; the paper's SUPS definition, PAPER.md
  Tables II/III, lines 115-133).
* A bench "step" is one hlb_step(S) call: S (= --inner) consecutive LB time steps, each ONE
  launch of the fused collide-and-stream kernel over every fluid site of the workload (all
  rows S1..S8 of SURVEY.md section 8(a)). The default workload is BASELINE configs[4]
  ("the largest geometry", the one north_star's roofline target is stated on).
* value: device-timed (CUDA events on the launching stream, populations resident in HBM).
* e2e: the same metric through the C-ABI with HOST buffers: every step uploads the initial
  rho/u from pinned host memory (hlb_set_state), runs hlb_step(S), and reads rho/u back to
  pinned host memory (hlb_get_macroscopic); the copies are inside the timed region.
* roofline: algorithmic bytes per launch / average launch duration of the dominant kernel,
  against MEASURED_PEAKS.json's hbm_gbs (fallback 6650 GB/s, B200_PROFILING.md).
* cpu_baseline: the oracle (oracle/, as it stands, 1 thread) timed on a bounded crop of the
  same geometry on this box's host cores. `--impl reference` times only that.
* Multi-GPU (--gpus N under torchrun): REPLICAS ONLY: every rank
  runs the same workload on its own GPU, no data-path collective; value = total site updates
  of all ranks / max-over-ranks time; "scaling": "weak".
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

METRIC = "fluid site updates/sec (MSUPS), D3Q15 LBGK sparse site update"
METRIC_Q19 = "fluid site updates/sec (MSUPS), D3Q19 LBGK sparse site update"
UNIT = "MSUPS"
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md "FALLBACK"
DEFAULT_SCHEME = {"pipe": "two_lattice", "cube": "two_lattice", "aneurysm": "two_lattice",
                  "paper_sized": "two_lattice", "paper_sized_23": "two_lattice",
                  "tree": "two_lattice", "bigtree": "aa", "cube672": "aa", "bigtree_x": "aa"}
WORKLOAD_DESC = {
    "pipe": "BASELINE configs[0]: pipe R=8 L=64",
    "cube": "BASELINE configs[1]: periodic 128^3 Taylor-Green",
    "aneurysm": "BASELINE configs[2]: sine vessel + sac, 480x160x160",
    "tree": "BASELINE configs[3]: 5-level tree, 1024^3 box, r0=32",
    "bigtree": "BASELINE configs[4]: 5-level tree, 2048x2048x1024 box, r0=64",
    "paper_sized": "context only: aneurysm recipe scaled to ~297k sites (the paper's Subject 16, Table II)",
    "paper_sized_23": "context only: aneurysm recipe scaled to ~133k sites (the paper's Subject 23, Table II)",
    "cube672": "context only: periodic 672^3 cube, 303.5 M sites (64-bit flat offsets: Q N > 2^32)",
    "bigtree_x": "context only: configs[4] generator at 77 um voxels (box and r0 x 1.3), 85.5 M sites "
                 "(BASELINE's nominal 80-100 M)",
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="bigtree", choices=list(WORKLOAD_DESC))
    ap.add_argument("--scheme", default=None, choices=["aa", "two_lattice", "auto"])
    ap.add_argument("--store", default="f64", choices=["f64", "f32"])
    ap.add_argument("--order", default="auto", choices=["auto", "morton", "raster", "tiled"])
    ap.add_argument("--links", default="auto", choices=["auto", "table", "records"])
    ap.add_argument("--lattice", default="d3q15", choices=["d3q15", "d3q19"],
                    help="d3q15 = BASELINE.json's metric; d3q19 = the lattice the paper ran (NEXT-1)")
    ap.add_argument("--inlet", default="pressure", choices=["pressure", "velocity", "waveform", "host_waveform"],
                    help="velocity: iolet 0 becomes a Ladd velocity inlet (the paper's LADDIOLET); "
                         "waveform: the same, driven by a device-resident pulsatile waveform "
                         "(hlb_set_iolet_waveform, period 1000 steps); host_waveform: the same "
                         "waveform handed over by hlb_set_iolet_velocity before every LB step")
    ap.add_argument("--walls", default="bounce_back",
                    choices=["bounce_back", "bfl_random", "bfl_none", "bfl_one_direction"],
                    help="bfl_random: interpolated (BFL) walls with seeded random distances on every "
                         "wall link -- the kernel work of the paper's BFL option; bfl_none: the kernels with "
                         "interpolated walls but no link flagged; bfl_one_direction: d = 0.3 on the links of one "
                         "lattice direction (the cost split of profiles/r02_tuning.md sections 12 and 15)")
    ap.add_argument("--render", type=int, default=0, metavar="PIXELS",
                    help="also time the ray-marching renderer (NEXT-4) on the final state: PIXELS x "
                         "PIXELS frames of the speed field, rotating view; adds a \"render\" object")
    ap.add_argument("--render-view", default="rotate", choices=["rotate", "axis", "oblique1", "oblique2", "oblique3"],
                    help="rotate: the view turns about the y axis over the frames; else one fixed view "
                         "(the ones profiles/render_inst.csv has instruction counts for)")
    ap.add_argument("--no-prefetch", action="store_true", help="HLB_NO_PREFETCH (ablation)")
    ap.add_argument("--no-pdl", action="store_true", help="HLB_NO_PDL (ablation)")
    ap.add_argument("--index64", action="store_true",
                    help="HLB_INDEX64: run the 64-bit-offset kernels at any size (tuning)")
    ap.add_argument("--readouts", action="store_true",
                    help="also time the read-out kernels (hlb_get_macroscopic_device, hlb_get_stress_device) "
                         "after an even and after an odd step count: 'readouts' in the JSON line")
    ap.add_argument("--no-resident", action="store_true",
                    help="HLB_NO_RESIDENT (ablation: small geometries step by graph replay instead "
                         "of the resident multi-step kernel)")
    ap.add_argument("--inner", type=int, default=50, help="LB time steps per bench step (even)")
    ap.add_argument("--sweep", default="auto", choices=["auto", "on", "off"],
                    help="after the headline, time the other configs / variants shortly and attach "
                         "them as \"configs\" (auto: with the default workload and flags at 1 GPU)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--small", action="store_true", help="scaled-down geometry (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0,
                    help="CPU work budget of the cpu_baseline leg")
    ap.add_argument("--ref-seconds", type=float, default=120.0,
                    help="total budget of an --impl reference run")
    return ap.parse_args()


# --------------------------------------------------------------------------- helpers
def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            v = float(json.load(fh)["hbm_gbs"])
        return v, "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock and throttle reasons with nvidia-smi while the timed region runs."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.15] or [l for _, l in self.lines]
        for l in rows:
            p = [x.strip() for x in l.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0]))
                smax = float(p[1])
                power.append(float(p[2]))
            except ValueError:
                continue
            for n, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm),
                "power_w_max": max(power) if power else None}


def crop_sample(wl, max_sites=1_200_000):
    """A bounded sample of the workload for the CPU legs: the sub-box of the voxel array,
    starting at the low-x end of the fluid's bounding box (the inlet side), that holds about
    max_sites fluid sites. Outside the crop counts as solid, like outside the full box."""
    st = wl.site_type
    if wl.n_sites <= max_sites:
        return st, wl.periodic, "whole geometry"
    per_x = np.count_nonzero(st == 1, axis=(0, 1)).astype(np.int64)     # fluid per x-slab
    cum = np.cumsum(per_x)
    x1 = int(np.searchsorted(cum, max_sites)) + 1
    x0 = int(np.argmax(per_x > 0))
    x0 = max(0, x0 - 2)                                               # keep the inlet ghost slab
    sub = st[:, :, x0:x1]
    zs = np.flatnonzero(np.any(sub != 0, axis=(1, 2)))
    ys = np.flatnonzero(np.any(sub != 0, axis=(0, 2)))
    sub = np.ascontiguousarray(sub[zs[0]:zs[-1] + 1, ys[0]:ys[-1] + 1, :])
    return sub, 0, f"crop x in [{x0},{x1}) of the same voxel array (outside = solid)"


def time_oracle(wl, budget_s, threads=1, lattice="d3q15"):
    """Oracle MSUPS on the bounded sample: 1 calibration step, then as many steps as fit
    the budget. Returns (msups, n_sites, steps, seconds, sample description)."""
    import oracle
    st, periodic, what = crop_sample(wl)
    o = oracle.Oracle(st, periodic, wl.tau, wl.iolet_rho, threads=threads, lattice=lattice)
    n = o.n_sites
    t0 = time.perf_counter()
    o.step(1)
    t1 = time.perf_counter() - t0
    steps = int(max(2, min(200, budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    return n * steps / dt / 1e6, n, steps, dt, what, o.threads


def max_over_ranks(values, world, device):
    """Element-wise maximum of a list of floats over all ranks (replicas: no data-path
    collective, only this reduction of the timings)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def replicas_value(n_sites, lb_steps, world, seconds):
    """Whole-job MSUPS of `world` replicas that each did n_sites x lb_steps site updates in
    at most `seconds` (the max over ranks)."""
    return world * n_sites * lb_steps / seconds / 1e6


RENDER_VIEWS = {   # rotations (degrees about x, then about y) of the fixed views of --render-view
    "rotate": None, "axis": (0.0, 0.0), "oblique1": (20.0, 30.0), "oblique2": (-35.0, 60.0), "oblique3": (50.0, -20.0)}
SM_ISSUE_PEAK = 148 * 4 * 1.965e9   # warp instructions / s: 148 SMs x 4 schedulers x 1965 MHz


def render_inst_count(workload, pixels, view, texture):
    """Warp instructions of one k_raymarch launch from the committed ncu capture of exactly this
    frame (profiles/render_inst.csv: workload,pixels,view,texture,smsp__inst_executed.sum,source)."""
    path = os.path.join(ROOT, "profiles", "render_inst.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        parts = [p.strip() for p in line.split(",")]
        if parts[:4] == [workload, str(pixels), view, "texture" if texture else "linear"]:
            return float(parts[4])
    return None


def time_renderer(hlb, g, wl, workload, pixels, view_name="rotate", frames=12, cpu_pixels=96):
    """Frames per second of hlb_render_device on the geometry's current state (speed field,
    orthographic view, sample step 0.5 voxel, image kept on the device), the ray marcher alone
    (CUDA events around it are not possible from here, so: frame time minus the time of the same
    calls with a 16 x 16 image), the oracle renderer timed on a cpu_pixels^2 frame of the same
    view as the CPU baseline, and -- for the fixed views with a committed instruction count --
    the issue-slot roofline of k_raymarch."""
    import math
    import torch
    nx, ny, nz = wl.shape
    lut = np.stack([np.linspace(0, 1, 256)] * 3 + [np.full(256, 0.02)], axis=1).astype(np.float32)
    lut[0, 3] = 0.0          # value 0 (solid voxels, fluid at rest) is transparent: empty cells are skipped
    rho, u = g.hlb_get_macroscopic()
    speed = np.linalg.norm(u, axis=1)
    umax = float(np.max(speed)) or 1.0

    def rot_of(k):
        if RENDER_VIEWS[view_name] is None:
            ax, ay = 0.0, 360.0 * k / frames
        else:
            ax, ay = RENDER_VIEWS[view_name]
        ax, ay = math.radians(ax), math.radians(ay)
        rx = np.array([[1, 0, 0], [0, math.cos(ax), -math.sin(ax)], [0, math.sin(ax), math.cos(ax)]])
        ry = np.array([[math.cos(ay), 0, math.sin(ay)], [0, 1, 0], [-math.sin(ay), 0, math.cos(ay)]])
        return ry @ rx

    def view(k, px):
        return hlb.make_view(px, px, rot=rot_of(k), zoom=px / float(max(nx, ny, nz)), step=0.5,
                             tf_scale=1.0 / umax, tf_offset=0.0, opacity=1.0, field=0)

    def timed(px):
        g.hlb_render_device(view(0, px), lut)                       # builds the volume
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(torch.cuda.current_stream())
        for k in range(frames):
            img = g.hlb_render_device(view(k, px), lut)
        ev1.record(torch.cuda.current_stream())
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / frames, img

    ms_small, _ = timed(16)          # read-out + scatter + a negligible march
    ms, img = timed(pixels)
    ms_march = max(ms - ms_small, 1e-6)
    texture = not os.environ.get("HLB_RENDER_LINEAR", "0").strip("0")
    out = {"pixels": [pixels, pixels], "frames": frames, "view": view_name, "ms_per_frame": ms, "fps": 1e3 / ms,
           "ms_ray_march": ms_march, "ms_readout_and_scatter": ms_small,
           "rays_per_s": pixels * pixels / (ms_march * 1e-3),
           "volume_voxels": nx * ny * nz, "sample_step": 0.5, "volume_through": "texture" if texture else "linear",
           "includes": "macroscopic read-out + scatter into the voxel volume + ray march, per frame",
           "empty_space_skipping": not os.environ.get("HLB_RENDER_NO_SKIP", "0").strip("0"),
           "max_alpha": float(img[..., 3].max())}
    inst = render_inst_count(workload, pixels, view_name, texture)
    out["roofline"] = {"bound": "alu", "kernel": "k_raymarch", "unit": "Gwarp-inst/s",
                       "peak": SM_ISSUE_PEAK / 1e9, "peak_source": "148 SMs x 4 schedulers x 1965 MHz (issue slots)",
                       "warp_inst_per_frame": inst,
                       "achieved": (inst / (ms_march * 1e-3) / 1e9) if inst else None,
                       "frac": (inst / (ms_march * 1e-3) / SM_ISSUE_PEAK) if inst else None}
    # CPU baseline: the oracle renderer (oracle/render_oracle.cpp, 1 core) on the same volume and
    # view at cpu_pixels^2 rays -- a bounded sample of the frame, centred on the same axis
    import oracle
    vol = np.zeros(nx * ny * nz, dtype=np.float32)
    vol[wl.fluid_voxels()] = speed.astype(np.float32)
    vol = vol.reshape(nz, ny, nx)
    v = view(0, cpu_pixels)
    t0 = time.perf_counter()
    _, n_samples = oracle.render(vol, cpu_pixels, cpu_pixels, rot_of(0), v.zoom, v.step, v.tf_scale,
                                 v.tf_offset, v.opacity, lut)
    dt = time.perf_counter() - t0
    del vol
    out["cpu_baseline"] = {"kind": "oracle", "cores": 1, "value": cpu_pixels * cpu_pixels / dt, "unit": "rays/s",
                           "samples_inside_the_box_per_s": n_samples / dt,
                           "sample": f"{cpu_pixels} x {cpu_pixels} rays of the same view (zoom scaled to the frame) "
                                     f"in {dt:.1f} s; the oracle visits every sample, the GPU skips empty cells"}
    return out


def host_cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


# --------------------------------------------------------------------------- reference arm
def run_reference(args, rank, world):
    if rank != 0:
        return 0
    import workloads as W
    import oracle
    wl = W.by_name(args.workload, small=args.small)
    scheme = args.scheme or DEFAULT_SCHEME[args.workload]
    st, periodic, what = crop_sample(wl)
    o = oracle.Oracle(st, periodic, wl.tau, wl.iolet_rho, threads=1, lattice=args.lattice)
    n = o.n_sites
    t0 = time.perf_counter()
    o.step(1)
    t1 = time.perf_counter() - t0
    total = args.steps + args.warmup
    lb_per_step = int(max(1, min(args.inner, args.ref_seconds / total / max(t1, 1e-6))))
    for _ in range(args.warmup):
        o.step(lb_per_step)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(lb_per_step)
    dt = time.perf_counter() - t0
    o.close()
    value = n * lb_per_step * args.steps / dt / 1e6
    sample = f"{what}: {n} sites x {lb_per_step} LB steps per bench step"
    out = {
        "impl": "reference", "metric": METRIC if args.lattice == "d3q15" else METRIC_Q19, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": WORKLOAD_DESC[args.workload] + (" (small)" if args.small else ""),
                   "scheme": scheme, "store": args.store, "lattice": args.lattice,
                   "n_sites_full": wl.n_sites,
                   "n_sites_sample": n, "lb_steps_per_step": lb_per_step, "tau": wl.tau,
                   "host_cpu": host_cpu_model(), "host_cores": os.cpu_count()},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)
    return 0


def time_readouts(g, N, nq, store):
    """Device time of the read-out kernels on the state as it stands and one LB
    step later (A-A: own slots after an even step count, gathered after an odd one; two-lattice:
    always gathered): CUDA events around the C-ABI call with device outputs, best of 5, and the
    rate in the bytes the read-out has to move at least (populations + outputs)."""
    import torch
    pop = nq * (4 if store == "f32" else 8)
    res = []
    for _ in range(2):
        for name, fn, out_bytes in (("hlb_get_macroscopic_device", g.hlb_get_macroscopic_device, 32),
                                    ("hlb_get_stress_device", g.hlb_get_stress_device, 48)):
            fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            best = 1e30
            for _ in range(5):
                e0.record()
                fn()
                e1.record()
                torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1))
            res.append({"call": name, "steps_done": g.hlb_steps_done(), "ms": best,
                        "min_bytes_per_site": pop + out_bytes, "gbs": N * (pop + out_bytes) / best / 1e6})
        g.hlb_step(1)
    g.hlb_step(1)      # back to an even step count
    return res


# --------------------------------------------------------------------------- our arm
def variant_flags(hlb, v):
    return {"aa": hlb.HLB_AA, "two_lattice": hlb.HLB_TWO_LATTICE, "auto": hlb.HLB_SCHEME_AUTO}[v["scheme"]] | \
        (hlb.HLB_STORE_F32 if v["store"] == "f32" else hlb.HLB_STORE_F64) | \
        {"auto": hlb.HLB_ORDER_AUTO, "morton": hlb.HLB_ORDER_MORTON, "raster": hlb.HLB_ORDER_RASTER,
         "tiled": hlb.HLB_ORDER_TILED}[v["order"]] | \
        {"auto": hlb.HLB_LINKS_AUTO, "table": hlb.HLB_LINKS_TABLE,
         "records": hlb.HLB_LINKS_RECORDS}[v["links"]] | \
        (0 if v["prefetch"] else hlb.HLB_NO_PREFETCH) | (0 if v["pdl"] else hlb.HLB_NO_PDL) | \
        (0 if v["resident"] else hlb.HLB_NO_RESIDENT) | (hlb.HLB_INDEX64 if v.get("index64") else 0) | \
        (hlb.HLB_LATTICE_D3Q19 if v["lattice"] == "d3q19" else hlb.HLB_LATTICE_D3Q15)


def default_variant(**kw):
    v = {"scheme": "two_lattice", "store": "f64", "lattice": "d3q15", "order": "auto", "links": "auto",
         "prefetch": True, "pdl": True, "resident": True, "inlet": "pressure", "walls": "bounce_back"}
    v.update(kw)
    return v


class Run:
    """One geometry on the device in one variant, with the timing helpers of a bench line."""

    def __init__(self, hlb, W, wl, name, v, world=1, local_rank=0, copy_stream=False):
        import torch
        self.torch, self.hlb, self.W, self.name, self.v = torch, hlb, W, name, v
        self.world, self.local_rank = world, local_rank
        t0 = time.perf_counter()
        self.g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, variant_flags(hlb, v),
                                         copy_stream=torch.cuda.Stream() if copy_stream else None)
        torch.cuda.synchronize()
        self.t_create = time.perf_counter() - t0
        g = self.g
        self.N, self.nq = g.n_sites, g.hlb_num_q()
        if v["scheme"] == "auto":          # report what HLB_SCHEME_AUTO took
            self.v = v = dict(v, scheme="aa" if g.hlb_uses_aa() else "two_lattice", scheme_auto=True)
        if wl.rho0 is not None or wl.u0 is not None:
            g.hlb_set_state(wl.rho0, wl.u0)
        self.wave = None
        if v["inlet"] != "pressure" and wl.n_iolets > 0:
            wl = W.with_velocity_inlet(wl)
            g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
            if v["inlet"] in ("waveform", "host_waveform"):
                self.wave = W.pulsatile_waveform(wl, 1000)
                if v["inlet"] == "waveform":
                    g.hlb_set_iolet_waveform(self.wave)
        if v["walls"] == "bfl_random":
            d27 = np.random.default_rng(1906).uniform(0.05, 1.0, size=(self.N, 27))
            g.hlb_set_wall_distance(d27)
            del d27
        elif v["walls"] in ("bfl_none", "bfl_one_direction"):
            d27 = np.full((self.N, 27), -1.0)
            if v["walls"] == "bfl_one_direction":
                d27[:, 14] = 0.3                 # lattice vector (+1, 0, 0)
            g.hlb_set_wall_distance(d27)
            del d27
        self.wl = wl
        self.stream = torch.cuda.current_stream()

    def advance(self, n):
        g = self.g
        if self.v["inlet"] == "host_waveform" and self.wave is not None:
            for _ in range(n):       # the time-varying inlet without the device-resident table
                g.hlb_set_iolet_velocity(self.wl.iolet_kind, self.wave[g.hlb_steps_done() % len(self.wave)])
                g.hlb_step(1)
        else:
            g.hlb_step(n)

    def barrier(self):
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        self.torch.cuda.synchronize()

    def timed(self, S, K, warmup):
        """K x hlb_step(S) between CUDA events on the launching stream, clocks sampled during it.
        Returns (milliseconds of the K steps, launches inside them, clocks)."""
        torch = self.torch
        for _ in range(warmup):
            self.advance(S)
        self.barrier()
        sampler = ClockSampler(self.local_rank)
        sampler.start()
        time.sleep(0.25)
        l0 = self.g.hlb_launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.barrier()
        w0 = time.time()
        ev0.record(self.stream)
        for _ in range(K):
            self.advance(S)
        ev1.record(self.stream)
        self.barrier()
        w1 = time.time()
        clocks = sampler.stop(w0, w1)
        return ev0.elapsed_time(ev1), self.g.hlb_launch_count() - l0, clocks

    def kernel_times(self, reps, S, timed_ms, K, launches):
        """Average duration of every step kernel (events around single launches on the same
        stream) with its bytes per site in both models; the resident multi-step kernel is one
        launch per hlb_step(S), so its duration is the timed region's own."""
        torch, g, v, nq = self.torch, self.g, self.v, self.nq
        scheme, store = v["scheme"], v["store"]
        rec, sf = bool(g.hlb_uses_records()), g.hlb_record_sentinel_fraction()
        bfl = self.g.hlb_num_bfl_sites() / float(self.N)
        moved = lambda phase: self.hlb.moved_bytes_per_site(scheme, store, nq, rec, sf, phase, bfl)  # noqa: E731
        pop_bytes = nq * 2 * (4 if store == "f32" else 8)
        if launches < S * K:
            name = "k_aa_resident" if scheme == "aa" else "k_pull_resident"
            return {name: {"ms": timed_ms / K, "steps_per_launch": S,
                           "bytes_per_site": S * self.hlb.algorithmic_bytes_per_site(scheme, store, nq),
                           "moved_bytes_per_site": S * moved("step")}}
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(2 * reps)]
        torch.cuda.synchronize()
        parity0 = g.hlb_steps_done() & 1
        for a, b in evs:
            a.record(self.stream)
            g.hlb_step(1)
            b.record(self.stream)
        torch.cuda.synchronize()
        per = np.array([a.elapsed_time(b) for a, b in evs])
        if scheme == "aa":
            phase = (parity0 + np.arange(per.size)) & 1          # 0: even-phase kernel, 1: odd-phase
            return {"k_aa<even>": {"ms": float(np.mean(per[phase == 0])), "bytes_per_site": pop_bytes,
                                   "moved_bytes_per_site": moved("even")},
                    "k_aa<odd>": {"ms": float(np.mean(per[phase == 1])), "bytes_per_site": pop_bytes + 4 * (nq - 1),
                                  "moved_bytes_per_site": moved("odd")}}
        return {"k_pull": {"ms": float(np.mean(per)), "bytes_per_site": pop_bytes + 4 * (nq - 1),
                           "moved_bytes_per_site": moved("step")}}

    def close(self):
        self.g.close()


def traffic_key(name, v, nq):
    return [name + ("_d3q19" if nq == 19 else ""), v["scheme"], v["store"], v["order"], v["links"],
            "prefetch" if v["prefetch"] else "no_prefetch", v["inlet"], v["walls"]]


def committed_traffic(name, v, nq, kernel):
    """dram bytes per launch from the committed ncu --set full capture of EXACTLY this
    configuration (profiles/traffic.csv: workload,scheme,store,order,links,prefetch,inlet,walls,
    kernel,n_sites,dram_bytes_per_launch,source), else None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    if v.get("index64"):
        return None         # other kernels (64-bit offsets) than the captured ones
    key = traffic_key(name, v, nq) + [kernel]
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        parts = [p.strip() for p in line.split(",")]
        if parts[:9] == key:
            try:
                return float(parts[10])
            except (ValueError, IndexError):
                return None
    return None


def roofline_of(run, kernels, name):
    """The roofline object of the dominant kernel. `achieved` is ALGORITHMIC bytes (SURVEY.md
    section 8(d): Q populations read + written + the int32 table) over the measured launch
    duration -- with link records the kernels read less than that model charges, so it can
    exceed the copy peak; `frac_moved_model` uses the bytes the variant really has to move and
    `frac_traffic` the DRAM bytes ncu counted for exactly this configuration (None if that was
    not captured)."""
    peak, peak_src = measured_peak()
    dom = max(kernels, key=lambda k: kernels[k]["ms"])
    k = kernels[dom]
    sec = k["ms"] * 1e-3
    N = run.N
    achieved = k["bytes_per_site"] * N / sec / 1e9
    moved = k["moved_bytes_per_site"] * N / sec / 1e9
    traffic = committed_traffic(name, run.v, run.nq, dom)
    return {"bound": "hbm", "kernel": dom, "achieved": achieved, "achieved_is": "algorithmic bytes (SURVEY 8(d) model)",
            "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
            "moved_model_gbs": moved, "frac_moved_model": moved / peak,
            "traffic": traffic, "traffic_gbs": (traffic / sec / 1e9) if traffic else None,
            "frac_traffic": (traffic / sec / 1e9 / peak) if traffic else None,
            "overfetch": (traffic / (k["bytes_per_site"] * N)) if traffic else None,
            "bytes_per_site": k["bytes_per_site"], "moved_bytes_per_site": k["moved_bytes_per_site"],
            "sites_per_launch": N, "ms_per_launch": k["ms"],
            "kernels": {n: dict(kk, gbs=kk["bytes_per_site"] * N / (kk["ms"] * 1e-3) / 1e9,
                                moved_gbs=kk["moved_bytes_per_site"] * N / (kk["ms"] * 1e-3) / 1e9)
                        for n, kk in kernels.items()}}


# The other configurations the driver's single run should observe (north_star: "reported at 1
# GPU on the synthetic geometries below"; SURVEY.md section 8(d) "per config and variant"):
# (workload, variant overrides, LB steps per hlb_step call, calls) sized for ~0.5 s each.
SWEEP = [
    ("pipe", {}, 2000, 100),
    ("cube", {}, 200, 30),
    ("aneurysm", {}, 400, 35),
    ("paper_sized", {"lattice": "d3q19", "scheme": "auto"}, 500, 50),
    ("paper_sized_23", {"lattice": "d3q19", "scheme": "auto"}, 1000, 60),
    ("tree", {}, 100, 24),
    ("tree", {"store": "f32"}, 100, 32),
    ("tree", {"store": "f32", "scheme": "auto"}, 100, 36),
    ("bigtree", {"scheme": "two_lattice"}, 50, 7),
    ("bigtree", {"scheme": "aa", "store": "f32"}, 50, 10),
    ("bigtree", {"scheme": "two_lattice", "store": "f32"}, 50, 9),
    ("bigtree", {"scheme": "aa", "lattice": "d3q19"}, 50, 6),
]


def run_sweep(hlb, W, have):
    """Short timed runs of SWEEP; `have` maps workload name -> Workload already generated."""
    out = []
    cache = dict(have)
    for name, over, S, K in SWEEP:
        if name not in cache:
            for k in list(cache):          # one big voxel array at a time
                if k != name:
                    del cache[k]
            cache[name] = W.by_name(name)
        wl = cache[name]
        v = default_variant(scheme=DEFAULT_SCHEME[name])
        v.update(over)
        try:
            run = Run(hlb, W, wl, name, v)
            v = run.v
            ms, launches, clocks = run.timed(S, K, 3)
            kernels = run.kernel_times(6, S, ms, K, launches)
            rf = roofline_of(run, kernels, name)
            value = run.N * S * K / (ms * 1e-3) / 1e6
            step_bytes = hlb.algorithmic_bytes_per_site(v["scheme"], v["store"], run.nq)
            out.append({"workload": name, "n_sites": run.N, "scheme": v["scheme"], "store": v["store"],
                        "lattice": v["lattice"], "links": "records" if run.g.hlb_uses_records() else "table",
                        "resident_kernel": bool(launches < S * K),
                        "value": value, "unit": UNIT, "lb_steps": S * K, "ms_per_lb_step": ms / (S * K),
                        "algorithmic_gbs": value * 1e6 * step_bytes / 1e9,
                        "roofline": {k: rf[k] for k in ("kernel", "frac", "frac_moved_model", "frac_traffic",
                                                        "ms_per_launch", "bytes_per_site", "moved_bytes_per_site")},
                        "hbm_bound": bool(run.g.hlb_device_bytes() > 4 * 126e6),
                        "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons", "power_w_max")}})
            run.close()
        except Exception as e:   # one failing entry must not take the headline down with it
            out.append({"workload": name, "variant": over, "error": repr(e)})
    return out


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank, world)
    if args.inner < 2 or args.inner % 2:
        raise SystemExit("--inner must be even and >= 2 (A-A alternates two kernels)")
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the site update has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    import paper_1906_11925_b200 as hlb
    import workloads as W

    scheme = args.scheme or DEFAULT_SCHEME[args.workload]
    v = default_variant(scheme=scheme, store=args.store, lattice=args.lattice, order=args.order,
                        links=args.links, prefetch=not args.no_prefetch, pdl=not args.no_pdl,
                        resident=not args.no_resident, inlet=args.inlet, walls=args.walls)
    if args.index64:
        v["index64"] = True
    t_gen = time.perf_counter()
    wl = W.by_name(args.workload, small=args.small)
    t_gen = time.perf_counter() - t_gen
    run = Run(hlb, W, wl, args.workload, v, world, local_rank, copy_stream=not args.no_e2e)
    g, N, S, nq = run.g, run.N, args.inner, run.nq
    scheme = run.v["scheme"]          # what HLB_SCHEME_AUTO took, if that was asked for

    # ---------------- device-resident timing: K x hlb_step(S)
    ms, launches, clocks = run.timed(S, args.steps, args.warmup)
    # ---------------- per-kernel durations (events around single launches, same stream)
    kernels = run.kernel_times(max(6, min(40, 2 * args.steps)) // 2, S, ms, args.steps, launches)

    # ---------------- end to end through the C-ABI with host buffers
    e2e = None
    if not args.no_e2e and 128 * N > 16e9:
        args.no_e2e = True          # four pinned host arrays of 32 N bytes: not at this size
    if not args.no_e2e:
        # pinned host buffers: the inputs of every step, and two sets of outputs (the read-out of
        # step k is copied back on the copy stream while step k + 1 uploads and runs)
        rho_in = torch.ones(N, dtype=torch.float64).pin_memory()
        u_in = torch.zeros((N, 3), dtype=torch.float64).pin_memory()
        if wl.rho0 is not None:
            rho_in.numpy()[:] = wl.rho0
        if wl.u0 is not None:
            u_in.numpy()[:] = wl.u0
        outs = [(torch.empty(N, dtype=torch.float64).pin_memory(), torch.empty((N, 3), dtype=torch.float64).pin_memory())
                for _ in range(2)]
        outs_np = [(r.numpy(), uu.numpy()) for r, uu in outs]
        rin_np, uin_np = rho_in.numpy(), u_in.numpy()

        def e2e_step(k):
            g.hlb_set_state_staged()                          # the state uploaded by hlb_stage_state
            run.advance(S)
            g.hlb_stage_state(rin_np, uin_np)                 # H2D of the NEXT step: rho [N], u [N][3]
            g.hlb_get_macroscopic_async(*outs_np[k & 1])      # D2H: rho [N], u [N][3], on the copy stream

        e2e_steps = max(2, min(args.steps, 20))    # the last read-out copy has nothing to hide under: amortised over the steps
        g.hlb_stage_state(rin_np, uin_np)
        e2e_step(0)
        g.hlb_wait_copies()
        run.barrier()
        t0 = time.perf_counter()
        for k in range(e2e_steps):                            # e2e_steps uploads, runs and read-outs
            e2e_step(k)
        g.hlb_wait_copies()                                   # every step's result is on the host
        run.barrier()
        t_e2e = time.perf_counter() - t0
        e2e = (t_e2e, e2e_steps)
        assert np.all(np.isfinite(outs_np[(e2e_steps - 1) & 1][0][:1000]))
        del rho_in, u_in, outs, outs_np

    # ---------------- aggregate over ranks (max time; total work)
    ms_all, e2e_all = max_over_ranks([ms, e2e[0] if e2e else 0.0], world, dev)
    value = replicas_value(N, S * args.steps, world, ms_all * 1e-3)

    peak, peak_src = measured_peak()
    step_bytes = hlb.algorithmic_bytes_per_site(scheme, args.store, nq)
    moved_step = hlb.moved_bytes_per_site(scheme, args.store, nq, bool(g.hlb_uses_records()),
                                          g.hlb_record_sentinel_fraction(), "step",
                                          g.hlb_num_bfl_sites() / float(N))
    out = {
        "metric": METRIC if nq == 15 else METRIC_Q19, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_all / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {
            "workload": WORKLOAD_DESC[args.workload] + (" (small)" if args.small else ""),
            "n_sites": N, "lattice": args.lattice, "lb_steps_per_step": S, "scheme": scheme, "store": args.store,
            "order": args.order, "links": "records" if g.hlb_uses_records() else "table",
            "l2_prefetch": not args.no_prefetch, "pdl": not args.no_pdl,
            "resident_kernel": bool(launches < S * args.steps), "inlet": args.inlet, "walls": args.walls,
            "bfl_sites": g.hlb_num_bfl_sites(),
            "record_sentinel_fraction": round(g.hlb_record_sentinel_fraction(), 4), "tau": wl.tau, "n_iolets": wl.n_iolets,
            "box": list(wl.shape), "seed": wl.info.get("seed"),
            "device_bytes": g.hlb_device_bytes(), "offset_bits": g.hlb_offset_bits(),
            "l2": "no flush: the populations + table (device_bytes) exceed the 126 MB L2"
                  if g.hlb_device_bytes() > 4 * 126e6 else "working set is L2-sized: not an HBM measurement",
            "parallelism": "replicas" if world > 1 else "single GPU",
            "geometry_seconds": {"generate": round(t_gen, 2), "create": round(run.t_create, 2)},
        },
        "algorithmic_gbs": value * 1e6 * step_bytes / 1e9 / world,
        "frac_of_measured_hbm": value * 1e6 * step_bytes / 1e9 / world / peak,
        "frac_of_nominal_8000": value * 1e6 * step_bytes / 1e9 / world / 8000.0,
        "moved_model_gbs": value * 1e6 * moved_step / 1e9 / world,
        "frac_moved_model_of_measured_hbm": value * 1e6 * moved_step / 1e9 / world / peak,
        "roofline": roofline_of(run, kernels, args.workload),
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if e2e:
        out["e2e"] = {"value": replicas_value(N, S * e2e[1], world, e2e_all), "unit": UNIT,
                      "h2d_bytes_per_step": 32 * N, "d2h_bytes_per_step": 32 * N,
                      "steps": e2e[1], "ms_per_step": e2e_all / e2e[1] * 1e3,
                      "what": "per step: hlb_set_state_staged() + hlb_step(S) + hlb_stage_state(host rho,u of the next "
                              "step) + hlb_get_macroscopic_async(host rho,u), pinned buffers, through the C-ABI; "
                              "both copies of every step are inside the timed region, on a second stream under "
                              "the LB steps; hlb_wait_copies() before the clock stops"}
    if args.render > 0:
        out["render"] = time_renderer(hlb, g, wl, args.workload, args.render, args.render_view)
    if args.readouts:
        out["readouts"] = time_readouts(g, N, nq, args.store)
    run.close()
    sweep = args.sweep == "on" or (args.sweep == "auto" and world == 1 and args.workload == "bigtree"
                                   and not args.small and run.v == default_variant(scheme="aa"))
    if sweep and rank == 0:
        out["configs"] = run_sweep(hlb, W, {args.workload: wl})
        # the same numbers as scalars (MSUPS, fraction of the measured copy peak in moved bytes)
        out["config"]["sweep"] = "; ".join(
            f"{c['workload']}/{c['scheme']}/{c['store']}/{c['lattice']}={c['value']:.0f}"
            f"@{c['roofline']['frac_moved_model']:.2f}" for c in out["configs"] if "value" in c)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        val, n, st, dt, what, thr = time_oracle(wl, args.cpu_seconds, threads=1, lattice=args.lattice)
        out["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": thr, "kind": "oracle",
                               "sample": f"{what}: {n} sites x {st} LB steps in {dt:.1f} s",
                               "host_cpu": host_cpu_model(), "host_cores": os.cpu_count()}
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
