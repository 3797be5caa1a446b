#!/usr/bin/env python
"""bench.py — ms/frame of the whole hot path (per-brick ray casting + sort-last composite) at 1024^2
on the GASS-sized 2048x2048x1600 float32 cube (26.8 GB), BASELINE.json configs[3]: 2x2x2 bricks,
perspective 45 deg, step 1 voxel, early termination at alpha 0.995, 36-view orbit about the y axis.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..3]

A step is one frame (one view of the orbit; view k uses azimuth 10*(k mod 36) degrees).  The cube is
synthetic (workloads.cube_gass_like, seed 3), generated on the device, re-laid once by
vr_create_volume (reported separately as `relayout`, a load-time cost like the paper's file load,
PAPER.md:136) and then resident in HBM.  The cube is 26.8 GB >> the 126 MB L2, so nothing survives
between frames and no L2 flush is needed.  N > 1: replicas only — every
rank holds the whole cube and renders its own K frames of the orbit; no data-path collective.

--impl reference times the CPU oracle (oracle/, double precision, OpenMP) on the host cores on the
same workload; each step renders every 4th pixel in x and y of the frame and scales the time by 16.
"""
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

import numpy as np
import torch

from paper_1008_0135_b200 import replicas
from paper_1008_0135_b200 import workloads as wl

METRIC = "ms_per_frame_1024x1024"
UNIT = "ms/frame"
# Per-launch DRAM traffic of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full`
# capture) lives in profiles/traffic.csv, one row per captured run, written by `bench.py --record-traffic` from the
# ncu CSV and stamped with a hash of paper_1008_0135_b200/csrc/.  A bench line carries the figure only when the row's
# hash is the hash of the tree it runs on; after any kernel edit it reports traffic = null until re-captured.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "traffic.csv")
TRAFFIC_FIELDS = ["config", "image", "mode", "bricks", "skipping", "kernel", "bytes_per_launch", "launches", "csrc_sha256",
                  "captured_after_commit", "source"]


def csrc_hash():
    import glob
    import hashlib
    h = hashlib.sha256()
    for p in sorted(glob.glob(os.path.join(ROOT, "paper_1008_0135_b200", "csrc", "*"))):
        h.update(os.path.basename(p).encode() + b"\0")
        with open(p, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def traffic_key(config, W, H, mode, bricks, skipping):
    return (str(config), str(W if W == H else -1), str(mode), "x".join(str(b) for b in bricks), "1" if skipping else "0")


def read_traffic(key):
    """(bytes per launch or None, text saying where the figure comes from or why there is none)."""
    import csv
    if not os.path.exists(TRAFFIC_CSV):
        return None, "no profiles/traffic.csv"
    tree = csrc_hash()
    stale = None
    with open(TRAFFIC_CSV, newline="") as f:
        for row in csv.DictReader(f):
            if (row["config"], row["image"], row["mode"], row["bricks"], row["skipping"]) != key:
                continue
            if row["csrc_sha256"] == tree:
                return float(row["bytes_per_launch"]), f"{row['source']} ({row['kernel']}, mean of {row['launches']} launches, csrc {tree})"
            stale = f"stale: profiles/traffic.csv holds a capture of csrc {row['csrc_sha256']}, this tree is {tree} (re-capture and --record-traffic)"
    return None, stale or "this run was never captured under ncu"


def record_traffic(args):
    """bench.py --record-traffic NCU.csv --traffic-source profiles/x.md [--config N --no-skip --image S]: NCU.csv is
    `ncu -i REPORT.ncu-rep --page raw --csv --print-units base` of a capture of THIS bench command on THIS tree."""
    import csv
    with open(args.record_traffic, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    head = next(k for k, r in enumerate(rows) if "Kernel Name" in r)
    h = rows[head]
    kn, rd, wr = h.index("Kernel Name"), h.index("dram__bytes_read.sum"), h.index("dram__bytes_write.sum")
    per = {}
    for r in rows[head + 1:]:
        try:
            b = float(r[rd].replace(",", "")) + float(r[wr].replace(",", ""))
        except (ValueError, IndexError):
            continue                                              # the units row
        name = r[kn].split("(")[0]
        if "cast" in name:
            per.setdefault(name, []).append(b)
    if not per:
        raise SystemExit("bench.py --record-traffic: no caster launch in " + args.record_traffic)
    kernel = max(per, key=lambda k: sum(per[k]))                  # the dominant caster of the capture
    w, _ = workload_for(args)
    skipping = (not args.no_skip) and w.mode == 0
    key = traffic_key(args.config, w.W, w.H, w.mode, w.bricks, skipping)
    commit = subprocess.run(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    new = dict(zip(TRAFFIC_FIELDS, list(key) + [kernel, f"{sum(per[kernel]) / len(per[kernel]):.0f}", str(len(per[kernel])),
                                                csrc_hash(), commit, args.traffic_source or args.record_traffic]))
    old = []
    if os.path.exists(TRAFFIC_CSV):
        with open(TRAFFIC_CSV, newline="") as f:
            old = [r for r in csv.DictReader(f) if tuple(r[k] for k in TRAFFIC_FIELDS[:5]) != key]
    with open(TRAFFIC_CSV, "w", newline="") as f:
        wtr = csv.DictWriter(f, fieldnames=TRAFFIC_FIELDS)
        wtr.writeheader()
        for r in old + [new]:
            wtr.writerow(r)
    print(json.dumps(new))


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons of one GPU, sampled every 200 ms while running."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
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
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.lines if t0 - 0.1 <= t <= t1 + 0.3] or [l for (_, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


class NvmlSampler:
    """The same clocks and throttle reasons read in-process through NVML (nvidia-ml-py) every 20 ms: no child process,
    and many samples inside a timed region of ~0.2 s.  Falls back to ClockSampler (nvidia-smi) when NVML is missing."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.stop_flag = False
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(self._physical_index(index))
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.fallback = ClockSampler(index)

    @staticmethod
    def _physical_index(index):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
        ids = [v for v in vis.split(",") if v.strip() != ""]
        try:
            return int(ids[index]) if ids else index
        except (ValueError, IndexError):
            return index

    def start(self):
        if not self.ok:
            return self.fallback.start()
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()

    def _run(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    rs = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    rs = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.rows.append((time.time(), sm, rs))
            except Exception:
                pass
            time.sleep(0.02)

    def stop(self, t0, t1):
        if not self.ok:
            return self.fallback.stop(t0, t1)
        self.stop_flag = True
        self.thread.join(timeout=2)
        rows = [r for r in self.rows if t0 <= r[0] <= t1] or self.rows
        sm = [r[1] for r in rows]
        reasons = sorted(n for n, bit in self.REASONS.items() if any(r[2] & bit for r in rows))
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": self.max_sm, "reasons": reasons,
                "samples": len(sm), "source": "NVML in-process, 20 ms period, samples inside the timed region"}


def workload_for(args):
    w = wl.config(args.config)
    if getattr(args, "image", None):
        w.W = w.H = int(args.image)
    views = wl.orbit_azimuths() if args.config in (3, 5) else [w.az_deg]   # 5: rotation about y at el 0 (Fig 7)
    return w, views


def describe(w, views):
    B = w.bricks[0] * w.bricks[1] * w.bricks[2]
    return {"workload": w.name, "cube": "x".join(str(d) for d in w.dims) + " f32", "seed": w.seed,
            "cube_GB": round(4e-9 * w.dims[0] * w.dims[1] * w.dims[2], 2), "bricks": "x".join(map(str, w.bricks)),
            "n_bricks": B, "image": f"{w.W}x{w.H}", "projection": "perspective45" if w.projection else "orthographic",
            "step_voxels": w.step, "mode": "EA" if w.mode == 0 else "MIP", "ert_alpha": w.ert_alpha,
            "views": f"{len(views)}-view orbit about y, el {w.el_deg} deg" if len(views) > 1 else f"az {w.az_deg} el {w.el_deg}",
            "views_timed": None,
            "l2": "cube >> 126 MB L2: inputs larger than L2, no flush" if w.dims[0] * w.dims[1] * w.dims[2] * 4 > 4e8
                  else "cube fits L2; 512 MB scratch written between frames to flush it"}


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    from paper_1008_0135_b200 import vr                      # fails loudly without the CUDA library
    vr.lib()
    rank, world = env_int("RANK", 0), env_int("WORLD_SIZE", 1)
    local = env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w, views = workload_for(args)
    K, Wm = args.steps, args.warmup
    cube = w.cube("cuda")
    torch.cuda.synchronize()
    vol = vr.Volume(cube)
    relayout_ms, tiled_bytes = vol.vr_volume_info()
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    vol.vr_set_bricks(*w.bricks)
    vol.vr_set_empty_space_skipping(not args.no_skip)
    if args.slab is not None:
        vol.vr_set_slab_staging(args.slab)
    skip_info = vol.vr_get_skip_info()                           # builds the occupancy mask once (a per-table step)
    B = w.bricks[0] * w.bricks[1] * w.bricks[2]
    cams = [vr.camera_from_spec(w.camera(az_deg=a)) for a in views]
    out = torch.empty((w.H, w.W, 4), dtype=torch.float32, device="cuda")
    small = w.dims[0] * w.dims[1] * w.dims[2] * 4 <= 4e8
    scratch = torch.empty(128 << 20, dtype=torch.float32, device="cuda") if small else None

    def view_of(step_idx):
        # ranks start at different points of the orbit (replicas render different views)
        return replicas.view_of(step_idx, rank, world, len(views))

    def frame(k):
        if scratch is not None:
            scratch.fill_(float(k))                              # L2 flush (outside the per-frame events)
        vol.vr_render(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, out=out)

    # warm-up frames are spread over the orbit (views 0, n/W, 2n/W, ...): per-volume preparations that depend on the
    # view direction (the slab caster's linear copies, one per memory order) then happen before the timed region, as
    # the re-layout and the mask build do
    for k in range(Wm):
        frame((k * len(views)) // Wm)
    barrier()
    sampler = NvmlSampler(local)
    if rank == 0:
        sampler.start()
    time.sleep(0.3)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K)]
    cast_ms, comp_ms = [], []
    launches = 0
    slab_frames = []                                               # per timed frame: rendered by the slab-staged caster?
    barrier()
    t_wall0 = time.time()
    for k in range(K):
        if scratch is not None:
            scratch.fill_(float(k))
        ev[2 * k].record()
        vol.vr_render(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, out=out)
        ev[2 * k + 1].record()
        slab_frames.append(vol.vr_get_slab_info()["used"])         # host-side state, no synchronisation
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    per_frame = [ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(K)]
    total_ms = ev[0].elapsed_time(ev[2 * K - 1]) if scratch is None else float(sum(per_frame))
    total_ms = replicas.max_over_ranks(total_ms, dist, "cuda")

    # ---- stage split: second, untimed-for-the-headline pass with the library's own events ----
    for k in range(K):
        if scratch is not None:
            scratch.fill_(float(k))
        vol.vr_render(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, out=out)
        c, m = vol.vr_get_stage_ms()
        cast_ms.append(c); comp_ms.append(m)
        launches += 1 + (1 if m > 0.0 else 0)                     # vr_get_stage_ms reports 0 when no compositor ran

    # ---- end to end through the public call with HOST frame buffers (pinned), D2H inside ----
    # e2e: vr_render_to_host_async per frame (plan upload, kernels, D2H of the frame), two host buffers used
    # alternately, one vr_wait_frames at the end: the copy of frame k overlaps the casting of frame k+1.
    # e2e_latency: the blocking call vr_render_to_host per frame (each frame fully delivered before the next starts).
    host_out = [torch.empty((w.H, w.W, 4), dtype=torch.float32).pin_memory() for _ in range(2)]
    for k in range(min(Wm, 3)):
        vol.vr_render_to_host(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, host_out[0])
    barrier()
    t0 = time.perf_counter()
    for k in range(K):
        if scratch is not None:
            scratch.fill_(float(k))
        vol.vr_render_to_host_async(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, host_out[k & 1])
    vol.vr_wait_frames()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms = replicas.max_over_ranks(e2e_ms, dist, "cuda")
    barrier()
    t0 = time.perf_counter()
    for k in range(K):
        if scratch is not None:
            scratch.fill_(float(k))
        vol.vr_render_to_host(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, host_out[0])
    torch.cuda.synchronize()
    e2e_lat_ms = (time.perf_counter() - t0) * 1e3
    e2e_lat_ms = replicas.max_over_ranks(e2e_lat_ms, dist, "cuda")

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- untimed instrumented pass: samples and distinct 32-byte sectors (cube + occupancy mask) per view ----
    used_views = sorted(set(view_of(k) for k in range(K)))
    # frames the slab-staged caster rendered evaluate every lattice sample: they are measured with skipping off
    slab_views = sorted(set(view_of(k) for k in range(K) if slab_frames[k]))
    meas = {v: vol.vr_measure_units(cams[v], w.W, w.H, w.step, w.mode, w.ert_alpha) for v in used_views if v not in slab_views}
    if slab_views:
        vol.vr_set_empty_space_skipping(False)
        meas.update({v: vol.vr_measure_units(cams[v], w.W, w.H, w.step, w.mode, w.ert_alpha) for v in slab_views})
        vol.vr_set_empty_space_skipping(not args.no_skip)
    samples = sum(meas[view_of(k)][0][0] for k in range(K))           # lattice samples visited (the oracle's count)
    evaluated = sum(meas[view_of(k)][0][1] for k in range(K))         # of which not passed over by empty-space skipping
    alg_bytes = 32.0 * sum(meas[view_of(k)][1][0] + meas[view_of(k)][1][3] for k in range(K))
    cast_total_ms = float(sum(cast_ms))
    peak, peak_src = measured_peak_gbs()
    achieved = alg_bytes / (cast_total_ms * 1e-3) / 1e9
    ms_per_frame = replicas.aggregate_ms_per_frame(total_ms, K, world)   # whole job: all ranks' frames

    # ---- the same frames with skipping off (dense walk), untimed for the headline: what skipping buys ----
    dense = None
    if skip_info["active"]:
        vol.vr_set_empty_space_skipping(False)
        d_cast = []
        for k in range(K):
            vol.vr_render(cams[view_of(k)], w.W, w.H, w.step, w.mode, w.ert_alpha, out=out)
            d_cast.append(vol.vr_get_stage_ms()[0])
        d_meas = {v: vol.vr_measure_units(cams[v], w.W, w.H, w.step, w.mode, w.ert_alpha) for v in used_views}
        d_bytes = 32.0 * sum(d_meas[view_of(k)][1][0] for k in range(K))
        vol.vr_set_empty_space_skipping(True)
        d_ach = d_bytes / (sum(d_cast) * 1e-3) / 1e9
        dense = {"cast_ms": float(sum(d_cast)) / K, "algorithmic_bytes_per_launch": d_bytes / K, "achieved": d_ach,
                 "frac": d_ach / peak, "note": "vr_set_empty_space_skipping(0): every lattice sample is evaluated; same frames bit for bit"}

    # ---- the oracle beside it: one full frame (view az 30 deg) on the host cores ----
    cpu = None
    parity = None
    if not args.no_cpu_baseline:
        from oracle import vro                                    # cpu_baseline leg only
        host_cube = cube.cpu().numpy()
        az = 30.0
        cs = w.camera(az_deg=az)
        ocam = vro.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
        stride = args.cpu_stride
        xs = np.arange(0, w.W, stride, dtype=np.int32)
        ys = np.arange(0, w.H, stride, dtype=np.int32)
        yy, xx = np.meshgrid(ys, xs, indexing="ij")
        t0 = time.perf_counter()
        ref = vro.render_pixels(host_cube, w.table, w.vmin, w.vmax, w.bricks, ocam, w.W, w.H, w.step, w.mode,
                                w.ert_alpha, 1, xx.reshape(-1), yy.reshape(-1))
        cpu_s = time.perf_counter() - t0
        frac = xx.size / float(w.W * w.H)
        cpu = {"value": cpu_s * 1e3 / frac, "unit": UNIT, "cores": vro.max_threads(), "kind": "oracle",
               "sample": f"view az {az:g} deg, every {stride}th pixel in x and y ({xx.size} rays, "
                         f"{ref['samples']} samples, {cpu_s:.1f} s of wall time), scaled by {1 / frac:g}",
               "msamples_per_s": ref["samples"] / cpu_s / 1e6}
        got = vol.vr_render(vr.camera_from_spec(cs), w.W, w.H, w.step, w.mode, w.ert_alpha)
        torch.cuda.synchronize()
        g = got.cpu().numpy()[::stride, ::stride].reshape(-1, 4)
        parity = {"max_abs_err_vs_oracle": float(np.abs(g - ref["rgba"]).max()), "pixels": int(xx.size),
                  "gate": 5e-3 if w.ert_alpha > 0 else 1e-4}
        del host_cube

    traffic, traffic_src = read_traffic(traffic_key(args.config, w.W, w.H, w.mode, w.bricks, bool(skip_info["active"])))
    cfg = describe(w, views)
    cfg["views_timed"] = {"count": len(used_views), "azimuths_deg": [views[v] for v in used_views],
                          "note": "view k of the timed region is azimuth views[k mod len(views)]; steps < len(views) time a prefix of the orbit"}
    line = {
        "metric": METRIC, "value": ms_per_frame, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": total_ms / K, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": cfg,
        "frames_per_s_all_gpus": world * K / (total_ms * 1e-3),
        "ms_per_frame_min": min(per_frame), "ms_per_frame_max": max(per_frame),
        "ms_per_view": {str(int(views[view_of(k)])): round(per_frame[k], 3) for k in range(K)},
        "gsamples_evaluated_per_s": evaluated / (total_ms * 1e-3) / 1e9 * world,     # samples interpolated and classified
        "gsamples_lattice_per_s": samples / (total_ms * 1e-3) / 1e9 * world,         # incl. those empty-space skipping passed over
        "samples_evaluated_per_frame": evaluated / K, "samples_lattice_per_frame": samples / K,
        "empty_space_skipping": dict(skip_info, dense=dense),
        "stages_ms": {"cast": cast_total_ms / K, "composite": float(sum(comp_ms)) / K},
        "caster": {"slab_staged_frames": int(sum(slab_frames)), "row_cache_frames": int(K - sum(slab_frames)),
                   "slab_info_last_frame": vol.vr_get_slab_info()},
        "relayout": {"ms": relayout_ms, "GBps_read_plus_write": (4.0 * cube.numel() + tiled_bytes) / (relayout_ms * 1e-3) / 1e9
                     if relayout_ms > 0 else None},
        "clocks": clocks,
        "e2e": {"value": replicas.aggregate_ms_per_frame(e2e_lat_ms, K, world), "unit": UNIT, "h2d_bytes_per_step": B * (72 + 4) + 256,
                "d2h_bytes_per_step": w.W * w.H * 16,
                "pipelined_value": replicas.aggregate_ms_per_frame(e2e_ms, K, world),
                "note": "value: the blocking vr_render_to_host per frame (plan upload + kernels + D2H of the RGBA frame into pinned "
                        "host memory, each frame fully delivered before the next starts; the round-1 definition); pipelined_value: "
                        "vr_render_to_host_async per frame + one vr_wait_frames, the copy of frame k overlapping the casting of "
                        "frame k+1 (what BENCH_r02 reported as value)"},
        "gpu_launches": launches,          # counted per frame of the stage pass: the caster, + composite_kernel when its events fired
        "roofline": {"bound": "hbm", "kernel": ("cast_slab_kernel" if sum(slab_frames) * 2 > K else "cast_kernel") + ("<EA>" if w.mode == 0 else "<MIP>"),
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": alg_bytes / K,
                     "cube_bytes": 4.0 * cube.numel(), "avg_launch_ms": cast_total_ms / K,
                     "definition": "32 B x distinct sectors of the tiled cube and of the occupancy mask touched by the "
                                   "frame's evaluated samples (instrumented pass, untimed) / cast kernel time (CUDA events)"},
        "cpu_baseline": cpu, "parity": parity,
        "paper_context": "< 0.3 s per 1024^2 frame of the 26 GB GASS cube on 3 workstations / 8 Tesla C1060 "
                         "(PAPER.md:9,304): another machine and the real cube, context only",
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle as it stands, timed on the host cores (rank 0 only)."""
    if env_int("RANK", 0) != 0:
        return
    from oracle import vro
    w, views = workload_for(args)
    K, Wm = args.steps, args.warmup
    dev = "cuda" if torch.cuda.is_available() else "cpu"         # generation only; not timed
    host_cube = w.cube(dev).cpu().numpy()
    stride = args.cpu_stride
    xs = np.arange(0, w.W, stride, dtype=np.int32)
    ys = np.arange(0, w.H, stride, dtype=np.int32)
    yy, xx = np.meshgrid(ys, xs, indexing="ij")
    px, py = xx.reshape(-1), yy.reshape(-1)
    frac = px.size / float(w.W * w.H)

    def step(k):
        cs = w.camera(az_deg=views[k % len(views)])
        ocam = vro.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
        return vro.render_pixels(host_cube, w.table, w.vmin, w.vmax, w.bricks, ocam, w.W, w.H, w.step, w.mode,
                                 w.ert_alpha, 1, px, py)["samples"]

    for k in range(Wm):
        step(k)
    t0 = time.perf_counter()
    samples = 0
    for k in range(K):
        samples += step(k)
    dt = time.perf_counter() - t0
    ms = dt * 1e3 / K / frac
    sample = (f"each step: every {stride}th pixel in x and y of one orbit view ({px.size} rays), time scaled by "
              f"{1 / frac:g} to a full frame")
    cfg = describe(w, views)
    timed = sorted(set(k % len(views) for k in range(K)))
    cfg["views_timed"] = {"count": len(timed), "azimuths_deg": [views[v] for v in timed]}
    line = {"impl": "reference", "metric": METRIC, "value": ms, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": Wm, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": cfg,
            "cpu_baseline": {"value": ms, "unit": UNIT, "kind": "oracle", "cores": vro.max_threads(), "sample": sample,
                             "msamples_per_s": samples / dt / 1e6},
            "e2e": {"value": ms, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def run_sweep(args):
    """BASELINE.json configs[4]: MIP point + EA sweep (bricks 1/8/64 x step 1/4,1/2,1 x image 512/1024/2048) on
    config 3's cube, orthographic az 30 el 20, early termination off.  One JSON line per point (1 GPU)."""
    from paper_1008_0135_b200 import vr
    vr.lib()
    torch.cuda.set_device(0)
    w = wl.config(3)
    cube = w.cube("cuda")
    torch.cuda.synchronize()
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    vol.vr_set_empty_space_skipping(not args.no_skip)
    if args.slab is not None:
        vol.vr_set_slab_staging(args.slab)
    cs = wl.orbit_camera(w.dims, 30.0, 20.0, wl.PROJ_PERSP if args.sweep_persp else wl.PROJ_ORTHO)
    cam = vr.camera_from_spec(cs)
    peak, peak_src = measured_peak_gbs()
    reps = max(3, min(args.steps, 10))
    host_cube, ocam = None, None
    if not args.no_cpu_baseline:                                   # parity per point against the oracle (128x128-pixel lattice)
        from oracle import vro
        host_cube = cube.cpu().numpy()
        ocam = vro.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    for pt in wl.sweep_points():
        size, step, mode, bricks = pt["size"], pt["step"], pt["mode"], pt["bricks"]
        if args.sweep_filter:
            want = args.sweep_filter.split(":")
            have = ["MIP" if mode else "EA", str(bricks[0] * bricks[1] * bricks[2]), f"{step:g}", str(size)]
            if len(want) != 4 or any(a != "*" and a != b for a, b in zip(want, have)):
                continue
        vol.vr_set_bricks(*bricks)
        out = torch.empty((size, size, 4), dtype=torch.float32, device="cuda")
        for _ in range(3):
            vol.vr_render(cam, size, size, step, mode, 0.0, out=out)
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * reps)]
        cast = []
        for k in range(reps):
            ev[2 * k].record()
            vol.vr_render(cam, size, size, step, mode, 0.0, out=out)
            ev[2 * k + 1].record()
            cast.append(vol.vr_get_stage_ms()[0])
        torch.cuda.synchronize()
        ms = sorted(ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(reps))
        (samples, evaluated), units = vol.vr_measure_units(cam, size, size, step, mode, 0.0)
        sectors = units[0] + units[3]
        best, med = ms[0], ms[len(ms) // 2]
        cast_med = sorted(cast)[len(cast) // 2]
        B = bricks[0] * bricks[1] * bricks[2]
        parity = None
        if host_cube is not None:
            stride = size // 128
            xs = np.arange(stride // 2, size, stride, dtype=np.int32)
            yy, xx = np.meshgrid(xs, xs, indexing="ij")
            px, py = xx.reshape(-1), yy.reshape(-1)
            ref = vro.render_pixels(host_cube, w.table, w.vmin, w.vmax, bricks, ocam, size, size, step, mode, 0.0, 0, px, py)
            got = out.cpu().numpy()[py, px]
            parity = {"max_abs_err_vs_oracle": float(np.abs(got - ref["rgba"]).max()), "pixels": int(px.size), "gate": 1e-4}
        print(json.dumps({"sweep_point": {"mode": "MIP" if mode else "EA", "bricks": B, "step_voxels": step,
                                          "image": f"{size}x{size}", "projection": "perspective45" if args.sweep_persp else "orthographic"},
                          "ms_per_frame_best": best, "ms_per_frame_median": med, "cast_ms_median": cast_med,
                          "samples_evaluated": evaluated, "samples_lattice": samples,
                          "gsamples_evaluated_per_s": evaluated / (med * 1e-3) / 1e9, "gsamples_lattice_per_s": samples / (med * 1e-3) / 1e9,
                          "algorithmic_GB": 32e-9 * sectors, "bytes_per_sample": 32.0 * sectors / samples,
                          "hbm_GBps_algorithmic": 32e-9 * sectors / (cast_med * 1e-3),
                          "frac_of_peak": 32e-9 * sectors / (cast_med * 1e-3) / peak, "peak": peak,
                          "side_of_ridge": "hbm" if 32.0 * sectors / samples > 14.0 else "alu/lsu",
                          "slab": vol.vr_get_slab_info(), "parity": parity}), flush=True)
        del out
    vol.close()


def launch_ranks_if_needed(args):
    """--gpus N must mean N ranks.  Under torchrun (WORLD_SIZE set) the two have to agree; started by hand with N > 1
    the script re-launches itself as N ranks, one per GPU, the way the driver does (torch.distributed.run on
    127.0.0.1), and exits with that job's status — it never prints an n_gpus: 1 line for --gpus 8."""
    world = os.environ.get("WORLD_SIZE")
    if world is not None:
        if int(world) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch as many ranks as --gpus says")
        return
    if args.gpus <= 1 or args.sweep:
        return
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=36)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (0..3), 3 is the headline; 5 = N-body-like 1024^3 cube")
    ap.add_argument("--cpu-stride", type=int, default=None,
                    help="oracle legs render every n-th pixel in x and y (default 1 = the full frame for cpu_baseline, 4 for --impl reference)")
    ap.add_argument("--image", type=int, default=None, help="override the image size (W = H), e.g. 512 for Fig 12's comparison")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-skip", action="store_true", help="vr_set_empty_space_skipping(0): the dense walk (same frames)")
    ap.add_argument("--sweep-persp", action="store_true", help="with --sweep: perspective 45 deg camera instead of the orthographic one")
    ap.add_argument("--sweep-filter", default=None,
                    help="with --sweep: run only the points matching MODE:BRICKS:STEP:SIZE (e.g. EA:8:0.25:2048; * = any)")
    ap.add_argument("--slab", type=int, default=None, choices=[0, 1, 2],
                    help="vr_set_slab_staging: 0 never, 1 auto (library default), 2 whenever the window fits")
    ap.add_argument("--sweep", action="store_true", help="run BASELINE.json configs[4] (28 points) instead of the headline")
    ap.add_argument("--record-traffic", default=None, metavar="NCU_CSV",
                    help="no benchmark: store the caster's mean DRAM bytes per launch of an ncu raw CSV in profiles/traffic.csv")
    ap.add_argument("--traffic-source", default=None, help="with --record-traffic: the profiles/ file that describes the capture")
    args = ap.parse_args()
    if args.record_traffic:
        record_traffic(args)
        return
    launch_ranks_if_needed(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.cpu_stride is None:
        args.cpu_stride = 4 if args.impl == "reference" else 1
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
